"""Step batching and the list-free path on the GPU.

mdpd_step(n) replays the captured step graph (k_integrate with the second half kick of step k fused with the first half
kick of step k + 1, Algorithm 1 lines 7 and 1; the rebuild chain inside a device-set IF node); n calls
of mdpd_step(1) go through the same kernels one call at a time.  Both must give the same trajectory BIT FOR BIT, with
and without the voxel mask, with and without graphs, on the Verlet-list path and on the list-free path
(MDPD_FLAG_DIRECT).  (A force pass that also integrates was built and measured in round 2: correct,
no faster -- DESIGN.md section 10.)"""
import numpy as np
import pytest

import mdpd_workloads as wl

pytestmark = pytest.mark.gpu

FLAG_NO_GRAPH, FLAG_DIRECT, FLAG_TMA, FLAG_CPASYNC = 1, 2, 4, 8


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def make_sim(pk, c, flags):
    prm = dict(c["params"])
    prm["flags"] = flags
    md = None if c.get("mask") is None else c["mask"].shape[::-1]
    sim = pk.Simulation(prm, device=0)
    sim.load_particles(c["pos"], c["vel"], c["type"], mask_dims=md)
    if c.get("mask") is not None:
        sim.load_wall_mask(c["mask"], c["voxel"])
    return sim


def same_state(a, b):
    for k in ("pos", "vel", "force", "rho"):
        assert np.array_equal(a[k], b[k]), k
    assert a["step"] == b["step"]


@pytest.mark.parametrize("cfg,nsteps", [(0, 13), (2, 25)])
@pytest.mark.parametrize("flags", [0, FLAG_NO_GRAPH, FLAG_DIRECT, FLAG_DIRECT | FLAG_NO_GRAPH, FLAG_TMA])
def test_fused_steps_equal_single_steps_bitwise(gpu, cfg, nsteps, flags):
    c = wl.make_config(cfg)
    a = make_sim(gpu, c, flags)
    b = make_sim(gpu, c, flags)
    a.step(nsteps)                      # graph replays
    for _ in range(nsteps):
        b.step(1)
    sa, sb = a.get_state(), b.get_state()
    same_state(sa, sb)
    ca, cb = a.counters(), b.counters()
    for k in ("steps", "rebuilds", "bounces"):
        assert ca[k] == cb[k], k
    assert ca["steps"] == nsteps and ca["rebuilds"] >= 2
    if cfg == 2:
        assert ca["bounces"] > 0
    # and a second call continues both the same way (the pending half kick is applied by the next call)
    a.step(3)
    b.step(2)
    b.step(1)
    same_state(a.get_state(), b.get_state())
    a.close()
    b.close()


@pytest.mark.parametrize("cfg", [0, 2])
def test_direct_path_equals_list_path(gpu, cfg):
    """The list-free path finds the r < rc neighbours straight from the cells every step; the Verlet-list path filters
    its list.  Same pair sets => rho identical up to summation order, forces too; trajectories stay together for a few
    steps to fp32 rounding (they are not bitwise equal: the order of the sums differs)."""
    c = wl.make_config(cfg)
    a = make_sim(gpu, c, 0)
    b = make_sim(gpu, c, FLAG_DIRECT)
    sa, sb = a.get_state(), b.get_state()
    f_rms = np.sqrt(np.mean((sa["force"] ** 2).sum(1)))
    assert np.abs(sa["rho"] - sb["rho"]).max() <= 2e-6 * np.abs(sa["rho"]).max()
    assert np.sqrt(((sa["force"] - sb["force"]) ** 2).sum(1)).max() <= 2e-6 * f_rms
    for rcut in (c["params"]["rd"], c["params"]["rc"], c["params"]["rc"] + c["params"]["skin"]):
        pa, pb = a.get_pairs(rcut), b.get_pairs(rcut)
        assert np.array_equal(pa, pb)
    a.step(5)
    b.step(5)
    sa, sb = a.get_state(), b.get_state()
    assert np.abs(sa["pos"] - sb["pos"]).max() < 2e-4
    assert np.abs(sa["vel"] - sb["vel"]).max() < 2e-3
    assert a.counters()["rebuilds"] == b.counters()["rebuilds"]
    a.close()
    b.close()


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_tma_staging_equals_cp_async_staging_bitwise(gpu, cfg):
    """MDPD_FLAG_TMA_STAGING: the density / force passes stage their tile with cp.async.bulk (one bulk copy per
    contiguous run, mbarrier completion) instead of per-particle cp.async copies.  The staged image is the same, so
    every result is bit-identical."""
    c = wl.make_config(cfg)
    sims = [make_sim(gpu, c, f) for f in (0, FLAG_TMA, FLAG_CPASYNC)]   # default (mixed), all bulk, all cp.async
    for s in sims[1:]:
        same_state(sims[0].get_state(), s.get_state())
    for s in sims:
        s.step(9)
    for s in sims[1:]:
        same_state(sims[0].get_state(), s.get_state())
    for s in sims:
        s.close()
