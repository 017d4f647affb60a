"""Randomised GPU-vs-oracle parity over box shapes, densities, vacuum regions, frozen fractions and skins: the tile /
staging-recipe / hand-out machinery must give the same pair sets, densities and forces for partial tiles, tiles that
wrap a short periodic dimension, empty cells and very uneven occupancy.  Seeds are fixed; every case is small enough for
the oracle to finish in about a second."""
import numpy as np
import pytest

import mdpd_workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def make_case(seed):
    rng = np.random.default_rng(wl.BASE_SEED + 100 + seed)
    box = tuple(float(v) for v in rng.uniform(4.0, 19.0, 3).round(2))
    skin = float(rng.choice([0.15, 0.25, 0.4]))
    # particles fill a random sub-block of the box at a random density: the rest stays empty (vacuum cells)
    lo = rng.uniform(0.0, 0.5, 3) * np.asarray(box)
    hi = lo + rng.uniform(0.45, 1.0, 3) * (np.asarray(box) - lo)
    dens = float(rng.uniform(2.0, 8.0))
    n = int(min(9000, max(50, dens * np.prod(hi - lo))))
    pos = (lo + rng.random((n, 3)) * (hi - lo)).astype(np.float32)
    vel = wl.maxwell_velocities(rng, n)
    typ = (rng.random(n) < float(rng.choice([0.0, 0.3]))).astype(np.uint8)
    vel[typ != 0] = 0.0
    p = wl.default_params(box, skin=skin, g=(float(rng.choice([0.0, 0.05])), 0.0, 0.0), seed=int(rng.integers(1, 2 ** 31)))
    return dict(params=p, pos=pos, vel=vel, type=typ)


@pytest.mark.parametrize("direct", [False, True])
@pytest.mark.parametrize("seed", range(12))
def test_random_case(gpu, seed, direct):
    from oracle.mdpd_ref import RefSim
    c = make_case(seed)
    if direct:
        c["params"]["flags"] = 2   # MDPD_FLAG_DIRECT: the list-free path
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    r = RefSim(c["params"])
    r.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    x = c["pos"].astype(np.float64)
    box = np.asarray(c["params"]["box"])
    for rcut in (0.75, 1.0, 1.0 + c["params"]["skin"]):         # pair sets right after the build
        pg, pr = s.get_pairs(rcut), r.get_pairs(rcut)
        kg = (pg[:, 0].astype(np.uint64) << np.uint64(32)) | pg[:, 1].astype(np.uint64)
        kr = (pr[:, 0].astype(np.uint64) << np.uint64(32)) | pr[:, 1].astype(np.uint64)
        for k in np.setxor1d(kg, kr):                             # only pairs within 4 ulp of the cut-off may differ
            a, b = int(k >> np.uint64(32)), int(k & np.uint64(0xFFFFFFFF))
            d = x[a] - x[b]
            d -= box * np.round(d / box)
            assert abs((d * d).sum() / rcut ** 2 - 1.0) < 4 * 2.0 ** -23, (seed, rcut, a, b)

    def check(g, o, what):
        rho_rms = max(np.sqrt(np.mean(o["rho"] ** 2)), 1e-12)
        f_rms = max(np.sqrt(np.mean((o["force"] ** 2).sum(1))), 1e-12)
        e_rho = np.abs(g["rho"] - o["rho"]).max() / rho_rms
        e_f = np.sqrt(((g["force"] - o["force"]) ** 2).sum(1)).max() / f_rms
        assert e_rho <= TOL and e_f <= TOL, (seed, what, e_rho, e_f)

    check(s.get_state(), r.get_state(), "load")
    s.step(7)                                                    # through rebuilds (the random state moves fast)
    st = s.get_state()
    s.compute_forces()
    r2 = RefSim(c["params"])
    r2.load_particles(st["pos"].astype(np.float64), st["vel"].astype(np.float64), c["type"])
    r2.set_step(st["step"])
    r2.compute_forces()
    check(s.get_state(), r2.get_state(), "after 7 steps")
    assert s.counters()["faults"] == 0
