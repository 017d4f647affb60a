"""GPU-vs-oracle parity (the -m gpu suite): every call goes through the C-ABI of include/mdpd.h.

Three-way comparison of BASELINE.json's north_star on the same seeded inputs:
  (1) neighbour pair sets and the RNG stream bit-exact,
  (2) per-particle density and force within 1e-4 of the RMS (fp32 kernels vs the fp64 oracle, identical positions),
  (3) long-run observables within 1 % (tests/test_gpu_observables.py).
P:L<n> = /root/reference/PAPER.md line n (cited, never read at run time); R<n> = DESIGN.md reading n.
"""
import numpy as np
import pytest

import mdpd_workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-4  # relative to the RMS of the oracle's values (BASELINE.json north_star)


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def ref_sim(c, step=0, brute=False):
    from oracle.mdpd_ref import RefSim
    s = RefSim(c["params"], brute_force=brute)
    s.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    if c.get("mask") is not None:
        s.load_wall_mask(c["mask"], c["voxel"])
    if step:
        s.set_step(step)
        s.compute_forces()
    return s


def gpu_sim(pk, c, step=0, direct=False):
    prm = dict(c["params"])
    if direct:
        prm["flags"] = 2        # MDPD_FLAG_DIRECT: the list-free path
    s = pk.Simulation(prm)
    md = None if c.get("mask") is None else c["mask"].shape[::-1]
    s.load_particles(c["pos"], c["vel"], c["type"], mask_dims=md)
    if c.get("mask") is not None:
        s.load_wall_mask(c["mask"], c["voxel"])
    if step:
        s.set_step_counter(step)
        s.compute_forces()
    return s


def assert_rho_force_parity(g, r, typ=None, what=""):
    rho_rms = np.sqrt(np.mean(r["rho"] ** 2))
    f_rms = np.sqrt(np.mean((r["force"] ** 2).sum(1)))
    d_rho = np.abs(g["rho"].astype(np.float64) - r["rho"]).max()
    d_f = np.sqrt(((g["force"].astype(np.float64) - r["force"]) ** 2).sum(1)).max()
    assert d_rho <= TOL * rho_rms, (what, d_rho, rho_rms)
    assert d_f <= TOL * f_rms, (what, d_f, f_rms)
    return d_rho / rho_rms, d_f / f_rms


# ---------------------------------------------------------------------------------------------- (1) RNG stream
def test_rng_stream_bit_exact(gpu):
    """the device hash kernel and the oracle's hash give the same uint32 for every
    (pair, step, seed); symmetric in the pair."""
    from oracle.mdpd_ref import ref_rng_fill
    rng = np.random.default_rng(11)
    pairs = rng.integers(0, 2 ** 31 - 1, size=(200_000, 2), dtype=np.int64).astype(np.uint32)
    pairs[:1000] = rng.integers(0, 50, size=(1000, 2))          # small tags, many ties a == b excluded below
    pairs = pairs[pairs[:, 0] != pairs[:, 1]]
    c = wl.make_liquid(4.0, seed=1)
    for seed in (0, 12345, 0xFFFFFFFF):
        c["params"]["seed"] = seed
        s = gpu_sim(gpu, c)
        for step in (0, 1, 999, 0xFFFFFFFF):
            h_gpu = s.rng_fill(pairs, step)
            h_ref = ref_rng_fill(seed, pairs, step)
            assert np.array_equal(h_gpu, h_ref), (seed, step)
            assert np.array_equal(s.rng_fill(pairs[:, ::-1], step), h_gpu)
        s.close()


# ---------------------------------------------------------------------------------------------- (1) pair sets
@pytest.mark.parametrize("box,n,seed", [((4.0, 4.0, 4.0), 400, 3), ((5.0, 5.0, 5.0), 900, 4),
                                        ((4.0, 5.0, 7.0), 1100, 5), ((16.0, 16.0, 16.0), 24000, 6)])
def test_pair_sets_quantised_inputs_identical(gpu, box, n, seed):
    """coordinates on a 2^-7 grid in boxes <= 16 make r^2 exact in fp32 and fp64 alike, so the pair
    sets at rd, rc and rc + skin must be IDENTICAL (pairs exactly at a cut-off included: strict <, R3)."""
    c = wl.make_liquid(box, n=n, seed=seed)
    c["pos"] = wl.quantise_positions(c["pos"], box)
    # plant pairs at exactly rd, rc, rc+skin along axes and across the periodic boundary
    c["pos"][0] = (0.0, 1.0, 1.0); c["pos"][1] = (box[0] - 0.75, 1.0, 1.0)
    c["pos"][2] = (2.0, 2.0, 0.5); c["pos"][3] = (2.0, 2.0, box[2] - 0.5)
    c["pos"][4] = (1.0, 0.25, 3.0); c["pos"][5] = (1.0, box[1] - 1.0, 3.0)
    c["pos"][6] = (3.0, 3.0, 3.0); c["pos"][7] = (3.0, 3.0, 3.0)          # coincident pair
    g, r = gpu_sim(gpu, c), ref_sim(c, brute=n <= 2000)
    for rcut in (0.75, 1.0, 1.25):
        pg, pr = g.get_pairs(rcut), r.get_pairs(rcut)
        assert pg.shape == pr.shape and np.array_equal(pg, pr), (rcut, pg.shape, pr.shape)
    g.close()


@pytest.mark.parametrize("direct", [False, True])
@pytest.mark.parametrize("cfg", [0, 1])
def test_pair_sets_random_fp32_inputs(gpu, cfg, direct):
    """random fp32 positions; the oracle gets the same values upcast.  Sets identical except pairs
    within 4 ulp of a cut-off (|r^2/rcut^2 - 1| < 4 * 2^-23), which are listed and must be few."""
    c = wl.make_config(cfg)
    g, r = gpu_sim(gpu, c, direct=direct), ref_sim(c)
    x = c["pos"].astype(np.float64)
    box = np.asarray(c["params"]["box"])
    for rcut in (0.75, 1.0, 1.25):
        pg, pr = g.get_pairs(rcut), r.get_pairs(rcut)
        kg = (pg[:, 0].astype(np.uint64) << np.uint64(32)) | pg[:, 1].astype(np.uint64)
        kr = (pr[:, 0].astype(np.uint64) << np.uint64(32)) | pr[:, 1].astype(np.uint64)
        diff = np.setxor1d(kg, kr)
        assert len(diff) <= 4, (rcut, len(diff))
        for k in diff:
            a, b = int(k >> np.uint64(32)), int(k & np.uint64(0xFFFFFFFF))
            d = x[a] - x[b]
            d -= box * np.round(d / box)
            assert abs((d * d).sum() / rcut ** 2 - 1.0) < 4 * 2.0 ** -23, (rcut, a, b)
    g.close()


# --------------------------------------------------------------------------- (2) density and force, same state
@pytest.mark.parametrize("direct", [False, True])
@pytest.mark.parametrize("cfg,step", [(0, 0), (0, 17), (1, 3), (2, 5)])
def test_density_force_parity_configs(gpu, cfg, step, direct):
    """rho and F (Eq. 1 + dissipative + hashed random, P:L186 body force) on BASELINE configs
    0, 1, 2 from identical fp32-valued positions / velocities: max error <= 1e-4 RMS."""
    c = wl.make_config(cfg)
    g, r = gpu_sim(gpu, c, step, direct=direct), ref_sim(c, step)
    sg, sr = g.get_state(), r.get_state()
    assert_rho_force_parity(sg, sr, what=f"cfg{cfg}")
    # frozen particles: v = 0 (R8); wall-wall forces skipped, so a wall particle deep in the wall feels only fluid
    if cfg == 2:
        w = c["type"] == 1
        assert (sg["vel"][w] == 0).all()
    g.close()


@pytest.mark.parametrize("direct", [False, True])
def test_density_force_parity_pore_network_small(gpu, direct):
    """Config 3's recipe at 32^3 voxels (box 16^3, ~8.6 k fluid + wall shell): mask, frozen shell, body force."""
    c = wl.make_pore_network(nvox=32, corr=3.0, seed=wl.BASE_SEED + 3)
    g, r = gpu_sim(gpu, c, 2, direct=direct), ref_sim(c, 2)
    assert_rho_force_parity(g.get_state(), r.get_state(), what="pore32")
    g.close()


def test_force_terms_separately(gpu):
    """Each term of Eq. 1 on its own (others switched off) so that a wrong sign / weight in one term cannot hide
    behind the random force that dominates the RMS."""
    base = wl.make_config(0)
    for name, over in [("A", dict(B=0.0, gamma=0.0, sigma=0.0, kT=0.0)),
                       ("B", dict(A=0.0, gamma=0.0, sigma=0.0, kT=0.0)),
                       ("D", dict(A=0.0, B=0.0, sigma=0.0, kT=0.0)),
                       ("R", dict(A=0.0, B=0.0, gamma=0.0, kT=0.0)),
                       ("g", dict(A=0.0, B=0.0, gamma=0.0, sigma=0.0, kT=0.0, g=(0.1, -0.2, 0.3)))]:
        c = dict(base, params=dict(base["params"], **over))
        g, r = gpu_sim(gpu, c, 4), ref_sim(c, 4)
        assert_rho_force_parity(g.get_state(), r.get_state(), what=name)
        g.close()


def test_pairwise_forces_antisymmetric_bitwise(gpu):
    """Full list + symmetric hash: F_ij = -F_ji bitwise, so the total pairwise force sums to ~0 (momentum
    conservation, P:L75 'central pairwise'); fp32 sum of 6000 vectors of RMS 47 stays below 1e-2."""
    c = wl.make_config(0)
    g = gpu_sim(gpu, c, 9)
    f = g.get_state()["force"].astype(np.float64)
    assert np.abs(f.sum(0)).max() < 2e-2, f.sum(0)
    g.close()


# ------------------------------------------------------------------------------------ closed forms on the GPU
def test_closed_form_two_particles(gpu, golden_dir):
    """tests/golden/closed_form_pairs.txt (Eq. 1; two particles, v = 0, sigma = 0) through the CUDA path."""
    import os
    rows = [l.split() for l in open(os.path.join(golden_dir, "closed_form_pairs.txt")) if l.strip() and l[0] != "#"]
    p = wl.default_params((10.0, 10.0, 10.0), sigma=0.0, kT=0.0)
    for r_, rho, F in [(float(a), float(b), float(c_)) for a, b, c_ in rows]:
        pos = np.array([[3.0, 4.0, 5.0], [3.0 + r_, 4.0, 5.0]], np.float32)
        s = gpu.Simulation(p)
        s.load_particles(pos, np.zeros_like(pos))
        st = s.get_state()
        assert np.allclose(st["rho"], rho, atol=3e-6 * max(1.0, rho)), (r_, st["rho"], rho)
        assert np.allclose(st["force"][0], [-F, 0, 0], atol=2e-5 * max(1.0, abs(F))), (r_, st["force"], F)
        assert np.array_equal(st["force"][1], -st["force"][0])
        s.close()


def test_simple_cubic_lattice_sum(gpu):
    """Periodic simple-cubic lattice a = 0.5 (number density 8): every rho = 6 w(.5) + 12 w(.7071) = 3.9946693043,
    26 neighbours inside rc (the 6 at exactly r = 1 excluded by strict <), zero net conservative force."""
    n1 = 12
    idx = np.stack(np.meshgrid(*(np.arange(n1),) * 3, indexing="ij"), -1).reshape(-1, 3)
    pos = (idx * 0.5).astype(np.float32)
    p = wl.default_params((6.0, 6.0, 6.0), sigma=0.0, gamma=0.0, kT=0.0)
    s = gpu.Simulation(p)
    s.load_particles(pos, np.zeros_like(pos))
    st = s.get_state()
    assert np.allclose(st["rho"], 3.9946693043, atol=2e-5)
    assert np.abs(st["force"]).max() < 2e-3
    assert len(s.get_pairs(1.0)) == len(pos) * 26 // 2
    assert len(s.get_pairs(0.75)) == len(pos) * 18 // 2
    s.close()


# ------------------------------------------------------------------------------------------ integrator parity
@pytest.mark.parametrize("cfg", [0, 2])
def test_short_trajectory_parity(gpu, cfg):
    """After 1 and 5 steps from the identical state, x and v agree with the oracle to fp32 rounding accumulated
    over the steps (chaos has not yet amplified it: R18); bounce-back counts agree (R7)."""
    c = wl.make_config(cfg)
    if cfg == 2:   # make sure bounce-backs happen: fast fluid next to the walls
        c["vel"] = (c["vel"] * np.float32(3.0)).astype(np.float32)
    g, r = gpu_sim(gpu, c), ref_sim(c)
    box = np.asarray(c["params"]["box"])
    for nstep, tol_x, tol_v in [(1, 2e-6, 2e-4), (4, 2e-5, 2e-3)]:
        g.step(nstep)
        r.step(nstep)
        sg, sr = g.get_state(), r.get_state()
        assert sg["step"] == sr["step"]
        d = sg["pos"].astype(np.float64) - sr["pos"]
        d -= box * np.round(d / box)
        assert np.abs(d).max() < tol_x * box.max(), (nstep, np.abs(d).max())
        assert np.abs(sg["vel"] - sr["vel"]).max() < tol_v * 10, (nstep, np.abs(sg["vel"] - sr["vel"]).max())
    if cfg == 2:
        assert g.counters()["bounces"] == r.counters()["bounces"] > 0
        w = c["type"] == 1
        assert np.array_equal(g.get_state()["pos"][w], c["pos"][w])
    g.close()


def test_verlet_list_stays_valid_over_rebuilds(gpu):
    """a3/a4: the list (skin 0.25, rebuilt on the max-displacement trigger) must yield exactly the r < rc and
    r < rd pair sets of a fresh O(N) search at every step (R17): the oracle recomputes from the GPU's positions."""
    from oracle.mdpd_ref import RefSim
    c = wl.make_liquid(8.0, seed=21)
    g = gpu_sim(gpu, c)
    rebuilds = []
    for it in range(12):
        g.step(3)
        st = g.get_state()
        r = RefSim(c["params"])
        r.load_particles(st["pos"].astype(np.float64), st["vel"].astype(np.float64), c["type"])
        for rcut in (0.75, 1.0):
            pg, pr = g.get_pairs(rcut), r.get_pairs(rcut)
            kg = (pg[:, 0].astype(np.uint64) << np.uint64(32)) | pg[:, 1].astype(np.uint64)
            kr = (pr[:, 0].astype(np.uint64) << np.uint64(32)) | pr[:, 1].astype(np.uint64)
            assert len(np.setxor1d(kg, kr)) <= 2, (it, rcut)
        # and the forces the stepper holds are the forces of these positions (half-step velocities differ from
        # the full-step ones get_state returns, so compare through compute_forces on both sides)
        g.compute_forces()
        r.set_step(st["step"])
        r.compute_forces()
        assert_rho_force_parity(g.get_state(), r.get_state(), what=f"it{it}")
        rebuilds.append(g.counters()["rebuilds"])
    assert rebuilds[-1] > 3, rebuilds            # the trigger fired several times in 36 steps
    assert rebuilds[-1] < 36, rebuilds           # ... but not every step
    g.close()


@pytest.mark.parametrize("s_exp", [0.5, 0.25, 2.0])
def test_density_force_parity_general_exponent_s(gpu, s_exp):
    """wR = (1 - r/rc)^s, wD = wR^2 with s != 1 (R15): rho and F against the oracle at load and after stepping."""
    from oracle.mdpd_ref import RefSim
    c = wl.make_config(0, s=s_exp)
    g = gpu.Simulation(c["params"])
    g.load_particles(c["pos"], c["vel"], c["type"])
    r = RefSim(c["params"])
    r.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])

    # For s < 1/2 the random force sigma w^s xi / sqrt(dt) is ill-conditioned at the cut-off in ANY fp32 evaluation:
    # d(w^s) = s w^(s-1) dw with dw ~ 1e-7 from r itself, so the few pairs with w ~ 1e-5 carry errors ~1e-3 of the RMS
    # force.  The maximum norm is therefore relaxed to 2e-3 for s = 1/4 and the RMS error to 5e-5 (R15).
    tol_max, tol_rms = (TOL, 1e-5) if s_exp >= 0.5 else (2e-3, 5e-5)

    def check(a, b, what):
        f_rms = np.sqrt(np.mean((b["force"] ** 2).sum(1)))
        err = np.sqrt(((a["force"] - b["force"]) ** 2).sum(1))
        e_rho = np.abs(a["rho"] - b["rho"]).max() / np.sqrt(np.mean(b["rho"] ** 2))
        assert err.max() / f_rms <= tol_max and np.sqrt(np.mean(err ** 2)) / f_rms <= tol_rms and e_rho <= TOL, \
            (what, s_exp, err.max() / f_rms, np.sqrt(np.mean(err ** 2)) / f_rms, e_rho)

    check(g.get_state(), r.get_state(), "load")
    # the exponent really enters: the s = 1 forces of the same state differ
    g1 = gpu.Simulation(dict(c["params"], s=1.0))
    g1.load_particles(c["pos"], c["vel"], c["type"])
    assert np.abs(g1.get_state()["force"] - g.get_state()["force"]).max() > 1.0
    g.step(12)
    st = g.get_state()
    g.compute_forces()
    r2 = RefSim(c["params"])
    r2.load_particles(st["pos"].astype(np.float64), st["vel"].astype(np.float64), c["type"])
    r2.set_step(st["step"])
    r2.compute_forces()
    check(g.get_state(), r2.get_state(), "after 12 steps")
