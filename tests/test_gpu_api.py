"""C-ABI behaviour on the GPU: call order, error codes, edge cases (empty / tiny / degenerate inputs), ownership,
checkpoint-resume, determinism.  Every call goes through include/mdpd.h via the ctypes binding."""
import ctypes as C

import numpy as np
import pytest

import mdpd_workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def ref_state(c, step=0):
    from oracle.mdpd_ref import RefSim
    s = RefSim(c["params"])
    s.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    if step:
        s.set_step(step)
        s.compute_forces()
    return s.get_state()


def test_call_order_and_bad_arguments(gpu):
    L = gpu.lib()
    h = C.c_void_p()
    assert L.mdpd_create(C.byref(h), 0, None) == 0
    assert L.mdpd_step(h, 1) == -5                                   # MDPD_ESTATE: nothing loaded
    assert L.mdpd_get_state(h, None, None, None, None, None) == -5
    assert L.mdpd_load_particles(h, 1, None, None, None) == -5       # set_params first
    assert b"set_params" in L.mdpd_last_error(h)
    p = gpu.make_params(wl.default_params((10.0, 10.0, 10.0), s=-0.5))
    assert L.mdpd_set_params(h, C.byref(p)) == -1                    # MDPD_EINVAL: s must be in (0, 4] (R15)
    p = gpu.make_params(wl.default_params((10.0, 10.0, 10.0), sigma=2.0))
    assert L.mdpd_set_params(h, C.byref(p)) == -1                    # sigma^2 != 2 gamma kT
    p = gpu.make_params(wl.default_params((10.0, 10.0, 10.0)))
    assert L.mdpd_set_params(h, C.byref(p)) == 0
    assert L.mdpd_load_particles(h, 4, None, None, None) == -1       # NULL arrays with n > 0
    assert L.mdpd_create(C.byref(C.c_void_p()), 99, None) == -3      # no such device
    assert L.mdpd_destroy(h) == 0
    assert L.mdpd_destroy(None) == -1


@pytest.mark.parametrize("n", [0, 1, 2])
def test_tiny_systems(gpu, n):
    """N = 0, 1, 2 (the degenerate cases): zero / single particle feel nothing but the body force; two particles
    reproduce the oracle; stepping works."""
    p = wl.default_params((5.0, 5.0, 5.0), g=(0.0, 0.0, 0.5))
    pos = np.array([[1.0, 1.0, 1.0], [1.3, 1.4, 1.1]], np.float32)[:n]
    vel = np.array([[0.5, 0.0, 0.0], [-0.5, 0.2, 0.0]], np.float32)[:n]
    s = gpu.Simulation(p)
    s.load_particles(pos, vel)
    st = s.get_state()
    assert st["pos"].shape == (n, 3) and st["rho"].shape == (n,)
    if n == 1:
        assert st["rho"][0] == 0.0 and np.allclose(st["force"][0], [0, 0, 0.5])
    if n == 2:
        r = ref_state(dict(params=p, pos=pos, vel=vel, type=np.zeros(2, np.uint8)))
        assert np.allclose(st["rho"], r["rho"], rtol=2e-6) and np.allclose(st["force"], r["force"], rtol=1e-5, atol=1e-4)
    s.step(5)
    st = s.get_state()
    assert st["step"] == 5 and np.isfinite(st["pos"]).all()
    if n == 1:   # free flight under gravity, velocity Verlet is exact for constant force
        t = 0.05
        assert np.allclose(st["pos"][0], [1.0 + 0.5 * t, 1.0, 1.0 + 0.25 * t * t], atol=2e-6)
        assert np.allclose(st["vel"][0], [0.5, 0.0, 0.5 * t], atol=1e-6)
    s.close()


def test_all_particles_in_one_cell_and_periodic_faces(gpu):
    """Degenerate occupancy: everything in one cell next to a box corner, so neighbours are found across three
    periodic faces; minimum box (3 cells per dimension)."""
    rng = np.random.default_rng(3)
    n = 60
    pos = ((rng.random((n, 3)) - 0.5) * 1.2) % 3.75
    pos = pos.astype(np.float32)
    c = dict(params=wl.default_params((3.75, 3.75, 3.75), max_neigh=128), pos=pos,
             vel=rng.standard_normal((n, 3)).astype(np.float32), type=np.zeros(n, np.uint8))
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"])
    g, r = s.get_state(), ref_state(c)
    assert np.abs(g["rho"] - r["rho"]).max() <= 1e-4 * np.sqrt((r["rho"] ** 2).mean())
    assert np.sqrt(((g["force"] - r["force"]) ** 2).sum(1)).max() <= 1e-4 * np.sqrt((r["force"] ** 2).sum(1).mean())
    s.close()


def test_list_capacity_overflow_is_reported(gpu):
    c = wl.make_liquid(5.0, seed=9, max_neigh=16)     # ~49 neighbours needed
    s = gpu.Simulation(c["params"])
    with pytest.raises(gpu.MdpdError) as e:
        s.load_particles(c["pos"], c["vel"])
    assert e.value.code == -4                          # MDPD_EOVERFLOW
    s.close()
    with pytest.raises(gpu.MdpdError) as e:            # capacity above the hard limit
        gpu.Simulation(wl.default_params((5.0, 5.0, 5.0), max_neigh=256))
    assert e.value.code == -1


def test_fluid_inside_solid_is_reported(gpu):
    c = wl.make_poiseuille(L=12.0, wall=2.0, Lxy=6.0, seed=4)
    c["pos"][0] = (1.0, 1.0, 0.5)                      # a fluid particle inside the lower wall
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"], c["type"], mask_dims=c["mask"].shape[::-1])
    with pytest.raises(gpu.MdpdError) as e:
        s.load_wall_mask(c["mask"], c["voxel"])
    assert e.value.code == -7                          # MDPD_EINSOLID
    s.close()


def test_nan_input_is_reported(gpu):
    c = wl.make_liquid(5.0, seed=10)
    c["vel"][5, 0] = np.nan
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"])
    s.step(1)
    with pytest.raises(gpu.MdpdError) as e:
        s.get_state()
    assert e.value.code == -6                          # MDPD_ENAN
    s.close()


def test_determinism_and_checkpoint_resume(gpu):
    """Two runs from the same input are bitwise identical; a checkpoint (pos, vel, force, step) resumes the
    trajectory (the force of a time level was evaluated with the half-step velocities, R6, so it is part of the
    state: mdpd.h 'Checkpoint / resume')."""
    c = wl.make_liquid(8.0, seed=12)
    a = gpu.Simulation(c["params"])
    a.load_particles(c["pos"], c["vel"])
    a.step(7)
    mid = a.get_state()
    a.step(9)
    fa = a.get_state()
    b = gpu.Simulation(c["params"])
    b.load_particles(c["pos"], c["vel"])
    b.step(16)
    fb = b.get_state()
    for k in ("pos", "vel", "force", "rho"):
        assert np.array_equal(fa[k], fb[k]), k
    # resume from the step-7 state
    r = gpu.Simulation(c["params"])
    r.load_particles(mid["pos"], mid["vel"])
    r.set_step_counter(7)
    r.set_forces(mid["force"])
    r.step(9)
    fr = r.get_state()
    assert fr["step"] == 16
    # the resumed run re-sorts from the saved positions, so its list order can differ: same trajectory to rounding
    assert np.abs(fr["vel"] - fa["vel"]).max() < 5e-4
    d = np.abs(fr["pos"] - fa["pos"])
    assert np.minimum(d, 8.0 - d).max() < 5e-5
    for s in (a, b, r):
        s.close()


def test_device_pointers_and_caller_owned_outputs(gpu):
    """load_particles / get_state accept device pointers (torch CUDA tensors): 'host or device' in mdpd.h."""
    import torch
    c = wl.make_liquid(6.0, seed=13)
    s = gpu.Simulation(c["params"])
    dpos = torch.from_numpy(c["pos"]).cuda()
    dvel = torch.from_numpy(c["vel"]).cuda()
    s.load_particles(dpos, dvel, None)
    out = {"pos": torch.empty_like(dpos), "rho": torch.empty(len(c["pos"]), device="cuda")}
    st = s.get_state(vel=False, force=False, out=out)
    h = gpu.Simulation(c["params"])
    h.load_particles(c["pos"], c["vel"])
    sh = h.get_state()
    assert np.array_equal(st["pos"].cpu().numpy(), sh["pos"]) and np.array_equal(st["rho"].cpu().numpy(), sh["rho"])
    s.close()
    h.close()


def test_parameters_can_change_between_steps(gpu):
    """g, dt, seed, A, B, gamma, sigma may change after load (mdpd.h); box / cut-offs / skin may not."""
    c = wl.make_liquid(6.0, seed=14)
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"])
    s.set_params(g=(0.0, 0.3, 0.0), seed=99)
    s.compute_forces()
    c2 = dict(c, params=dict(c["params"], g=(0.0, 0.3, 0.0), seed=99))
    r = ref_state(c2)
    g = s.get_state()
    assert np.sqrt(((g["force"] - r["force"]) ** 2).sum(1)).max() <= 1e-4 * np.sqrt((r["force"] ** 2).sum(1).mean())
    with pytest.raises(gpu.MdpdError) as e:
        s.set_params(skin=0.4)
    assert e.value.code == -5
    s.close()


def test_counters_and_profile(gpu):
    c = wl.make_liquid(8.0, seed=15)
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"])
    c0 = s.counters()
    s.profile_begin()
    s.step(10)
    prof = s.profile_end()
    c1 = s.counters()
    assert c1["steps"] == 10 and c1["launches"] - c0["launches"] >= 30
    assert prof["k_force"][1] == 10 and prof["k_density"][1] == 10 and prof["k_force"][0] > 0
    n = len(c["pos"])
    assert 40 < c1["sum_nbr"] / n < 60                                   # ~49 listed neighbours at skin 0.25
    assert 20 < (c1["sum_act"] - c0["sum_act"]) / (10 * n) < 30          # ~25 inside rc
    assert c1["density_passes"] - c0["density_passes"] == 10
    s.close()


def test_reload_with_more_particles_reallocates_the_workspace(gpu):
    """A second load_particles with a larger n needs a larger workspace: the binding hands the handle a new tensor
    (mdpd_set_workspace on a loaded handle drops the loaded state) and the results are those of a fresh handle."""
    small, big = wl.make_liquid((6.0, 6.0, 6.0), seed=5), wl.make_config(0)
    s = gpu.Simulation(big["params"])
    s.load_particles(small["pos"], small["vel"], small["type"])      # 1296 particles in the 10^3 box
    s.step(3)
    s.load_particles(big["pos"], big["vel"], big["type"])            # 6000 particles: more memory
    s.step(4)
    a = s.get_state()
    f = gpu.Simulation(big["params"])
    f.load_particles(big["pos"], big["vel"], big["type"])
    f.step(4)
    b = f.get_state()
    for k in ("pos", "vel", "force", "rho"):
        assert np.array_equal(a[k], b[k]), k
    s.close()
    f.close()
    # the C-ABI without a caller workspace: the library's own allocation grows too
    L = gpu.lib()
    h = C.c_void_p()
    assert L.mdpd_create(C.byref(h), 0, None) == 0
    p = gpu.make_params(big["params"])
    assert L.mdpd_set_params(h, C.byref(p)) == 0
    assert L.mdpd_load_particles(h, len(small["pos"]), small["pos"].ctypes.data, small["vel"].ctypes.data, None) == 0
    assert L.mdpd_load_particles(h, len(big["pos"]), big["pos"].ctypes.data, big["vel"].ctypes.data, None) == 0
    assert L.mdpd_step(h, 2) == 0
    assert L.mdpd_get_state(h, None, None, None, None, None) == 0
    assert L.mdpd_destroy(h) == 0


def test_set_params_rejects_general_exponent_with_pair_params(gpu):
    """s != 1 runs the one-material force kernel: with per-type-pair parameters it must be refused after load as well
    as before (the A_ij, B_ij table would silently be ignored)."""
    c = wl.make_species_mixture()
    s = gpu.Simulation(c["params"])
    s.set_pair_params(c["pair_A"], c["pair_B"], c["frozen_mask"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    with pytest.raises(gpu.MdpdError) as e:
        s.set_params(s=0.5)
    assert e.value.code == -1
    s.set_params(s=1.0)
    s.step(2)                       # the handle is still usable with its old parameters
    s.close()


def test_runaway_particle_with_mask_is_a_latched_fault_not_a_crash(gpu):
    """A particle whose trial position leaves [-L, 2L) (or is not finite) must latch MDPD_ENAN; the voxel lookup must
    not read outside the mask (advisor finding of round 1: the index was clamped above only)."""
    c = wl.make_poiseuille(L=12.0, wall=2.0, gx=0.05, seed=3, Lxy=8.0)
    for bad_v in (-1.0e6, 1.0e6, np.float32("-inf")):
        vel = c["vel"].copy()
        vel[0] = (bad_v, bad_v, bad_v)
        s = gpu.Simulation(c["params"])
        s.load_particles(c["pos"], vel, c["type"], mask_dims=c["mask"].shape[::-1])
        s.load_wall_mask(c["mask"], c["voxel"])
        s.step(2)
        with pytest.raises(gpu.MdpdError) as e:
            s.get_state()
        assert e.value.code == -6, e.value
        s.close()
    good = gpu.Simulation(c["params"])      # the CUDA context survived
    good.load_particles(c["pos"], c["vel"], c["type"], mask_dims=c["mask"].shape[::-1])
    good.load_wall_mask(c["mask"], c["voxel"])
    good.step(3)
    good.get_state()
    good.close()


def test_dense_system_takes_the_multi_window_list_build(gpu):
    """Number density 9.5: the 27-cell stencil of a cell holds ~500 particles, more than one register window of the
    list build (384 candidates), while the lists (~78 entries) still fit: pair sets, rho and F against the oracle."""
    from oracle.mdpd_ref import RefSim
    c = wl.make_liquid((7.5, 6.3, 5.1), density=9.5, seed=21)
    for flags in (0, 2):
        prm = dict(c["params"])
        prm["flags"] = flags
        s = gpu.Simulation(prm)
        s.load_particles(c["pos"], c["vel"], c["type"])
        r = RefSim(c["params"])
        r.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
        for rcut in (0.75, 1.0, 1.25):
            pg, pr = s.get_pairs(rcut), r.get_pairs(rcut)
            assert abs(len(pg) - len(pr)) <= 2 and len(pg) > 10000
        g, o = s.get_state(), r.get_state()
        assert np.abs(g["rho"] - o["rho"]).max() <= 1e-4 * np.sqrt(np.mean(o["rho"] ** 2))
        assert np.sqrt(((g["force"] - o["force"]) ** 2).sum(1)).max() <= 1e-4 * np.sqrt(np.mean((o["force"] ** 2).sum(1)))
        ctr = s.counters()
        assert ctr["faults"] == 0 and (flags or ctr["max_nbr"] <= 128)
        s.close()


@pytest.mark.parametrize("flags", [0, 2])
def test_collapsed_cluster_overflows_cleanly(gpu, flags):
    """600 particles inside a sphere of radius 0.3 (R10 allows coincident and near-coincident particles): every one of
    them has ~600 candidates inside rc + skin, more than the 392 entries of a warp's row in the list build, and the row
    fill is carried across the windows of the stencil.  The write address has to saturate inside the row: the answer
    is MDPD_EOVERFLOW, not an illegal address that poisons the CUDA context -- the second simulation proves the
    context is still alive."""
    c = wl.make_liquid(6.0, seed=31)
    rng = np.random.default_rng(32)
    u = rng.normal(size=(600, 3))
    u *= (0.3 * rng.random((600, 1)) ** (1 / 3)) / np.linalg.norm(u, axis=1, keepdims=True)
    c["pos"][:600] = (np.array([3.1, 2.9, 3.3]) + u).astype(np.float32)
    prm = dict(c["params"])
    prm["flags"] = flags
    s = gpu.Simulation(prm)
    with pytest.raises(gpu.MdpdError) as e:
        s.load_particles(c["pos"], c["vel"], c["type"])
        s.step(1)
        s.get_state()
    assert e.value.code == -4, e.value                  # MDPD_EOVERFLOW
    s.close()
    ok = wl.make_liquid(5.0, seed=33)
    s = gpu.Simulation(ok["params"])
    s.load_particles(ok["pos"], ok["vel"], ok["type"])
    s.step(2)
    assert np.isfinite(s.get_state()["pos"]).all() and s.counters()["faults"] == 0
    s.close()


def test_two_handles_with_different_tile_sizes(gpu):
    """The opt-in to large dynamic shared memory is a property of the kernel FUNCTION on the device.  A handle with big
    tiles (dense liquid) must keep working after a second handle with small tiles (dilute gas) has been loaded: pair
    search, force evaluation and stepping, interleaved."""
    big = wl.make_liquid((7.5, 6.3, 5.1), density=9.5, seed=21)
    small = wl.make_liquid(5.0, density=3.0, seed=22)
    a = gpu.Simulation(big["params"])
    a.load_particles(big["pos"], big["vel"], big["type"])
    pa, sa = a.get_pairs(1.0), a.get_state()
    assert len(pa) > 10000
    b = gpu.Simulation(small["params"])
    b.load_particles(small["pos"], small["vel"], small["type"])
    pb = b.get_pairs(1.0)
    assert 0 < len(pb) < len(pa)
    assert np.array_equal(a.get_pairs(1.0), pa)              # a's kernels still launch after b's load
    a.compute_forces()
    s2 = a.get_state()
    assert np.array_equal(s2["rho"], sa["rho"]) and np.array_equal(s2["force"], sa["force"])
    for _ in range(3):
        a.step(2)
        b.step(2)
    assert a.counters()["faults"] == 0 and b.counters()["faults"] == 0
    assert np.array_equal(b.get_pairs(0.75), b.get_pairs_static(0.75))
    assert np.array_equal(a.get_pairs(0.75), a.get_pairs_static(0.75))
    a.close()
    b.close()


def test_tile_that_outgrows_its_capacity_is_reported(gpu):
    """headroom = 1.0: the shared-memory capacity of a tile is the fullest tile of the LOADED state.  A dilute gas that
    condenses (A = -40 at number density 3) outgrows it; the run must end in MDPD_EOVERFLOW, not in silent missing
    forces."""
    c = wl.make_liquid((16.0, 16.0, 16.0), density=3.0, seed=9, headroom=1.0)
    s = gpu.Simulation(c["params"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    with pytest.raises(gpu.MdpdError) as e:
        for _ in range(40):
            s.step(50)
            s.counters()
    assert e.value.code == -4, e.value
    s.close()
