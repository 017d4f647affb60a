"""GPU-vs-oracle parity of the per-type-pair dissipative / random amplitudes gamma_ij, sigma_ij
(mdpd_set_pair_gamma_sigma, with the two parameter sets of L89 and L141): force of every particle within
1e-4 of the RMS on the five-species mixture, from the load state, after stepping, through the virial pass and after the
values were changed on a loaded handle; uniform matrices reproduce the uniform path bit for bit; a cold two-fluid mixture
with its own thermostat per pair of species heats to kT = 1."""
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


def sym(rng, nt, lo, hi):
    m = lo + (hi - lo) * rng.random((nt, nt))
    return (0.5 * (m + m.T)).astype(np.float32)


def oracle_for(c, G, S, pos, vel, step):
    from oracle.mdpd_ref import RefSim
    r = RefSim(c["params"])
    r.set_pair_params(c["pair_A"].astype(np.float64), c["pair_B"].astype(np.float64), c["frozen_mask"])
    if G is not None:
        r.set_pair_gamma_sigma(G.astype(np.float64), S.astype(np.float64))
    r.load_particles(np.asarray(pos, np.float64), np.asarray(vel, np.float64), c["type"])
    if step:
        r.set_step(step)
        r.compute_forces()
    return r


def check(g, r, what):
    rho_rms = np.sqrt(np.mean(r["rho"] ** 2))
    f_rms = np.sqrt(np.mean((r["force"] ** 2).sum(1)))
    e_rho = np.abs(g["rho"] - r["rho"]).max() / rho_rms
    e_f = np.sqrt(((g["force"] - r["force"]) ** 2).sum(1)).max() / f_rms
    assert e_rho <= TOL and e_f <= TOL, (what, e_rho, e_f)
    return e_f


@pytest.mark.parametrize("direct", [False, True])
def test_five_species_force_parity(gpu, direct):
    c = wl.make_species_mixture()
    nt = c["pair_A"].shape[0]
    rng = np.random.default_rng(77)
    G, S = sym(rng, nt, 1.0, 13.0), sym(rng, nt, 0.5, 5.0)
    prm = dict(c["params"], flags=2 if direct else 0)
    s = gpu.Simulation(prm)
    s.set_pair_params(c["pair_A"], c["pair_B"], c["frozen_mask"])
    s.set_pair_gamma_sigma(G, S)
    s.load_particles(c["pos"], c["vel"], c["type"])
    check(s.get_state(), oracle_for(c, G, S, c["pos"], c["vel"], 0).get_state(), "load")
    # the matrices matter: against the uniform amplitudes the same state is far outside the tolerance
    r_uni = oracle_for(c, None, None, c["pos"], c["vel"], 0).get_state()
    assert np.sqrt(((s.get_state()["force"] - r_uni["force"]) ** 2).sum(1)).max() > 1.0
    s.step(15)
    st = s.get_state()
    s.compute_forces()
    check(s.get_state(), oracle_for(c, G, S, st["pos"], st["vel"], st["step"]).get_state(), "after 15 steps")
    s.compute_virial()                                    # the virial instantiation of the force pass reads the same table
    check(s.get_state(), oracle_for(c, G, S, st["pos"], st["vel"], st["step"]).get_state(), "virial pass")
    # new values on a loaded handle enter the next force evaluation
    G2, S2 = sym(rng, nt, 2.0, 9.0), sym(rng, nt, 1.0, 4.0)
    s.set_pair_gamma_sigma(G2, S2)
    s.compute_forces()
    check(s.get_state(), oracle_for(c, G2, S2, st["pos"], st["vel"], st["step"]).get_state(), "changed after load")
    # and NULL returns to the uniform gamma, sigma of mdpd_params
    s.set_pair_gamma_sigma(None, None)
    s.compute_forces()
    check(s.get_state(), oracle_for(c, None, None, st["pos"], st["vel"], st["step"]).get_state(), "cleared")
    assert s.counters()["faults"] == 0
    s.close()


def test_uniform_matrices_are_the_uniform_path_bitwise(gpu):
    c = wl.make_species_mixture()
    nt = c["pair_A"].shape[0]
    out = []
    for with_gs in (False, True):
        s = gpu.Simulation(c["params"])
        s.set_pair_params(c["pair_A"], c["pair_B"], c["frozen_mask"])
        if with_gs:
            s.set_pair_gamma_sigma(np.full((nt, nt), c["params"]["gamma"], np.float32),
                                   np.full((nt, nt), c["params"]["sigma"], np.float32))
        s.load_particles(c["pos"], c["vel"], c["type"])
        s.step(25)
        out.append(s.get_state())
        s.close()
    for key in ("pos", "vel", "force", "rho"):
        assert np.array_equal(out[0][key], out[1][key]), key


def test_two_fluids_with_their_own_thermostats_reach_kT_1(gpu):
    """sigma^2 = 2 gamma kT per pair.  gamma = 4.5 (L89), 12.4 (water, L141), 8.0 for unlike pairs; started
    cold, 16^3 box (24 576 particles): kT = 1 +- 2 % overall and per species."""
    from helpers import kinetic_temperature
    c = wl.make_liquid(16.0, seed=43)
    n = len(c["pos"])
    sp = (np.arange(n) % 2).astype(np.uint8)
    G = np.array([[4.5, 8.0], [8.0, 12.4]], np.float32)
    S = np.sqrt(2.0 * G).astype(np.float32)
    s = gpu.Simulation(c["params"])
    s.set_pair_params(np.full((2, 2), -40.0, np.float32), np.full((2, 2), 25.0, np.float32), 0)
    s.set_pair_gamma_sigma(G, S)
    s.load_particles(c["pos"], np.zeros((n, 3), np.float32), sp)
    s.step(600)
    kts = []
    for _ in range(40):
        s.step(10)
        v = s.get_state()["vel"]
        kts.append([kinetic_temperature(v), kinetic_temperature(v[sp == 0]), kinetic_temperature(v[sp == 1])])
    kt = np.mean(kts, axis=0)
    assert np.abs(kt - 1.0).max() < 0.02, kt
    assert s.counters()["faults"] == 0
    s.close()


def test_bad_arguments_are_rejected(gpu):
    c = wl.make_species_mixture()
    nt = c["pair_A"].shape[0]
    s = gpu.Simulation(c["params"])
    ok = np.full((nt, nt), 4.5, np.float32)
    with pytest.raises(gpu.MdpdError) as e:                # no species set yet
        s.set_pair_gamma_sigma(ok, ok)
    assert e.value.code == -1
    s.set_pair_params(c["pair_A"], c["pair_B"], c["frozen_mask"])
    with pytest.raises(gpu.MdpdError):
        s.set_pair_gamma_sigma(np.full((2, 2), 4.5, np.float32), np.full((2, 2), 3.0, np.float32))    # another ntypes
    bad = ok.copy()
    bad[0, 1] = 5.0
    with pytest.raises(gpu.MdpdError):
        s.set_pair_gamma_sigma(bad, ok)                    # not symmetric
    with pytest.raises(gpu.MdpdError):
        s.set_pair_gamma_sigma(-ok, ok)                    # negative friction
    s.set_pair_gamma_sigma(ok, ok)
    s.load_particles(c["pos"], c["vel"], c["type"])
    s.step(2)
    assert s.counters()["faults"] == 0
    s.close()
