"""Conservative virial tensor sum_pairs r_a F^C_b (the configurational part of the stress used for the interfacial tension
of section 4.1): oracle against an independent numpy O(N^2) evaluation, CUDA path against the oracle."""
import math

import numpy as np
import pytest

import mdpd_workloads as wl

from helpers import brute_density, minimg_all


def brute_virial(pos, typ, p, species=None, Amat=None, Bmat=None):
    """Eq. (1) of the paper, conservative part only, every pair once: W_ab = sum r_a F_b, F = F^C(r) r / r."""
    pos = np.asarray(pos, np.float64)
    frozen = np.asarray(typ).astype(bool)
    rho = brute_density(pos, p["box"], p["rd"])
    d = minimg_all(pos, p["box"])
    r = np.sqrt((d * d).sum(-1))
    n = len(pos)
    iu = np.triu_indices(n, 1)
    rr, dd = r[iu], d[iu]
    ok = (rr < p["rc"]) & (rr > 1e-10) & ~(frozen[iu[0]] & frozen[iu[1]])
    A = p["A"] if species is None else Amat[species[iu[0]], species[iu[1]]]
    B = p["B"] if species is None else Bmat[species[iu[0]], species[iu[1]]]
    FC = A * (1.0 - rr / p["rc"]) + B * (rho[iu[0]] + rho[iu[1]]) * np.maximum(0.0, 1.0 - rr / p["rd"])
    c = np.where(ok, FC / np.where(rr > 0, rr, 1.0), 0.0)
    W = np.einsum("k,ka,kb->ab", c, dd, dd)
    return np.array([W[0, 0], W[1, 1], W[2, 2], W[0, 1], W[0, 2], W[1, 2]])


def test_oracle_virial_vs_numpy_brute_force():
    from oracle.mdpd_ref import RefSim
    p = dict(wl.default_params((4.0, 5.0, 7.0)))
    rng = np.random.default_rng(21)
    n = 700
    pos = rng.random((n, 3)) * np.asarray(p["box"])
    vel = rng.standard_normal((n, 3))
    typ = (rng.random(n) < 0.2).astype(np.uint8)
    s = RefSim(p)
    s.load_particles(pos, vel, typ)
    want = brute_virial(pos, typ, p)
    got = s.virial()
    assert np.allclose(got, want, rtol=0, atol=1e-8 * np.abs(want).max())
    assert abs(got[:3].sum() - s.counters()["virial_c"]) < 1e-9 * abs(got[:3].sum())     # trace = the scalar virial
    # two particles on the x axis: only W_xx, equal to r F^C(r)  (closed form, golden value of Eq. (1) at r = 0.5)
    s2 = RefSim(dict(p, sigma=0.0))
    s2.load_particles([[1.0, 1.0, 1.0], [1.5, 1.0, 1.0]], np.zeros((2, 3)))
    assert np.allclose(s2.virial(), [0.5 * (-9.5206621832), 0, 0, 0, 0, 0], atol=1e-9)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 2, "mixture"])
def test_gpu_virial_matches_the_oracle(cfg):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    import paper_1903_10134_b200 as pk
    from oracle.mdpd_ref import RefSim
    pk.build()
    c = wl.make_species_mixture() if cfg == "mixture" else wl.make_config(cfg)
    s = pk.Simulation(c["params"])
    r = RefSim(c["params"])
    if cfg == "mixture":
        s.set_pair_params(c["pair_A"], c["pair_B"], c["frozen_mask"])
        r.set_pair_params(c["pair_A"].astype(np.float64), c["pair_B"].astype(np.float64), c["frozen_mask"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    s.step(10)
    st = s.get_state()
    f_before = st["force"].copy()
    W = s.compute_virial()
    r.load_particles(st["pos"].astype(np.float64), st["vel"].astype(np.float64), c["type"])
    want = r.virial()
    scale = np.abs(want[:3]).max()
    assert np.abs(W - want).max() < 1e-4 * scale, (W, want)
    # the same pass refreshes rho and f like mdpd_compute_forces (full-step velocities now, so only close to before)
    g = s.get_state()
    mobile = np.abs(st["vel"]).sum(1) > 0        # frozen particles have v = 0 (and get a force only in this diagnostic pass)
    assert np.isfinite(g["force"]).all() and np.abs(g["force"] - f_before)[mobile].max() < 50.0
