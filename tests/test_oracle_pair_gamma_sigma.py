"""Pins of the oracle's per-type-pair dissipative and random amplitudes gamma_ij, sigma_ij.

PAPER.md L75 gives every pair F^D = -gamma wD(r) (e.v) e and F^R = sigma wR(r) xi e with wD = wR^2 and sigma^2 = 2 gamma kT
(the 1/sqrt(dt) of the discrete random force is DESIGN.md R2).  The paper runs water at gamma = 12.4 (L141) and its other
fluids at 4.5 (L89, L186): a system of two fluids needs the amplitudes per pair of species, like A_SL and B_SL (L152).
No GPU.  Nothing here comes from the CUDA path."""
import math

import numpy as np
import pytest

import mdpd_workloads as wl
from oracle.mdpd_ref import RefSim

from helpers import brute_forces, hash_py, kinetic_temperature, xi_py

BOX = (10.0, 10.0, 10.0)


def two_particle_sim(r, v0, v1, G, S, species=(0, 1), step=7, seed=99, A=0.0, B=0.0):
    """Two particles r apart along a tilted axis; conservative force off unless asked."""
    p = dict(wl.default_params(BOX), A=A, B=B, gamma=4.5, sigma=3.0, seed=seed)
    s = RefSim(p)
    s.set_pair_params(np.full((2, 2), A), np.full((2, 2), B), 0)
    s.set_pair_gamma_sigma(G, S)
    e = np.array([2.0, -1.0, 2.0]) / 3.0
    x0 = np.array([4.0, 5.0, 6.0])
    s.load_particles([x0, x0 - r * e], [v0, v1], np.array(species, np.uint8))     # d = x0 - x1 = r e
    s.set_step(step)
    s.compute_forces()
    return s, e, p


@pytest.mark.parametrize("r", [0.2, 0.5, 0.8, 0.95])
def test_single_unlike_pair_closed_forms(r):
    """F^D on particle 0 = -gamma_SL (1 - r)^2 (e.v01) e, F^R = sigma_SL (1 - r) xi / sqrt(dt) e, each alone; the like
    entries of the matrices (deliberately different) must not leak into the unlike pair, and vice versa."""
    G = np.array([[4.5, 12.4], [12.4, 7.0]])
    S = np.array([[3.0, 0.0], [0.0, 1.0]])
    v0, v1 = np.array([0.3, -0.2, 0.5]), np.array([-0.1, 0.4, 0.2])
    s, e, p = two_particle_sim(r, v0, v1, G, S)                    # sigma_SL = 0: dissipative force alone
    ev = float(e @ (v0 - v1))
    want = -12.4 * (1.0 - r) ** 2 * ev * e
    f = s.get_state()["force"]
    assert np.allclose(f[0], want, rtol=0, atol=1e-12) and np.allclose(f[1], -want, rtol=0, atol=1e-12)
    S2 = np.array([[3.0, 5.0], [5.0, 1.0]])
    G2 = np.array([[4.5, 0.0], [0.0, 7.0]])
    s, e, p = two_particle_sim(r, v0, v1, G2, S2)                  # gamma_SL = 0: random force alone
    xi = xi_py(hash_py(0, 1, 7, 99))                               # independent restatement of the hash
    want = 5.0 * (1.0 - r) * xi / math.sqrt(p["dt"]) * e
    f = s.get_state()["force"]
    assert abs(xi) > 1e-3
    assert np.allclose(f[0], want, rtol=0, atol=1e-11) and np.allclose(f[1], -want, rtol=0, atol=1e-11)
    # a LIKE pair of species 1 takes the (1, 1) entries
    s, e, p = two_particle_sim(r, v0, v1, G, S, species=(1, 1))
    want = (-7.0 * (1.0 - r) ** 2 * ev + 1.0 * (1.0 - r) * xi / math.sqrt(p["dt"])) * e
    assert np.allclose(s.get_state()["force"][0], want, rtol=0, atol=1e-11)


def test_beyond_rc_nothing_and_linear_in_gamma():
    v0, v1 = np.array([1.0, 0.0, 0.0]), np.array([0.0, 0.0, 0.0])
    G = np.array([[4.5, 9.0], [9.0, 4.5]])
    Z = np.zeros((2, 2))
    s, e, _ = two_particle_sim(1.0, v0, v1, G, Z)
    assert np.all(s.get_state()["force"] == 0.0)                   # strict r < rc
    f1 = two_particle_sim(0.5, v0, v1, G, Z)[0].get_state()["force"][0]
    f2 = two_particle_sim(0.5, v0, v1, 3.0 * G, Z)[0].get_state()["force"][0]
    assert np.allclose(f2, 3.0 * f1, rtol=1e-14, atol=0)


def random_state(n, box, seed, nspecies):
    rng = np.random.default_rng(seed)
    pos = rng.random((n, 3)) * np.asarray(box)
    vel = rng.standard_normal((n, 3))
    sp = rng.integers(0, nspecies, n).astype(np.uint8)
    return pos, vel, sp


def test_uniform_matrices_equal_the_uniform_path_bit_for_bit():
    p = dict(wl.default_params((5.0, 5.0, 5.0)))
    pos, vel, sp = random_state(600, p["box"], 31, 3)
    Am, Bm = np.full((3, 3), p["A"]), np.full((3, 3), p["B"])
    a = RefSim(p)
    a.set_pair_params(Am, Bm, 0b100)
    a.load_particles(pos, vel, sp)
    b = RefSim(p)
    b.set_pair_params(Am, Bm, 0b100)
    b.set_pair_gamma_sigma(np.full((3, 3), p["gamma"]), np.full((3, 3), p["sigma"]))
    b.load_particles(pos, vel, sp)
    for k in range(3):
        sa, sb = a.get_state(), b.get_state()
        for key in ("pos", "vel", "force", "rho"):
            assert np.array_equal(sa[key], sb[key]), (k, key)
        a.step(1)
        b.step(1)
    # and clearing the matrices returns to the uniform amplitudes
    c = RefSim(p)
    c.set_pair_params(Am, Bm, 0b100)
    c.set_pair_gamma_sigma(np.full((3, 3), 1.0), np.full((3, 3), 0.5))
    c.set_pair_gamma_sigma(None, None)
    c.load_particles(pos, vel, sp)
    d = RefSim(p)
    d.set_pair_params(Am, Bm, 0b100)
    d.load_particles(pos, vel, sp)
    assert np.array_equal(c.get_state()["force"], d.get_state()["force"])


def test_five_species_vs_numpy_brute_force():
    """Five species, two frozen, random symmetric A, B, gamma, sigma: forces against the independent
    O(N^2) numpy evaluation of tests/helpers.py (its own hash restatement), at a non-zero step; sum of pair forces 0."""
    p = dict(wl.default_params((4.0, 5.0, 7.0)), g=(0.02, 0.0, 0.0))
    rng = np.random.default_rng(6)
    nt = 5

    def sym(lo, hi):
        m = lo + (hi - lo) * rng.random((nt, nt))
        return 0.5 * (m + m.T)

    Am, Bm, Gm, Sm = sym(-40.0, -15.0), sym(20.0, 30.0), sym(1.0, 13.0), sym(0.5, 5.0)
    frozen_mask = 0b01010
    pos, vel, sp = random_state(700, p["box"], 13, nt)
    frozen = ((frozen_mask >> sp) & 1).astype(bool)
    s = RefSim(p)
    s.set_pair_params(Am, Bm, frozen_mask)
    s.set_pair_gamma_sigma(Gm, Sm)
    s.load_particles(pos, vel, sp)
    s.set_step(3)
    s.compute_forces()
    f, fpair, rho = brute_forces(pos, vel, frozen, p, 3, species=sp, Amat=Am, Bmat=Bm, Gmat=Gm, Smat=Sm)
    st = s.get_state()
    assert np.allclose(st["force"], f, rtol=0, atol=1e-8)
    assert np.allclose(s.pair_force(), fpair, rtol=0, atol=1e-8)
    assert np.abs(s.pair_force().sum(0)).max() < 1e-9 * np.abs(fpair).sum()
    # the matrices matter: the uniform amplitudes give a different force field
    f_uni, _, _ = brute_forces(pos, vel, frozen, p, 3, species=sp, Amat=Am, Bmat=Bm)
    assert np.abs(f_uni - f).max() > 1.0


def test_two_fluids_with_their_own_thermostats_reach_kT_1():
    """Fluctuation-dissipation per pair (sigma^2 = 2 gamma kT): species 0 with gamma = 4.5, species 1 with
    the water value 12.4 (L141), unlike pairs 8.0, every sigma_ij = sqrt(2 gamma_ij kT).  Started COLD (v = 0) the mixture
    must heat to kT = 1 +- 2 % -- with any sigma_ij inconsistent with its gamma_ij it would settle elsewhere (second
    half: sigma doubled for the unlike pairs only raises the temperature measurably)."""
    box = (6.0, 6.0, 6.0)
    c = wl.make_liquid(box, seed=41)
    n = len(c["pos"])
    sp = (np.arange(n) % 2).astype(np.uint8)
    Gm = np.array([[4.5, 8.0], [8.0, 12.4]])

    def run(Sm, nsteps=700, navg=400):
        s = RefSim(c["params"])
        s.set_pair_params(np.full((2, 2), -40.0), np.full((2, 2), 25.0), 0)
        s.set_pair_gamma_sigma(Gm, Sm)
        s.load_particles(c["pos"].astype(np.float64), np.zeros((n, 3)), sp)
        s.step(nsteps - navg)
        kts = []
        for _ in range(navg // 10):
            s.step(10)
            v = s.get_state()["vel"]
            kts.append([kinetic_temperature(v), kinetic_temperature(v[sp == 0]), kinetic_temperature(v[sp == 1])])
        return np.mean(kts, axis=0)

    kt = run(np.sqrt(2.0 * Gm * 1.0))
    # dt = 0.01 velocity-Verlet runs ~1 % warm at gamma = 4.5 (tests/test_oracle_statistics.py); each species separately too
    assert abs(kt[0] - 1.0) < 0.02, kt
    assert abs(kt[1] - 1.0) < 0.03 and abs(kt[2] - 1.0) < 0.03, kt
    Sbad = np.sqrt(2.0 * Gm * 1.0)
    Sbad[0, 1] = Sbad[1, 0] = 2.0 * Sbad[0, 1]
    assert run(Sbad, nsteps=400, navg=200)[0] > 1.5


def test_bad_arguments_are_rejected():
    p = dict(wl.default_params(BOX))
    s = RefSim(p)
    with pytest.raises(Exception):
        s.set_pair_gamma_sigma(np.full((2, 2), 4.5), np.full((2, 2), 3.0))          # no species set yet
    s.set_pair_params(np.full((2, 2), -40.0), np.full((2, 2), 25.0), 0)
    with pytest.raises(Exception):
        s.set_pair_gamma_sigma(np.full((3, 3), 4.5), np.full((3, 3), 3.0))          # another number of species
    with pytest.raises(Exception):
        s.set_pair_gamma_sigma(np.array([[4.5, 1.0], [2.0, 4.5]]), np.full((2, 2), 3.0))   # not symmetric
    with pytest.raises(Exception):
        s.set_pair_gamma_sigma(np.full((2, 2), -1.0), np.full((2, 2), 3.0))         # negative friction
    s.set_pair_gamma_sigma(np.full((2, 2), 4.5), np.full((2, 2), 3.0))
