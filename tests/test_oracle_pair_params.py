"""Pins of the oracle's per-type-pair conservative parameters A_ij, B_ij ("the particle interaction
force between two types of materials such as solid and liquid can be modified by adjusting A_SL, B_SL"; Table 1,
PAPER.md L155-160: A_SS = A_SL' = -40, A_LL in {-35, -30, -20}; B = 25).  No GPU.  Nothing here comes from the CUDA path."""
import math

import numpy as np
import pytest

import mdpd_workloads as wl
from oracle.mdpd_ref import RefSim

from helpers import brute_forces

P0 = dict(wl.default_params((10.0, 10.0, 10.0)), sigma=0.0, gamma=0.0)
K_RHO = 15.0 / (2.0 * math.pi * 0.75 ** 3)


def pair_force_on_0(r, A, B, species=(0, 1), ntypes=2):
    s = RefSim(P0)
    Am = np.full((ntypes, ntypes), -40.0)
    Bm = np.full((ntypes, ntypes), 25.0)
    Am[0, 1] = Am[1, 0] = A      # the unlike pair; like pairs keep (-40, 25)
    Bm[0, 1] = Bm[1, 0] = B
    s.set_pair_params(Am, Bm, 0)
    s.load_particles([[3.0, 4.0, 5.0], [3.0 + r, 4.0, 5.0]], np.zeros((2, 3)), np.array(species, np.uint8))
    return -s.get_state()["force"][0][0]      # radial, + = repulsive


@pytest.mark.parametrize("A_SL", [-35.0, -30.0, -20.0])      # Table 1
def test_two_species_closed_form(A_SL):
    """Eq. (1) for one pair of unlike particles: F = A_SL (1 - r/rc) + B_SL * 2 rho(r) * (1 - r/rd),
    rho(r) = K (1 - r/rd)^2, values typed out per r."""
    for r in (0.25, 0.375, 0.5, 0.6, 0.75, 0.9, 1.0, 1.1):
        want = 0.0
        if r < 1.0:
            want = A_SL * (1.0 - r)
            if r < 0.75:
                want += 25.0 * 2.0 * K_RHO * (1.0 - r / 0.75) ** 3
        assert abs(pair_force_on_0(r, A_SL, 25.0) - want) < 5e-9, (r, A_SL)
    # like pairs keep their own entry: two liquid particles at r = 0.5 feel A_LL = -40 (golden value of Eq. (1))
    assert abs(pair_force_on_0(0.5, A_SL, 25.0, species=(0, 0)) - (-9.5206621832)) < 5e-9


def test_force_is_affine_in_A_and_B():
    """Eq. (1) is linear in A_ij and in B_ij: dF/dA = 1 - r/rc, dF/dB = (rho_i + rho_j)(1 - r/rd)."""
    for r in (0.3, 0.55, 0.7, 0.85):
        f0 = pair_force_on_0(r, -40.0, 25.0)
        assert abs(pair_force_on_0(r, -17.0, 25.0) - f0 - 23.0 * (1.0 - r)) < 5e-9
        rho2 = 2.0 * K_RHO * max(0.0, 1.0 - r / 0.75) ** 2
        assert abs(pair_force_on_0(r, -40.0, 31.0) - f0 - 6.0 * rho2 * max(0.0, 1.0 - r / 0.75)) < 5e-9


def random_state(n, box, seed, nspecies):
    rng = np.random.default_rng(seed)
    pos = rng.random((n, 3)) * np.asarray(box)
    vel = rng.standard_normal((n, 3))
    sp = rng.integers(0, nspecies, n).astype(np.uint8)
    return pos, vel, sp


def test_uniform_matrix_equals_single_material():
    """A matrix whose entries all equal (A, B) with species 1 frozen is the one-material path, bit for bit."""
    p = dict(wl.default_params((5.0, 5.0, 5.0)))
    pos, vel, sp = random_state(600, p["box"], 11, 2)
    a = RefSim(p)
    a.load_particles(pos, vel, sp)
    b = RefSim(p)
    b.set_pair_params(np.full((2, 2), p["A"]), np.full((2, 2), p["B"]), frozen_mask=0b10)
    b.load_particles(pos, vel, sp)
    for k in range(3):
        sa, sb = a.get_state(), b.get_state()
        for key in ("pos", "vel", "force", "rho"):
            assert np.array_equal(sa[key], sb[key]), (k, key)
        a.step(1)
        b.step(1)


def test_five_species_vs_numpy_brute_force():
    """Five material types, two of them frozen, random symmetric A_ij, B_ij: total and pairwise forces
    against an independent O(N^2) numpy evaluation; pairwise forces sum to zero; frozen species never move."""
    p = dict(wl.default_params((4.0, 5.0, 7.0)), g=(0.02, 0.0, 0.0))
    rng = np.random.default_rng(5)
    nt = 5
    Am = -40.0 + 25.0 * rng.random((nt, nt))
    Am = 0.5 * (Am + Am.T)
    Bm = 20.0 + 10.0 * rng.random((nt, nt))
    Bm = 0.5 * (Bm + Bm.T)
    frozen_mask = 0b01010
    pos, vel, sp = random_state(700, p["box"], 12, nt)
    frozen = ((frozen_mask >> sp) & 1).astype(bool)
    s = RefSim(p)
    s.set_pair_params(Am, Bm, frozen_mask)
    s.load_particles(pos, vel, sp)
    f, fpair, rho = brute_forces(pos, vel, frozen, p, 0, species=sp, Amat=Am, Bmat=Bm)
    st = s.get_state()
    assert np.allclose(st["rho"], rho, rtol=0, atol=1e-10)
    assert np.allclose(st["force"], f, rtol=0, atol=1e-8)
    assert np.allclose(s.pair_force(), fpair, rtol=0, atol=1e-8)
    assert np.abs(s.pair_force().sum(0)).max() < 1e-9 * np.abs(fpair).sum()
    x0 = st["pos"].copy()
    s.step(5)
    st = s.get_state()
    assert np.array_equal(st["pos"][frozen], x0[frozen]) and not np.array_equal(st["pos"][~frozen], x0[~frozen])
    assert np.all(st["vel"][frozen] == 0.0)


def test_bad_arguments_are_rejected():
    s = RefSim(P0)
    A = np.array([[-40.0, -30.0], [-31.0, -40.0]])
    with pytest.raises(Exception):
        s.set_pair_params(A, np.full((2, 2), 25.0), 0)            # not symmetric
    s.set_pair_params(np.full((2, 2), -40.0), np.full((2, 2), 25.0), 0)
    with pytest.raises(Exception):
        s.load_particles(np.ones((2, 3)), np.zeros((2, 3)), np.array([0, 2], np.uint8))   # species 2 of 2
