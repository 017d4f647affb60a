"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage it checks: P:L<n> = /root/reference/PAPER.md line n;
R<n> = DESIGN.md reading n.  Nothing here comes from the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import mdpd_workloads as wl
from oracle.mdpd_ref import RefSim, ref_hash, ref_rng_fill, ref_xi

from helpers import brute_density, brute_forces, brute_pairs, hash_py, kinetic_temperature, xi_py

P0 = wl.default_params((10.0, 10.0, 10.0))
K_RHO = 15.0 / (2.0 * math.pi * 0.75 ** 3)


def two_particles(r, params, v0=(0, 0, 0), v1=(0, 0, 0), direction=(1.0, 0.0, 0.0), origin=(3.0, 4.0, 5.0)):
    d = np.asarray(direction, float)
    d /= np.linalg.norm(d)
    x0 = np.asarray(origin, float)
    s = RefSim(params)
    s.load_particles([x0, x0 + r * d], [v0, v1])
    return s, d


# ------------------------------------------------------------------ closed forms (Eq. 1)
def test_w_rho_constant_and_golden_pairs(golden_dir):
    assert abs(K_RHO - 5.6588424210451675) < 1e-14
    rows = [l.split() for l in open(os.path.join(golden_dir, "closed_form_pairs.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 8
    p = dict(P0, sigma=0.0)
    for r, rho, F in [(float(a), float(b), float(c)) for a, b, c in rows]:
        for direction in [(1, 0, 0), (0, -1, 0), (1, 2, -3)]:
            s, d = two_particles(r, p, direction=direction)
            st = s.get_state()
            assert np.allclose(st["rho"], rho, rtol=0, atol=2e-10), (r, st["rho"])
            # particle 0 sits at the origin, particle 1 at +r d: repulsive F pushes particle 0 along -d
            f0 = st["force"][0]
            assert np.allclose(f0, -F * d, rtol=0, atol=5e-9), (r, f0, F)
            assert np.allclose(st["force"][1], -f0, rtol=0, atol=1e-12)


def test_w_rho_normalisation_integral():
    """int_0^inf 4 pi r^2 w_rho(r) dr = 1 -- integrate the oracle's own two-particle rho(r)
    (composite Simpson on [0, rd], 160 panels: the integrand is a quartic, error ~ 6e-9)."""
    m = 160
    rs = np.linspace(0.0, 0.75, m + 1)
    vals = []
    p = dict(P0, sigma=0.0)
    for r in rs:
        s, _ = two_particles(max(r, 1e-9), p)
        vals.append(4 * math.pi * r * r * s.get_state()["rho"][0])
    vals = np.array(vals)
    h = rs[1] - rs[0]
    integral = h / 3 * (vals[0] + vals[-1] + 4 * vals[1:-1:2].sum() + 2 * vals[2:-1:2].sum())
    assert abs(integral - 1.0) < 5e-8
    # and nothing outside rd
    s, _ = two_particles(0.7500001, p)
    assert s.get_state()["rho"][0] == 0.0


def test_dissipative_and_random_single_pair():
    """F^D = -gamma wD (e.v) e with wD = wR^2; F^R = sigma wR xi e (/sqrt(dt), R2).
    r = 0.5, e.v_ij = 1  =>  F^D = -4.5 * 0.25 = -1.125 on particle i along e_ij."""
    p = dict(P0, A=0.0, B=0.0, sigma=0.0)
    # e_ij = (x0 - x1)/r = -d ; v_ij = v0 - v1 ; choose v0 = -d  => e.v = 1
    s, d = two_particles(0.5, p, v0=(-1, 0, 0))
    f0 = s.get_state()["force"][0]
    e = -d
    assert np.allclose(f0, -1.125 * e, atol=1e-13)
    # random force: magnitude sigma * 0.5 * xi / sqrt(0.01) = 15 xi, xi from the hash of tags (0, 1)
    p = dict(P0, A=0.0, B=0.0, gamma=0.0, seed=77)
    s, d = two_particles(0.5, p)
    s.set_step(5)
    s.compute_forces()
    f0 = s.get_state()["force"][0]
    xi = xi_py(hash_py(0, 1, 5, 77))
    assert abs(xi) <= math.sqrt(3.0)
    assert np.allclose(f0, 15.0 * xi * (-d), atol=1e-12)
    # exponent s: wR = w^s (R15): s = 0.5 at r = 0.75 -> wR = 0.5, wD = 0.25
    p = dict(P0, A=0.0, B=0.0, sigma=0.0, s=0.5)
    s, d = two_particles(0.75, p, v0=(-1, 0, 0))
    assert np.allclose(s.get_state()["force"][0], -4.5 * 0.25 * (-d), atol=1e-13)


def test_three_collinear_and_triangle():
    """three collinear particles spacing .5; equilateral triangle side .5 (Eq. 1 + P:L81)."""
    p = dict(P0, sigma=0.0)
    s = RefSim(p)
    s.load_particles([[2, 2, 2], [2.5, 2, 2], [3, 2, 2]], np.zeros((3, 3)))
    st = s.get_state()
    assert np.allclose(st["rho"], [0.6287602690, 1.2575205380, 0.6287602690], atol=2e-10)
    # end-mid radial F = -4.2809932749 (attractive): particle 0 is pulled toward +x
    assert np.allclose(st["force"][0], [4.2809932749, 0, 0], atol=5e-9)
    assert np.allclose(st["force"][1], 0.0, atol=1e-12)
    assert np.allclose(st["force"][2], [-4.2809932749, 0, 0], atol=5e-9)
    a = 0.5
    tri = np.array([[0, 0, 0], [a, 0, 0], [a / 2, a * math.sqrt(3) / 2, 0]]) + 4.0
    s = RefSim(p)
    s.load_particles(tri, np.zeros((3, 3)))
    st = s.get_state()
    assert np.allclose(st["rho"], 1.2575205380, atol=2e-10)
    cen = tri.mean(0)
    for i in range(3):
        out = (tri[i] - cen) / np.linalg.norm(tri[i] - cen)
        assert np.allclose(st["force"][i], 1.6604749052 * out, atol=5e-9)


def test_simple_cubic_lattice_sums():
    """periodic simple-cubic lattice a = .5: rho = 6 w(.5) + 12 w(.7071) = 3.9946693043;
    18 neighbours r < rd, 26 neighbours r < rc (the 6 at r == 1 excluded by strict <, R3); net force 0."""
    m = 12
    a = 0.5
    g = np.arange(m) * a
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    p = dict(wl.default_params((m * a,) * 3), sigma=0.0)
    s = RefSim(p)
    s.load_particles(pos, np.zeros_like(pos))
    st = s.get_state()
    assert np.allclose(st["rho"], 3.9946693043, atol=2e-9)
    assert np.abs(st["force"]).max() < 1e-9
    n = len(pos)
    assert len(s.get_pairs(0.75)) == 18 * n // 2
    assert len(s.get_pairs(1.0)) == 26 * n // 2
    assert len(s.get_pairs(1.0 + 1e-9)) == 32 * n // 2


# ------------------------------------------------------------------ brute force on tiny boxes
@pytest.mark.parametrize("box,n,seed", [((4.0, 4.0, 4.0), 400, 1), ((5.0, 5.0, 5.0), 700, 2), ((4.0, 5.0, 7.0), 800, 3),
                                        ((3.0, 3.0, 3.0), 150, 4)])
def test_pairs_density_force_vs_numpy_brute_force(box, n, seed):
    rng = np.random.default_rng(seed)
    pos = (rng.random((n, 3)) * box).astype(np.float32).astype(np.float64)
    vel = rng.standard_normal((n, 3))
    typ = (rng.random(n) < 0.2).astype(np.uint8)
    p = wl.default_params(box, seed=99 + seed, g=(0.05, 0.0, -0.01))
    s = RefSim(p)
    s.load_particles(pos, vel, typ)
    s.set_step(17)
    s.compute_forces()
    for rcut in (0.75, 1.0, 1.25):
        bp = brute_pairs(pos, box, rcut)
        op = s.get_pairs(rcut)
        assert op.shape == bp.shape and (op == bp).all()
    st = s.get_state()
    rho = brute_density(pos, box, 0.75)
    assert np.allclose(st["rho"], rho, rtol=1e-12, atol=1e-12)
    f, fpair, _ = brute_forces(pos, vel, typ, p, 17)
    scale = np.sqrt((f * f).sum(1).mean())
    assert np.abs(st["force"] - f).max() < 1e-11 * scale
    assert np.abs(s.pair_force() - fpair).max() < 1e-11 * scale
    # the oracle's own O(N^2) mode agrees with its cell-list mode
    sb = RefSim(p, brute_force=True)
    sb.load_particles(pos, vel, typ)
    sb.set_step(17)
    sb.compute_forces()
    assert np.abs(sb.get_state()["force"] - st["force"]).max() < 1e-11 * scale
    assert (sb.get_pairs(1.0) == s.get_pairs(1.0)).all()


def test_adversarial_pair_sets():
    """Particles on box faces, cell faces, exactly at rc and rd, all in one cell, N = 1, 2 (R3, R12)."""
    box = (4.0, 4.0, 4.0)
    p = wl.default_params(box)
    pos = np.array([[0.0, 0.0, 0.0], [4.0 - 2 ** -20, 0.0, 0.0], [1.0, 0.0, 0.0], [0.75, 0.0, 0.0],
                    [2.0, 2.0, 2.0], [2.0, 2.0, 3.0], [2.0, 2.75, 2.0], [1.0, 1.0, 1.0], [1.0, 1.0, 1.0 + 2 ** -10],
                    [3.999, 3.999, 3.999], [0.001, 0.001, 0.001]])
    s = RefSim(p)
    s.load_particles(pos, np.zeros_like(pos))
    for rcut in (0.75, 1.0, 1.25):
        assert (s.get_pairs(rcut) == brute_pairs(pos, box, rcut)).all()
    pr = {tuple(x) for x in s.get_pairs(1.0).tolist()}
    assert (0, 2) not in pr and (4, 5) not in pr          # r == rc exactly: excluded (strict <)
    assert (0, 1) in pr and (9, 10) in pr                 # across the periodic boundary
    pd = {tuple(x) for x in s.get_pairs(0.75).tolist()}
    assert (0, 3) not in pd and (4, 6) not in pd          # r == rd exactly: excluded
    # all particles in one cell
    rng = np.random.default_rng(5)
    pos = 1.0 + 0.9 * rng.random((60, 3))
    s = RefSim(p)
    s.load_particles(pos, np.zeros_like(pos))
    assert (s.get_pairs(1.0) == brute_pairs(pos, box, 1.0)).all()
    for n in (1, 2):
        s = RefSim(p)
        s.load_particles(pos[:n], np.zeros((n, 3)))
        assert len(s.get_pairs(1.25)) == len(brute_pairs(pos[:n], box, 1.25))
        assert np.isfinite(s.get_state()["force"]).all()
    s = RefSim(p)
    s.load_particles(np.zeros((0, 3)), np.zeros((0, 3)))
    s.step(2)
    assert s.get_state()["pos"].shape == (0, 3)


def test_zero_beyond_cutoffs_and_momentum():
    c = wl.make_liquid(6.0, seed=11)
    s = RefSim(c["params"])
    s.load_particles(c["pos"], c["vel"])
    s.step(3)
    fp = s.pair_force()
    assert np.abs(fp.sum(0)).max() <= 1e-12 * np.abs(fp).sum()      # sum of pairwise forces = 0
    # a pair with rd <= r < rc: no density contribution, no B term (force = A w only)
    p = dict(P0, sigma=0.0, B=1e6)
    s2, d = two_particles(0.8, p)
    st = s2.get_state()
    assert (st["rho"] == 0).all()
    assert np.allclose(st["force"][0], -(-40 * (1 - 0.8)) * d, atol=1e-9)
    s3, _ = two_particles(1.0, dict(P0))
    assert (s3.get_state()["force"] == 0).all()


def test_poisson_statistics_of_random_state():
    """uniform-random points at number density 6: E[rho] = 6 (normalisation),
    Var[rho] = 6 K^2 4 pi rd^3/105 = 9.7009, E[#r<rc] = 25.13, E|F^R|^2 = (sigma^2/dt) 6 4pi/30 = 2261.9."""
    c = wl.make_config(0)
    p = dict(c["params"], A=0.0, B=0.0, gamma=0.0)
    s = RefSim(p)
    s.load_particles(c["pos"], c["vel"])
    st = s.get_state()
    n = len(c["pos"])
    assert abs(st["rho"].mean() - 6.0) < 4 * 3.1146 / math.sqrt(n) * 1.5
    assert abs(st["rho"].var() - 9.7009) < 0.6
    assert abs(2 * s.counters()["pairs_rc"] / n - 25.13) < 0.3
    f2 = (st["force"] ** 2).sum(1).mean()
    assert abs(f2 / 2261.9 - 1) < 0.05


# ------------------------------------------------------------------ hash / RNG (R5)
def test_hash_symmetry_and_python_restatement(golden_dir):
    rng = np.random.default_rng(0)
    for _ in range(300):
        a, b, k, sd = (int(x) for x in rng.integers(0, 2 ** 32, 4))
        if a == b:
            continue
        h = ref_hash(a, b, k, sd)
        assert h == ref_hash(b, a, k, sd) == hash_py(a, b, k, sd)
        assert abs(ref_xi(h) - xi_py(h)) < 1e-15
    rows = [l.split() for l in open(os.path.join(golden_dir, "rng_vectors.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) >= 32
    for a, b, k, sd, h in rows:
        assert hash_py(int(a), int(b), int(k), int(sd)) == int(h, 16) == ref_hash(int(a), int(b), int(k), int(sd))
    assert ref_xi(0) == -math.sqrt(3.0) and ref_xi(0x80000000) == 0.0
    assert ref_xi(0xFFFFFFFF) < math.sqrt(3.0)


def test_hash_statistics():
    """Acceptance tests of R5 on the oracle's stream: mean, variance, chi^2 of the top byte,
    lag-1 correlations across b, a, step, seed; avalanche per input bit."""
    n = 1 << 21
    idx = np.arange(n, dtype=np.uint32)
    thr = 4.0 / math.sqrt(n)

    def xi_of(h):
        return math.sqrt(3.0) * ((h >> 8).astype(np.float64) - 2 ** 23) / 2 ** 23

    def stream(kind):
        if kind == "b":
            return ref_rng_fill(7, np.stack([np.full(n, 3, np.uint32), idx + 4], 1), 11)
        if kind == "a":
            return ref_rng_fill(7, np.stack([idx, np.full(n, 0x7FFFFFF0, np.uint32)], 1), 11)
        raise ValueError

    for kind in ("a", "b"):
        h = stream(kind)
        xi = xi_of(h)
        assert abs(xi.mean()) < thr * 1.0
        assert abs(xi.var() - 1.0) < 0.005
        cnt = np.bincount(h >> 24, minlength=256)
        chi2 = ((cnt - n / 256) ** 2 / (n / 256)).sum()
        assert chi2 < 255 + 5 * math.sqrt(2 * 255)          # p > ~1e-6 ; typical 255 +- 22.6
        assert abs(np.corrcoef(xi[:-1], xi[1:])[0, 1]) < thr
    # across step and across seed (scalar loop through the C function, smaller n)
    m = 200000
    hs = np.array([ref_hash(5, 9, k, 7) for k in range(m)], dtype=np.uint64)
    xs = xi_of(hs)
    assert abs(np.corrcoef(xs[:-1], xs[1:])[0, 1]) < 4 / math.sqrt(m)
    hs = np.array([ref_hash(5, 9, 3, sd) for sd in range(m)], dtype=np.uint64)
    xs = xi_of(hs)
    assert abs(np.corrcoef(xs[:-1], xs[1:])[0, 1]) < 4 / math.sqrt(m)
    # the same pair at consecutive steps and different pairs at the same step are uncorrelated
    h1 = ref_rng_fill(7, np.stack([idx, idx + 1], 1), 100).astype(np.float64)
    h2 = ref_rng_fill(7, np.stack([idx, idx + 1], 1), 101).astype(np.float64)
    assert abs(np.corrcoef(h1, h2)[0, 1]) < thr
    # avalanche: flipping any input bit flips each output bit with probability 0.5 +- 0.02
    rng = np.random.default_rng(3)
    q = 1 << 16
    a = rng.integers(0, 1 << 24, q, dtype=np.uint32)
    b = a + 1 + rng.integers(0, 1 << 24, q, dtype=np.uint32)
    base = ref_rng_fill(1234, np.stack([a, b], 1), 77)

    def flips(h2):
        d = base ^ h2
        return np.unpackbits(d.view(np.uint8).reshape(-1, 4), axis=1).mean(0)

    for bit in range(0, 32, 1):
        fk = flips(ref_rng_fill(1234, np.stack([a, b], 1), 77 ^ (1 << bit)))
        fs = flips(ref_rng_fill(1234 ^ (1 << bit), np.stack([a, b], 1), 77))
        assert np.abs(fk - 0.5).max() < 0.02, ("step", bit)
        assert np.abs(fs - 0.5).max() < 0.02, ("seed", bit)
    # single-bit flips of a and of b with the order a < b preserved (a < 2^24 <= b after the offset)
    b2 = (b & np.uint32((1 << 24) - 1)) | np.uint32(1 << 28)
    base2 = ref_rng_fill(1234, np.stack([a, b2], 1), 77)
    for bit in range(0, 24):
        da = base2 ^ ref_rng_fill(1234, np.stack([a ^ np.uint32(1 << bit), b2], 1), 77)
        db = base2 ^ ref_rng_fill(1234, np.stack([a, b2 ^ np.uint32(1 << bit)], 1), 77)
        for dlt, nm in ((da, "a"), (db, "b")):
            pr = np.unpackbits(dlt.view(np.uint8).reshape(-1, 4), axis=1).mean(0)
            assert np.abs(pr - 0.5).max() < 0.02, (nm, bit)


# ------------------------------------------------------------------ integrator ("standard velocity Verlet"; R6, R7, R8)
def test_velocity_verlet_constant_force_is_exact():
    """No pair forces, body force g: velocity Verlet reproduces x0 + v0 t + g t^2/2 and v0 + g t exactly
    (up to rounding) -- pins half-kick / drift / half-kick and the body-force term."""
    p = wl.default_params((10.0, 10.0, 10.0), A=0.0, B=0.0, gamma=0.0, sigma=0.0, g=(0.3, -0.2, 0.1))
    s = RefSim(p)
    x0 = np.array([[1.0, 2.0, 3.0], [7.0, 7.0, 7.0]])
    v0 = np.array([[0.5, 0.0, -0.25], [0.0, 0.1, 0.0]])
    s.load_particles(x0, v0)
    s.step(40)
    t = 40 * 0.01
    st = s.get_state()
    g = np.array(p["g"])
    assert np.allclose(st["vel"], v0 + g * t, atol=1e-13)
    assert np.allclose(st["pos"], x0 + v0 * t + 0.5 * g * t * t, atol=1e-13)
    assert st["step"] == 40


def test_velocity_verlet_time_reversible_and_wrap():
    """Without the thermostat (gamma = sigma = 0) velocity Verlet is time reversible: n steps, flip v,
    n steps returns to the start.  Also exercises the periodic wrap (R12)."""
    c = wl.make_liquid(4.0, seed=21, density=3.0)
    p = dict(c["params"], gamma=0.0, sigma=0.0)
    s = RefSim(p)
    s.load_particles(c["pos"], c["vel"])
    x0 = s.get_state()["pos"]
    s.step(25)
    st = s.get_state()
    assert (st["pos"] >= 0).all() and (st["pos"] < 4.0).all()
    moved = np.abs(st["pos"] - x0).max()
    assert moved > 0.05
    s2 = RefSim(p)
    s2.load_particles(st["pos"], -st["vel"])
    s2.step(25)
    d = s2.get_state()["pos"] - x0
    d -= 4.0 * np.round(d / 4.0)
    assert np.abs(d).max() < 1e-9


def test_bounce_back_and_frozen_walls():
    """R7: a fluid particle whose trial position is in a solid voxel keeps its position and reverses its
    velocity; R8: frozen particles never move, carry v = 0, feel no body force, interact with fluid only."""
    box = (4.0, 4.0, 4.0)
    p = wl.default_params(box, A=0.0, B=0.0, gamma=0.0, sigma=0.0)
    mask = np.zeros((8, 8, 8), np.uint8)
    mask[0, :, :] = 1  # solid for z < 0.5
    s = RefSim(p)
    s.load_particles([[2.0, 2.0, 0.52]], [[0.3, 0.0, -1.0]])
    s.load_wall_mask(mask, 0.5)
    s.step(1)  # z* = 0.51, still pore
    st = s.get_state()
    assert np.allclose(st["pos"], [[2.003, 2.0, 0.51]]) and s.counters()["bounces"] == 0
    s.step(1)  # z* = 0.50 -> voxel 1 (pore): floor(0.5/0.5) = 1
    s.step(1)  # z* = 0.49 -> solid: bounce
    st = s.get_state()
    assert s.counters()["bounces"] == 1
    assert np.allclose(st["vel"], [[-0.3, 0.0, 1.0]])
    assert np.allclose(st["pos"], [[2.006, 2.0, 0.50]], atol=1e-12)
    # frozen wall particle + fluid particle
    p2 = wl.default_params(box, sigma=0.0, g=(0.1, 0.0, 0.0))
    s = RefSim(p2)
    s.load_particles([[1.0, 1.0, 1.0], [1.5, 1.0, 1.0], [1.2, 1.4, 1.0]], [[1, 1, 1], [0, 0, 0], [2, 2, 2]], [1, 0, 1])
    st0 = s.get_state()
    assert (st0["vel"][0] == 0).all() and (st0["vel"][2] == 0).all()
    s.step(5)
    s.compute_forces()  # re-evaluate at the full-step velocities (the step itself used the half-step ones, R6)
    st = s.get_state()
    assert (st["pos"][0] == [1.0, 1.0, 1.0]).all() and (st["pos"][2] == [1.2, 1.4, 1.0]).all()
    assert (st["vel"][[0, 2]] == 0).all()
    # wall-wall pair (0, 2) exchanges no force: the force on wall 0 is exactly minus the 0-1 pair force
    f, fpair, _ = brute_forces(st["pos"], st["vel"], [1, 0, 1], p2, st["step"])
    assert np.allclose(st["force"], f, atol=1e-12)
    assert st["rho"][0] > 0  # walls do get a density, from fluid and wall neighbours alike
    assert abs(st["rho"][0] - brute_density(st["pos"], box, 0.75)[0]) < 1e-13


def test_bounce_back_mask_axis_order():
    """The voxel mask is mask[nz][ny][nx] (include/mdpd.h, R7): on a NON-cubic box with three different voxel
    counts, one mask solid for x >= 5 only and one solid for y >= 3.5 only.  A particle driven in +x must bounce at
    the x-wall (and nowhere in the y-wall mask until it wraps), a particle driven in +y the other way round; a
    transposed index (x <-> y, or any other permutation of the three axes) fails one of the four cases."""
    box = (6.0, 4.0, 5.0)
    p = wl.default_params(box, A=0.0, B=0.0, gamma=0.0, sigma=0.0)
    nx, ny, nz = 12, 8, 10
    mx = np.zeros((nz, ny, nx), np.uint8)
    mx[:, :, 10:] = 1                      # solid for x >= 5.0
    my = np.zeros((nz, ny, nx), np.uint8)
    my[:, 7:, :] = 1                       # solid for y >= 3.5
    start = [[4.005, 2.605, 1.2]]         # off the voxel faces: no trial position lands on a boundary

    def run(mask, vel, nsteps):
        s = RefSim(p)
        s.load_particles(start, [vel])
        s.load_wall_mask(mask, 0.5)
        s.step(nsteps)
        st = s.get_state()
        return st["pos"][0], st["vel"][0], s.counters()["bounces"]

    # +x at speed 2: x* = 4.005 + 0.02 k passes 5.0 at step 50 -> first bounce there (x stays 4.985, v reversed)
    x, v, nb = run(mx, [2.0, 0.0, 0.0], 49)
    assert nb == 0 and abs(x[0] - 4.985) < 1e-9
    x, v, nb = run(mx, [2.0, 0.0, 0.0], 50)
    assert nb == 1 and abs(x[0] - 4.985) < 1e-9 and v[0] == -2.0
    # the same particle in the y-wall mask flies on (x = 5.405 is pore there): 70 steps, no bounce
    x, v, nb = run(my, [2.0, 0.0, 0.0], 70)
    assert nb == 0 and abs(x[0] - 5.405) < 1e-9
    # +y at speed 2: y* = 2.605 + 0.02 k passes 3.5 at step 45 -> bounce there in the y-wall mask, none in the x-wall mask
    x, v, nb = run(my, [0.0, 2.0, 0.0], 44)
    assert nb == 0 and abs(x[1] - 3.485) < 1e-9
    x, v, nb = run(my, [0.0, 2.0, 0.0], 45)
    assert nb == 1 and abs(x[1] - 3.485) < 1e-9 and v[1] == -2.0
    x, v, nb = run(mx, [0.0, 2.0, 0.0], 60)
    assert nb == 0 and abs(x[1] - 3.805) < 1e-9
    # +z: neither mask has a z-wall
    x, v, nb = run(mx, [0.0, 0.0, 2.0], 150)
    assert nb == 0
    x, v, nb = run(my, [0.0, 0.0, 2.0], 150)
    assert nb == 0


def test_subset_with_tags_evaluates_the_whole_systems_random_force():
    """DESIGN.md section 4 / R5: the hashed random force of a pair is a function of the two TAGS, the step and the seed.
    mdpd_ref_set_tags lets a SUBSET of a larger system keep the tags it has there (used by the 32 M-particle parity
    test, where the oracle can only afford a sub-cube).  Pins: (a) one pair with tags (70001, 12) against the
    independent Python restatement of the hash, both orders; (b) a sub-cube of a periodic liquid, loaded alone with its
    original tags, reproduces the whole system's forces on every particle whose neighbours (and their neighbours inside
    rd) are all present -- and does NOT without the tags."""
    p = dict(P0, A=0.0, B=0.0, gamma=0.0, seed=77)
    for tags in ((70001, 12), (12, 70001)):
        s, d = two_particles(0.5, p)
        s.set_step(5)
        s.set_tags(np.array(tags, np.uint32))
        f0 = s.get_state()["force"][0]
        xi = xi_py(hash_py(12, 70001, 5, 77))
        assert np.allclose(f0, 15.0 * xi * (-d), atol=1e-12)
        s.set_tags(None)                                   # back to tag == index
        assert np.allclose(s.get_state()["force"][0], 15.0 * xi_py(hash_py(0, 1, 5, 77)) * (-d), atol=1e-12)
    c = wl.make_liquid(9.0, seed=4242)
    whole = RefSim(c["params"])
    whole.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    whole.set_step(3)
    whole.compute_forces()
    W = whole.get_state()
    pos = c["pos"].astype(np.float64)
    inside = ((pos >= 1.0) & (pos < 8.0)).all(1)           # a 7^3 sub-cube, away from the periodic faces
    idx = np.nonzero(inside)[0]
    core = ((pos[idx] >= 1.0 + 1.75) & (pos[idx] < 8.0 - 1.75)).all(1)   # rc + rd inside: neighbours and their rho complete
    assert core.sum() > 100
    sub = RefSim(dict(c["params"], box=(12.0, 12.0, 12.0)))   # no periodic image of the sub-cube is within reach
    sub.load_particles(pos[idx] + 1.0, c["vel"][idx].astype(np.float64), None)
    sub.set_step(3)
    sub.compute_forces()
    S0 = sub.get_state()                                    # tags = load index of the subset: another random force
    sub.set_tags(idx.astype(np.uint32))
    S1 = sub.get_state()
    frms = np.sqrt((W["force"] ** 2).sum(1).mean())
    assert np.abs(S1["rho"][core] - W["rho"][idx][core]).max() < 1e-12
    assert np.abs(S1["force"][core] - W["force"][idx][core]).max() < 1e-10 * frms
    assert np.abs(S0["force"][core] - W["force"][idx][core]).max() > 0.05 * frms
