"""Input generators.  No mDPD arithmetic lives here (see package docstring)."""
from __future__ import annotations

import numpy as np

BASE_SEED = 190310134  # "1903_10134" as a Python integer


def default_params(box, **over):
    """Parameter set of BASELINE.json config 0 (kBT=1, gamma=4.5, rc=1,
    rd=0.75, A=-40, B=25; L186: dt=0.01).  Keys mirror ``mdpd_params`` in include/mdpd.h."""
    p = dict(
        box=tuple(float(b) for b in box),
        rc=1.0, rd=0.75, A=-40.0, B=25.0,
        gamma=4.5, sigma=3.0, kT=1.0, s=1.0,
        mass=1.0, dt=0.01, g=(0.0, 0.0, 0.0),
        skin=0.25, seed=12345, max_neigh=0, reorder_every=1, flags=0,
    )
    p.update(over)
    return p


def _clip_into_box(pos, box):
    """float32 positions strictly inside [0, L) per dimension."""
    pos = np.asarray(pos, dtype=np.float32)
    for d in range(3):
        L = np.float32(box[d])
        hi = np.nextafter(L, np.float32(0.0), dtype=np.float32)
        np.clip(pos[:, d], np.float32(0.0), hi, out=pos[:, d])
    return pos


def maxwell_velocities(rng, n, kT=1.0, mass=1.0):
    """v ~ N(0, kT/m) per component, mean removed, rescaled so that
    m*sum|v|^2/(3n-3) == kT exactly (in fp64, then rounded to float32)."""
    if n == 0:
        return np.zeros((0, 3), np.float32)
    v = rng.standard_normal((n, 3)) * np.sqrt(kT / mass)
    v -= v.mean(axis=0, keepdims=True)
    if n > 1:
        cur = mass * (v * v).sum() / (3 * n - 3)
        v *= np.sqrt(kT / cur)
    return v.astype(np.float32)


def make_liquid(box, density=6.0, seed=BASE_SEED, n=None, **pover):
    """Configs 0 / 4a / 4b: periodic box, uniform-random positions, Maxwell velocities."""
    box = tuple(float(b) for b in (box if np.ndim(box) else (box,) * 3))
    rng = np.random.default_rng(seed)
    if n is None:
        n = int(round(density * box[0] * box[1] * box[2]))
    pos = rng.random((n, 3), dtype=np.float32) * np.asarray(box, np.float32)
    pos = _clip_into_box(pos, box)
    vel = maxwell_velocities(rng, n)
    return dict(name="liquid", params=default_params(box, **pover), pos=pos, vel=vel,
                type=np.zeros(n, np.uint8), mask=None, voxel=0.0)


def make_slab(box=(40.0, 20.0, 20.0), half_width=10.0, density=6.0, seed=BASE_SEED + 1, lattice=False, **pover):
    """Config 1: liquid slab |x - Lx/2| < half_width in vacuum (the |x|<10 slab shifted by Lx/2).
    lattice=False (the config's recipe): uniform-random positions.  lattice=True: a jittered lattice at the same
    number density -- a gentle start without the pressure shock of overlapping random points, for tests that compare
    a stationary profile after a short equilibration."""
    rng = np.random.default_rng(seed)
    if lattice:
        lo = (box[0] / 2 - half_width, 0.0, 0.0)
        hi = (box[0] / 2 + half_width, box[1], box[2])
        sp = density ** (-1.0 / 3.0)
        counts = [max(1, int(round((hi[d] - lo[d]) / sp))) for d in range(3)]
        pos = _clip_into_box(_jittered_lattice(rng, lo, hi, counts).astype(np.float32), box)
        n = len(pos)
    else:
        n = int(round(density * 2 * half_width * box[1] * box[2]))
        u = rng.random((n, 3), dtype=np.float32)
        pos = np.empty((n, 3), np.float32)
        pos[:, 0] = np.float32(box[0] / 2 - half_width) + u[:, 0] * np.float32(2 * half_width)
        pos[:, 1] = u[:, 1] * np.float32(box[1])
        pos[:, 2] = u[:, 2] * np.float32(box[2])
        pos = _clip_into_box(pos, box)
    vel = maxwell_velocities(rng, n)
    return dict(name="slab", params=default_params(box, **pover), pos=pos, vel=vel,
                type=np.zeros(n, np.uint8), mask=None, voxel=0.0)


def _jittered_lattice(rng, lo, hi, counts, jitter=0.2):
    """Lattice of counts[d] sites per dimension filling [lo, hi), jittered by U(+-jitter*spacing)."""
    lo = np.asarray(lo, np.float64)
    hi = np.asarray(hi, np.float64)
    counts = np.asarray(counts, np.int64)
    sp = (hi - lo) / counts
    gx, gy, gz = np.meshgrid(*(np.arange(c) for c in counts), indexing="ij")
    sites = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1).astype(np.float64)
    pts = lo + (sites + 0.5) * sp
    pts += (rng.random(pts.shape) * 2 - 1) * jitter * sp
    return pts


def make_poiseuille(L=20.0, wall=2.0, density=6.0, gx=0.05, seed=BASE_SEED + 2,
                    voxel=0.5, Lxy=None, **pover):
    """Config 2: fluid in wall < z < L - wall, two frozen walls (jittered lattice, type 1) in
    0 <= z < wall and L - wall <= z < L; voxel mask solid where the walls are; body force gx."""
    Lxy = L if Lxy is None else float(Lxy)   # box is Lxy x Lxy x L (config 2: cubic)
    box = (Lxy, Lxy, L)
    rng = np.random.default_rng(seed)
    nf = int(round(density * Lxy * Lxy * (L - 2 * wall)))
    u = rng.random((nf, 3), dtype=np.float32)
    pf = np.empty((nf, 3), np.float32)
    pf[:, 0] = u[:, 0] * np.float32(Lxy)
    pf[:, 1] = u[:, 1] * np.float32(Lxy)
    pf[:, 2] = np.float32(wall) + u[:, 2] * np.float32(L - 2 * wall)
    # keep fluid strictly inside the pore voxels
    zlo = np.nextafter(np.float32(wall), np.float32(L))
    zhi = np.nextafter(np.float32(L - wall), np.float32(0))
    np.clip(pf[:, 2], zlo, zhi, out=pf[:, 2])
    vf = maxwell_velocities(rng, nf)
    # wall lattice: nxy x nxy x nz sites per wall at number density ~density
    nz = max(1, int(round(wall / 0.5)))
    nxy = int(round(np.sqrt(density * Lxy * Lxy * wall / nz)))
    w0 = _jittered_lattice(rng, (0, 0, 0), (Lxy, Lxy, wall), (nxy, nxy, nz))
    w1 = _jittered_lattice(rng, (0, 0, L - wall), (Lxy, Lxy, L), (nxy, nxy, nz))
    pw = np.concatenate([w0, w1]).astype(np.float32)
    pw[:, 0] %= np.float32(Lxy)
    pw[:, 1] %= np.float32(Lxy)
    np.clip(pw[:w0.shape[0], 2], 0, np.nextafter(np.float32(wall), np.float32(0)), out=pw[:w0.shape[0], 2])
    np.clip(pw[w0.shape[0]:, 2], np.float32(L - wall), np.nextafter(np.float32(L), np.float32(0)),
            out=pw[w0.shape[0]:, 2])
    pos = _clip_into_box(np.concatenate([pf, pw]), box)
    vel = np.concatenate([vf, np.zeros_like(pw)])
    typ = np.concatenate([np.zeros(nf, np.uint8), np.ones(pw.shape[0], np.uint8)])
    nv = int(round(L / voxel))
    nvxy = int(round(Lxy / voxel))
    mask = np.zeros((nv, nvxy, nvxy), np.uint8)  # [nz][ny][nx]
    kw = int(round(wall / voxel))
    mask[:kw, :, :] = 1
    mask[nv - kw:, :, :] = 1
    return dict(name="poiseuille", params=default_params(box, g=(gx, 0.0, 0.0), **pover),
                pos=pos, vel=vel, type=typ, mask=mask, voxel=float(voxel))


def _periodic_gaussian_field(rng, nvox, corr):
    """White noise N(0,1) on nvox^3, periodic Gaussian filter with std `corr` voxels (FFT)."""
    w = rng.standard_normal((nvox, nvox, nvox))
    k = np.fft.fftfreq(nvox)
    kk = np.fft.rfftfreq(nvox)
    k2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + kk[None, None, :] ** 2
    filt = np.exp(-2.0 * (np.pi ** 2) * (corr ** 2) * k2)
    return np.fft.irfftn(np.fft.rfftn(w) * filt, s=w.shape, axes=(0, 1, 2))


def _periodic_dilate(ind, radius):
    """Voxels within Euclidean `radius` voxels (periodic) of any set voxel of `ind`."""
    n = ind.shape[0]
    ax = np.minimum(np.arange(n), n - np.arange(n)).astype(np.float64)
    ball = (ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2) <= radius ** 2
    conv = np.fft.irfftn(np.fft.rfftn(ind.astype(np.float64)) * np.fft.rfftn(ball.astype(np.float64)),
                         s=ind.shape, axes=(0, 1, 2))
    return conv > 0.5


def make_pore_network(nvox=128, voxel=0.5, corr=6.0, porosity=0.35, density=6.0, gx=0.02,
                      wall_depth=2.0, seed=BASE_SEED + 3, **pover):
    """Config 3: thresholded periodic Gaussian random field -> pore mask; fluid uniform in pore
    voxels; frozen wall particles on a jittered lattice in solid voxels within wall_depth of a pore."""
    rng = np.random.default_rng(seed)
    L = nvox * voxel
    box = (L, L, L)
    field = _periodic_gaussian_field(rng, nvox, corr)
    thr = np.quantile(field, porosity)
    pore = field < thr                                  # [z][y][x]
    mask = (~pore).astype(np.uint8)
    # fluid: uniform in pore voxels
    pz, py, px = np.nonzero(pore)
    npore = pz.size
    nf = int(round(density * npore * voxel ** 3))
    pick = rng.integers(0, npore, nf)
    u = rng.random((nf, 3), dtype=np.float32)
    # keep a small margin from voxel faces so float32 rounding cannot move a point to a neighbour voxel
    u = np.float32(0.001) + u * np.float32(0.998)
    pf = np.empty((nf, 3), np.float32)
    pf[:, 0] = (px[pick].astype(np.float32) + u[:, 0]) * np.float32(voxel)
    pf[:, 1] = (py[pick].astype(np.float32) + u[:, 1]) * np.float32(voxel)
    pf[:, 2] = (pz[pick].astype(np.float32) + u[:, 2]) * np.float32(voxel)
    vf = maxwell_velocities(rng, nf)
    # wall: lattice spacing density^(-1/3), keep solid sites within wall_depth of a pore voxel
    m = int(round(L / density ** (-1.0 / 3.0)))
    pts = _jittered_lattice(rng, (0, 0, 0), box, (m, m, m)).astype(np.float32)
    pts = _clip_into_box(pts % np.float32(L), box)
    iv = np.minimum((pts / np.float32(voxel)).astype(np.int64), nvox - 1)
    shell = _periodic_dilate(pore, wall_depth / voxel) & (~pore)
    keep = shell[iv[:, 2], iv[:, 1], iv[:, 0]]
    pw = pts[keep]
    pos = _clip_into_box(np.concatenate([pf, pw]), box)
    vel = np.concatenate([vf, np.zeros_like(pw)])
    typ = np.concatenate([np.zeros(nf, np.uint8), np.ones(pw.shape[0], np.uint8)])
    return dict(name="pore_network", params=default_params(box, g=(gx, 0.0, 0.0), **pover),
                pos=pos, vel=vel, type=typ, mask=mask, voxel=float(voxel))


def make_liquid_vacuum(L=100.0, Lyz=None, half_width=10.0, A=-50.0, gamma=12.4, seed=BASE_SEED + 7, **pover):
    """Section 4.1's liquid-vacuum interface: periodic box L x Lyz x Lyz, particles on an fcc lattice of
    spacing rc in the slab |x - L/2| <= half_width (the paper's box [-50, 50]^3 shifted by +50: 820 000 particles for
    L = Lyz = 100, half_width = 10), A = -50, B = 25, rd = 0.75, gamma = 12.4 (sigma^2 = 2 gamma kT), Maxwell velocities
    at kT = 1."""
    Lyz = L if Lyz is None else float(Lyz)
    box = (float(L), Lyz, Lyz)
    rng = np.random.default_rng(seed)
    nx = int(round(2 * half_width + 0.5)) + 1                 # whole cells 0 .. 2 hw, the last one contributes half a cell
    ny = int(round(Lyz))
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(ny), indexing="ij")
    cells = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], 1).astype(np.float32)
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], np.float32)
    sites = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3)
    sites = sites[sites[:, 0] < 2 * half_width + 0.5]          # x in [0, 20.5): 41 half-layers, 4 * ny^2 * 20.5 sites
    pos = sites + np.array([L / 2 - half_width, 0.25, 0.25], np.float32)
    pos = _clip_into_box(pos.astype(np.float32), box)
    n = len(pos)
    vel = maxwell_velocities(rng, n)
    sigma = float(np.sqrt(2.0 * gamma * 1.0))
    return dict(name="liquid_vacuum", params=default_params(box, A=A, gamma=gamma, sigma=sigma, **pover),
                pos=pos, vel=vel, type=np.zeros(n, np.uint8))


def make_species_mixture(box=(12.0, 10.0, 9.0), nspecies=5, frozen_mask=0b01010, density=6.0, seed=BASE_SEED + 5, **pover):
    """A liquid of `nspecies` material types drawn uniformly (type byte = species index), the species of `frozen_mask`
    frozen, with random symmetric pair matrices A_ij in [-40, -20], B_ij in [22, 28]: stands in for the five material
    types of the paper's kerogen case, whose parameter table is not in the text."""
    c = make_liquid(box, density=density, seed=seed, **pover)
    rng = np.random.default_rng(seed + 1000)
    n = len(c["pos"])
    c["type"] = rng.integers(0, nspecies, n).astype(np.uint8)
    A = (-40.0 + 20.0 * rng.random((nspecies, nspecies))).astype(np.float32)
    B = (22.0 + 6.0 * rng.random((nspecies, nspecies))).astype(np.float32)
    c["pair_A"] = np.maximum(A, A.T)
    c["pair_B"] = np.maximum(B, B.T)
    c["frozen_mask"] = int(frozen_mask)
    frozen = ((c["frozen_mask"] >> c["type"]) & 1).astype(bool)
    c["vel"][frozen] = 0.0
    c["name"] = "species_mixture"
    return c


def make_slit_wetting(A_SL=-30.0, seed=BASE_SEED + 6, **pover):
    """Section 4.2's slit pore shifted into [0, L): box 60 x 10 x 5, 3 500 solid particles (species 1,
    frozen) uniformly random in each of the wall regions 0 <= y < 1 and 9 <= y < 10, 4 000 liquid particles (species 0)
    in a block 20 <= x < 40, 1 < y < 9; A_SS = A_LL = -40, the unlike pair A_SL from Table 1, B = 25 (R19); the
    wall regions are also solid voxels of a 0.5-voxel mask (the bounce-back wall of BASELINE.json in place of the paper's
    anti-penetration model, R7)."""
    box = (60.0, 10.0, 5.0)
    rng = np.random.default_rng(seed)
    def block(n, lo, hi):
        u = rng.random((n, 3), dtype=np.float32)
        return (np.asarray(lo, np.float32) + u * (np.asarray(hi, np.float32) - np.asarray(lo, np.float32))).astype(np.float32)
    w0 = block(3500, (0, 0, 0), (60, 1, 5))
    w1 = block(3500, (0, 9, 0), (60, 10, 5))
    liq = block(4000, (20, 1.05, 0), (40, 8.95, 5))
    pos = _clip_into_box(np.concatenate([liq, w0, w1]), box)
    vel = np.concatenate([maxwell_velocities(rng, 4000), np.zeros((7000, 3), np.float32)])
    typ = np.concatenate([np.zeros(4000, np.uint8), np.ones(7000, np.uint8)])
    A = np.array([[-40.0, A_SL], [A_SL, -40.0]], np.float32)
    B = np.full((2, 2), 25.0, np.float32)
    voxel = 0.5
    mask = np.zeros((10, 20, 120), np.uint8)   # [nz][ny][nx]: the wall regions are solid voxels (no-slip bounce-back)
    mask[:, :2, :] = 1
    mask[:, 18:, :] = 1
    return dict(name="slit_wetting", params=default_params(box, **pover), pos=pos, vel=vel, type=typ,
                pair_A=A, pair_B=B, frozen_mask=0b10, mask=mask, voxel=voxel)


def quantise_positions(pos, box, bits=7):
    """Round coordinates to multiples of 2^-bits (and keep them inside the box): with boxes <= 16,
    every r^2 is then exact in fp32 and fp64 alike."""
    q = np.float32(2.0 ** bits)
    out = np.floor(np.asarray(pos, np.float64) * q) / q
    for d in range(3):
        out[:, d] = np.minimum(out[:, d], box[d] - 1.0 / q)
        out[:, d] = np.maximum(out[:, d], 0.0)
    return out.astype(np.float32)


def make_config(idx, **over):
    """BASELINE.json configs: 0, 1, 2, 3, '4a' (175^3, 32.2 M), '4b' (55^3, 1 M)."""
    if idx in (0, "0"):
        return make_liquid(10.0, seed=BASE_SEED + 0, **over)
    if idx in (1, "1"):
        return make_slab(seed=BASE_SEED + 1, **over)
    if idx in (2, "2"):
        return make_poiseuille(seed=BASE_SEED + 2, **over)
    if idx in (3, "3"):
        return make_pore_network(seed=BASE_SEED + 3, **over)
    if idx in ("4a",):
        return make_liquid(175.0, seed=BASE_SEED + 4, **over)
    if idx in (4, "4", "4b"):
        return make_liquid(55.0, seed=BASE_SEED + 4, **over)
    raise ValueError(f"unknown config {idx!r}")
