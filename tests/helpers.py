"""Test-side helpers: an independent brute-force O(N^2) evaluation written in numpy, an
independent pure-Python restatement of the hash from DESIGN.md's text, and observables.
None of this is imported by the oracle or by the CUDA path."""
from __future__ import annotations

import math

import numpy as np

M32 = 0xFFFFFFFF


def hash_py(a, b, step, seed):
    """DESIGN.md 'RNG specification' restated with Python integers (arbitrary precision, masked)."""
    a, b = (a, b) if a < b else (b, a)
    x, y = a & M32, b & M32
    for r in range(6):
        if r % 2 == 0:
            key = (step + (r // 2) * 0x9E3779B9) & M32
        else:
            key = (seed + (r // 2) * 0xBB67AE85) & M32
        p = 0xD256D193 * x
        x, y = ((p >> 32) ^ y ^ key) & M32, p & M32
    return x


def xi_py(h):
    return math.sqrt(3.0) * (((h >> 8) - (1 << 23)) / float(1 << 23))


def minimg_all(pos, box):
    """d[i, j] = minimum image of pos[i] - pos[j] (fp64)."""
    pos = np.asarray(pos, np.float64)
    d = pos[:, None, :] - pos[None, :, :]
    L = np.asarray(box, np.float64)
    d = np.where(d > 0.5 * L, d - L, d)
    d = np.where(d < -0.5 * L, d + L, d)
    return d


def brute_pairs(pos, box, rcut):
    d = minimg_all(pos, box)
    r2 = (d * d).sum(-1)
    i, j = np.nonzero(np.triu(r2 < rcut * rcut, k=1))
    return np.stack([i, j], 1).astype(np.uint32)


def brute_density(pos, box, rd):
    d = minimg_all(pos, box)
    r = np.sqrt((d * d).sum(-1))
    n = len(pos)
    K = 15.0 / (2.0 * math.pi * rd ** 3)
    w = np.where(r < rd, K * (1.0 - r / rd) ** 2, 0.0)
    w[np.arange(n), np.arange(n)] = 0.0
    return w.sum(1)


def brute_forces(pos, vel, typ, p, step, rho=None, species=None, Amat=None, Bmat=None, Gmat=None, Smat=None):
    """O(N^2) total force per particle (pairwise part + m g on fluid), fp64, python-loop hash.
    typ: frozen flags.  species / Amat / Bmat: per-type-pair A_ij, B_ij (Tables 1-2); default one material.
    Gmat / Smat: per-type-pair gamma_ij, sigma_ij; default the uniform gamma, sigma of p."""
    pos = np.asarray(pos, np.float64)
    vel = np.asarray(vel, np.float64).copy()
    typ = np.asarray(typ).astype(bool)
    vel[typ] = 0.0
    n = len(pos)
    box = p["box"]
    if rho is None:
        rho = brute_density(pos, box, p["rd"])
    d = minimg_all(pos, box)
    r2 = (d * d).sum(-1)
    f = np.zeros((n, 3))
    ii, jj = np.nonzero(np.triu(r2 < p["rc"] ** 2, k=1))
    for i, j in zip(ii.tolist(), jj.tolist()):
        if typ[i] and typ[j]:
            continue
        if r2[i, j] < 1e-20:
            continue
        r = math.sqrt(r2[i, j])
        e = d[i, j] / r
        w = 1.0 - r / p["rc"]
        wd = max(0.0, 1.0 - r / p["rd"])
        wR = w ** p["s"]
        xi = xi_py(hash_py(i, j, step, p["seed"]))
        A, B = (p["A"], p["B"]) if species is None else (Amat[species[i]][species[j]], Bmat[species[i]][species[j]])
        gam = p["gamma"] if Gmat is None else Gmat[species[i]][species[j]]
        sig = p["sigma"] if Smat is None else Smat[species[i]][species[j]]
        F = (A * w + B * (rho[i] + rho[j]) * wd
             - gam * wR * wR * float(e @ (vel[i] - vel[j]))
             + sig * wR * xi / math.sqrt(p["dt"]))
        f[i] += F * e
        f[j] -= F * e
    fpair = f.copy()
    g = np.asarray(p["g"], np.float64) * p["mass"]
    f[~typ] += g
    return f, fpair, rho


def kinetic_temperature(vel, typ=None, mass=1.0):
    """kT = m sum_fluid |v - vbar|^2 / (3 Nf - 3)   (R9)."""
    v = np.asarray(vel, np.float64)
    if typ is not None:
        v = v[np.asarray(typ) == 0]
    v = v - v.mean(0, keepdims=True)
    return mass * (v * v).sum() / (3 * len(v) - 3)


def profile(coord, values, lo, hi, nbins):
    """mean of `values` in equal bins of `coord`; returns (centres, mean, count)."""
    edges = np.linspace(lo, hi, nbins + 1)
    idx = np.clip(np.digitize(coord, edges) - 1, 0, nbins - 1)
    cnt = np.bincount(idx, minlength=nbins).astype(np.float64)
    s = np.bincount(idx, weights=values, minlength=nbins)
    with np.errstate(invalid="ignore", divide="ignore"):
        m = np.where(cnt > 0, s / cnt, 0.0)
    return 0.5 * (edges[1:] + edges[:-1]), m, cnt
