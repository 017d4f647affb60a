"""ctypes binding of the fp64 CPU oracle (oracle/mdpd_ref.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_1903_10134_b200/ (the
product path has no CPU fallback).  Shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mdpd_ref.c")
_LIB = os.path.join(_HERE, "libmdpd_ref.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, no OpenMP, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O3", "-std=c11", "-D_GNU_SOURCE", "-fPIC", "-shared", "-ffp-contract=off",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("box", C.c_double * 3), ("rc", C.c_double), ("rd", C.c_double), ("A", C.c_double),
                ("B", C.c_double), ("gamma", C.c_double), ("sigma", C.c_double), ("kT", C.c_double),
                ("s", C.c_double), ("mass", C.c_double), ("dt", C.c_double), ("g", C.c_double * 3),
                ("seed", C.c_uint32), ("pad", C.c_uint32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, u64, u32, dp = C.c_void_p, C.c_uint64, C.c_uint32, C.POINTER(C.c_double)
        L.mdpd_ref_hash.restype = C.c_uint32
        L.mdpd_ref_hash.argtypes = [u32, u32, u32, u32]
        L.mdpd_ref_xi.restype = C.c_double
        L.mdpd_ref_xi.argtypes = [u32]
        L.mdpd_ref_rng_fill.argtypes = [u32, u64, vp, u32, vp]
        L.mdpd_ref_create.argtypes = [C.POINTER(vp)]
        L.mdpd_ref_destroy.argtypes = [vp]
        L.mdpd_ref_set_params.argtypes = [vp, C.POINTER(_Params)]
        L.mdpd_ref_set_brute_force.argtypes = [vp, C.c_int]
        L.mdpd_ref_set_pair_params.argtypes = [vp, C.c_int, vp, vp, u32]
        L.mdpd_ref_set_pair_gamma_sigma.argtypes = [vp, C.c_int, vp, vp]
        L.mdpd_ref_compute_forces.argtypes = [vp]
        L.mdpd_ref_load_particles.argtypes = [vp, u64, vp, vp, vp]
        L.mdpd_ref_load_wall_mask.argtypes = [vp, vp, vp, C.c_double]
        L.mdpd_ref_set_step.argtypes = [vp, u64]
        L.mdpd_ref_set_tags.argtypes = [vp, vp]
        L.mdpd_ref_set_velocities.argtypes = [vp, vp]
        L.mdpd_ref_step.argtypes = [vp, u32]
        L.mdpd_ref_get_state.argtypes = [vp, vp, vp, vp, vp, vp]
        L.mdpd_ref_get_pair_force.argtypes = [vp, vp]
        L.mdpd_ref_get_counters.argtypes = [vp, vp, vp]
        L.mdpd_ref_get_virial.argtypes = [vp, vp]
        L.mdpd_ref_get_pairs.argtypes = [vp, C.c_double, vp, vp, u64]
        _lib = L
    return _lib


def ref_hash(a, b, step, seed) -> int:
    a, b = int(a), int(b)
    return int(lib().mdpd_ref_hash(min(a, b), max(a, b), int(step) & 0xFFFFFFFF, int(seed) & 0xFFFFFFFF))


def ref_xi(h) -> float:
    return float(lib().mdpd_ref_xi(int(h)))


def ref_rng_fill(seed, pairs, step) -> np.ndarray:
    pairs = np.ascontiguousarray(pairs, np.uint32).reshape(-1, 2)
    out = np.empty(pairs.shape[0], np.uint32)
    lib().mdpd_ref_rng_fill(int(seed), pairs.shape[0], pairs.ctypes.data, int(step), out.ctypes.data)
    return out


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


class RefSim:
    """fp64 oracle simulation; same logical API as the product's Simulation (get_state in tag order)."""

    def __init__(self, params: dict, brute_force: bool = False):
        self._L = lib()
        self._h = C.c_void_p()
        _check(self._L.mdpd_ref_create(C.byref(self._h)), "create")
        p = _Params()
        p.box[:] = [float(b) for b in params["box"]]
        for k in ("rc", "rd", "A", "B", "gamma", "sigma", "kT", "s", "mass", "dt"):
            setattr(p, k, float(params[k]))
        p.g[:] = [float(b) for b in params["g"]]
        p.seed = int(params["seed"]) & 0xFFFFFFFF
        _check(self._L.mdpd_ref_set_params(self._h, C.byref(p)), "set_params")
        self._L.mdpd_ref_set_brute_force(self._h, 1 if brute_force else 0)
        self.n = 0

    def close(self):
        if self._h:
            self._L.mdpd_ref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_pair_params(self, A, B, frozen_mask=0):
        """Per-type-pair A_ij, B_ij ([nt][nt], symmetric; Tables 1-2) and the set of frozen species (bit s);
        call before load_particles, whose type byte is then the species index.  A = None: back to one material."""
        if A is None:
            _check(self._L.mdpd_ref_set_pair_params(self._h, 0, None, None, 0), "set_pair_params")
            return
        A = np.ascontiguousarray(A, np.float64)
        B = np.ascontiguousarray(B, np.float64)
        nt = A.shape[0]
        assert A.shape == (nt, nt) and B.shape == (nt, nt)
        _check(self._L.mdpd_ref_set_pair_params(self._h, nt, A.ctypes.data, B.ctypes.data, int(frozen_mask)),
               "set_pair_params")

    def set_pair_gamma_sigma(self, G, S):
        """Per-type-pair gamma_ij, sigma_ij ([nt][nt], symmetric, the two parameter sets of P:L89 and P:L141) for
        the species set of the last set_pair_params; G = None: back to the uniform gamma, sigma.  Takes effect at the
        next force evaluation."""
        if G is None or S is None:
            _check(self._L.mdpd_ref_set_pair_gamma_sigma(self._h, 0, None, None), "set_pair_gamma_sigma")
            return
        G = np.ascontiguousarray(G, np.float64)
        S = np.ascontiguousarray(S, np.float64)
        nt = G.shape[0]
        assert G.shape == (nt, nt) and S.shape == (nt, nt)
        _check(self._L.mdpd_ref_set_pair_gamma_sigma(self._h, nt, G.ctypes.data, S.ctypes.data), "set_pair_gamma_sigma")

    def load_particles(self, pos, vel, type=None):
        pos = np.ascontiguousarray(pos, np.float64).reshape(-1, 3)
        vel = np.ascontiguousarray(vel, np.float64).reshape(-1, 3)
        n = pos.shape[0]
        t = None if type is None else np.ascontiguousarray(type, np.uint8)
        _check(self._L.mdpd_ref_load_particles(self._h, n, pos.ctypes.data, vel.ctypes.data,
                                               None if t is None else t.ctypes.data), "load_particles")
        self.n = n

    def load_wall_mask(self, mask, voxel):
        if mask is None:
            _check(self._L.mdpd_ref_load_wall_mask(self._h, None, None, 0.0), "load_wall_mask")
            return
        mask = np.ascontiguousarray(mask, np.uint8)
        nz, ny, nx = mask.shape
        dims = np.array([nx, ny, nz], np.uint32)
        _check(self._L.mdpd_ref_load_wall_mask(self._h, mask.ctypes.data, dims.ctypes.data, float(voxel)),
               "load_wall_mask")

    def set_step(self, k):
        _check(self._L.mdpd_ref_set_step(self._h, int(k)), "set_step")

    def set_tags(self, tags):
        """The loaded particles are a subset of a larger system: they keep the tags they have there (hash input, DESIGN.md
        section 4).  None returns to tag == load index.  Forces are re-evaluated."""
        if tags is None:
            _check(self._L.mdpd_ref_set_tags(self._h, None), "set_tags")
            return
        t = np.ascontiguousarray(tags, np.uint32)
        assert t.shape == (self.n,)
        _check(self._L.mdpd_ref_set_tags(self._h, t.ctypes.data), "set_tags")

    def set_velocities(self, vel):
        vel = np.ascontiguousarray(vel, np.float64).reshape(-1, 3)
        _check(self._L.mdpd_ref_set_velocities(self._h, vel.ctypes.data), "set_velocities")

    def compute_forces(self):
        _check(self._L.mdpd_ref_compute_forces(self._h), "compute_forces")

    def step(self, n=1):
        _check(self._L.mdpd_ref_step(self._h, int(n)), "step")

    def get_state(self):
        n = self.n
        pos = np.empty((n, 3)); vel = np.empty((n, 3)); f = np.empty((n, 3)); rho = np.empty(n)
        step = C.c_uint64()
        _check(self._L.mdpd_ref_get_state(self._h, pos.ctypes.data, vel.ctypes.data, f.ctypes.data,
                                          rho.ctypes.data, C.addressof(step)), "get_state")
        return dict(pos=pos, vel=vel, force=f, rho=rho, step=int(step.value))

    def pair_force(self):
        f = np.empty((self.n, 3))
        _check(self._L.mdpd_ref_get_pair_force(self._h, f.ctypes.data), "get_pair_force")
        return f

    def virial(self):
        """sum over interacting pairs of r_a F^C_b at the last force evaluation: [xx, yy, zz, xy, xz, yz]."""
        out = np.zeros(6, np.float64)
        _check(self._L.mdpd_ref_get_virial(self._h, out.ctypes.data), "get_virial")
        return out

    def counters(self):
        out = np.zeros(4, np.uint64); outf = np.zeros(2)
        _check(self._L.mdpd_ref_get_counters(self._h, out.ctypes.data, outf.ctypes.data), "get_counters")
        return dict(steps=int(out[0]), bounces=int(out[1]), pairs_rc=int(out[2]), n=int(out[3]),
                    virial_c=float(outf[0]))

    def get_pairs(self, rcut):
        cnt = C.c_uint64()
        _check(self._L.mdpd_ref_get_pairs(self._h, float(rcut), C.addressof(cnt), None, 0), "get_pairs")
        m = int(cnt.value)
        pairs = np.empty((max(m, 1), 2), np.uint32)
        _check(self._L.mdpd_ref_get_pairs(self._h, float(rcut), C.addressof(cnt), pairs.ctypes.data, m), "get_pairs")
        return pairs[:m]
