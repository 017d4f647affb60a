"""Thin ctypes binding of libmdpd_b200.so (include/mdpd.h): argument marshalling only.

Every step of the mDPD timestep (Eq. (1), L125-133 Algorithm 1) runs in the CUDA kernels of
``csrc/mdpd_b200.cu``; PyTorch supplies device memory (the workspace tensor) and the stream, nothing else.
There is NO CPU fallback: without the built library or without a CUDA device this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libmdpd_b200.so")

MDPD_OK, MDPD_EINVAL, MDPD_ENOMEM, MDPD_ECUDA = 0, -1, -2, -3
MDPD_EOVERFLOW, MDPD_ESTATE, MDPD_ENAN, MDPD_EINSOLID = -4, -5, -6, -7
MDPD_FLAG_NO_GRAPH = 1
MDPD_FLAG_DIRECT = 2

_ERRNAME = {-1: "MDPD_EINVAL", -2: "MDPD_ENOMEM", -3: "MDPD_ECUDA", -4: "MDPD_EOVERFLOW", -5: "MDPD_ESTATE",
            -6: "MDPD_ENAN", -7: "MDPD_EINSOLID"}

# every symbol include/mdpd.h declares
SYMBOLS = ("mdpd_create", "mdpd_destroy", "mdpd_set_params", "mdpd_set_pair_params", "mdpd_set_pair_gamma_sigma", "mdpd_workspace_bytes", "mdpd_set_workspace",
           "mdpd_load_particles", "mdpd_load_wall_mask", "mdpd_step", "mdpd_get_state", "mdpd_set_step_counter",
           "mdpd_set_forces",
           "mdpd_compute_forces", "mdpd_compute_virial", "mdpd_get_pairs", "mdpd_get_pairs_static", "mdpd_rng_fill", "mdpd_get_counters", "mdpd_last_error",
           "mdpd_profile_begin", "mdpd_profile_end", "mdpd_profile_name", "mdpd_build_flags", "mdpd_probe_issue_rates")
MDPD_PROF_SLOTS = 16
MDPD_STATIC_PAIRS_MAX = 524288   # include/mdpd.h: pairs the fixed scratch of mdpd_get_pairs_static holds


class MdpdError(RuntimeError):
    def __init__(self, code, what, text=""):
        self.code = code
        super().__init__(f"{what}: {_ERRNAME.get(code, code)} {text}".strip())


class mdpd_params(C.Structure):
    """Mirror of ``mdpd_params`` in include/mdpd.h (field order and types must match)."""
    _fields_ = [("box", C.c_float * 3), ("rc", C.c_float), ("rd", C.c_float), ("A", C.c_float), ("B", C.c_float),
                ("gamma", C.c_float), ("sigma", C.c_float), ("kT", C.c_float), ("s", C.c_float),
                ("mass", C.c_float), ("dt", C.c_float), ("g", C.c_float * 3), ("skin", C.c_float),
                ("headroom", C.c_float),
                ("seed", C.c_uint32), ("max_neigh", C.c_uint32), ("reorder_every", C.c_uint32),
                ("flags", C.c_uint32)]


def make_params(d: dict) -> mdpd_params:
    p = mdpd_params()
    p.box[:] = [float(b) for b in d["box"]]
    for k in ("rc", "rd", "A", "B", "gamma", "sigma", "kT", "s", "mass", "dt", "skin"):
        setattr(p, k, float(d[k]))
    p.g[:] = [float(b) for b in d["g"]]
    p.headroom = float(d.get("headroom", 0.0))
    for k in ("seed", "max_neigh", "reorder_every", "flags"):
        setattr(p, k, int(d.get(k, 0)) & 0xFFFFFFFF)
    return p


_lib = None


def lib():
    """Load libmdpd_b200.so (built in-tree by ``paper_1903_10134_b200/build.py``); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1903_10134_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, u64, u32, i32, f32 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int, C.c_float
        pp = C.POINTER(mdpd_params)
        L.mdpd_create.argtypes = [C.POINTER(vp), i32, vp]
        L.mdpd_destroy.argtypes = [vp]
        L.mdpd_set_params.argtypes = [vp, pp]
        L.mdpd_set_pair_params.argtypes = [vp, u32, vp, vp, u32]
        L.mdpd_set_pair_gamma_sigma.argtypes = [vp, u32, vp, vp]
        L.mdpd_workspace_bytes.argtypes = [pp, u64, i32, vp]
        L.mdpd_workspace_bytes.restype = C.c_size_t
        L.mdpd_set_workspace.argtypes = [vp, vp, C.c_size_t]
        L.mdpd_load_particles.argtypes = [vp, u64, vp, vp, vp]
        L.mdpd_load_wall_mask.argtypes = [vp, vp, vp, f32]
        L.mdpd_step.argtypes = [vp, u32]
        L.mdpd_get_state.argtypes = [vp, vp, vp, vp, vp, vp]
        L.mdpd_set_step_counter.argtypes = [vp, u64]
        L.mdpd_set_forces.argtypes = [vp, vp]
        L.mdpd_compute_forces.argtypes = [vp]
        L.mdpd_compute_virial.argtypes = [vp, vp]
        L.mdpd_get_pairs.argtypes = [vp, f32, vp, vp, u64]
        L.mdpd_get_pairs_static.argtypes = [vp, f32, vp, vp, u64]
        L.mdpd_rng_fill.argtypes = [vp, u64, vp, u32, vp]
        L.mdpd_get_counters.argtypes = [vp, vp]
        L.mdpd_last_error.argtypes = [vp]
        L.mdpd_last_error.restype = C.c_char_p
        L.mdpd_profile_begin.argtypes = [vp]
        L.mdpd_profile_end.argtypes = [vp, vp, vp]
        L.mdpd_profile_name.argtypes = [i32]
        L.mdpd_profile_name.restype = C.c_char_p
        L.mdpd_probe_issue_rates.argtypes = [i32, vp, vp]
        L.mdpd_build_flags.argtypes = []
        L.mdpd_build_flags.restype = C.c_char_p
        for s in SYMBOLS:
            getattr(L, s).restype = getattr(L, s).restype  # touch: AttributeError if a symbol is missing
        _lib = L
    return _lib


def _ptr(a):
    """Host numpy array or torch tensor (host or device) -> raw pointer; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()  # torch tensor


COUNTER_NAMES = ("steps", "rebuilds", "bounces", "max_nbr", "sum_nbr", "max_staged", "faults", "launches",
                 "sum_act", "density_passes", "tile_shape", "ntiles")


def build_flags() -> str:
    """``mdpd_build_flags``: the extra -D options of the loaded library ("" = the plain build)."""
    return lib().mdpd_build_flags().decode()


def probe_issue_rates(device: int = 0, stream=None):
    """mdpd_probe_issue_rates: measured warp-instructions/s of the whole GPU for FFMA, the logic pipe and IMAD.WIDE."""
    import torch
    st = (stream or torch.cuda.current_stream(device)).cuda_stream
    out = np.zeros(4, np.float64)
    rc = lib().mdpd_probe_issue_rates(int(device), C.c_void_p(st), out.ctypes.data)
    if rc != MDPD_OK:
        raise MdpdError(rc, "mdpd_probe_issue_rates")
    return {"ffma": float(out[0]), "logic": float(out[1]), "imad_wide": float(out[2]), "sm_clock_hz": float(out[3])}


class Simulation:
    """One mDPD simulation on one GPU.  Methods carry the C-ABI's names and only marshal arguments."""

    def __init__(self, params: dict, device: int = 0, stream=None):
        import torch  # device memory + streams only
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the mDPD path has no CPU fallback")
        self._torch = torch
        self._L = lib()
        self.device = int(device)
        self.params = dict(params)
        self._p = make_params(params)
        torch.cuda.set_device(self.device)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        rc = self._L.mdpd_create(C.byref(self._h), self.device, C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            self._h = None
            raise MdpdError(rc, "mdpd_create")
        self._ws = None
        self.n = 0
        self._ck(self._L.mdpd_set_params(self._h, C.byref(self._p)), "mdpd_set_params")

    # -- plumbing ---------------------------------------------------------------------------------------------
    def _ck(self, rc, what):
        if rc != 0:
            txt = self._L.mdpd_last_error(self._h)
            raise MdpdError(rc, what, txt.decode() if txt else "")

    def close(self):
        if getattr(self, "_h", None):
            self._L.mdpd_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- C-ABI calls ------------------------------------------------------------------------------------------
    def set_params(self, **changes):
        self.params.update(changes)
        self._p = make_params(self.params)
        self._ck(self._L.mdpd_set_params(self._h, C.byref(self._p)), "mdpd_set_params")

    def set_pair_gamma_sigma(self, gamma, sigma):
        """mdpd_set_pair_gamma_sigma: per-type-pair gamma_ij, sigma_ij ([nt][nt], symmetric) for the species set of the last
        set_pair_params; None returns to the uniform amplitudes."""
        if gamma is None or sigma is None:
            self._ck(self._L.mdpd_set_pair_gamma_sigma(self._h, 0, None, None), "mdpd_set_pair_gamma_sigma")
            return
        G = np.ascontiguousarray(gamma, np.float32)
        S = np.ascontiguousarray(sigma, np.float32)
        nt = G.shape[0]
        if G.shape != (nt, nt) or S.shape != (nt, nt):
            raise ValueError("gamma and sigma must be [ntypes][ntypes]")
        self._ck(self._L.mdpd_set_pair_gamma_sigma(self._h, nt, G.ctypes.data, S.ctypes.data), "mdpd_set_pair_gamma_sigma")

    def set_pair_params(self, A, B, frozen_mask=0):
        """mdpd_set_pair_params: per-type-pair A_ij, B_ij ([nt][nt], symmetric) and the frozen species (bit s)."""
        if A is None:
            self._ck(self._L.mdpd_set_pair_params(self._h, 0, None, None, 0), "mdpd_set_pair_params")
            return
        A = np.ascontiguousarray(A, np.float32)
        B = np.ascontiguousarray(B, np.float32)
        nt = A.shape[0]
        if A.shape != (nt, nt) or B.shape != (nt, nt):
            raise ValueError("A, B must be [nt][nt]")
        self._ck(self._L.mdpd_set_pair_params(self._h, nt, A.ctypes.data, B.ctypes.data, int(frozen_mask)),
                 "mdpd_set_pair_params")

    def workspace_bytes(self, n, mask_dims=None):
        md = None if mask_dims is None else (C.c_uint32 * 3)(*[int(x) for x in mask_dims])
        return int(self._L.mdpd_workspace_bytes(C.byref(self._p), int(n), 0 if md is None else 1, md))

    def load_particles(self, pos, vel, type=None, mask_dims=None):
        """pos, vel: [n][3] float32 (numpy, or torch host/device); type: [n] uint8 or None.  The workspace is a
        torch uint8 tensor owned by this object (PyTorch owns device memory)."""
        torch = self._torch
        if isinstance(pos, np.ndarray):
            pos = np.ascontiguousarray(pos, np.float32).reshape(-1, 3)
            vel = np.ascontiguousarray(vel, np.float32).reshape(-1, 3)
            if type is not None:
                type = np.ascontiguousarray(type, np.uint8)
        n = int(pos.shape[0])
        need = self.workspace_bytes(n, mask_dims)
        if need == 0:
            self._ck(MDPD_EINVAL, "mdpd_workspace_bytes (bad parameters)")
        if self._ws is None or self._ws.numel() < need + 256:
            # the old tensor stays alive until the handle has accepted the new one (the handle points into it)
            ws = torch.empty(need + 256, dtype=torch.uint8, device=f"cuda:{self.device}")
            ptr = (ws.data_ptr() + 255) // 256 * 256
            self._ck(self._L.mdpd_set_workspace(self._h, C.c_void_p(ptr), need), "mdpd_set_workspace")
            self._ws, self._ws_ptr = ws, ptr
        self._ck(self._L.mdpd_load_particles(self._h, n, _ptr(pos), _ptr(vel), _ptr(type)), "mdpd_load_particles")
        self.n = n

    def load_wall_mask(self, mask, voxel):
        if mask is None:
            self._ck(self._L.mdpd_load_wall_mask(self._h, None, None, 0.0), "mdpd_load_wall_mask")
            return
        if isinstance(mask, np.ndarray):
            mask = np.ascontiguousarray(mask, np.uint8)
        nz, ny, nx = mask.shape
        dims = (C.c_uint32 * 3)(nx, ny, nz)
        self._ck(self._L.mdpd_load_wall_mask(self._h, _ptr(mask), dims, float(voxel)), "mdpd_load_wall_mask")

    def step(self, n=1):
        self._ck(self._L.mdpd_step(self._h, int(n)), "mdpd_step")

    def compute_forces(self):
        self._ck(self._L.mdpd_compute_forces(self._h), "mdpd_compute_forces")

    def compute_virial(self):
        """mdpd_compute_virial: [xx, yy, zz, xy, xz, yz] of sum over pairs r_a F^C_b (also refreshes rho and f)."""
        out = np.zeros(6, np.float64)
        self._ck(self._L.mdpd_compute_virial(self._h, out.ctypes.data), "mdpd_compute_virial")
        return out

    def set_step_counter(self, k):
        self._ck(self._L.mdpd_set_step_counter(self._h, int(k)), "mdpd_set_step_counter")

    def set_forces(self, force):
        if isinstance(force, np.ndarray):
            force = np.ascontiguousarray(force, np.float32).reshape(-1, 3)
        self._ck(self._L.mdpd_set_forces(self._h, _ptr(force)), "mdpd_set_forces")

    def get_state(self, pos=True, vel=True, force=True, rho=True, out=None):
        """Returns numpy arrays in TAG order (host).  ``out``: optional dict of preallocated host/device buffers."""
        n = self.n
        res = {}
        bufs = {}
        for key, want, shape in (("pos", pos, (n, 3)), ("vel", vel, (n, 3)), ("force", force, (n, 3)),
                                 ("rho", rho, (n,))):
            if out is not None and key in out:
                bufs[key] = out[key]
            elif want:
                bufs[key] = np.empty(shape, np.float32)
            else:
                bufs[key] = None
        step = C.c_uint64()
        self._ck(self._L.mdpd_get_state(self._h, _ptr(bufs["pos"]), _ptr(bufs["vel"]), _ptr(bufs["force"]),
                                        _ptr(bufs["rho"]), C.addressof(step)), "mdpd_get_state")
        for k, v in bufs.items():
            if v is not None:
                res[k] = v
        res["step"] = int(step.value)
        return res

    def get_pairs(self, rcut):
        cnt = C.c_uint64()
        self._ck(self._L.mdpd_get_pairs(self._h, float(rcut), C.addressof(cnt), None, 0), "mdpd_get_pairs")
        m = int(cnt.value)
        pairs = np.empty((max(m, 1), 2), np.uint32)
        self._ck(self._L.mdpd_get_pairs(self._h, float(rcut), C.addressof(cnt), pairs.ctypes.data, m),
                 "mdpd_get_pairs")
        return pairs[:min(m, int(cnt.value))]

    def get_pairs_static(self, rcut, cap=None):
        """``mdpd_get_pairs_static``: the pairs of :meth:`get_pairs`, found without a single device allocation (the
        scratch is a fixed array inside the library; see include/mdpd.h for who needs that and for the sharing rules).
        cap = None counts first and then fetches exactly that many; more than MDPD_STATIC_PAIRS_MAX pairs raise
        MdpdError(MDPD_EINVAL).  Returns the sorted [m][2] uint32 tag pairs."""
        cnt = C.c_uint64()
        if cap is None:
            self._ck(self._L.mdpd_get_pairs_static(self._h, float(rcut), C.addressof(cnt), None, 0),
                     "mdpd_get_pairs_static")
            cap = int(cnt.value)
        cap = int(cap)
        pairs = np.empty((max(cap, 1), 2), np.uint32)
        self._ck(self._L.mdpd_get_pairs_static(self._h, float(rcut), C.addressof(cnt), pairs.ctypes.data, cap),
                 "mdpd_get_pairs_static")
        return pairs[:min(cap, int(cnt.value))]

    def rng_fill(self, pairs, step):
        pairs = np.ascontiguousarray(pairs, np.uint32).reshape(-1, 2)
        out = np.empty(pairs.shape[0], np.uint32)
        self._ck(self._L.mdpd_rng_fill(self._h, pairs.shape[0], pairs.ctypes.data, int(step) & 0xFFFFFFFF,
                                       out.ctypes.data), "mdpd_rng_fill")
        return out

    def counters(self):
        out = np.zeros(16, np.uint64)
        self._ck(self._L.mdpd_get_counters(self._h, out.ctypes.data), "mdpd_get_counters")
        return {k: int(v) for k, v in zip(COUNTER_NAMES, out)}

    def profile_begin(self):
        self._ck(self._L.mdpd_profile_begin(self._h), "mdpd_profile_begin")

    def profile_end(self):
        """{kernel name: (summed device ms, launches)} since profile_begin."""
        ms = np.zeros(MDPD_PROF_SLOTS, np.float64)
        cnt = np.zeros(MDPD_PROF_SLOTS, np.uint64)
        self._ck(self._L.mdpd_profile_end(self._h, ms.ctypes.data, cnt.ctypes.data), "mdpd_profile_end")
        out = {}
        for k in range(MDPD_PROF_SLOTS):
            nm = self._L.mdpd_profile_name(k).decode()
            if nm:
                out[nm] = (float(ms[k]), int(cnt[k]))
        return out

    def synchronize(self):
        self._stream.synchronize()
