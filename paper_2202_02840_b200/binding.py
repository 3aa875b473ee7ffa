"""ctypes binding of libcrk.so (include/crk.h).  Marshals torch CUDA tensors to device pointers; nothing else."""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("CRK_LIB") or os.path.join(_HERE, "libcrk.so")   # CRK_LIB: e.g. the range-checked build libcrk_checked.so

EXPORTED_SYMBOLS = (
    "crk_create", "crk_destroy", "crk_build_cells", "crk_volumes", "crk_rk_coefficients", "crk_hydro_derivs",
    "crk_step_derivs", "crk_step_derivs_host", "crk_hydro_derivs_active", "crk_compatible_energy", "crk_evolve_h", "crk_timestep", "crk_kdk_step", "crk_last_error", "crk_get_perm", "crk_get_gradv", "crk_get_leaf_segments", "crk_get_stats",
    "crk_reset_stats", "crk_set_timing", "crk_get_leaf_list", "crk_measure_fp32_peak", "crk_measure_fp32_peak_3reg",
    "crk_sfc_order_noalloc",
)
NOALLOC_MAX_N = 262144       # CRK_NOALLOC_MAX_N of include/crk.h

_ERR = {0: "CRK_OK", -1: "CRK_EINVAL", -2: "CRK_ERANGE", -3: "CRK_ENOMEM", -4: "CRK_ECUDA", -5: "CRK_ESTATE"}


class CrkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERR.get(code, code)}: {msg}")
        self.code = code


class _Params(C.Structure):
    _fields_ = [("box", C.c_float), ("gamma", C.c_float), ("n_h", C.c_float), ("C_l", C.c_float), ("C_q", C.c_float),
                ("eps", C.c_float), ("leaf_size", C.c_int), ("flags", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_leaves", C.c_int64), ("n_leaf_pairs", C.c_int64),
                ("n_leaf_pairs_gather", C.c_int64), ("launches", C.c_int64), ("scratch_bytes", C.c_int64), ("list_bytes", C.c_int64),
                ("ms_build", C.c_float), ("ms_volumes", C.c_float), ("ms_rk", C.c_float), ("ms_hydro", C.c_float),
                ("ms_sort", C.c_float), ("ms_tree", C.c_float), ("ms_gradv", C.c_float), ("ms_forces", C.c_float),
                ("ms_lists", C.c_float), ("timed_steps", C.c_int32), ("sort_passes", C.c_int32),
                ("n_active_leaves", C.c_int64), ("n_halo_leaves", C.c_int64), ("rebuilds", C.c_int32), ("n_fallback", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def library_path() -> str:
    return _LIB_PATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        # build in-tree with nvcc (cross-compiles without a GPU); no fallback of any kind if that fails
        from . import build as _build
        _build.build()
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2202_02840_b200.build`")
    L = C.CDLL(_LIB_PATH)
    vp, i64 = C.c_void_p, C.c_int64
    L.crk_create.argtypes = [C.POINTER(vp), C.POINTER(_Params), vp]
    L.crk_destroy.argtypes = [vp]
    L.crk_destroy.restype = None
    L.crk_build_cells.argtypes = [vp, i64, vp, vp, vp, vp]
    L.crk_volumes.argtypes = [vp, vp, vp, vp, vp]
    L.crk_rk_coefficients.argtypes = [vp, vp, vp, vp, vp]
    L.crk_hydro_derivs.argtypes = [vp] + [vp] * 9
    L.crk_step_derivs.argtypes = [vp, i64] + [vp] * 13
    L.crk_hydro_derivs_active.argtypes = [vp] + [vp] * 9
    L.crk_step_derivs_host.argtypes = [vp, i64] + [vp] * 13
    L.crk_last_error.argtypes = [vp]
    L.crk_last_error.restype = C.c_char_p
    L.crk_get_perm.argtypes = [vp, vp]
    L.crk_get_gradv.argtypes = [vp, vp]
    L.crk_compatible_energy.argtypes = [vp, C.c_float, vp]
    L.crk_evolve_h.argtypes = [vp, vp]
    L.crk_timestep.argtypes = [vp, C.c_float, vp]
    L.crk_kdk_step.argtypes = [vp, i64] + [vp] * 9 + [C.c_float]
    L.crk_get_leaf_segments.argtypes = [vp, vp]
    L.crk_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.crk_reset_stats.argtypes = [vp]
    L.crk_set_timing.argtypes = [vp, C.c_int]
    L.crk_get_leaf_list.argtypes = [vp, i64, vp, i64]
    L.crk_get_leaf_list.restype = i64
    L.crk_measure_fp32_peak.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    L.crk_measure_fp32_peak.restype = C.c_double
    L.crk_measure_fp32_peak_3reg.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    L.crk_measure_fp32_peak_3reg.restype = C.c_double
    L.crk_sfc_order_noalloc.argtypes = [vp, i64, vp, vp, vp, vp, C.c_float, vp, C.c_char_p, C.c_int]
    _lib = L
    return L


def _dev(t: torch.Tensor, dtype=torch.float32):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    return C.c_void_p(t.data_ptr())


def _opt(t, dtype=torch.float32):
    return None if t is None else _dev(t, dtype)


class Crk:
    """One library context (crk_ctx) bound to the current torch CUDA stream."""

    def __init__(self, box=1.0, gamma=5.0 / 3.0, n_h=2.4, C_l=2.0, C_q=1.0, eps=0.1, stream=None, timestep=False, kdk_reuse=False, kdk_compatible=False,
                 tree_per_leaf=False):
        L = _load()
        if not torch.cuda.is_available():
            raise RuntimeError("libcrk needs a CUDA device; there is no CPU fallback")
        self._L = L
        self._p = _Params(box, gamma, n_h, C_l, C_q, eps, 32, (1 if timestep else 0) | (2 if kdk_reuse else 0) | (4 if kdk_compatible else 0)
                          | (8 if tree_per_leaf else 0))   # CRK_FLAG_TIMESTEP | _KDK_REUSE | _KDK_COMPATIBLE | _TREE_PER_LEAF
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = C.c_void_p()
        rc = L.crk_create(C.byref(h), C.byref(self._p), C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise CrkError(rc, "crk_create failed")
        self._h = h
        self.n = 0
        self._dev = torch.device("cuda", torch.cuda.current_device())

    def close(self):
        if getattr(self, "_h", None):
            self._L.crk_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            raise CrkError(rc, self._L.crk_last_error(self._h).decode())

    # ---- the five entry points (same names as the C ABI, minus the prefix)
    def build_cells(self, x, y, z, h):
        self.n = int(x.numel())
        self._dev = x.device
        self._chk(self._L.crk_build_cells(self._h, self.n, *[self._len(t) for t in (x, y, z, h)]))

    def volumes(self, m, want_count=True):
        n, d = self.n, self._dev
        V = torch.empty(n, device=d)
        rho = torch.empty(n, device=d)
        cnt = torch.empty(n, device=d, dtype=torch.int32) if want_count else None
        self._chk(self._L.crk_volumes(self._h, self._len(m), _dev(V), _dev(rho), _opt(cnt, torch.int32)))
        return V, rho, cnt

    def rk_coefficients(self, want=True):
        n, d = self.n, self._dev
        if not want:
            self._chk(self._L.crk_rk_coefficients(self._h, None, None, None, None))
            return None
        A = torch.empty(n, device=d)
        B = torch.empty((3, n), device=d)
        gA = torch.empty((3, n), device=d)
        gB = torch.empty((9, n), device=d)
        self._chk(self._L.crk_rk_coefficients(self._h, _dev(A), _dev(B), _dev(gA), _dev(gB)))
        return A, B, gA, gB

    def hydro_derivs(self, vx, vy, vz, u, want_count=True):
        n, d = self.n, self._dev
        out = [torch.empty(n, device=d) for _ in range(4)]
        cnt = torch.empty(n, device=d, dtype=torch.int32) if want_count else None
        self._chk(self._L.crk_hydro_derivs(self._h, *[self._len(t) for t in (vx, vy, vz, u)], *[_dev(o) for o in out],
                                           _opt(cnt, torch.int32)))
        return out[0], out[1], out[2], out[3], cnt

    def hydro_derivs_active(self, active, vx, vy, vz, u, out=None):
        """Eqs. 17-18 for the particles with active[i] != 0 (uint8 tensor); other entries of `out` are left as
        they are (NaN in freshly made outputs)"""
        n, d = self.n, self._dev
        if out is None:
            out = [torch.full((n,), float("nan"), device=d) for _ in range(4)]
        self._chk(self._L.crk_hydro_derivs_active(self._h, self._len(active, torch.uint8), *[self._len(t) for t in (vx, vy, vz, u)],
                                                  *[self._len(o) for o in out]))
        return out

    def _len(self, t, dtype=torch.float32):
        """device pointer of a per-particle tensor; its length must be the particle count of the last build"""
        if self.n > 0 and int(t.numel()) != self.n:     # before any build the library itself reports CRK_ESTATE
            raise ValueError(f"per-particle tensor has {int(t.numel())} elements, the context holds {self.n} particles")
        return _dev(t, dtype)

    def step_derivs(self, x, y, z, h, vx, vy, vz, m, u, out=None):
        n = int(x.numel())
        self.n, self._dev = n, x.device
        if out is None:
            out = [torch.empty(n, device=x.device) for _ in range(4)]
        self._chk(self._L.crk_step_derivs(self._h, n, *[self._len(t) for t in (x, y, z, h, vx, vy, vz, m, u)],
                                          *[self._len(o) for o in out]))
        return out

    def step_derivs_host(self, x, y, z, h, vx, vy, vz, m, u, out):
        """All arguments are HOST float32 tensors (pinned recommended); `out` = [ax, ay, az, dudt] host tensors."""
        n = int(x.numel())
        self.n = n
        for t in (x, y, z, h, vx, vy, vz, m, u, *out):
            if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or int(t.numel()) != n:
                raise TypeError("expected contiguous host float32 tensors of one length")
        self._chk(self._L.crk_step_derivs_host(self._h, n, *[C.c_void_p(t.data_ptr()) for t in (x, y, z, h, vx, vy, vz, m, u)],
                                               *[C.c_void_p(t.data_ptr()) for t in out]))
        return out

    def kdk_step(self, x, y, z, h, vx, vy, vz, m, u, dt: float):
        """Eq. 43: one velocity-Verlet step, x, y, z, vx, vy, vz, u advanced in place"""
        n = int(x.numel())
        self.n = n
        self._chk(self._L.crk_kdk_step(self._h, n, *[self._len(t) for t in (x, y, z, h, vx, vy, vz, m, u)], C.c_float(dt)))

    def timestep(self, C_cfl: float = 0.25, out=None):
        """Eqs. 46-50 after hydro_derivs on a context created with timestep=True"""
        dt = out if out is not None else torch.empty(self.n, device=self._dev)
        self._chk(self._L.crk_timestep(self._h, C.c_float(C_cfl), _dev(dt)))
        return dt

    def evolve_h(self, out=None):
        """Eqs. 51-53 after volumes(): adjusted support radii, caller order"""
        h = out if out is not None else torch.empty(self.n, device=self._dev)
        self._chk(self._L.crk_evolve_h(self._h, _dev(h)))
        return h

    def compatible_energy(self, dt: float, out=None):
        """Eqs. 19-23 after hydro_derivs: Delta u over dt, caller order"""
        du = out if out is not None else torch.empty(self.n, device=self._dev)
        self._chk(self._L.crk_compatible_energy(self._h, C.c_float(dt), _dev(du)))
        return du

    # ---- diagnostics
    def perm(self):
        p = torch.empty(self.n, device=self._dev, dtype=torch.int32)
        self._chk(self._L.crk_get_perm(self._h, _dev(p, torch.int32)))
        return p

    def leaf_segments(self):
        """uint32 [n_leaves, 4]: {next, C | Kg << 16, K, arena unit} of every leaf's first neighbour-list segment"""
        nl = (self.n + 31) // 32
        t = torch.empty((nl, 4), device=self._dev, dtype=torch.int32)
        self._chk(self._L.crk_get_leaf_segments(self._h, _dev(t, torch.int32)))
        return t

    def gradv(self):
        g = torch.empty((9, self.n), device=self._dev)
        self._chk(self._L.crk_get_gradv(self._h, _dev(g)))
        return g

    def stats(self) -> dict:
        s = Stats()
        self._chk(self._L.crk_get_stats(self._h, C.byref(s)))
        return s.as_dict()

    def reset_stats(self):
        self._chk(self._L.crk_reset_stats(self._h))

    def set_timing(self, on: bool):
        self._chk(self._L.crk_set_timing(self._h, int(bool(on))))

    def leaf_list(self, leaf: int):
        import numpy as np
        cnt = self._L.crk_get_leaf_list(self._h, int(leaf), None, 0)
        if cnt < 0:
            self._chk(int(cnt))
        buf = np.empty(max(int(cnt), 1), dtype=np.uint32)
        self._L.crk_get_leaf_list(self._h, int(leaf), C.c_void_p(buf.ctypes.data), int(cnt))
        return buf[:cnt]


# module-level aliases with the C names
def crk_create(**kw):
    return Crk(**kw)


def crk_destroy(ctx: Crk):
    ctx.close()


def crk_build_cells(ctx: Crk, x, y, z, h):
    return ctx.build_cells(x, y, z, h)


def crk_volumes(ctx: Crk, m):
    return ctx.volumes(m)


def crk_rk_coefficients(ctx: Crk):
    return ctx.rk_coefficients()


def crk_hydro_derivs(ctx: Crk, vx, vy, vz, u):
    return ctx.hydro_derivs(vx, vy, vz, u)


def crk_step_derivs(ctx: Crk, x, y, z, h, vx, vy, vz, m, u):
    return ctx.step_derivs(x, y, z, h, vx, vy, vz, m, u)


def crk_step_derivs_host(ctx: Crk, x, y, z, h, vx, vy, vz, m, u, out):
    return ctx.step_derivs_host(x, y, z, h, vx, vy, vz, m, u, out)


def crk_sfc_order_noalloc(x, y, z, h, box: float, perm, stream=None):
    """Curve order of up to NOALLOC_MAX_N particles for callers that must not allocate device memory (a host code whose own
    arena already holds the whole GPU, or one that cannot take the device-wide stall of a cudaMalloc inside a time step):
    the library works in a fixed array that is part of its device image instead of cudaMalloc'ed buffers.  x, y, z, h:
    float32 CUDA tensors of one length n; perm: an int32 CUDA tensor of n elements that the CALLER provides (this wrapper
    makes no tensor either) and that receives what Crk.perm() gives after build_cells of the same input.  Calls share the
    array: do not let two of them overlap on the GPU.  The first call on a device looks the array up; make it outside any
    stream capture.  Raises CrkError with the library's message (n too large, input out of range, CUDA failure)."""
    L = _load()
    if not torch.cuda.is_available():
        raise RuntimeError("libcrk needs a CUDA device; there is no CPU fallback")
    n = int(x.numel())
    for t in (y, z, h, perm):
        if int(t.numel()) != n:
            raise ValueError("x, y, z, h and perm must have one length")
    st = stream if stream is not None else torch.cuda.current_stream()
    msg = C.create_string_buffer(256)
    if n == 0:
        args = [None] * 4 + [C.c_float(box), None]
    else:
        args = [_dev(t) for t in (x, y, z, h)] + [C.c_float(box), _dev(perm, torch.int32)]
    rc = L.crk_sfc_order_noalloc(C.c_void_p(st.cuda_stream), n, *args, msg, len(msg))
    if rc != 0:
        raise CrkError(rc, msg.value.decode())
    return perm


def crk_measure_fp32_peak(repeats=5, three_reg=False):
    """achieved FP32 rate (flop/s) of a register-resident FFMA loop; three_reg: a = b * c + a with three register operands"""
    L = _load()
    ms = C.c_float()
    fn = L.crk_measure_fp32_peak_3reg if three_reg else L.crk_measure_fp32_peak
    f = fn(C.c_void_p(torch.cuda.current_stream().cuda_stream), int(repeats), C.byref(ms))
    return float(f), float(ms.value)
