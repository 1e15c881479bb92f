"""Thin binding of libpimpc.so (include/pimpc.h): argument marshalling only.

Every step of Algorithm 1 runs in the CUDA kernels behind the C ABI; nothing in
this file computes.  Function names follow the C entry points.  Arrays may be numpy arrays (host)
or torch tensors (host or CUDA); they are passed as raw pointers.  There is no CPU fallback: if
libpimpc.so is missing or no CUDA device is present, this module raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

try:  # torch is optional plumbing (device memory, streams); the library itself does not need it
    import torch
except Exception:  # pragma: no cover
    torch = None

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("PIMPC_LIB") or os.path.join(_HERE, "libpimpc.so")   # PIMPC_LIB: another build of the same ABI

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENOTPD = 0, -1, -2, -3, -4, -5
F64, F32 = 0, 1
ENGINE_AUTO, ENGINE_STAGED, ENGINE_RESIDENT, ENGINE_STREAM, ENGINE_COOP = 0, 1, 2, 3, 4
ENGINES = {"auto": 0, "staged": 1, "resident": 2, "stream": 3, "coop": 4}
SETS = {"none": 0, "halfspace": 1, "hyperplane": 2, "soc": 3, "l1ball": 4}
X, Z, V, TH, BE, LA, D, DE, DU = range(9)
STATE = {"X": X, "Z": Z, "V": V, "TH": TH, "BE": BE, "LA": LA, "D": D, "DE": DE, "DU": DU}


class pimpc_tune(ctypes.Structure):
    _fields_ = [("grid", ctypes.c_int), ("ctas_per_sm", ctypes.c_int), ("ring_slots", ctypes.c_int),
                ("stages_per_group", ctypes.c_int), ("cluster", ctypes.c_int), ("rows_per_lane", ctypes.c_int),
                ("lookahead", ctypes.c_int), ("reserved_", ctypes.c_int)]


class pimpc_opts(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("engine", ctypes.c_int), ("rho", ctypes.c_double),
                ("eta", ctypes.c_double), ("c0", ctypes.c_double), ("history", ctypes.c_int),
                ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
                ("tune", pimpc_tune)]


class pimpc_result(ctypes.Structure):
    _fields_ = [("c", ctypes.c_double), ("alpha", ctypes.c_double), ("r_prim2", ctypes.c_double),
                ("r_dual2", ctypes.c_double), ("iters", ctypes.c_int), ("restarts", ctypes.c_int),
                ("converged", ctypes.c_int), ("pad_", ctypes.c_int)]


class pimpc_info(ctypes.Structure):
    _fields_ = [("engine", ctypes.c_int), ("launches", ctypes.c_int), ("total_launches", ctypes.c_longlong),
                ("device_bytes", ctypes.c_size_t), ("sm_count", ctypes.c_int), ("grid", ctypes.c_int),
                ("block", ctypes.c_int), ("smem_bytes", ctypes.c_size_t), ("setup_ms", ctypes.c_double),
                ("iter_ms", ctypes.c_double)]


class pimpc_peaks(ctypes.Structure):
    _fields_ = [("ffma_tflops", ctypes.c_double), ("ffma2_tflops", ctypes.c_double), ("dfma_tflops", ctypes.c_double),
                ("smem_gbs", ctypes.c_double), ("sm_count", ctypes.c_int), ("pad_", ctypes.c_int),
                ("lat_ffma2_cycles", ctypes.c_double), ("lat_dadd_cycles", ctypes.c_double), ("lat_shfl_cycles", ctypes.c_double),
                ("lat_lds_cycles", ctypes.c_double), ("lds128_bcast_cycles", ctypes.c_double)]


RESULT_DTYPE = np.dtype([("c", "f8"), ("alpha", "f8"), ("r_prim2", "f8"), ("r_dual2", "f8"), ("iters", "i4"),
                         ("restarts", "i4"), ("converged", "i4"), ("pad_", "i4")])

# name -> (restype, argtypes); every symbol include/pimpc.h declares
_vp, _i, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
SYMBOLS = {
    "pimpc_version": (ctypes.c_char_p, []),
    "pimpc_measure_peaks": (_i, [ctypes.POINTER(pimpc_peaks), _vp]),
    "pimpc_default_opts": (None, [ctypes.POINTER(pimpc_opts)]),
    "pimpc_workspace_bytes": (ctypes.c_size_t, [_i, _i, _i, _i, ctypes.POINTER(pimpc_opts)]),
    "pimpc_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, ctypes.POINTER(pimpc_opts)]),
    "pimpc_destroy": (_i, [_vp]),
    "pimpc_set_stage": (_i, [_vp, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "pimpc_set_stages": (_i, [_vp, _vp, _vp, _vp]),
    "pimpc_set_cost": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _i]),
    "pimpc_set_bounds": (_i, [_vp, _vp, _vp, _vp, _vp, _i]),
    "pimpc_set_tracking": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _vp, _i]),
    "pimpc_set_stage_terms": (_i, [_vp, _vp, _vp, _vp, _i]),
    "pimpc_set_constraint": (_i, [_vp, _i, _i, _i, _vp, _d]),
    "pimpc_set_x0": (_i, [_vp, _vp, _vp]),
    "pimpc_solve": (_i, [_vp, _i, _d]),
    "pimpc_get": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "pimpc_get_state": (_i, [_vp, _i, _vp]),
    "pimpc_set_state": (_i, [_vp, _i, _vp]),
    "pimpc_get_history": (_i, [_vp, _vp, _vp]),
    "pimpc_get_cache": (_i, [_vp, _vp, _vp]),
    "pimpc_reset": (_i, [_vp]),
    "pimpc_shift": (_i, [_vp, _i]),
    "pimpc_sync": (_i, [_vp]),
    "pimpc_get_info": (_i, [_vp, ctypes.POINTER(pimpc_info)]),
    "pimpc_last_error": (ctypes.c_char_p, [_vp]),
    "pimpc_rprim2_noalloc": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _d, _vp, _vp]),
    "pimpc_noalloc_last_error": (ctypes.c_char_p, []),
}

_lib = None


def load():
    """dlopen libpimpc.so and declare every entry point.  Raises if the library was not built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: run `python -m paper_2601_14414_b200.build` "
                               "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


class PimpcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pimpc error {code}: {msg}")
        self.code = code


def _ptr(a):
    """Raw pointer of a numpy array / torch tensor / None / int."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if torch is not None and isinstance(a, torch.Tensor):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    raise TypeError(type(a))


class Solver:
    """One libpimpc handle.  Methods mirror the C entry points (without the `pimpc_` prefix)."""

    def __init__(self, nx, nu, N, batch=1, *, dtype="f64", engine="auto", rho=1.0, eta=0.999, c0=1.0,
                 history=0, stream=None, workspace=None, tune=None):
        """workspace: a CUDA tensor (uint8 / any dtype) of at least workspace_bytes(...) bytes, kept alive by the
        Solver; tune: dict of pimpc_tune fields (launch-shape overrides, see include/pimpc.h)."""
        self.lib = load()
        self.nx, self.nu, self.N, self.batch, self.nb = nx, nu, N, batch, nx + nu
        self.dtype = dtype
        self.np_dtype = np.float64 if dtype == "f64" else np.float32
        self.history = history
        o = pimpc_opts()
        self.lib.pimpc_default_opts(ctypes.byref(o))
        o.dtype = F64 if dtype == "f64" else F32
        o.engine = ENGINES[engine] if isinstance(engine, str) else int(engine)
        o.rho, o.eta, o.c0, o.history = float(rho), float(eta), float(c0), int(history)
        if stream is None and torch is not None and torch.cuda.is_available():
            stream = torch.cuda.current_stream().cuda_stream
        o.stream = stream
        self._workspace = workspace              # keeps the caller's tensor alive as long as the handle
        if workspace is not None:
            o.workspace = workspace.data_ptr()
            o.workspace_bytes = workspace.numel() * workspace.element_size()
        for k, v in (tune or {}).items():
            if not hasattr(o.tune, k):
                raise KeyError(f"unknown pimpc_tune field {k!r}")
            setattr(o.tune, k, int(v))
        h = ctypes.c_void_p()
        rc = self.lib.pimpc_create(ctypes.byref(h), nx, nu, N, batch, ctypes.byref(o))
        if rc != OK:
            raise PimpcError(rc, self.lib.pimpc_last_error(None).decode())
        self.h = h

    # ---- helpers -------------------------------------------------------------------------
    def _ck(self, rc):
        if rc != OK:
            raise PimpcError(rc, self.lib.pimpc_last_error(self.h).decode())

    def _in(self, a, shape=None):
        """Host inputs are converted to the handle's dtype (marshalling); device tensors must match."""
        if a is None:
            return None
        if torch is not None and isinstance(a, torch.Tensor):
            want = torch.float64 if self.dtype == "f64" else torch.float32
            if a.dtype != want:
                raise TypeError(f"tensor dtype {a.dtype} does not match handle dtype {self.dtype}")
            return a
        a = np.ascontiguousarray(np.asarray(a), dtype=self.np_dtype)
        if shape is not None:
            a = a.reshape(shape)
        return a

    def close(self):
        if getattr(self, "h", None):
            self.lib.pimpc_destroy(self.h)
            self.h = None

    __del__ = close

    # ---- setters -------------------------------------------------------------------------
    def set_stage(self, b, k, A_k=None, B_k=None, e_k=None, Q=None, R=None, bounds=None, x0=None):
        args = [self._in(v) for v in (A_k, B_k, e_k, Q, R, bounds, x0)]
        self._ck(self.lib.pimpc_set_stage(self.h, b, k, *[_ptr(v) for v in args]))

    def set_stages(self, A, B, e=None):
        nst = (self.batch, self.N)
        A = self._in(A, (*nst, self.nx, self.nx)); B = self._in(B, (*nst, self.nx, self.nu))
        e = self._in(e, (*nst, self.nx))
        self._ck(self.lib.pimpc_set_stages(self.h, _ptr(A), _ptr(B), _ptr(e)))

    def set_cost(self, Q, R, P=None, Wdu=None, qbar=None, per_instance=False):
        a = [self._in(v) for v in (Q, R, P, Wdu, qbar)]
        self._ck(self.lib.pimpc_set_cost(self.h, *[_ptr(v) for v in a], int(per_instance)))

    def set_bounds(self, lo, hi, du_lo=None, du_hi=None, per_instance=False):
        a = [self._in(v) for v in (lo, hi, du_lo, du_hi)]
        self._ck(self.lib.pimpc_set_bounds(self.h, *[_ptr(v) for v in a], int(per_instance)))

    def set_tracking(self, C, Wy, Wu, ry=None, ru=None, per_stage=False):
        C = self._in(C); ny = C.shape[0]
        Wy = self._in(Wy, (ny, ny)); Wu = self._in(Wu, (self.nu, self.nu))
        ry = self._in(ry, (self.N, ny) if per_stage else (ny,)); ru = self._in(ru, (self.N, self.nu) if per_stage else (self.nu,))
        self._ck(self.lib.pimpc_set_tracking(self.h, int(ny), _ptr(C), _ptr(Wy), _ptr(Wu), _ptr(ry), _ptr(ru), int(per_stage)))

    def set_stage_terms(self, lo=None, hi=None, qbar=None, per_instance=False):
        a = [self._in(v) for v in (lo, hi, qbar)]
        self._ck(self.lib.pimpc_set_stage_terms(self.h, *[_ptr(v) for v in a], int(per_instance)))

    def set_constraint(self, kind, i0=0, length=0, a=None, b=0.0):
        a = self._in(a)
        if a is not None:
            length = int(np.asarray(a).size) if not (torch is not None and isinstance(a, torch.Tensor)) else a.numel()
        self._ck(self.lib.pimpc_set_constraint(self.h, SETS[kind] if isinstance(kind, str) else int(kind), int(i0), int(length),
                                               _ptr(a), float(b if b is not None else 0.0)))

    def set_x0(self, x0, u_prev=None):
        x0 = self._in(x0, (self.batch, self.nx)); u_prev = self._in(u_prev, (self.batch, self.nu))
        self._ck(self.lib.pimpc_set_x0(self.h, _ptr(x0), _ptr(u_prev)))

    def set_problem(self, p):
        """All setters for a workloads.Problem (marshalling convenience)."""
        self.set_stages(p.A, p.B, p.e)
        self.set_cost(p.Q, p.R, p.P, p.Wdu, p.qbar)
        self.set_bounds(p.lo, p.hi, p.du_lo, p.du_hi)
        self.set_x0(p.x0, p.u_prev)
        lo_k, hi_k, qbar_k, cset = (getattr(p, n, None) for n in ("lo_k", "hi_k", "qbar_k", "cset"))
        self.set_stage_terms(lo_k, hi_k, qbar_k)
        if cset is None:
            self.set_constraint("none")
        else:
            kind, i0, a, b = cset
            if isinstance(a, (int, np.integer)):
                self.set_constraint(kind, i0, int(a), None, b)
            else:
                self.set_constraint(kind, i0, 0, a, b)

    # ---- solve / results -------------------------------------------------------------------
    def solve(self, max_iters, tol=0.0):
        self._ck(self.lib.pimpc_solve(self.h, int(max_iters), float(tol)))

    def sync(self):
        self._ck(self.lib.pimpc_sync(self.h))

    def reset(self):
        self._ck(self.lib.pimpc_reset(self.h))

    def shift(self, steps=1):
        self._ck(self.lib.pimpc_shift(self.h, int(steps)))

    def get(self, x=None, u=None, du=None, res=None):
        """Fill caller-provided buffers (numpy or torch); returns (x, u, du, res) with numpy defaults."""
        nst = (self.batch, self.N)
        x = np.empty((*nst, self.nx), self.np_dtype) if x is None else x
        u = np.empty((*nst, self.nu), self.np_dtype) if u is None else u
        du = np.empty((*nst, self.nu), self.np_dtype) if du is None else du
        res = np.zeros(self.batch, RESULT_DTYPE) if res is None else res
        self._ck(self.lib.pimpc_get(self.h, _ptr(x), _ptr(u), _ptr(du), _ptr(res)))
        return x, u, du, res

    def get_state(self, which, out=None):
        w = STATE[which] if isinstance(which, str) else which
        width = self.nu if w in (D, DE, DU) else self.nb
        out = np.empty((self.batch, self.N, width), self.np_dtype) if out is None else out
        self._ck(self.lib.pimpc_get_state(self.h, w, _ptr(out)))
        return out

    def set_state(self, which, arr):
        w = STATE[which] if isinstance(which, str) else which
        arr = self._in(arr)
        self._ck(self.lib.pimpc_set_state(self.h, w, _ptr(arr)))

    def get_history(self):
        c = np.zeros((self.batch, self.history)); a = np.zeros((self.batch, self.history), np.uint8)
        self._ck(self.lib.pimpc_get_history(self.h, _ptr(c), _ptr(a)))
        return c, a

    def get_cache(self):
        M = np.empty((self.batch, self.N, self.nu, self.nu), self.np_dtype)
        H = np.empty((self.batch, self.N, self.nb, self.nb), self.np_dtype)
        self._ck(self.lib.pimpc_get_cache(self.h, _ptr(M), _ptr(H)))
        return M, H

    def get_info(self):
        info = pimpc_info()
        self._ck(self.lib.pimpc_get_info(self.h, ctypes.byref(info)))
        return {f: getattr(info, f) for f, _ in pimpc_info._fields_}


def workspace_bytes(nx, nu, N, batch=1, *, dtype="f64", history=0) -> int:
    o = pimpc_opts()
    load().pimpc_default_opts(ctypes.byref(o))
    o.dtype = F64 if dtype == "f64" else F32
    o.history = int(history)
    return int(load().pimpc_workspace_bytes(nx, nu, N, batch, ctypes.byref(o)))


def measure_peaks(stream=None) -> dict:
    """pimpc_measure_peaks on the current device: measured FP32 / FP64 FMA TFLOP/s and shared-memory GB/s."""
    pk = pimpc_peaks()
    rc = load().pimpc_measure_peaks(ctypes.byref(pk), stream)
    if rc != OK:
        raise PimpcError(rc, "pimpc_measure_peaks failed")
    return {f: getattr(pk, f) for f, _ in pimpc_peaks._fields_ if f != "pad_"}


NOALLOC_MAX_PARTS = 32768      # PIMPC_NOALLOC_MAX_PARTS of include/pimpc.h


def rprim2_noalloc(dtype, nx, nu, N, batch, A, B, e, x0, u_prev, X, DU, Z, V, D, rho, r_prim2, stream=None):
    """pimpc_rprim2_noalloc: r_prim2[b] of the iterate in the caller's DEVICE arrays (torch tensors or raw device pointers),
    into the caller's device double[batch]; no allocation, no synchronisation, asynchronous on `stream`.  Calls on one
    device share a static scratch array: do not let them overlap on the GPU."""
    rc = load().pimpc_rprim2_noalloc(F64 if dtype == "f64" else (F32 if dtype == "f32" else int(dtype)), nx, nu, N, batch,
                                     _ptr(A), _ptr(B), _ptr(e), _ptr(x0), _ptr(u_prev), _ptr(X), _ptr(DU), _ptr(Z), _ptr(V),
                                     _ptr(D), float(rho), _ptr(r_prim2), stream)
    if rc != OK:
        raise PimpcError(rc, load().pimpc_noalloc_last_error().decode())
    return r_prim2


def version() -> str:
    return load().pimpc_version().decode()
