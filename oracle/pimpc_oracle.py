"""ctypes wrapper of oracle/pimpc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It marshals arguments; all arithmetic of Algorithm 1
is in the C file.  It imports nothing from paper_2601_14414_b200/.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pimpc_oracle.c")
_LIB = os.path.join(_HERE, "libpimpc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        dp = ctypes.c_void_p
        _lib.pimpc_oracle_solve.restype = ctypes.c_int
        _lib.pimpc_oracle_solve.argtypes = (
            [ctypes.c_int] * 3 + [dp] * 14 + [ctypes.c_double] * 3 + [ctypes.c_int, ctypes.c_double]
            + [dp, ctypes.c_int] + [dp] * 9 + [dp, dp] + [dp, dp, dp] + [ctypes.POINTER(_Ext)])
        _lib.pimpc_oracle_project.restype = ctypes.c_int
        _lib.pimpc_oracle_project.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp, ctypes.c_double, dp]
        _lib.pimpc_oracle_tracking.restype = ctypes.c_int
        _lib.pimpc_oracle_tracking.argtypes = [ctypes.c_int] * 3 + [dp] * 8
        _lib.pimpc_oracle_cache.restype = ctypes.c_int
        _lib.pimpc_oracle_cache.argtypes = (
            [ctypes.c_int] * 3 + [dp] * 6 + [ctypes.c_int, ctypes.c_double] + [dp, dp])
    return _lib


SETS = {"none": 0, "halfspace": 1, "hyperplane": 2, "soc": 3, "l1ball": 4}


class _Ext(ctypes.Structure):
    """pimpc_oracle_ext of pimpc_oracle.c."""
    _fields_ = [("set_kind", ctypes.c_int), ("set_i0", ctypes.c_int), ("set_len", ctypes.c_int),
                ("set_a", ctypes.c_void_p), ("set_b", ctypes.c_double), ("lo_k", ctypes.c_void_p),
                ("hi_k", ctypes.c_void_p), ("qbar_k", ctypes.c_void_p)]


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f64(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


@dataclass
class OracleResult:
    X: np.ndarray
    DU: np.ndarray
    Z: np.ndarray
    V: np.ndarray
    TH: np.ndarray
    BE: np.ndarray
    LA: np.ndarray
    D: np.ndarray | None
    DE: np.ndarray | None
    c_hist: np.ndarray
    acc_hist: np.ndarray
    iters: int
    restarts: int
    c_last: float
    r_prim2: float = 0.0                  # rho ||F p + G q - h||^2 half of c_last
    r_dual2: float = 0.0                  # rho ||G (q - qhat)||^2 half of c_last
    x: np.ndarray = field(default=None)   # x_1..x_N  = Z[:, :nx]  (bound-feasible copy)
    u: np.ndarray = field(default=None)   # u_0..u_{N-1} = Z[:, nx:]


def solve(A, B, Q, R, lo, hi, x0, *, e=None, P=None, Wdu=None, qbar=None, du_lo=None, du_hi=None,
          u_prev=None, rho=1.0, eta=0.999, c0=1.0, max_iters=100, tol=0.0, forced=None,
          warm=None, cset=None, lo_k=None, hi_k=None, qbar_k=None) -> OracleResult:
    """One invocation of Algorithm 1 for one instance.  `warm` = dict of Z,V,TH,BE,LA[,D,DE].
    cset = (kind, i0, a or None, b): components [i0, i0 + len) of every z lie in a halfspace / hyperplane a^T z <= / = b,
    a second-order cone (len given by a tuple ("soc", i0, len, None)) or an l1 ball of radius b; lo_k, hi_k, qbar_k
    [N][nb]: per-stage boxes / linear terms."""
    lib = _load()
    A = _f64(A); B = _f64(B)
    N, nx, _ = A.shape
    nu = B.shape[2]
    nb = nx + nu
    e = _f64(e, (N, nx)); Q = _f64(Q, (nx, nx)); R = _f64(R, (nu, nu))
    P = _f64(P, (nx, nx)); Wdu = _f64(Wdu, (nu, nu)); qbar = _f64(qbar, (nb,))
    lo = _f64(lo, (nb,)); hi = _f64(hi, (nb,))
    du_lo = _f64(du_lo, (nu,)); du_hi = _f64(du_hi, (nu,))
    x0 = _f64(x0, (nx,)); u_prev = _f64(u_prev, (nu,))
    has_du = du_lo is not None
    st = {}
    for name, w in (("Z", nb), ("V", nb), ("TH", nb), ("BE", nb), ("LA", nb), ("D", nu), ("DE", nu)):
        if warm is not None and name in warm and warm[name] is not None:
            st[name] = np.array(warm[name], dtype=np.float64).reshape(N, w).copy()
        else:
            st[name] = np.zeros((N, w))
    X = np.zeros((N, nb)); DU = np.zeros((N, nu))
    c_hist = np.zeros(max(max_iters, 1)); acc_hist = np.zeros(max(max_iters, 1), dtype=np.uint8)
    info = np.zeros(2, dtype=np.int32); c_last = np.zeros(1); r_parts = np.zeros(2)
    if forced is not None:
        forced = np.ascontiguousarray(np.asarray(forced, dtype=np.uint8))
    ext, keep = None, []
    if cset is not None or lo_k is not None or hi_k is not None or qbar_k is not None:
        ext = _Ext()
        if cset is not None:
            kind, i0, a, b = cset
            ext.set_kind, ext.set_i0 = SETS[kind], int(i0)
            if isinstance(a, (int, np.integer)):
                ext.set_len, a = int(a), None
            else:
                a = _f64(a); keep.append(a)
                ext.set_len, ext.set_a = a.size, a.ctypes.data
            ext.set_b = 0.0 if b is None else float(b)
        for name, arr in (("lo_k", lo_k), ("hi_k", hi_k), ("qbar_k", qbar_k)):
            if arr is not None:
                arr = _f64(arr, (N, nb)); keep.append(arr)
                setattr(ext, name, arr.ctypes.data)
    rc = lib.pimpc_oracle_solve(
        nx, nu, N, _p(A), _p(B), _p(e), _p(Q), _p(R), _p(P), _p(Wdu), _p(qbar),
        _p(lo), _p(hi), _p(du_lo), _p(du_hi), _p(x0), _p(u_prev),
        float(rho), float(eta), float(c0), int(max_iters), float(tol),
        _p(forced), 0 if forced is None else int(forced.size),
        _p(st["Z"]), _p(st["V"]), _p(st["TH"]), _p(st["BE"]), _p(st["LA"]), _p(st["D"]), _p(st["DE"]),
        _p(X), _p(DU), _p(c_hist), _p(acc_hist), _p(info), _p(c_last), _p(r_parts),
        None if ext is None else ctypes.byref(ext))
    if rc != 0:
        raise RuntimeError(f"pimpc_oracle_solve failed: {rc}")
    it = int(info[0])
    return OracleResult(
        X=X, DU=DU, Z=st["Z"], V=st["V"], TH=st["TH"], BE=st["BE"], LA=st["LA"],
        D=st["D"] if has_du else None, DE=st["DE"] if has_du else None,
        c_hist=c_hist[:it].copy(), acc_hist=acc_hist[:it].copy(), iters=it, restarts=int(info[1]),
        c_last=float(c_last[0]), r_prim2=float(r_parts[0]), r_dual2=float(r_parts[1]), x=st["Z"][:, :nx].copy(), u=st["Z"][:, nx:].copy())


def project(kind, t, a=None, b=0.0):
    """Projection of t onto one of the sets of PAPER.md:166 ("halfspace", "hyperplane", "soc", "l1ball")."""
    lib = _load()
    t = _f64(t).ravel(); a = None if a is None else _f64(a).ravel()
    out = np.zeros_like(t)
    rc = lib.pimpc_oracle_project(SETS[kind], t.size, _p(t), _p(a), float(b), _p(out))
    if rc != 0:
        raise RuntimeError(f"pimpc_oracle_project failed: {rc}")
    return out


def tracking(C, Wy, Wu, ry=None, ru=None):
    """(Q, R, qbar) of the tracking cost (1a): Q = C'W_y C, R = W_u, qbar = (C'W_y r_y; W_u r_u)."""
    lib = _load()
    C = _f64(C); ny, nx = C.shape
    Wu = _f64(Wu); nu = Wu.shape[0]
    Wy = _f64(Wy, (ny, ny)); ry = _f64(ry, (ny,)); ru = _f64(ru, (nu,))
    Q = np.zeros((nx, nx)); R = np.zeros((nu, nu)); q = np.zeros(nx + nu)
    rc = lib.pimpc_oracle_tracking(nx, nu, ny, _p(C), _p(Wy), _p(Wu), _p(ry), _p(ru), _p(Q), _p(R), _p(q))
    if rc != 0:
        raise RuntimeError(f"pimpc_oracle_tracking failed: {rc}")
    return Q, R, q


def cache(A, B, Q, R, *, P=None, Wdu=None, has_du=False, rho=1.0):
    """The per-solve cache of Alg. 1: returns (M [N][nu][nu], H [N][nb][nb])."""
    lib = _load()
    A = _f64(A); B = _f64(B)
    N, nx, _ = A.shape
    nu = B.shape[2]
    nb = nx + nu
    Q = _f64(Q, (nx, nx)); R = _f64(R, (nu, nu)); P = _f64(P, (nx, nx)); Wdu = _f64(Wdu, (nu, nu))
    M = np.zeros((N, nu, nu)); H = np.zeros((N, nb, nb))
    rc = lib.pimpc_oracle_cache(nx, nu, N, _p(A), _p(B), _p(Q), _p(R), _p(P), _p(Wdu),
                                int(bool(has_du)), float(rho), _p(M), _p(H))
    if rc != 0:
        raise RuntimeError(f"pimpc_oracle_cache failed: {rc}")
    return M, H


def shift_warm(warm, steps=1):
    """Receding-horizon warm start (reading R18): stage k takes the iterate of stage
    k + steps, the last `steps` stages repeat the old last stage.  `warm` = dict of [N, w] arrays."""
    out = {}
    for name, a in warm.items():
        if a is None:
            out[name] = None
            continue
        a = np.asarray(a, dtype=np.float64)
        N = a.shape[0]
        idx = np.minimum(np.arange(N) + steps, N - 1)
        out[name] = a[idx].copy()
    return out
