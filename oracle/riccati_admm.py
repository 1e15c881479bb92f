"""Riccati-ADMM (Eq. (5)-(6)) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A SECOND, independent CPU oracle for CONVERGED solutions of problem (1): the structure-exploiting ADMM
the paper compares against.  It shares nothing with pimpc_oracle.c -- a different splitting (copies V of U and Z of X,
Eq. (5)), a different primal step (one affine finite-horizon LQR solved by the backward Riccati recursion, Eq. (6a),
instead of per-stage closed forms) -- so agreement of the two converged (x, u) cross-checks both.  Plain numpy, float64,
pure loops over the horizon.  Only tests/ may import it.

Problem (1) with box sets:  min sum_k 1/2 x_{k+1}' Q_{k+1} x_{k+1} - qx' x_{k+1} + 1/2 u_k' R u_k - qu' u_k
                            s.t. x_{k+1} = A_k x_k + B_k u_k + e_k,  x_lo <= x_{k+1} <= x_hi,  u_lo <= u_k <= u_hi,
with Q_j = Q (j < N), Q_N = P (terminal weight; P = Q if not given).  No Delta-u terms: the paper's Riccati-ADMM has none.
"""
from __future__ import annotations

import numpy as np


def lqr_step(A, B, e, Qs, qs, Rt, rs, x0):
    """Eq. (6a): min sum_k 1/2 x_{k+1}' Qs[k] x_{k+1} - qs[k]' x_{k+1} + 1/2 u_k' Rt u_k - rs[k]' u_k subject to the
    dynamics, by the backward Riccati recursion on the cost-to-go W_j(x) = 1/2 x' P_j x - p_j' x (W_N = 0) and a forward
    roll-out.  Qs [N][nx][nx], qs [N][nx] weigh x_1..x_N.  Returns (x [N][nx] = x_1..x_N, u [N][nu])."""
    N, nx, nu = A.shape[0], A.shape[1], B.shape[2]
    P = np.zeros((nx, nx)); p = np.zeros(nx)
    K = np.zeros((N, nu, nx)); d = np.zeros((N, nu))
    for k in range(N - 1, -1, -1):
        Pi = Qs[k] + P                       # Hessian / linear term of everything that depends on x_{k+1}
        pi = qs[k] + p
        S = Rt + B[k].T @ Pi @ B[k]
        K[k] = np.linalg.solve(S, B[k].T @ Pi @ A[k])
        d[k] = np.linalg.solve(S, rs[k] + B[k].T @ (pi - Pi @ e[k]))
        P = A[k].T @ Pi @ (A[k] - B[k] @ K[k])
        P = 0.5 * (P + P.T)
        p = A[k].T @ (pi - Pi @ (B[k] @ d[k] + e[k]))
    x = np.zeros((N, nx)); u = np.zeros((N, nu))
    xk = np.asarray(x0, float)
    for k in range(N):
        u[k] = -K[k] @ xk + d[k]
        xk = A[k] @ xk + B[k] @ u[k] + e[k]
        x[k] = xk
    return x, u


def solve(A, B, Q, R, lo, hi, x0, *, e=None, P=None, qbar=None, rho=1.0, max_iters=100000, tol=1e-12):
    """Riccati-ADMM, Eq. (6a)-(6c), scaled duals Phi (for U = V) and Psi (for X = Z).  Stops when the primal residual
    max(|U - V|, |X - Z|) and the dual residual rho max(|V - V_prev|, |Z - Z_prev|) are both below tol.
    Returns dict(x, u, iters, r_prim, r_dual) with (x, u) = the projected copies (Z, V)."""
    A = np.asarray(A, float); B = np.asarray(B, float)
    N, nx, nu = A.shape[0], A.shape[1], B.shape[2]
    e = np.zeros((N, nx)) if e is None else np.asarray(e, float)
    P = Q if P is None else P
    qbar = np.zeros(nx + nu) if qbar is None else np.asarray(qbar, float)
    lo = np.asarray(lo, float); hi = np.asarray(hi, float)
    Qs = np.stack([Q] * (N - 1) + [P]) + rho * np.eye(nx)          # x_1..x_N: Q + rho I, terminal P + rho I
    Rt = R + rho * np.eye(nu)
    V = np.zeros((N, nu)); Z = np.zeros((N, nx)); Phi = np.zeros((N, nu)); Psi = np.zeros((N, nx))
    it, r_prim, r_dual = 0, np.inf, np.inf
    for it in range(1, max_iters + 1):
        X, U = lqr_step(A, B, e, Qs, qbar[:nx] + rho * (Z - Psi), Rt, qbar[nx:] + rho * (V - Phi), x0)       # (6a)
        Vn = np.clip(U + Phi, lo[nx:], hi[nx:]); Zn = np.clip(X + Psi, lo[:nx], hi[:nx])                     # (6b)
        Phi = Phi + U - Vn; Psi = Psi + X - Zn                                                             # (6c)
        r_prim = max(np.max(np.abs(U - Vn)), np.max(np.abs(X - Zn)))
        r_dual = rho * max(np.max(np.abs(Vn - V)), np.max(np.abs(Zn - Z)))
        V, Z = Vn, Zn
        if r_prim < tol and r_dual < tol:
            break
    return dict(x=Z, u=V, iters=it, r_prim=r_prim, r_dual=r_dual)
