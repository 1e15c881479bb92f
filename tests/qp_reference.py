"""Plain-definition solvers of QP (1) used ONLY to pin the oracle.

Nothing here implements ADMM; these are the textbook objects the converged iteration must reach:
  * dense_kkt        -- equality-constrained QP by one dense KKT solve (closed form),
  * riccati_lqr      -- finite-horizon affine LTV LQR by the backward Riccati recursion (textbook),
  * active_set_bruteforce -- condensed QP, enumeration of active sets, KKT sign checks.
The cost is  sum_k 1/2 x_{k+1}' Q_k x_{k+1} - qx' x_{k+1} + 1/2 u_k' R u_k - qu' u_k
             + 1/2 du_k' Wdu du_k,   Q_k = Q (k < N-1), Q_{N-1} = P,  du_k = u_k - u_{k-1}, u_{-1} = u_prev.
"""
from __future__ import annotations

import itertools

import numpy as np


def _defaults(A, B, e, P, Q, Wdu, qbar, u_prev):
    N, nx, _ = A.shape
    nu = B.shape[2]
    e = np.zeros((N, nx)) if e is None else e
    P = Q if P is None else P
    Wdu = np.zeros((nu, nu)) if Wdu is None else Wdu
    qbar = np.zeros(nx + nu) if qbar is None else qbar
    u_prev = np.zeros(nu) if u_prev is None else u_prev
    return N, nx, nu, e, P, Wdu, qbar, u_prev


def condensed(A, B, Q, R, x0, e=None, P=None, Wdu=None, qbar=None, u_prev=None):
    """Eliminate the states: x_{k+1} = Phi[k] U + phi[k].  Returns (Hc, fc, Phi, phi, Dm, d0) with
    cost 1/2 U'Hc U + fc'U + const and du = Dm U + d0."""
    N, nx, nu, e, P, Wdu, qbar, u_prev = _defaults(A, B, e, P, Q, Wdu, qbar, u_prev)
    Phi = np.zeros((N, nx, N * nu))
    phi = np.zeros((N, nx))
    xk_lin = np.zeros((nx, N * nu))
    xk_off = np.array(x0, float)
    for k in range(N):
        xk_lin = A[k] @ xk_lin
        xk_lin[:, k * nu:(k + 1) * nu] += B[k]
        xk_off = A[k] @ xk_off + e[k]
        Phi[k] = xk_lin
        phi[k] = xk_off
    Dm = np.eye(N * nu)
    for k in range(1, N):
        Dm[k * nu:(k + 1) * nu, (k - 1) * nu:k * nu] = -np.eye(nu)
    d0 = np.zeros(N * nu)
    d0[:nu] = -u_prev
    Hc = np.zeros((N * nu, N * nu))
    fc = np.zeros(N * nu)
    for k in range(N):
        Qk = P if k == N - 1 else Q
        Hc += Phi[k].T @ Qk @ Phi[k]
        fc += Phi[k].T @ (Qk @ phi[k] - qbar[:nx])
        sl = slice(k * nu, (k + 1) * nu)
        Hc[sl, sl] += R
        fc[sl] -= qbar[nx:]
    bigW = np.kron(np.eye(N), Wdu)
    Hc += Dm.T @ bigW @ Dm
    fc += Dm.T @ bigW @ d0
    return Hc, fc, Phi, phi, Dm, d0


def dense_kkt(A, B, Q, R, x0, e=None, P=None, Wdu=None, qbar=None, u_prev=None):
    """Unconstrained (bounds = +-inf) problem: one KKT solve over y = (u_0..u_{N-1}, x_1..x_N, nu)."""
    N, nx, nu, e, P, Wdu, qbar, u_prev = _defaults(A, B, e, P, Q, Wdu, qbar, u_prev)
    nU, nX = N * nu, N * nx
    Hy = np.zeros((nU + nX, nU + nX))
    fy = np.zeros(nU + nX)
    for k in range(N):
        su = slice(k * nu, (k + 1) * nu)
        sx = slice(nU + k * nx, nU + (k + 1) * nx)
        Hy[su, su] += R
        fy[su] -= qbar[nx:]
        Hy[sx, sx] += P if k == N - 1 else Q
        fy[sx] -= qbar[:nx]
        # 1/2 (u_k - u_{k-1})' W (u_k - u_{k-1})
        Hy[su, su] += Wdu
        if k == 0:
            fy[su] -= Wdu @ u_prev
        else:
            sp = slice((k - 1) * nu, k * nu)
            Hy[sp, sp] += Wdu
            Hy[su, sp] -= Wdu
            Hy[sp, su] -= Wdu
    E = np.zeros((nX, nU + nX))
    d = np.zeros(nX)
    for k in range(N):
        r = slice(k * nx, (k + 1) * nx)
        E[r, nU + k * nx:nU + (k + 1) * nx] = np.eye(nx)          # x_{k+1}
        E[r, k * nu:(k + 1) * nu] = -B[k]                          # - B_k u_k
        if k == 0:
            d[r] = A[0] @ x0 + e[0]
        else:
            E[r, nU + (k - 1) * nx:nU + k * nx] = -A[k]            # - A_k x_k
            d[r] = e[k]
    K = np.block([[Hy, E.T], [E, np.zeros((nX, nX))]])
    sol = np.linalg.solve(K, np.concatenate([-fy, d]))
    return sol[:nU].reshape(N, nu), sol[nU:nU + nX].reshape(N, nx)


def riccati_lqr(A, B, Q, R, x0, e=None, P=None):
    """Textbook backward Riccati recursion for  min sum 1/2 x_{k+1}'Q_k x_{k+1} + 1/2 u_k'R u_k,
    x_{k+1} = A_k x_k + B_k u_k + e_k  (affine value function 1/2 x'S x + s'x)."""
    N, nx, _ = A.shape
    nu = B.shape[2]
    e = np.zeros((N, nx)) if e is None else e
    P = Q if P is None else P
    S = np.zeros((N + 1, nx, nx))
    s = np.zeros((N + 1, nx))
    Kk = np.zeros((N, nu, nx))
    kk = np.zeros((N, nu))
    for k in range(N - 1, -1, -1):
        Qn = P if k == N - 1 else Q          # weight on x_{k+1}
        Sn = S[k + 1] + Qn
        G = R + B[k].T @ Sn @ B[k]
        Kk[k] = -np.linalg.solve(G, B[k].T @ Sn @ A[k])
        kk[k] = -np.linalg.solve(G, B[k].T @ (Sn @ e[k] + s[k + 1]))
        Acl = A[k] + B[k] @ Kk[k]
        ecl = B[k] @ kk[k] + e[k]
        S[k] = Acl.T @ Sn @ Acl + Kk[k].T @ R @ Kk[k]
        s[k] = Acl.T @ (Sn @ ecl + s[k + 1]) + Kk[k].T @ R @ kk[k]
    x = np.array(x0, float)
    U = np.zeros((N, nu))
    Xs = np.zeros((N, nx))
    for k in range(N):
        U[k] = Kk[k] @ x + kk[k]
        x = A[k] @ x + B[k] @ U[k] + e[k]
        Xs[k] = x
    return U, Xs


def active_set_bruteforce(A, B, Q, R, lo, hi, x0, e=None, P=None, Wdu=None, qbar=None, u_prev=None,
                          du_lo=None, du_hi=None, tol=1e-9):
    """Enumerate active sets of the condensed, strictly convex QP; accept the (unique) one whose
    equality-constrained solution is primal feasible with non-negative multipliers.
    Returns (U [N][nu], X [N][nx], active_kinds = set of {'u','x','du'})."""
    N, nx, nu, e_, P_, W_, qb_, up_ = _defaults(A, B, e, P, Q, Wdu, qbar, u_prev)
    Hc, fc, Phi, phi, Dm, d0 = condensed(A, B, Q, R, x0, e, P, Wdu, qbar, u_prev)
    nU = N * nu
    rows, rhs, kinds = [], [], []

    def add(row, ub, lb, kind):
        if np.isfinite(ub):
            rows.append(row); rhs.append(ub); kinds.append(kind)
        if np.isfinite(lb):
            rows.append(-row); rhs.append(-lb); kinds.append(kind)

    for k in range(N):
        for j in range(nu):
            r = np.zeros(nU); r[k * nu + j] = 1.0
            add(r, hi[nx + j], lo[nx + j], "u")
        for i in range(nx):
            add(Phi[k][i].copy(), hi[i] - phi[k][i], lo[i] - phi[k][i], "x")
        if du_lo is not None:
            for j in range(nu):
                r = Dm[k * nu + j].copy()
                add(r, du_hi[j] - d0[k * nu + j], du_lo[j] - d0[k * nu + j], "du")
    G = np.array(rows); g = np.array(rhs)
    nc = len(g)
    best = None
    for size in range(0, nU + 1):
        for act in itertools.combinations(range(nc), size):
            act = list(act)
            if size:
                Ga = G[act]
                K = np.block([[Hc, Ga.T], [Ga, np.zeros((size, size))]])
                try:
                    sol = np.linalg.solve(K, np.concatenate([-fc, g[act]]))
                except np.linalg.LinAlgError:
                    continue
                U, mu = sol[:nU], sol[nU:]
                if not np.all(np.isfinite(sol)) or np.linalg.cond(K) > 1e12:
                    continue
            else:
                U, mu = np.linalg.solve(Hc, -fc), np.zeros(0)
            if np.all(G @ U <= g + tol) and np.all(mu >= -tol):
                best = (U, {kinds[a] for a, m in zip(act, mu) if m > 1e-7})
                break
        if best is not None:
            break
    if best is None:
        raise RuntimeError("no KKT active set found (infeasible problem?)")
    U = best[0]
    X = np.stack([Phi[k] @ U + phi[k] for k in range(N)])
    return U.reshape(N, nu), X, best[1]


# ------------------------------------------------------------------------------------------------
# general convex sets and the tracking cost: plain definitions, solved by library routines
# ------------------------------------------------------------------------------------------------
def set_constraints(kind, i0, a, b, n):
    """Inequality functions g(zeta) >= 0 (and equalities h(zeta) = 0) that DEFINE the set of PAPER.md:166 on the
    components [i0, i0 + n) of a stage vector zeta = (x_{k+1}; u_k).  Returns (list of ineq, list of eq)."""
    sl = slice(i0, i0 + n)
    if kind == "halfspace":
        return [lambda z: b - a @ z[sl]], []
    if kind == "hyperplane":
        return [], [lambda z: a @ z[sl] - b]
    if kind == "soc":                                  # ||x||_2 <= r (its gradient exists everywhere but on the axis)
        return [lambda z: z[sl][-1] - np.sqrt(np.sum(z[sl][:-1] ** 2) + 1e-300)], []
    if kind == "l1ball":                               # ||x||_1 <= r: one halfspace per sign pattern
        signs = [np.array(s) for s in itertools.product((-1.0, 1.0), repeat=n)]
        return [(lambda z, s=s: b - s @ z[sl]) for s in signs], []
    raise ValueError(kind)


def slsqp_qp(A, B, Q, R, lo, hi, x0, *, e=None, P=None, Wdu=None, qbar=None, u_prev=None, cset=None,
             lo_k=None, hi_k=None, qbar_k=None):
    """QP (1) with boxes (shared or per stage), an optional general set on part of (x_{k+1}; u_k) at every stage and
    optional per-stage linear terms, solved by scipy's SLSQP on the condensed problem in U.  Returns (x [N][nx], u [N][nu])."""
    from scipy.optimize import minimize
    N, nx, nu, e, P, Wdu, qbar, u_prev = _defaults(A, B, e, P, Q, Wdu, qbar, u_prev)
    Hc, fc, Phi, phi, Dm, d0 = condensed(A, B, Q, R, x0, e, P, Wdu, np.zeros(nx + nu), u_prev)
    qk = np.tile(qbar, (N, 1)) if qbar_k is None else np.asarray(qbar_k, float)
    for k in range(N):                                 # linear terms: - qx_k' x_{k+1} - qu_k' u_k
        fc = fc - Phi[k].T @ qk[k, :nx]
        fc[k * nu:(k + 1) * nu] -= qk[k, nx:]
    lo_s = np.tile(lo, (N, 1)) if lo_k is None else np.asarray(lo_k, float)
    hi_s = np.tile(hi, (N, 1)) if hi_k is None else np.asarray(hi_k, float)

    def stage(U, k):
        return np.concatenate([Phi[k] @ U + phi[k], U[k * nu:(k + 1) * nu]])

    cons = []
    for k in range(N):
        for i in range(nx + nu):
            if np.isfinite(lo_s[k, i]):
                cons.append({"type": "ineq", "fun": (lambda U, k=k, i=i: stage(U, k)[i] - lo_s[k, i])})
            if np.isfinite(hi_s[k, i]):
                cons.append({"type": "ineq", "fun": (lambda U, k=k, i=i: hi_s[k, i] - stage(U, k)[i])})
        if cset is not None:
            kind, i0, a, b = cset
            n = a if isinstance(a, (int, np.integer)) else len(a)
            ineq, eq = set_constraints(kind, i0, None if isinstance(a, (int, np.integer)) else np.asarray(a, float), b, n)
            cons += [{"type": "ineq", "fun": (lambda U, k=k, g=g: g(stage(U, k)))} for g in ineq]
            cons += [{"type": "eq", "fun": (lambda U, k=k, g=g: g(stage(U, k)))} for g in eq]
    best = None
    for start in (np.zeros(N * nu), 0.05 * np.ones(N * nu)):
        r = minimize(lambda U: 0.5 * U @ Hc @ U + fc @ U, start, jac=lambda U: Hc @ U + fc, constraints=cons,
                     method="SLSQP", options={"ftol": 1e-15, "maxiter": 2000})
        if best is None or (r.success and r.fun < best.fun):
            best = r
    U = best.x
    return np.stack([Phi[k] @ U + phi[k] for k in range(N)]), U.reshape(N, nu)


def tracking_least_squares(A, B, C, Wy, Wu, ry, ru, x0, e=None):
    """Unconstrained problem (1a)-(1b),(1d) as ONE linear least-squares problem in U:
    min sum_k 1/2 ||L_y' (C x_{k+1} - r_y)||^2 + 1/2 ||L_u' (u_k - r_u)||^2,  W = L L'.  Never forms C'W_yC or qbar."""
    N, nx, _ = A.shape
    nu = B.shape[2]
    _, _, Phi, phi, _, _ = condensed(A, B, np.eye(nx), np.eye(nu), x0, e)
    Ly, Lu = np.linalg.cholesky(Wy), np.linalg.cholesky(Wu)
    rows, rhs = [], []
    for k in range(N):
        rows.append(Ly.T @ C @ Phi[k]); rhs.append(Ly.T @ (ry - C @ phi[k]))
        sel = np.zeros((nu, N * nu)); sel[:, k * nu:(k + 1) * nu] = np.eye(nu)
        rows.append(Lu.T @ sel); rhs.append(Lu.T @ ru)
    U = np.linalg.lstsq(np.vstack(rows), np.concatenate(rhs), rcond=None)[0]
    return np.stack([Phi[k] @ U + phi[k] for k in range(N)]), U.reshape(N, nu)
