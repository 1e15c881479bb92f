"""Pins of the CPU oracle (oracle/pimpc_oracle.c) against what the paper and the mathematics fix.

None of these tests re-types the oracle's formulas: they compare with dense KKT solves, a Riccati
recursion, brute-force active-set enumeration, closed forms, library inverses, invariants of the
ADMM iteration, and numbers produced by an independent implementation (tests/golden/p_tiny.txt).
Chosen so that a dropped term, wrong sign/index or transposed operand fails at least one of them:
  index of Abar/ebar in h_k (R2)           -> P-KKT on LTV with distinct e_k
  z-update form (R1), v-update, duals      -> P-KKT, P-BF, invariants
  Delta-u copy block (R12), Wdu (R13)      -> P-BF with active du bounds, P-KKT with Wdu
  terminal weight (R14), qbar, u_prev      -> P-KKT / Riccati
  residual c (R7)                          -> closed form c^1, golden c^1..c^10
  accept / restart / momentum (R5, R6)     -> golden decision bits + c sequence, Lemma-2 monotonicity
"""
import os

import numpy as np
import pytest

from paper_2601_14414_b200 import workloads as wl
from tests import qp_reference as ref

GOLD = os.path.join(os.path.dirname(__file__), "golden", "p_tiny.txt")


def _golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            out[k] = np.array([float(t) for t in v])
    return out


def _solve(oracle, prob, b=0, **kw):
    args = prob.instance(b)
    args.update(kw)
    return oracle.solve(**args)


# ----------------------------------------------------------------------------------------------
# cache against numpy.linalg.inv of the printed definition
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("has_du,wdu", [(False, False), (True, True)])
def test_cache_matches_library_inverse(oracle, has_du, wdu):
    p = wl.random_ltv(5, 3, 4, seed=11, full_cost=True, wdu=wdu)
    rho = 0.7
    M, H = oracle.cache(p.A[0], p.B[0], p.Q, p.R, P=p.P, Wdu=p.Wdu, has_du=has_du, rho=rho)
    nx, nu, nb = p.nx, p.nu, p.nb
    for k in range(p.N):
        Bb = np.vstack([p.B[0, k], np.eye(nu)])
        S = Bb.T @ Bb + (p.Wdu / rho if wdu else 0) + (np.eye(nu) if has_du else 0)
        np.testing.assert_allclose(M[k], np.linalg.inv(S), rtol=1e-12, atol=1e-14)
        Qb = np.zeros((nb, nb)); Qb[:nx, :nx] = p.P if k == p.N - 1 else p.Q; Qb[nx:, nx:] = p.R
        S = Qb + rho * np.eye(nb)
        if k < p.N - 1:
            Ab = np.block([[p.A[0, k + 1], p.B[0, k + 1]], [np.zeros((nu, nx)), np.eye(nu)]])
            S = S + rho * Ab.T @ Ab
        np.testing.assert_allclose(H[k], np.linalg.inv(S), rtol=1e-12, atol=1e-14)


# ----------------------------------------------------------------------------------------------
# P-KKT: unconstrained LTV problem == one dense KKT solve == Riccati recursion
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["plain", "wdu_qbar_fullcost"])
def test_unconstrained_matches_dense_kkt(oracle, variant):
    full = variant != "plain"
    p = wl.random_ltv(3, 2, 6, seed=3, affine=True, u_prev=True, full_cost=full, wdu=full, qbar=full)
    a = p.instance(0)
    U, X = ref.dense_kkt(a["A"], a["B"], a["Q"], a["R"], a["x0"], e=a["e"], P=a["P"], Wdu=a["Wdu"],
                         qbar=a["qbar"], u_prev=a["u_prev"])
    r = _solve(oracle, p, max_iters=20000, tol=1e-24)
    assert r.iters < 20000, "oracle did not converge"
    assert np.max(np.abs(r.u - U)) <= 1e-9 * max(1.0, np.max(np.abs(U)))
    assert np.max(np.abs(r.x - X)) <= 1e-9 * max(1.0, np.max(np.abs(X)))
    # X (the unprojected copy) agrees with Z at convergence; DU is the increment of u
    np.testing.assert_allclose(r.X, r.Z, atol=1e-9)
    uu = np.vstack([a["u_prev"], r.u])
    np.testing.assert_allclose(r.DU, np.diff(uu, axis=0), atol=1e-9)


def test_unconstrained_matches_riccati(oracle):
    p = wl.random_ltv(4, 2, 8, seed=5, affine=True, u_prev=False, full_cost=True)
    a = p.instance(0)
    U, X = ref.riccati_lqr(a["A"], a["B"], a["Q"], a["R"], a["x0"], e=a["e"], P=a["P"])
    Uk, Xk = ref.dense_kkt(a["A"], a["B"], a["Q"], a["R"], a["x0"], e=a["e"], P=a["P"])
    np.testing.assert_allclose(U, Uk, atol=1e-10)          # the two textbook routes agree
    r = _solve(oracle, p, max_iters=30000, tol=1e-24)
    assert r.iters < 30000
    np.testing.assert_allclose(r.u, U, atol=1e-9)
    np.testing.assert_allclose(r.x, X, atol=1e-9)


def test_lti_e0_would_hide_index_bug_but_ltv_does_not(oracle):
    """R2: with the index of Abar/ebar in h_k shifted the LTV iteration converges to a wrong point;
    the KKT pin above is on an LTV system with distinct e_k, so it sees it.  Here: the KKT residual of
    the converged oracle solution on a strongly time-varying system is ~0 (stationarity of QP (1))."""
    p = wl.random_ltv(3, 1, 7, seed=21, affine=True, scale=1.0)
    a = p.instance(0)
    U, X = ref.dense_kkt(a["A"], a["B"], a["Q"], a["R"], a["x0"], e=a["e"], u_prev=a["u_prev"])
    r = _solve(oracle, p, max_iters=50000, tol=1e-24)
    assert r.iters < 50000
    np.testing.assert_allclose(r.u, U, atol=1e-8)


# ----------------------------------------------------------------------------------------------
# P-BF: constrained problems == brute-force active-set enumeration
# ----------------------------------------------------------------------------------------------
def test_constrained_matches_bruteforce_all_bound_kinds(oracle):
    """u-, x- and du-bounds all active at the solution (asserted), incl. affine e_k and u_prev."""
    p = wl.random_ltv(2, 1, 4, seed=43, affine=True, u_prev=True, bounds=None, du_bound=0.4)
    p.lo = np.array([-0.9, -0.9, -0.6]); p.hi = np.array([0.9, 0.9, 0.6])
    a = p.instance(0)
    U, X, kinds = ref.active_set_bruteforce(a["A"], a["B"], a["Q"], a["R"], a["lo"], a["hi"], a["x0"], e=a["e"],
                                            u_prev=a["u_prev"], du_lo=a["du_lo"], du_hi=a["du_hi"])
    assert kinds == {"u", "x", "du"}, kinds
    r = _solve(oracle, p, max_iters=200000, tol=1e-22)
    assert r.iters < 200000
    np.testing.assert_allclose(r.u, U, atol=1e-8)
    np.testing.assert_allclose(r.x, X, atol=1e-8)


def test_constrained_two_inputs_bruteforce(oracle):
    p = wl.random_ltv(2, 2, 2, seed=8, affine=True, u_prev=True, bounds=0.4, du_bound=0.3, wdu=True, qbar=True)
    a = p.instance(0)
    U, X, kinds = ref.active_set_bruteforce(a["A"], a["B"], a["Q"], a["R"], a["lo"], a["hi"], a["x0"], e=a["e"],
                                            Wdu=a["Wdu"], qbar=a["qbar"], u_prev=a["u_prev"],
                                            du_lo=a["du_lo"], du_hi=a["du_hi"])
    assert len(kinds) >= 1
    r = _solve(oracle, p, max_iters=200000, tol=1e-22)
    assert r.iters < 200000
    np.testing.assert_allclose(r.u, U, atol=1e-8)
    np.testing.assert_allclose(r.x, X, atol=1e-8)


def test_p_tiny_converged_matches_bruteforce_and_golden(oracle):
    g = _golden()
    for with_du, key in ((False, "ustar_nodu"), (True, "ustar_du")):
        p = wl.p_tiny(with_du)
        a = p.instance(0)
        U, X, kinds = ref.active_set_bruteforce(a["A"], a["B"], a["Q"], a["R"], a["lo"], a["hi"], a["x0"],
                                                P=a["P"], du_lo=a["du_lo"], du_hi=a["du_hi"])
        np.testing.assert_allclose(U.ravel(), g[key], atol=2e-10)       # golden == brute force
        r = _solve(oracle, p, max_iters=20000, tol=1e-26)
        np.testing.assert_allclose(r.u.ravel(), g[key], atol=2e-10)     # oracle == golden
        if not with_du:
            np.testing.assert_allclose(r.x.ravel(), g["xstar_nodu"], atol=2e-10)


# ----------------------------------------------------------------------------------------------
# fixed-count numbers: c sequence, decision bits, iterates (independent implementation, SURVEY P-tiny)
# ----------------------------------------------------------------------------------------------
def test_p_tiny_fixed_count_numbers(oracle):
    g = _golden()
    r = _solve(oracle, wl.p_tiny(False), max_iters=10, tol=0.0)
    np.testing.assert_allclose(r.c_hist, g["c_nodu"], rtol=2e-12)
    assert list(r.acc_hist) == [int(v) for v in g["acc_nodu"]]
    np.testing.assert_allclose(r.DU.ravel(), g["du10_nodu"], atol=2e-12)
    np.testing.assert_allclose(r.Z[0], g["z0_10_nodu"], atol=2e-12)
    r = _solve(oracle, wl.p_tiny(True), max_iters=5, tol=0.0)
    np.testing.assert_allclose(r.c_hist, g["c_du"], rtol=2e-12)


def test_c1_closed_form(oracle):
    """P-c1: cold start, qbar=0, e=0, projection inactive at i=0 => only stage 0 moves and
    c^1 = rho ||A_0 x0 + B_0 u_prev||^2 + rho ||u_prev||^2   (derived from Alg. 1)."""
    p = wl.random_ltv(4, 2, 5, seed=2, affine=False, u_prev=True, bounds=None)
    for rho in (1.0, 2.5):
        a = p.instance(0); a["rho"] = rho
        r = oracle.solve(**a, max_iters=1)
        expect = rho * (np.sum((a["A"][0] @ a["x0"] + a["B"][0] @ a["u_prev"]) ** 2) + np.sum(a["u_prev"] ** 2))
        assert abs(r.c_hist[0] - expect) <= 1e-13 * expect
        b0 = np.concatenate([a["A"][0] @ a["x0"] + a["B"][0] @ a["u_prev"], a["u_prev"]])
        np.testing.assert_allclose(r.Z[0], b0 / 3, atol=1e-14)
        np.testing.assert_allclose(r.V[0], -b0 / 3, atol=1e-14)
        np.testing.assert_allclose(r.TH[0], -b0 / 3, atol=1e-14)
        assert np.all(r.Z[1:] == 0) and np.all(r.DU == 0)


# ----------------------------------------------------------------------------------------------
# invariants of the iteration (every iteration)
# ----------------------------------------------------------------------------------------------
def test_invariants_every_iteration(oracle):
    p = wl.quadrotor_ltv(12, 1, iters=60)
    a = p.instance(0)
    warm = None
    for it in range(60):
        # one iteration at a time would reset alpha; instead run 1..60 from cold and check the end state
        r = oracle.solve(**a, max_iters=it + 1)
        # (i) beta + lambda = 0 (optimality in the unconstrained v, Eq. 15b)
        assert np.max(np.abs(r.BE + r.LA)) <= 1e-12
        # (ii) normal-cone condition (14c): Z = clip(Z + t (TH - LA)) for any t > 0
        for t in (0.5, 3.0):
            np.testing.assert_allclose(r.Z, np.clip(r.Z + t * (r.TH - r.LA), a["lo"], a["hi"]), atol=1e-12)
        # (iii) feasibility of the projected copies
        assert np.all(r.Z >= a["lo"]) and np.all(r.Z <= a["hi"])
        assert np.all(r.D >= a["du_lo"]) and np.all(r.D <= a["du_hi"])


def test_lemma2_plain_admm_monotone_and_restart_rule(oracle):
    p = wl.quadrotor_ltv(10, 1, iters=400)
    a = p.instance(0)
    # eta = 0 => never accept => plain ADMM: c is non-increasing (Lemma 2)
    r = oracle.solve(**{**a, "eta": 0.0}, max_iters=400)
    assert r.restarts == 400
    assert np.all(r.c_hist[1:] <= r.c_hist[:-1] * (1 + 1e-12))
    # accelerated: accepted steps satisfy c^{i+1} <= eta c^i by construction; the step after a rejected
    # step is a plain ADMM step from a plain iterate, so c does not increase there.
    r = oracle.solve(**a, max_iters=400)
    c, acc = r.c_hist, r.acc_hist
    cprev = np.concatenate([[1.0], c[:-1]])
    assert np.all(c[acc == 1] <= 0.999 * cprev[acc == 1])
    rej = np.where(acc == 0)[0]
    rej = rej[rej + 1 < len(c)]
    assert np.all(c[rej + 1] <= c[rej] * (1 + 1e-12))
    assert 0 < r.restarts < 400


def test_forced_decisions_replay(oracle):
    """P-flip protocol: forcing the oracle's own decision sequence reproduces the run bit for bit;
    flipping one decision changes the trajectory."""
    p = wl.quadrotor_ltv(8, 1)
    a = p.instance(0)
    r0 = oracle.solve(**a, max_iters=120)
    r1 = oracle.solve(**a, max_iters=120, forced=r0.acc_hist)
    assert np.array_equal(r0.Z, r1.Z) and np.array_equal(r0.c_hist, r1.c_hist)
    f = r0.acc_hist.copy(); f[40] ^= 1
    r2 = oracle.solve(**a, max_iters=120, forced=f)
    assert np.array_equal(r0.c_hist[:41], r2.c_hist[:41]) and not np.array_equal(r0.Z, r2.Z)


def test_convergence_residuals_and_stationarity(oracle):
    """P-conv: consensus residuals, KKT stationarity (14b) and c all -> 0 (Lemma 3)."""
    p = wl.random_ltv(3, 2, 5, seed=17, affine=True, bounds=0.8, du_bound=0.5)
    a = p.instance(0)
    r = oracle.solve(**a, max_iters=200000, tol=1e-24)
    assert r.iters < 200000 and r.c_last < 1e-24
    nx, nu, N = p.nx, p.nu, p.N
    xb = np.concatenate([a["x0"], a["u_prev"]])
    rho = a["rho"]
    Qb = np.zeros((nx + nu, nx + nu)); Qb[:nx, :nx] = a["Q"]; Qb[nx:, nx:] = a["R"]
    for k in range(N):
        Ab = np.block([[a["A"][k], a["B"][k]], [np.zeros((nu, nx)), np.eye(nu)]])
        Bb = np.vstack([a["B"][k], np.eye(nu)])
        eb = np.concatenate([a["e"][k], np.zeros(nu)])
        assert np.max(np.abs(r.X[k] - Ab @ xb - Bb @ r.DU[k] - eb)) < 1e-9      # dynamics consensus
        assert np.max(np.abs(r.X[k] - r.Z[k])) < 1e-9
        assert np.max(np.abs(Bb @ r.DU[k] - r.V[k])) < 1e-9
        # stationarity in Delta u: Bbar' beta + delta = 0 ; in xbar: Qbar x + rho theta - rho Abar_{k+1}' lambda_{k+1} = 0
        assert np.max(np.abs(Bb.T @ r.BE[k] + r.DE[k])) < 1e-9
        g = Qb @ r.X[k] + rho * r.TH[k]
        if k < N - 1:
            Ab1 = np.block([[a["A"][k + 1], a["B"][k + 1]], [np.zeros((nu, nx)), np.eye(nu)]])
            g = g - rho * Ab1.T @ r.LA[k + 1]
        assert np.max(np.abs(g)) < 1e-8
        xb = r.X[k]


def test_residual_halves_match_the_definition_of_the_primal_residual(oracle):
    """PAPER.md:259-263, (14a), (15c): the primal half of c is rho ||F p + G q - h||^2.  The oracle forms it from the
    dual differences s^{i+1} - shat^i; here it is rebuilt from the DEFINITION of the consensus constraints of
    Problem (11) on the returned X, DU, Z, V[, D] with dense Abar, Bbar -- a different formula that
    agrees only if every dual update (step 3) is the running sum of its constraint residual."""
    for du_bound, iters in ((None, 37), (0.3, 52)):
        p = wl.random_ltv(3, 2, 6, 1, seed=21, affine=True, u_prev=True, qbar=True, bounds=0.7, du_bound=du_bound)
        r = _solve(oracle, p, max_iters=iters, tol=0.0)
        nx, nu, N = p.nx, p.nu, p.N
        tot = 0.0
        xk = np.concatenate([p.x0[0], p.u_prev[0]])
        for k in range(N):
            Ab = np.block([[p.A[0, k], p.B[0, k]], [np.zeros((nu, nx)), np.eye(nu)]])
            Bb = np.vstack([p.B[0, k], np.eye(nu)])
            eb = np.concatenate([p.e[0, k], np.zeros(nu)])
            tot += np.sum((r.X[k] - r.Z[k]) ** 2) + np.sum((Bb @ r.DU[k] - r.V[k]) ** 2)
            tot += np.sum((r.Z[k] - Ab @ xk - r.V[k] - eb) ** 2)
            if du_bound is not None:
                tot += np.sum((r.DU[k] - r.D[k]) ** 2)
            xk = r.X[k]
        assert abs(p.rho * tot - r.r_prim2) <= 1e-12 * max(1.0, r.r_prim2)
        assert abs(r.r_prim2 + r.r_dual2 - r.c_last) <= 1e-13 * max(1.0, r.c_last)
        assert r.r_prim2 > 0 and r.r_dual2 > 0


def test_warm_start_is_a_fresh_alg1_invocation(oracle):
    """the output iterates seed the next invocation with hats = iterates, alpha_0 = 1."""
    p = wl.quadrotor_ltv(6, 1)
    a = p.instance(0)
    r1 = oracle.solve(**a, max_iters=30)
    warm = dict(Z=r1.Z, V=r1.V, TH=r1.TH, BE=r1.BE, LA=r1.LA, D=r1.D, DE=r1.DE)
    r2 = oracle.solve(**a, max_iters=1, warm=warm)
    # first iteration of a warm invocation uses kappa = 0: identical to forcing a restart at iteration 30
    f = np.concatenate([r1.acc_hist[:29], [0]]).astype(np.uint8)
    r3 = oracle.solve(**a, max_iters=31, forced=f)
    np.testing.assert_allclose(r2.Z, r3.Z, rtol=0, atol=1e-15)


def test_generators_are_deterministic_and_shaped():
    p = wl.config1()
    assert p.A.shape == (1, 20, 4, 4) and p.B.shape == (1, 20, 4, 2) and p.du_lo is None
    q = wl.config4(batch=3)
    assert q.A.shape == (3, 50, 12, 12) and np.array_equal(q.A, wl.config4(batch=3).A)
    assert np.array_equal(wl.config4(batch=2, first_instance=1).A[0], q.A[1])
    c5 = wl.config5(N=7, batch=2)
    assert c5.A.shape == (2, 7, 48, 48) and c5.nu == 12
    # forward-Euler chain: spectral radius close to 1 (SURVEY.md section 8(d) C5 probe: ~1.005)
    assert 0.99 < np.max(np.abs(np.linalg.eigvals(c5.A[0, 0]))) < 1.02


def test_shift_warm_start_definition_and_benefit(oracle):
    """Reading R18 (receding-horizon warm start): shift_warm is the index map k -> min(k + steps, N-1); on an LTI
    problem re-solved one step later from the plant's next state, the shifted warm start begins with a far smaller
    residual than the cold start (why Alg. 1 takes its initial iterates from the previous MPC step)."""
    a = np.arange(12.0).reshape(6, 2)
    w = oracle.shift_warm({"Z": a, "D": None}, 2)
    assert w["D"] is None
    np.testing.assert_array_equal(w["Z"], a[[2, 3, 4, 5, 5, 5]])
    p = wl.config1()
    o = oracle.solve(**p.instance(0), max_iters=3000, tol=0.0)
    x1 = p.A[0, 0] @ p.x0[0] + p.B[0, 0] @ o.u[0]
    kw = dict(p.instance(0)); kw["x0"] = x1; kw["u_prev"] = o.u[0]
    warm = oracle.shift_warm(dict(Z=o.Z, V=o.V, TH=o.TH, BE=o.BE, LA=o.LA), 1)
    cold = oracle.solve(**kw, max_iters=2, tol=0.0)
    hot = oracle.solve(**kw, max_iters=2, tol=0.0, warm=warm)
    assert hot.c_hist[0] < 0.2 * cold.c_hist[0]           # 0.42 vs 4.1 on config 1 (short horizon: the tail is new)


# ----------------------------------------------------------------------------------------------
# the other projections of PAPER.md:166, per-stage data, the tracking cost (1a)
# ----------------------------------------------------------------------------------------------
def _feasible(kind, y, a, b, tol=0.0):
    if kind == "halfspace":
        return a @ y <= b + tol
    if kind == "hyperplane":
        return abs(a @ y - b) <= tol
    if kind == "soc":
        return np.linalg.norm(y[:-1]) <= y[-1] + tol
    return np.sum(np.abs(y)) <= b + tol


@pytest.mark.parametrize("kind,n", [("halfspace", 4), ("hyperplane", 3), ("soc", 4), ("l1ball", 5)])
def test_projections_are_nearest_points(oracle, kind, n):
    """Each projection against what DEFINES it (not its closed form): the result is feasible, a fixed point of the map,
    satisfies the variational inequality <t - P t, y - P t> <= 0 for every feasible y (the optimality condition of the
    nearest-point problem), and equals scipy's numerical minimiser of ||y - t||^2 over the set."""
    from scipy.optimize import minimize
    rng = np.random.default_rng([2601, 14414, 166, n])
    a = rng.normal(size=n) if kind in ("halfspace", "hyperplane") else None
    b = {"halfspace": 0.3, "hyperplane": -0.2, "soc": 0.0, "l1ball": 1.1}[kind]
    moved = 0
    for trial in range(30):
        t = rng.normal(size=n) * (2.0 if trial % 3 else 0.3)
        p = oracle.project(kind, t, a, b)
        assert _feasible(kind, p, a, b, 1e-12)
        np.testing.assert_allclose(oracle.project(kind, p, a, b), p, atol=1e-13)          # idempotent
        moved += int(np.linalg.norm(p - t) > 1e-9)
        ys = rng.normal(size=(400, n)) * 2.0                                              # feasible test points
        if kind == "hyperplane":
            ys = ys - np.outer((ys @ a - b) / (a @ a), a)
        elif kind == "halfspace":
            ys = ys - np.outer(np.maximum(ys @ a - b, 0.0) / (a @ a), a) - np.outer(rng.uniform(0, 1, 400), a)
        elif kind == "soc":
            ys[:, -1] = np.linalg.norm(ys[:, :-1], axis=1) + rng.uniform(0, 1, 400)
        else:
            ys = ys * (b * rng.uniform(0, 1, 400) / np.sum(np.abs(ys), axis=1))[:, None]
        assert all(_feasible(kind, y, a, b, 1e-9) for y in ys)
        assert np.max((ys - p) @ (t - p)) <= 1e-10
        ineq, eq = ref.set_constraints(kind, 0, a, b, n)
        cons = [{"type": "ineq", "fun": g} for g in ineq] + [{"type": "eq", "fun": g} for g in eq]
        start = np.concatenate([np.zeros(n - 1), [1.0]]) if kind == "soc" else np.zeros(n)
        r = minimize(lambda y: np.sum((y - t) ** 2), start, jac=lambda y: 2 * (y - t), constraints=cons,
                     method="SLSQP", options={"ftol": 1e-16, "maxiter": 500})
        np.testing.assert_allclose(p, r.x, atol=2e-6)
    assert moved >= 10                                        # the set was really active
    # hand-worked cases of [22, Ch. 6]
    np.testing.assert_allclose(oracle.project("l1ball", [3.0, -1.0, 0.5], b=2.0), [2.0, 0.0, 0.0], atol=1e-15)
    np.testing.assert_allclose(oracle.project("soc", [3.0, 4.0, 1.0]), [1.8, 2.4, 3.0], atol=1e-15)
    np.testing.assert_allclose(oracle.project("soc", [3.0, 4.0, -6.0]), [0.0, 0.0, 0.0], atol=0)      # polar cone
    np.testing.assert_allclose(oracle.project("soc", [3.0, 4.0, 6.0]), [3.0, 4.0, 6.0], atol=0)       # inside


@pytest.mark.parametrize("cset", [("halfspace", 0, [1.0, 0.6, -0.8], -0.3), ("hyperplane", 1, [1.0, 2.0], 0.1),
                                  ("soc", 2, 3, None), ("l1ball", 2, 3, 0.15), ("l1ball", 2, 2, 0.3)])
def test_converged_solution_with_general_sets_matches_slsqp(oracle, cset):
    """Theorem 1: the z-update is Proj of the same argument for ANY closed convex set.  The converged
    oracle must reach the minimiser of QP (1) with that set on (x_{k+1}; u_k) -- computed here by scipy's SLSQP from the
    set's defining inequalities, with the box still on the remaining components."""
    kind, i0, a, b = cset
    # the cone ||(u_1, u_2)||_2 <= u_3 and the l1 balls sit on the inputs, where they are always feasible
    nu = a if isinstance(a, int) else 1
    p = wl.random_ltv(2, nu, 4, 1, seed=166, affine=True, u_prev=True, bounds=None, du_bound=None, scale=0.2)
    lo = np.concatenate([[-0.6, -0.6], -0.5 * np.ones(nu)]); hi = -lo
    n = a if isinstance(a, int) else len(a)
    for i in range(i0, i0 + n):                           # the set replaces the box on its components
        lo[i], hi[i] = -np.inf, np.inf
    if kind == "hyperplane" or (kind == "l1ball" and n == 2):      # keep the problem feasible: no state box
        lo[:], hi[:] = -np.inf, np.inf
    args = p.instance(0); args.update(lo=lo, hi=hi)
    r = oracle.solve(**args, max_iters=60000, tol=1e-22, cset=cset)
    assert r.c_last < 1e-22
    xs, us = ref.slsqp_qp(p.A[0], p.B[0], p.Q, p.R, lo, hi, p.x0[0], e=p.e[0], u_prev=p.u_prev[0], cset=cset)
    zs = np.hstack([xs, us])
    ineq, eq = ref.set_constraints(kind, i0, None if isinstance(a, int) else np.asarray(a, float), b, n)
    active = sum(int(min(abs(g(z)) for g in ineq + eq) < 1e-6) for z in zs)
    assert active >= 1, "the test problem does not exercise the set"
    np.testing.assert_allclose(r.x, xs, atol=2e-6)
    np.testing.assert_allclose(r.u, us, atol=2e-6)
    z = np.hstack([r.x, r.u])
    assert all(g(zk) >= -1e-9 for zk in z for g in ineq) and all(abs(g(zk)) <= 1e-9 for zk in z for g in eq)


def test_per_stage_boxes_and_linear_terms_match_slsqp(oracle):
    """x_{k+1} in X_k, u_k in U_k and time-varying references (qbar_k): PAPER.md:37-47 with stage-dependent data."""
    p = wl.random_ltv(2, 2, 5, 1, seed=37, affine=True, u_prev=True, bounds=None, du_bound=None, scale=0.2)
    rng = np.random.default_rng([2601, 14414, 37])
    hi_k = rng.uniform(0.15, 0.6, size=(5, 4)); lo_k = -rng.uniform(0.15, 0.6, size=(5, 4))
    qbar_k = 0.5 * rng.normal(size=(5, 4))
    r = oracle.solve(**p.instance(0), max_iters=60000, tol=1e-22, lo_k=lo_k, hi_k=hi_k, qbar_k=qbar_k)
    assert r.c_last < 1e-22
    xs, us = ref.slsqp_qp(p.A[0], p.B[0], p.Q, p.R, p.lo, p.hi, p.x0[0], e=p.e[0], u_prev=p.u_prev[0],
                          lo_k=lo_k, hi_k=hi_k, qbar_k=qbar_k)
    z = np.hstack([r.x, r.u])
    assert np.sum(np.isclose(z, lo_k, atol=1e-9) | np.isclose(z, hi_k, atol=1e-9)) >= 3       # several stage bounds active
    np.testing.assert_allclose(r.x, xs, atol=2e-6)
    np.testing.assert_allclose(r.u, us, atol=2e-6)


def test_tracking_cost_matches_least_squares_and_afti16_output_box(oracle):
    """(1a) -> (Q, R, qbar) = (C'W_yC, W_u, col(C'W_y r_y, W_u r_u)): the converged unconstrained
    iteration equals the least-squares solution of the tracking problem written with C, W_y, r_y, r_u directly.  Then the
    AFTI-16 model as printed (forward Euler here, the paper uses a zero-order hold) with its output
    constraint -0.5 <= y_1 <= 0.5, which is a box on x_2 because C selects states."""
    rng = np.random.default_rng([2601, 14414, 197])
    p = wl.random_ltv(3, 2, 5, 1, seed=197, affine=True, u_prev=False, bounds=None, du_bound=None, scale=0.2)
    C = rng.normal(size=(2, 3)); Ly = rng.normal(size=(2, 2)); Wy = Ly @ Ly.T + 0.3 * np.eye(2)
    Lu = rng.normal(size=(2, 2)); Wu = Lu @ Lu.T + 0.2 * np.eye(2)
    ry = rng.normal(size=2); ru = 0.3 * rng.normal(size=2)
    Q, R, qbar = oracle.tracking(C, Wy, Wu, ry, ru)
    np.testing.assert_allclose(Q, Q.T, atol=1e-15)
    args = p.instance(0); args.update(Q=Q, R=R, qbar=qbar, P=None)
    r = oracle.solve(**args, max_iters=60000, tol=1e-24)
    xs, us = ref.tracking_least_squares(p.A[0], p.B[0], C, Wy, Wu, ry, ru, p.x0[0], e=p.e[0])
    np.testing.assert_allclose(r.x, xs, atol=1e-8)
    np.testing.assert_allclose(r.u, us, atol=1e-8)
    # AFTI-16
    Ac = np.array([[-0.0151, -60.5651, 0.0, -32.174], [-0.0001, -1.3411, 0.9929, 0.0], [0.00018, 43.2541, -0.86939, 0.0],
                   [0.0, 0.0, 1.0, 0.0]])
    Bc = np.array([[-2.516, -13.136], [-0.1689, -0.2514], [-17.251, -1.5766], [0.0, 0.0]])
    Cy = np.array([[0.0, 1.0, 0.0, 0.0], [0.0, 0.0, 0.0, 1.0]])
    N, Ts = 5, 0.05
    A = np.tile(np.eye(4) + Ts * Ac, (N, 1, 1)); B = np.tile(Ts * Bc, (N, 1, 1))
    Q, R, qbar = oracle.tracking(Cy, np.diag([100.0, 100.0]), np.zeros((2, 2)), [0.0, 10.0], None)
    lo = np.array([-np.inf, -0.5, -np.inf, -100.0, -25.0, -25.0]); hi = -lo
    Wdu = np.diag([0.1, 0.1])
    r = oracle.solve(A, B, Q, R, lo, hi, np.zeros(4), Wdu=Wdu, qbar=qbar, rho=10.0, max_iters=200000, tol=1e-20)
    assert r.c_last < 1e-20 and 1000 < r.iters                 # thousands of iterations, as PAPER.md:331 reports
    xs, us = ref.slsqp_qp(A, B, Q, R, lo, hi, np.zeros(4), Wdu=Wdu, qbar=qbar)
    assert np.min(np.abs(np.abs(r.x[:, 1]) - 0.5)) < 1e-7      # the output constraint on y_1 is active
    np.testing.assert_allclose(r.x, xs, atol=5e-5, rtol=1e-5)
    np.testing.assert_allclose(r.u, us, atol=5e-5, rtol=1e-5)


# ----------------------------------------------------------------------------------------------
# Riccati-ADMM as a second, independent oracle for converged solutions
# ----------------------------------------------------------------------------------------------
def test_riccati_admm_primal_step_is_the_lqr_minimiser():
    """Eq. (6a) by the backward Riccati recursion == one dense KKT solve of the same unconstrained problem."""
    from oracle import riccati_admm as ra
    p = wl.random_ltv(3, 2, 6, 1, seed=79, affine=True, u_prev=False, full_cost=True, qbar=True)
    a = p.instance(0)
    N, nx = p.N, p.nx
    Qs = np.stack([a["Q"]] * (N - 1) + [a["P"]])
    x, u = ra.lqr_step(a["A"], a["B"], a["e"], Qs, np.tile(a["qbar"][:nx], (N, 1)), a["R"], np.tile(a["qbar"][nx:], (N, 1)), a["x0"])
    U, X = ref.dense_kkt(a["A"], a["B"], a["Q"], a["R"], a["x0"], e=a["e"], P=a["P"], qbar=a["qbar"])
    np.testing.assert_allclose(u, U, atol=1e-10)
    np.testing.assert_allclose(x, X, atol=1e-10)


def test_two_independent_admm_oracles_agree_at_convergence(oracle):
    """piMPC (Alg. 1) and Riccati-ADMM (Eq. 5-6) are different splittings of the same QP (1): their converged (x, u)
    must coincide (and equal the brute-force active-set solution on the tiny case), with x- and u-bounds active."""
    from oracle import riccati_admm as ra
    cases = [wl.p_tiny(False), wl.config1(),
             wl.random_ltv(3, 2, 7, 1, seed=80, affine=True, u_prev=False, qbar=True, bounds=0.7, du_bound=None, scale=0.2)]
    for p in cases:
        a = p.instance(0)
        r = oracle.solve(**a, max_iters=400000, tol=1e-24)
        assert r.c_last < 1e-24, p.name
        s = ra.solve(a["A"], a["B"], a["Q"], a["R"], a["lo"], a["hi"], a["x0"], e=a["e"], P=a["P"], qbar=a["qbar"],
                     rho=1.0, tol=1e-11)
        assert s["r_prim"] < 1e-11 and s["r_dual"] < 1e-11, (p.name, s["iters"])
        z = np.hstack([r.x, r.u])
        assert np.sum(np.isclose(z, a["lo"], atol=1e-8) | np.isclose(z, a["hi"], atol=1e-8)) >= 1, p.name   # a bound is active
        np.testing.assert_allclose(r.u, s["u"], atol=5e-8, err_msg=p.name)
        np.testing.assert_allclose(r.x, s["x"], atol=5e-8, err_msg=p.name)
