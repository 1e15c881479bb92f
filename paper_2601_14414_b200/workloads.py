"""Seeded synthetic MPC workloads (numpy only; none of the solver's arithmetic lives here).

These generators serve BOTH the CUDA path and the CPU oracle (tests and bench.py hand the same
arrays to each); neither solver imports the other.  They realise the five `configs` of
BASELINE.json as restated in SURVEY.md section 8(d), which stand in for the paper's own workloads
(random dense LTV systems with box constraints; long-horizon CSTR).
The recipe is restated in DESIGN.md "Input recipe".

All arrays are float64, row-major:  A [batch][N][nx][nx], B [batch][N][nx][nu], x0 [batch][nx].
Seeds: np.random.default_rng([2601, 14414, generator_id, instance]).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED = (2601, 14414)


@dataclass
class Problem:
    name: str
    nx: int
    nu: int
    N: int
    batch: int
    A: np.ndarray                 # [batch][N][nx][nx]
    B: np.ndarray                 # [batch][N][nx][nu]
    Q: np.ndarray                 # [nx][nx]
    R: np.ndarray                 # [nu][nu]
    lo: np.ndarray                # [nx+nu] = (x_lo; u_lo)
    hi: np.ndarray                # [nx+nu]
    x0: np.ndarray                # [batch][nx]
    e: np.ndarray | None = None   # [batch][N][nx]
    P: np.ndarray | None = None   # terminal weight (None = Q)
    Wdu: np.ndarray | None = None
    qbar: np.ndarray | None = None
    du_lo: np.ndarray | None = None
    du_hi: np.ndarray | None = None
    u_prev: np.ndarray | None = None   # [batch][nu]
    rho: float = 1.0
    iters: int = 100
    tol: float = 0.0
    dtypes: tuple = ("f64",)
    meta: dict = field(default_factory=dict)
    # SURVEY 8(f) row 2 (all shared by the instances): general set (kind, i0, a or length, b) on part of (x_{k+1}; u_k),
    # per-stage boxes [N][nb], per-stage linear terms [N][nb]
    cset: tuple | None = None
    lo_k: np.ndarray | None = None
    hi_k: np.ndarray | None = None
    qbar_k: np.ndarray | None = None

    @property
    def nb(self) -> int:
        return self.nx + self.nu

    def instance(self, b: int) -> dict:
        """Keyword arguments of one instance, in the naming both solvers' Python wrappers use."""
        kw = dict(A=self.A[b], B=self.B[b], Q=self.Q, R=self.R, lo=self.lo, hi=self.hi, x0=self.x0[b],
                  e=None if self.e is None else self.e[b], P=self.P, Wdu=self.Wdu, qbar=self.qbar,
                  du_lo=self.du_lo, du_hi=self.du_hi,
                  u_prev=None if self.u_prev is None else self.u_prev[b], rho=self.rho)
        for name in ("cset", "lo_k", "hi_k", "qbar_k"):
            if getattr(self, name) is not None:
                kw[name] = getattr(self, name)
        return kw

    def rounded(self, dtype: str) -> "Problem":
        """The same problem with every input rounded to `dtype` and promoted back to float64
        (what the oracle is fed for an fp32 GPU run, SURVEY.md section 8(c) parity metric)."""
        if dtype == "f64":
            return self
        r = lambda a: None if a is None else np.asarray(a, np.float32).astype(np.float64)
        cs = self.cset
        if cs is not None:
            cs = (cs[0], cs[1], cs[2] if isinstance(cs[2], (int, np.integer)) else r(cs[2]),
                  None if cs[3] is None else float(np.float32(cs[3])))
        return Problem(self.name, self.nx, self.nu, self.N, self.batch, r(self.A), r(self.B), r(self.Q),
                       r(self.R), r(self.lo), r(self.hi), r(self.x0), r(self.e), r(self.P), r(self.Wdu),
                       r(self.qbar), r(self.du_lo), r(self.du_hi), r(self.u_prev), self.rho, self.iters,
                       self.tol, self.dtypes, dict(self.meta), cs, r(self.lo_k), r(self.hi_k), r(self.qbar_k))


# --------------------------------------------------------------------------------------------
# mass-spring chains (configs 1 and 5)
# --------------------------------------------------------------------------------------------
def _chain_continuous(masses, springs, damping, input_masses):
    """wall - m_0 - m_1 - ... - m_{M-1} - wall with M+1 springs; state (p_0..p_{M-1}, v_0..v_{M-1}).
    springs may be [M+1] or [K][M+1] (K stage-wise stiffness sets). Returns A_c [K][2M][2M], B_c [2M][nu]."""
    masses = np.asarray(masses, float)
    springs = np.atleast_2d(np.asarray(springs, float))
    M = masses.size
    K = springs.shape[0]
    Ac = np.zeros((K, 2 * M, 2 * M))
    idx = np.arange(M)
    Ac[:, idx, M + idx] = 1.0                                            # p' = v
    Ac[:, M + idx, idx] = -(springs[:, :-1] + springs[:, 1:]) / masses   # own position
    Ac[:, M + idx[1:], idx[:-1]] = springs[:, 1:-1] / masses[1:]         # left neighbour
    Ac[:, M + idx[:-1], idx[1:]] = springs[:, 1:-1] / masses[:-1]        # right neighbour
    Ac[:, M + idx, M + idx] = -damping / masses                          # viscous damping
    Bc = np.zeros((2 * M, len(input_masses)))
    for j, mi in enumerate(input_masses):
        Bc[M + mi, j] = 1.0 / masses[mi]
    return Ac, Bc


def config1(seed_instance: int = 0) -> Problem:
    """C1: tiny LTI 2-mass chain, nx=4, nu=2, N=20, fp64, batch 1, 500 iterations, no du bounds."""
    nx, nu, N, dt = 4, 2, 20, 0.1
    Ac, Bc = _chain_continuous(np.ones(2), np.ones(3), 0.1, [0, 1])
    A1 = np.eye(nx) + dt * Ac[0]
    B1 = dt * Bc
    rng = np.random.default_rng([*SEED, 1, seed_instance])
    x0 = rng.uniform(-2.0, 2.0, size=(1, nx))
    A = np.broadcast_to(A1, (1, N, nx, nx)).copy()
    B = np.broadcast_to(B1, (1, N, nx, nu)).copy()
    lo = np.concatenate([-4.0 * np.ones(nx), -0.5 * np.ones(nu)])
    return Problem("C1", nx, nu, N, 1, A, B, np.eye(nx), 0.1 * np.eye(nu), lo, -lo, x0, P=np.eye(nx),
                   rho=1.0, iters=500, tol=0.0, dtypes=("f64",))


def config5(N: int = 2000, batch: int = 64, first_instance: int = 0) -> Problem:
    """C5: 24-mass chain, nx=48, nu=12, per-stage +-5 % stiffness, |du| <= 0.1, 500 iterations."""
    Mm, nu, dt = 24, 12, 0.05
    nx = 2 * Mm
    A = np.empty((batch, N, nx, nx))
    B = np.empty((batch, N, nx, nu))
    x0 = np.empty((batch, nx))
    for b in range(batch):
        rng = np.random.default_rng([*SEED, 5, first_instance + b])
        masses = rng.uniform(0.5, 2.0, size=Mm)
        springs = rng.uniform(0.5, 2.0, size=Mm + 1)
        pert = rng.uniform(-1.0, 1.0, size=(N, Mm + 1))
        x0[b] = rng.uniform(-1.0, 1.0, size=nx)
        Ac, Bc = _chain_continuous(masses, springs * (1.0 + 0.05 * pert), 0.1, list(range(0, Mm, 2)))
        A[b] = np.eye(nx) + dt * Ac
        B[b] = dt * Bc
    lo = np.concatenate([-3.0 * np.ones(nx), -1.0 * np.ones(nu)])
    return Problem("C5", nx, nu, N, batch, A, B, np.eye(nx), 0.1 * np.eye(nu), lo, -lo, x0,
                   du_lo=-0.1 * np.ones(nu), du_hi=0.1 * np.ones(nu), rho=1.0, iters=500, tol=0.0,
                   dtypes=("f64", "f32"))


# --------------------------------------------------------------------------------------------
# linearised quadrotor-like LTV system (configs 2, 3, 4)
# --------------------------------------------------------------------------------------------
def quadrotor_cost():
    """Shared diagonal Q ~ U[1,10]^12, R ~ U[0.01,0.1]^4 (cost rng)."""
    rng = np.random.default_rng([*SEED, 2, 10**6])
    return np.diag(rng.uniform(1.0, 10.0, size=12)), np.diag(rng.uniform(0.01, 0.1, size=4))


def quadrotor_ltv(N: int, batch: int = 1, first_instance: int = 0, *, iters: int = 2000, tol: float = 1e-4,
                  rho: float = 1.0, name: str = "C2", dtypes=("f64", "f32")) -> Problem:
    """State (p, phi/theta/psi, v, omega), inputs (thrust, tau_x, tau_y, tau_z);
    A_k = I + dt (J + dJ_k), B_k = dt (G + dG_k), dt = 0.02, dJ, dG ~ N(0, 0.05^2) per stage."""
    nx, nu, dt = 12, 4, 0.02
    J = np.zeros((nx, nx))
    J[0:3, 6:9] = np.eye(3)
    J[3:6, 9:12] = np.eye(3)
    J[6, 4] = 9.81
    J[7, 3] = -9.81
    G = np.zeros((nx, nu))
    G[8, 0] = 10.0
    G[9, 1] = 50.0
    G[10, 2] = 50.0
    G[11, 3] = 20.0
    Q, R = quadrotor_cost()
    A = np.empty((batch, N, nx, nx))
    B = np.empty((batch, N, nx, nu))
    x0 = np.empty((batch, nx))
    for b in range(batch):
        rng = np.random.default_rng([*SEED, 2, first_instance + b])
        dJ = rng.normal(0.0, 0.05, size=(N, nx, nx))
        dG = rng.normal(0.0, 0.05, size=(N, nx, nu))
        x0[b] = rng.uniform(-1.0, 1.0, size=nx)
        A[b] = np.eye(nx) + dt * (J + dJ)
        B[b] = dt * (G + dG)
    lo = np.concatenate([-5.0 * np.ones(nx), -1.0 * np.ones(nu)])
    return Problem(name, nx, nu, N, batch, A, B, Q, R, lo, -lo, x0, du_lo=-0.2 * np.ones(nu),
                   du_hi=0.2 * np.ones(nu), rho=rho, iters=iters, tol=tol, dtypes=tuple(dtypes))


def config2() -> Problem:
    return quadrotor_ltv(100, 1, iters=2000, tol=1e-4, name="C2")


def config3(N: int) -> Problem:
    return quadrotor_ltv(N, 1, iters=1000, tol=0.0, name=f"C3-N{N}", dtypes=("f32",))


C3_HORIZONS = (10, 100, 1000, 4000, 10000)


def config4(batch: int = 4096, first_instance: int = 0) -> Problem:
    return quadrotor_ltv(50, batch, first_instance, iters=200, tol=0.0, name="C4", dtypes=("f32",))


# --------------------------------------------------------------------------------------------
# small explicit / random systems used by the pins and the edge-case parity tests
# --------------------------------------------------------------------------------------------
def p_tiny(with_du_bounds: bool = False) -> Problem:
    """The explicit no-RNG problem of SURVEY.md section 8(c) 'P-tiny' (double integrator, N=4)."""
    nx, nu, N = 2, 1, 4
    A = np.broadcast_to(np.array([[1.0, 0.1], [0.0, 1.0]]), (1, N, nx, nx)).copy()
    B = np.broadcast_to(np.array([[0.005], [0.1]]), (1, N, nx, nu)).copy()
    lo = np.array([-4.0, -0.3, -0.5])
    hi = np.array([4.0, 0.3, 0.5])
    kw = dict(du_lo=np.array([-0.2]), du_hi=np.array([0.2])) if with_du_bounds else {}
    return Problem("P-tiny", nx, nu, N, 1, A, B, np.eye(2), np.array([[0.1]]), lo, hi,
                   np.array([[1.0, 0.0]]), P=np.eye(2), rho=1.0, iters=10, **kw)


def random_ltv(nx: int, nu: int, N: int, batch: int = 1, *, seed: int = 0, affine: bool = True,
               bounds: float | None = None, du_bound: float | None = None, u_prev: bool = True,
               full_cost: bool = False, wdu: bool = False, qbar: bool = False, scale: float = 0.3) -> Problem:
    """Small dense random LTV systems with distinct A_k, B_k, e_k per stage (pins P-KKT / P-BF and
    odd-shaped parity cases).  A_k = I + scale*N(0,1)/sqrt(nx), B_k = N(0,1), e_k = 0.1 N(0,1)."""
    rng = np.random.default_rng([*SEED, 99, seed])
    nb = nx + nu
    A = np.eye(nx) + scale * rng.normal(size=(batch, N, nx, nx)) / np.sqrt(nx)
    B = rng.normal(size=(batch, N, nx, nu))
    e = 0.1 * rng.normal(size=(batch, N, nx)) if affine else None
    x0 = rng.uniform(-1.0, 1.0, size=(batch, nx))
    up = 0.3 * rng.uniform(-1.0, 1.0, size=(batch, nu)) if u_prev else None
    if full_cost:
        Lq = rng.normal(size=(nx, nx)); Lr = rng.normal(size=(nu, nu))
        Q = Lq @ Lq.T / nx + 0.5 * np.eye(nx)
        R = Lr @ Lr.T / nu + 0.1 * np.eye(nu)
        P = 2.0 * Q
    else:
        Q = np.diag(rng.uniform(0.5, 2.0, size=nx)); R = np.diag(rng.uniform(0.05, 0.5, size=nu)); P = None
    W = np.diag(rng.uniform(0.05, 0.3, size=nu)) if wdu else None
    qb = 0.2 * rng.normal(size=nb) if qbar else None
    if bounds is None:
        lo = -np.inf * np.ones(nb); hi = np.inf * np.ones(nb)
    else:
        lo = -bounds * np.ones(nb); hi = bounds * np.ones(nb)
    kw = {}
    if du_bound is not None:
        kw = dict(du_lo=-du_bound * np.ones(nu), du_hi=du_bound * np.ones(nu))
    return Problem(f"rand-{nx}-{nu}-{N}", nx, nu, N, batch, A, B, Q, R, lo, hi, x0, e=e, P=P, Wdu=W, qbar=qb,
                   u_prev=up, rho=1.0, iters=200, **kw)


# --------------------------------------------------------------------------------------------
# CSTR with online linearisation: closed-loop / RTI stepping workload
# --------------------------------------------------------------------------------------------
CSTR = dict(CAi=10.0, k0=34930800.0, EaR=5963.6, Ts=0.5, x_init=(8.57, 311.27), u_init=300.0, ref=2.0,
            lo=(0.0, 250.0, 250.0), hi=(12.0, 450.0, 350.0), Wy=1.0, Wu=0.0, Wdu=0.1)


def cstr_f(x, u, t):
    """dC_A/dt, dT/dt of the CSTR as printed at PAPER.md:399; inlet disturbance T_i = 298.15 + 5 sin(0.05 t)."""
    ca, T = float(x[0]), float(x[1])
    r = CSTR["k0"] * np.exp(-CSTR["EaR"] / T) * ca
    Ti = 298.15 + 5.0 * np.sin(0.05 * t)
    return np.array([CSTR["CAi"] - ca - r, Ti + 0.3 * float(u[0]) - 1.3 * T + 11.92 * r])


def cstr_plant_step(x, u, t):
    """The plant, advanced by one sampling period with the paper's forward-Euler discretisation (T_s = 0.5 min)."""
    return np.asarray(x, np.float64) + CSTR["Ts"] * cstr_f(x, u, t)


def cstr_problem(x, u_prev, t0, N, *, rho=1.0, iters=1000, ref=None) -> Problem:
    """One MPC step: the model linearised around the current state and the previous input,
    x_{k+1} = A x_k + B u_k + e_k with the disturbance sampled along the horizon in e_k; output y = C_A tracked
    to `ref` (W_y = 1, W_u = 0, W_du = 0.1).  The reference value and the boxes are this build's choice (the paper
    shows them only in a figure); DESIGN.md "Input recipe"."""
    Ts, k0, EaR = CSTR["Ts"], CSTR["k0"], CSTR["EaR"]
    x = np.asarray(x, np.float64); u = np.asarray(u_prev, np.float64).reshape(1)
    ca, T = x
    kk = k0 * np.exp(-EaR / T)
    dk = kk * EaR / (T * T)                                  # d/dT of k0 exp(-EaR/T)
    J = np.array([[-1.0 - kk, -dk * ca], [11.92 * kk, -1.3 + 11.92 * dk * ca]])
    A = np.eye(2) + Ts * J
    B = np.array([[0.0], [Ts * 0.3]])
    e0 = x + Ts * cstr_f(x, u, t0) - A @ x - B @ u            # affine term of the linearisation at (x, u, t0)
    tk = t0 + Ts * np.arange(N)                               # the disturbance T_i(t) enters dT/dt additively
    e = np.tile(e0, (N, 1))
    e[:, 1] += Ts * 5.0 * (np.sin(0.05 * tk) - np.sin(0.05 * t0))
    r = CSTR["ref"] if ref is None else ref
    Q = np.diag([CSTR["Wy"], 0.0]); R = np.array([[CSTR["Wu"]]])
    qbar = np.array([CSTR["Wy"] * r, 0.0, 0.0])
    return Problem("CSTR", 2, 1, N, 1, np.tile(A, (1, N, 1, 1)), np.tile(B, (1, N, 1, 1)), Q, R,
                   np.array(CSTR["lo"]), np.array(CSTR["hi"]), x[None, :].copy(), e=e[None], Wdu=np.array([[CSTR["Wdu"]]]),
                   qbar=qbar, u_prev=u[None, :].copy(), rho=rho, iters=iters, tol=0.0, dtypes=("f64", "f32"),
                   meta=dict(t0=t0))


# --------------------------------------------------------------------------------------------
# AFTI-16: the printed model, output matrix, constraints and weights
# --------------------------------------------------------------------------------------------
AFTI16 = dict(
    Ac=((-0.0151, -60.5651, 0.0, -32.174), (-0.0001, -1.3411, 0.9929, 0.0), (0.00018, 43.2541, -0.86939, 0.0), (0.0, 0.0, 1.0, 0.0)),
    Bc=((-2.516, -13.136), (-0.1689, -0.2514), (-17.251, -1.5766), (0.0, 0.0)),
    C=((0.0, 1.0, 0.0, 0.0), (0.0, 0.0, 0.0, 1.0)), Ts=0.05, u_max=25.0, y_max=(0.5, 100.0), Wy=(100.0, 100.0), Wdu=(0.1, 0.1))


def afti16(N: int = 5, batch: int = 1, *, ref: float = 10.0, rho: float = 10.0, iters: int = 300, seed: int = 0):
    """The AFTI-16 tracking problem of PAPER.md:319-329 with the matrices as printed: y = C x, |u_i| <= 25, -0.5 <= y_1 <=
    0.5, -100 <= y_2 <= 100, W_y = diag(100, 100), W_u = 0, W_du = diag(0.1, 0.1), N = 5.  The paper discretises with a
    zero-order hold and does not print the reference signal or rho: forward Euler (T_s = 0.05 s) and a constant pitch
    reference `ref` stand in.  Because C selects states, the output constraints are a box on x_2 and x_4.  Returns
    (Problem, tracking) where tracking = dict(C, Wy, Wu, ry, ru) is what pimpc_set_tracking takes.  The Problem's Q, R are
    zero placeholders: forming (Q, R, qbar) from the tracking data is the solvers' arithmetic, not the generator's."""
    a = AFTI16
    A1 = np.eye(4) + a["Ts"] * np.array(a["Ac"]); B1 = a["Ts"] * np.array(a["Bc"])
    rng = np.random.default_rng([*SEED, 16, seed])
    x0 = 0.05 * rng.uniform(-1.0, 1.0, size=(batch, 4))
    C = np.array(a["C"]); Wy = np.diag(a["Wy"]); Wu = np.zeros((2, 2)); ry = np.array([0.0, ref])
    lo = np.array([-np.inf, -a["y_max"][0], -np.inf, -a["y_max"][1], -a["u_max"], -a["u_max"]])
    p = Problem("AFTI16", 4, 2, N, batch, np.tile(A1, (batch, N, 1, 1)), np.tile(B1, (batch, N, 1, 1)), np.zeros((4, 4)), Wu,
                lo, -lo, x0, Wdu=np.diag(a["Wdu"]), rho=rho, iters=iters, tol=0.0, dtypes=("f64", "f32"))
    return p, dict(C=C, Wy=Wy, Wu=Wu, ry=ry, ru=np.zeros(2))


def pad_problem(p: Problem, nx2: int, nu2: int) -> Problem:
    """Embed p in a larger shape by adding decoupled zero states / inputs (A, B blocks 0, unit weights, boxes
    [-1, 1], zero initial state): the added components stay exactly 0 in every iterate and add exactly 0 to the
    residual, so the original components are unchanged.  Lets a shape without a fused-engine instantiation
    (the CSTR's nx = 2, nu = 1) run on one that has (4, 2).  Pure data marshalling."""
    nx, nu, N, b = p.nx, p.nu, p.N, p.batch
    assert nx2 >= nx and nu2 >= nu
    A = np.zeros((b, N, nx2, nx2)); A[:, :, :nx, :nx] = p.A
    B = np.zeros((b, N, nx2, nu2)); B[:, :, :nx, :nu] = p.B

    def blk(M, n, n2, fill):
        if M is None:
            return None
        out = np.eye(n2) * fill
        out[:n, :n] = M
        return out

    def vec(xpart, upart, fx, fu):
        return np.concatenate([xpart, np.full(nx2 - nx, fx), upart, np.full(nu2 - nu, fu)])

    e = None
    if p.e is not None:
        e = np.zeros((b, N, nx2)); e[:, :, :nx] = p.e
    x0 = np.zeros((b, nx2)); x0[:, :nx] = p.x0
    up = None
    if p.u_prev is not None:
        up = np.zeros((b, nu2)); up[:, :nu] = p.u_prev
    qbar = None if p.qbar is None else vec(p.qbar[:nx], p.qbar[nx:], 0.0, 0.0)
    pad_u = lambda v, f: None if v is None else np.concatenate([v, np.full(nu2 - nu, f)])
    return Problem(p.name + "-pad", nx2, nu2, N, b, A, B, blk(p.Q, nx, nx2, 1.0), blk(p.R, nu, nu2, 1.0),
                   vec(p.lo[:nx], p.lo[nx:], -1.0, -1.0), vec(p.hi[:nx], p.hi[nx:], 1.0, 1.0), x0, e=e,
                   P=blk(p.P, nx, nx2, 1.0), Wdu=blk(p.Wdu, nu, nu2, 0.0), qbar=qbar,
                   du_lo=pad_u(p.du_lo, -1.0), du_hi=pad_u(p.du_hi, 1.0), u_prev=up, rho=p.rho, iters=p.iters,
                   tol=p.tol, dtypes=p.dtypes, meta=dict(p.meta, pad_of=(nx, nu)))


# --------------------------------------------------------------------------------------------
# the paper's scalability workload: random dense systems of Table I
# --------------------------------------------------------------------------------------------
TABLE1_SHAPES = ((10, 3), (20, 6), (30, 10), (50, 15))
TABLE1_HORIZONS = (20, 50, 100, 200, 500)


def paper_random(nx: int, nu: int, N: int, *, seed: int = 0, iters: int = 200) -> Problem:
    """A, B ~ N(0, 1) with A scaled to unit spectral radius, additive disturbance e_k ~ U[-0.3, 0.3], boxes
    |x_i| <= 5, |u_i| <= 0.1, W_y = W_u = I, W_du = 0, C = I; x0 ~ U[-1, 1].  The same (A, B) at
    every stage (LTI, as in the paper), stored per stage like every other workload."""
    rng = np.random.default_rng([*SEED, 7, nx, nu, seed])
    A = rng.standard_normal((nx, nx))
    A /= np.max(np.abs(np.linalg.eigvals(A)))
    B = rng.standard_normal((nx, nu))
    e = rng.uniform(-0.3, 0.3, (1, N, nx))
    x0 = rng.uniform(-1.0, 1.0, (1, nx))
    lo = np.concatenate([np.full(nx, -5.0), np.full(nu, -0.1)])
    return Problem(f"T1-{nx}-{nu}-{N}", nx, nu, N, 1, np.tile(A, (1, N, 1, 1)), np.tile(B, (1, N, 1, 1)), np.eye(nx),
                   np.eye(nu), lo, -lo, x0, e=e, rho=1.0, iters=iters, tol=0.0, dtypes=("f64", "f32"))
