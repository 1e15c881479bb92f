/*
 * pimpc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU restatement of Algorithm 1 of
 * "piMPC: A Parallel-in-horizon and Construction-free NMPC Solver"
 * (arxiv 2601.14414), i.e. the accelerated,
 * restarted ADMM iteration (Eq. 16) applied to the
 * velocity-form split problem (11) with the closed-form
 * updates (12) and Theorem 1.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this file.  It shares no code, header,
 * table or helper with the CUDA path under paper_2601_14414_b200/csrc/.
 *
 * It follows the algorithm step by step, in the paper's order and notation:
 * the dense matrices Abar_k, Bbar_k, Qbar are formed
 * explicitly and multiplied by plain triple loops; there is no blocking,
 * fusion or reordering.  Where the paper is garbled or silent the reading of
 * DESIGN.md "Readings of the paper" (R1..R17) is taken; each is marked below.
 *
 * Extensions: the other projections the paper lists (halfspace, hyperplane, second-order cone,
 * l1 ball), per-stage boxes and linear terms, and the tracking cost (1a) -> (Q, R, qbar).
 * Their pins: variational inequality + brute-force nearest point per set, scipy SLSQP on the QP with the set, and
 * a least-squares KKT solve of the tracking problem.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): dense KKT solve of QP (1)
 * (unconstrained LTV, affine e_k, u_prev), brute-force active-set enumeration
 * (u-, x- and du-bounds active), the closed form c^1, the SURVEY P-tiny
 * numbers, beta+lambda=0, projection fixed point, Lemma 2 monotonicity.
 * No function here is "parity unpinned".
 *
 * Stage-indexed storage (k = 0..N-1), nb = nx+nu:
 *   X[k]  = xbar_{k+1}   Z[k]  = z_{k+1}   V[k] = v_k
 *   TH[k] = theta_k      BE[k] = beta_k    LA[k] = lambda_k    DU[k] = Delta u_k
 *   D[k]  = d_k, DE[k] = delta_k : copy / scaled dual of the optional
 *   Delta-u consensus block (reading R12; only when du_lo/du_hi are given).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* y = M x, M is r x c row-major */
static void matvec(int r, int c, const double *M, const double *x, double *y)
{
    for (int i = 0; i < r; ++i) {
        double s = 0.0;
        for (int j = 0; j < c; ++j) s += M[i * c + j] * x[j];
        y[i] = s;
    }
}

/* y = M^T x, M is r x c row-major, x has r entries, y has c entries */
static void matTvec(int r, int c, const double *M, const double *x, double *y)
{
    for (int j = 0; j < c; ++j) {
        double s = 0.0;
        for (int i = 0; i < r; ++i) s += M[i * c + j] * x[i];
        y[j] = s;
    }
}

/* Inverse of a symmetric positive definite n x n matrix S (row-major) by
 * Cholesky S = L L^T followed by one forward/backward solve per unit vector.
 * Returns 0, or -1 if S is not positive definite. */
static int spd_inverse(int n, const double *S, double *Sinv)
{
    double *L = (double *)calloc((size_t)n * n, sizeof(double));
    double *y = (double *)calloc((size_t)n, sizeof(double));
    if (!L || !y) { free(L); free(y); return -2; }
    for (int j = 0; j < n; ++j) {
        double d = S[j * n + j];
        for (int p = 0; p < j; ++p) d -= L[j * n + p] * L[j * n + p];
        if (!(d > 0.0)) { free(L); free(y); return -1; }
        L[j * n + j] = sqrt(d);
        for (int i = j + 1; i < n; ++i) {
            double s = S[i * n + j];
            for (int p = 0; p < j; ++p) s -= L[i * n + p] * L[j * n + p];
            L[i * n + j] = s / L[j * n + j];
        }
    }
    for (int col = 0; col < n; ++col) {
        /* L y = e_col */
        for (int i = 0; i < n; ++i) {
            double s = (i == col) ? 1.0 : 0.0;
            for (int p = 0; p < i; ++p) s -= L[i * n + p] * y[p];
            y[i] = s / L[i * n + i];
        }
        /* L^T x = y */
        for (int i = n - 1; i >= 0; --i) {
            double s = y[i];
            for (int p = i + 1; p < n; ++p) s -= L[p * n + i] * Sinv[p * n + col];
            Sinv[i * n + col] = s / L[i * n + i];
        }
    }
    free(L); free(y);
    return 0;
}

static double clip(double t, double lo, double hi)
{
    /* Proj onto the box [lo,hi]; +-inf bounds allowed */
    if (t < lo) return lo;
    if (t > hi) return hi;
    return t;
}

static double sq(double x) { return x * x; }

/* ---- projections onto the closed convex sets the paper lists for Proj (closed forms of [22, Ch. 6]) ----
 * Each maps t (n entries) to the nearest point of the set, written to out (out may alias t). */

/* halfspace {x : a^T x <= b}: t if it is inside, else t - ((a^T t - b) / ||a||^2) a */
static void proj_halfspace(int n, const double *t, const double *a, double b, double *out)
{
    double at = 0.0, aa = 0.0;
    for (int i = 0; i < n; ++i) { at += a[i] * t[i]; aa += a[i] * a[i]; }
    double s = (at > b && aa > 0.0) ? (at - b) / aa : 0.0;
    for (int i = 0; i < n; ++i) out[i] = t[i] - s * a[i];
}

/* affine hyperplane {x : a^T x = b}: t - ((a^T t - b) / ||a||^2) a */
static void proj_hyperplane(int n, const double *t, const double *a, double b, double *out)
{
    double at = 0.0, aa = 0.0;
    for (int i = 0; i < n; ++i) { at += a[i] * t[i]; aa += a[i] * a[i]; }
    double s = aa > 0.0 ? (at - b) / aa : 0.0;
    for (int i = 0; i < n; ++i) out[i] = t[i] - s * a[i];
}

/* second-order cone {(x, r) : ||x||_2 <= r}, t = (x (n-1 entries), r):
 * inside: t;  ||x|| <= -r (polar cone): 0;  else ((||x|| + r) / 2) (x / ||x||, 1) */
static void proj_soc(int n, const double *t, double *out)
{
    double nx2 = 0.0, r = t[n - 1];
    for (int i = 0; i < n - 1; ++i) nx2 += t[i] * t[i];
    double nx = sqrt(nx2);
    if (nx <= r) { for (int i = 0; i < n; ++i) out[i] = t[i]; return; }
    if (nx <= -r) { for (int i = 0; i < n; ++i) out[i] = 0.0; return; }
    double s = 0.5 * (nx + r);
    for (int i = 0; i < n - 1; ++i) out[i] = s * t[i] / nx;
    out[n - 1] = s;
}

/* l1 ball {x : ||x||_1 <= r}, r >= 0: t if inside, else the soft threshold sign(t_i) max(|t_i| - tau, 0) with the tau
 * that makes the l1 norm r: sort |t| in descending order u_1 >= u_2 >= ..., m = the largest j with
 * u_j > (u_1 + ... + u_j - r) / j, tau = (u_1 + ... + u_m - r) / m. */
static void proj_l1ball(int n, const double *t, double r, double *out)
{
    double l1 = 0.0;
    for (int i = 0; i < n; ++i) l1 += fabs(t[i]);
    if (l1 <= r) { for (int i = 0; i < n; ++i) out[i] = t[i]; return; }
    double *u = (double *)malloc((size_t)n * sizeof(double));
    for (int i = 0; i < n; ++i) u[i] = fabs(t[i]);
    for (int i = 1; i < n; ++i) {                     /* insertion sort, descending */
        double v = u[i]; int j = i - 1;
        while (j >= 0 && u[j] < v) { u[j + 1] = u[j]; --j; }
        u[j + 1] = v;
    }
    double cs = 0.0, tau = 0.0;
    for (int j = 1; j <= n; ++j) {
        cs += u[j - 1];
        double cand = (cs - r) / j;
        if (u[j - 1] > cand) tau = cand;
    }
    free(u);
    for (int i = 0; i < n; ++i) {
        double m = fabs(t[i]) - tau;
        out[i] = m > 0.0 ? (t[i] > 0.0 ? m : -m) : 0.0;
    }
}

/* Optional extensions of problem (1).  All pointers may be NULL. */
enum { PIMPC_ORACLE_SET_NONE = 0, PIMPC_ORACLE_SET_HALFSPACE = 1, PIMPC_ORACLE_SET_HYPERPLANE = 2,
       PIMPC_ORACLE_SET_SOC = 3, PIMPC_ORACLE_SET_L1BALL = 4 };
typedef struct {
    int set_kind;            /* which closed convex set the components [set_i0, set_i0 + set_len) of z_{k+1} lie in;
                                the other components stay in the box [lo, hi]: Xbar = box x set (a product, so the
                                projection is the product of the projections)                                        */
    int set_i0, set_len;
    const double *set_a;     /* [set_len] normal vector a of the halfspace / hyperplane                              */
    double set_b;            /* offset b (halfspace, hyperplane) or radius r (l1 ball)                               */
    const double *lo_k, *hi_k;   /* per-stage boxes [N][nb] replacing lo / hi (x_{k+1} in X_k, u_k in U_k)           */
    const double *qbar_k;        /* per-stage linear terms [N][nb] replacing qbar (time-varying references r_y, r_u) */
} pimpc_oracle_ext;

/* Proj onto Xbar of one stage: t -> z (nb entries) */
static void proj_xbar(int nb, const double *t, const double *lo, const double *hi, const pimpc_oracle_ext *x, double *z)
{
    for (int i = 0; i < nb; ++i) z[i] = clip(t[i], lo[i], hi[i]);
    if (!x || x->set_kind == PIMPC_ORACLE_SET_NONE) return;
    const int i0 = x->set_i0, n = x->set_len;
    switch (x->set_kind) {
    case PIMPC_ORACLE_SET_HALFSPACE: proj_halfspace(n, t + i0, x->set_a, x->set_b, z + i0); break;
    case PIMPC_ORACLE_SET_HYPERPLANE: proj_hyperplane(n, t + i0, x->set_a, x->set_b, z + i0); break;
    case PIMPC_ORACLE_SET_SOC: proj_soc(n, t + i0, z + i0); break;
    case PIMPC_ORACLE_SET_L1BALL: proj_l1ball(n, t + i0, x->set_b, z + i0); break;
    default: break;
    }
}

/* The projections alone, for the pins of tests/test_oracle_pins.py: kind as above, a may be NULL. */
int pimpc_oracle_project(int kind, int n, const double *t, const double *a, double b, double *out)
{
    if (n <= 0 || !t || !out) return -1;
    switch (kind) {
    case PIMPC_ORACLE_SET_HALFSPACE: if (!a) return -1; proj_halfspace(n, t, a, b, out); return 0;
    case PIMPC_ORACLE_SET_HYPERPLANE: if (!a) return -1; proj_hyperplane(n, t, a, b, out); return 0;
    case PIMPC_ORACLE_SET_SOC: proj_soc(n, t, out); return 0;
    case PIMPC_ORACLE_SET_L1BALL: if (b < 0.0) return -1; proj_l1ball(n, t, b, out); return 0;
    default: return -1;
    }
}

/* Tracking cost of problem (1a) in the form of problem (11):
 *   Q = C^T W_y C [nx][nx],  R = W_u [nu][nu],  qbar = col(C^T W_y r_y, W_u r_u) [nx+nu];  C [ny][nx], W_y [ny][ny]. */
int pimpc_oracle_tracking(int nx, int nu, int ny, const double *C, const double *Wy, const double *Wu,
                          const double *ry, const double *ru, double *Q, double *R, double *qbar)
{
    if (nx <= 0 || nu <= 0 || ny <= 0 || !C || !Wy || !Wu) return -1;
    double *WC = (double *)calloc((size_t)ny * nx, sizeof(double));      /* W_y C */
    double *Wr = (double *)calloc((size_t)ny, sizeof(double));           /* W_y r_y */
    if (!WC || !Wr) { free(WC); free(Wr); return -2; }
    for (int i = 0; i < ny; ++i) {
        for (int j = 0; j < nx; ++j) {
            double s = 0.0;
            for (int p = 0; p < ny; ++p) s += Wy[i * ny + p] * C[p * nx + j];
            WC[i * nx + j] = s;
        }
        double s = 0.0;
        for (int p = 0; p < ny; ++p) s += Wy[i * ny + p] * (ry ? ry[p] : 0.0);
        Wr[i] = s;
    }
    for (int i = 0; i < nx; ++i) {
        for (int j = 0; j < nx; ++j) {
            double s = 0.0;
            for (int p = 0; p < ny; ++p) s += C[p * nx + i] * WC[p * nx + j];
            Q[i * nx + j] = s;
        }
        double s = 0.0;
        for (int p = 0; p < ny; ++p) s += C[p * nx + i] * Wr[p];
        qbar[i] = s;
    }
    for (int i = 0; i < nu; ++i) {
        double s = 0.0;
        for (int j = 0; j < nu; ++j) { R[i * nu + j] = Wu[i * nu + j]; s += Wu[i * nu + j] * (ru ? ru[j] : 0.0); }
        qbar[nx + i] = s;
    }
    free(WC); free(Wr);
    return 0;
}

/*
 * One invocation of Algorithm 1 for ONE problem instance.
 *
 * Inputs (all row-major, double):
 *   A [N][nx][nx], B [N][nx][nu], e [N][nx] or NULL (=0)      -- (1b) PAPER.md:41
 *   Q [nx][nx] = C^T W_y C, R [nu][nu] = W_u  (Qbar = diag(Q,R))
 *   P [nx][nx] or NULL: terminal weight replacing Q in stage N-1 (R14)
 *   Wdu [nu][nu] or NULL: weight on Delta u (R13)
 *   qbar [nb] or NULL (=0)                                     -- PAPER.md:197
 *   lo, hi [nb] = (x_lo;u_lo), (x_hi;u_hi): the box Xbar = X x U
 *   du_lo, du_hi [nu] or both NULL: box on Delta u (R12)
 *   x0 [nx], u_prev [nu] or NULL (=0): xbar_0 = (x(t); u(t-1)) (R10)
 *   rho > 0, eta (0.999), c0 (1.0)                             -- PAPER.md:287,339
 *   max_iters = K_max, tol = epsilon (<= 0: never stop early)  -- PAPER.md:339,370
 *   forced [n_forced] or NULL: if given, decision i (i < n_forced) of the
 *       accept/restart test is taken from forced[i] instead of the comparison
 *       (P-flip replay protocol); 1 = accept (step 6), 0 = restart (step 7)
 * In/out (warm start, "such as from warm-start", 381):
 *   Z,V,TH,BE,LA [N][nb];  D,DE [N][nu] (ignored/untouched if no du bounds)
 *   The hats start equal to these iterates, alpha_0 = 1, c^0 = c0.
 * Out:
 *   X [N][nb], DU [N][nu]: the primal block of the last executed iteration
 *   c_hist [max_iters], acc_hist [max_iters] (either may be NULL):
 *       c^{i+1} and the decision bit of iteration i (bit = 0 for the stopping iteration)
 *   info[0] = iterations executed, info[1] = number of restarts (step 7 taken)
 *   c_last = c of the last executed iteration
 *   r_parts [2] or NULL: the two halves of c_last:
 *       r_parts[0] = rho ||s^{i+1} - shat^i||^2  (primal residual F p + G q - h, by (15c))
 *       r_parts[1] = rho ||G (q^{i+1} - qhat^i)||^2  (dual residual)
 *   ext or NULL: general convex set on part of z, per-stage boxes, per-stage linear terms (see pimpc_oracle_ext)
 * Returns 0, -1 bad argument, -2 out of memory, -5 matrix not positive definite.
 */
int pimpc_oracle_solve(
    int nx, int nu, int N,
    const double *A, const double *B, const double *e,
    const double *Q, const double *R, const double *P, const double *Wdu,
    const double *qbar,
    const double *lo, const double *hi, const double *du_lo, const double *du_hi,
    const double *x0, const double *u_prev,
    double rho, double eta, double c0,
    int max_iters, double tol,
    const unsigned char *forced, int n_forced,
    double *Z, double *V, double *TH, double *BE, double *LA, double *D, double *DE,
    double *X, double *DU,
    double *c_hist, unsigned char *acc_hist,
    int *info, double *c_last, double *r_parts, const pimpc_oracle_ext *ext)
{
    if (nx <= 0 || nu <= 0 || N <= 0 || !(rho > 0.0) || max_iters < 0) return -1;
    if ((du_lo == NULL) != (du_hi == NULL)) return -1;
    const int nb = nx + nu;
    const int has_du = (du_lo != NULL);
    int rc = 0;

    /* ---- derived data: Abar_k, Bbar_k, ebar_k, Qbar, Qbar_N ---- */
    double *Abar = (double *)calloc((size_t)N * nb * nb, sizeof(double));
    double *Bbar = (double *)calloc((size_t)N * nb * nu, sizeof(double));
    double *ebar = (double *)calloc((size_t)N * nb, sizeof(double));
    double *Qbar = (double *)calloc((size_t)nb * nb, sizeof(double));
    double *QbarN = (double *)calloc((size_t)nb * nb, sizeof(double));
    double *qb = (double *)calloc((size_t)nb, sizeof(double));
    double *xbar0 = (double *)calloc((size_t)nb, sizeof(double));
    /* cache: M_k = (Bbar^T Bbar [+Wdu/rho] [+I])^-1 so that J_k = M_k Bbar_k^T; H_k */
    double *M = (double *)calloc((size_t)N * nu * nu, sizeof(double));
    double *H = (double *)calloc((size_t)N * nb * nb, sizeof(double));
    double *S = (double *)calloc((size_t)nb * nb, sizeof(double));
    /* hats and new iterates */
    size_t szb = (size_t)N * nb, szu = (size_t)N * nu;
    double *Zh = (double *)calloc(szb, sizeof(double)), *Vh = (double *)calloc(szb, sizeof(double));
    double *THh = (double *)calloc(szb, sizeof(double)), *BEh = (double *)calloc(szb, sizeof(double));
    double *LAh = (double *)calloc(szb, sizeof(double));
    double *Dh = (double *)calloc(szu, sizeof(double)), *DEh = (double *)calloc(szu, sizeof(double));
    double *Zn = (double *)calloc(szb, sizeof(double)), *Vn = (double *)calloc(szb, sizeof(double));
    double *THn = (double *)calloc(szb, sizeof(double)), *BEn = (double *)calloc(szb, sizeof(double));
    double *LAn = (double *)calloc(szb, sizeof(double));
    double *Dn = (double *)calloc(szu, sizeof(double)), *DEn = (double *)calloc(szu, sizeof(double));
    double *t1 = (double *)calloc((size_t)nb, sizeof(double)), *t2 = (double *)calloc((size_t)nb, sizeof(double));
    double *t3 = (double *)calloc((size_t)nb, sizeof(double)), *t4 = (double *)calloc((size_t)nb, sizeof(double));
    double *va = (double *)calloc((size_t)nb, sizeof(double)), *vb = (double *)calloc((size_t)nb, sizeof(double));
    double *vt = (double *)calloc((size_t)nb, sizeof(double)), *vz = (double *)calloc((size_t)nb, sizeof(double));
    if (ext && ext->set_kind != PIMPC_ORACLE_SET_NONE &&
        (ext->set_i0 < 0 || ext->set_len <= 0 || ext->set_i0 + ext->set_len > nb ||
         ((ext->set_kind == PIMPC_ORACLE_SET_HALFSPACE || ext->set_kind == PIMPC_ORACLE_SET_HYPERPLANE) && !ext->set_a))) { rc = -1; goto done; }
    if (!va || !vb || !vt || !vz) { rc = -2; goto done; }
    if (!Abar || !Bbar || !ebar || !Qbar || !QbarN || !qb || !xbar0 || !M || !H || !S || !Zh || !Vh ||
        !THh || !BEh || !LAh || !Dh || !DEh || !Zn || !Vn || !THn || !BEn || !LAn || !Dn || !DEn ||
        !t1 || !t2 || !t3 || !t4) { rc = -2; goto done; }

    for (int k = 0; k < N; ++k) {
        double *Ab = Abar + (size_t)k * nb * nb, *Bb = Bbar + (size_t)k * nb * nu;
        for (int i = 0; i < nx; ++i) {
            for (int j = 0; j < nx; ++j) Ab[i * nb + j] = A[((size_t)k * nx + i) * nx + j];
            for (int j = 0; j < nu; ++j) Ab[i * nb + nx + j] = B[((size_t)k * nx + i) * nu + j];
            for (int j = 0; j < nu; ++j) Bb[i * nu + j] = B[((size_t)k * nx + i) * nu + j];
            ebar[(size_t)k * nb + i] = e ? e[(size_t)k * nx + i] : 0.0;
        }
        for (int i = 0; i < nu; ++i) {
            Ab[(nx + i) * nb + nx + i] = 1.0;   /* [0 I] */
            Bb[(nx + i) * nu + i] = 1.0;        /* [B; I] */
        }
    }
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < nx; ++j) {
            Qbar[i * nb + j] = Q[i * nx + j];
            QbarN[i * nb + j] = P ? P[i * nx + j] : Q[i * nx + j];     /* R14 */
        }
    for (int i = 0; i < nu; ++i)
        for (int j = 0; j < nu; ++j) {
            Qbar[(nx + i) * nb + nx + j] = R[i * nu + j];
            QbarN[(nx + i) * nb + nx + j] = R[i * nu + j];
        }
    for (int i = 0; i < nb; ++i) qb[i] = qbar ? qbar[i] : 0.0;
    for (int i = 0; i < nx; ++i) xbar0[i] = x0[i];
    for (int i = 0; i < nu; ++i) xbar0[nx + i] = u_prev ? u_prev[i] : 0.0;   /* R10 */

    /* ---- cache ---- */
    for (int k = 0; k < N; ++k) {
        const double *Ab1 = Abar + (size_t)(k + 1) * nb * nb, *Bb = Bbar + (size_t)k * nb * nu;
        /* Bbar^T Bbar (= B^T B + I) [+ Wdu/rho (R13)] [+ I (R12)] */
        for (int i = 0; i < nu; ++i)
            for (int j = 0; j < nu; ++j) {
                double s = 0.0;
                for (int p = 0; p < nb; ++p) s += Bb[p * nu + i] * Bb[p * nu + j];
                if (Wdu) s += Wdu[i * nu + j] / rho;
                if (has_du && i == j) s += 1.0;
                S[i * nu + j] = s;
            }
        if (spd_inverse(nu, S, M + (size_t)k * nu * nu) != 0) { rc = -5; goto done; }
        /* H_k: (Qbar + rho I + rho Abar_{k+1}^T Abar_{k+1})^-1, k < N-1;
           (Qbar_N + rho I)^-1 for k = N-1 */
        for (int i = 0; i < nb; ++i)
            for (int j = 0; j < nb; ++j) {
                double s = (k == N - 1) ? QbarN[i * nb + j] : Qbar[i * nb + j];
                if (i == j) s += rho;
                if (k < N - 1) {
                    double a = 0.0;
                    for (int p = 0; p < nb; ++p) a += Ab1[p * nb + i] * Ab1[p * nb + j];
                    s += rho * a;
                }
                S[i * nb + j] = s;
            }
        if (spd_inverse(nb, S, H + (size_t)k * nb * nb) != 0) { rc = -5; goto done; }
    }

    /* ---- input of Alg. 1: hats = iterates, alpha_0 = 1, c^0 = c0 ---- */
    memcpy(Zh, Z, szb * sizeof(double)); memcpy(Vh, V, szb * sizeof(double));
    memcpy(THh, TH, szb * sizeof(double)); memcpy(BEh, BE, szb * sizeof(double));
    memcpy(LAh, LA, szb * sizeof(double));
    if (has_du) { memcpy(Dh, D, szu * sizeof(double)); memcpy(DEh, DE, szu * sizeof(double)); }
    double alpha = 1.0, c_prev = c0, c = c0, rp = 0.0, rd = 0.0;
    int iters = 0, restarts = 0;

    for (int it = 0; it < max_iters; ++it) {
        /* ---- step 1 (Eq. 12a) ---- */
        for (int k = 0; k < N; ++k) {
            const double *Bb = Bbar + (size_t)k * nb * nu;
            /* Delta u_k = M_k ( Bbar_k^T (vhat_k - betahat_k) [+ dhat_k - deltahat_k] ) */
            for (int i = 0; i < nb; ++i) t1[i] = Vh[(size_t)k * nb + i] - BEh[(size_t)k * nb + i];
            matTvec(nb, nu, Bb, t1, t2);
            if (has_du) for (int i = 0; i < nu; ++i) t2[i] += Dh[(size_t)k * nu + i] - DEh[(size_t)k * nu + i];
            matvec(nu, nu, M + (size_t)k * nu * nu, t2, DU + (size_t)k * nu);
            /* h_k = qbar + rho (zhat_{k+1} - thetahat_k)
                     [+ rho Abar_{k+1}^T (zhat_{k+2} - vhat_{k+1} - ebar_{k+1} + lambdahat_{k+1})]   (R2) */
            for (int i = 0; i < nb; ++i)
                t3[i] = ((ext && ext->qbar_k) ? ext->qbar_k[(size_t)k * nb + i] : qb[i])
                      + rho * (Zh[(size_t)k * nb + i] - THh[(size_t)k * nb + i]);
            if (k < N - 1) {
                const double *Ab1 = Abar + (size_t)(k + 1) * nb * nb;
                for (int i = 0; i < nb; ++i)
                    t1[i] = Zh[(size_t)(k + 1) * nb + i] - Vh[(size_t)(k + 1) * nb + i]
                          - ebar[(size_t)(k + 1) * nb + i] + LAh[(size_t)(k + 1) * nb + i];
                matTvec(nb, nb, Ab1, t1, t4);
                for (int i = 0; i < nb; ++i) t3[i] += rho * t4[i];
            }
            matvec(nb, nb, H + (size_t)k * nb * nb, t3, X + (size_t)k * nb);   /* xbar_{k+1} = H_k h_k */
        }
        /* ---- steps 2, 3 (Thm 1 proof PAPER.md:150-164, R1) and 4 (R7) ---- */
        double csum = 0.0, psum = 0.0, dsum = 0.0;
        for (int k = 0; k < N; ++k) {
            const double *Ab = Abar + (size_t)k * nb * nb, *Bb = Bbar + (size_t)k * nb * nu;
            const double *xk = (k == 0) ? xbar0 : X + (size_t)(k - 1) * nb;    /* xbar_k^{i+1} */
            matvec(nb, nu, Bb, DU + (size_t)k * nu, t1);       /* Bbar_k Delta u_k */
            matvec(nb, nb, Ab, xk, t2);                        /* Abar_k xbar_k   */
            for (int i = 0; i < nb; ++i) {
                size_t q = (size_t)k * nb + i;
                va[i] = t1[i] + BEh[q];                        /* a = Bbar du + betahat            */
                vb[i] = t2[i] + ebar[q] - LAh[q];              /* b = Abar xbar + ebar - lambdahat */
                double gamma = va[i] - vb[i];
                vt[i] = (2.0 * (X[q] + THh[q] + vb[i]) + gamma) / 3.0;      /* argument of Proj */
            }
            /* z_{k+1} = Proj_Xbar(.) (Thm 1: exact for any closed convex set) */
            proj_xbar(nb, vt, (ext && ext->lo_k) ? ext->lo_k + (size_t)k * nb : lo,
                      (ext && ext->hi_k) ? ext->hi_k + (size_t)k * nb : hi, ext, vz);
            for (int i = 0; i < nb; ++i) {
                size_t q = (size_t)k * nb + i;
                double a = va[i], b = vb[i], gamma = a - b, zn = vz[i];
                double vn = 0.5 * (zn + gamma);
                Zn[q] = zn; Vn[q] = vn;
                THn[q] = THh[q] + X[q] - zn;
                BEn[q] = a - vn;                               /* = betahat + Bbar du - v */
                LAn[q] = zn - b - vn;                          /* = lambdahat + z - Abar xbar - v - ebar */
                csum += sq(THn[q] - THh[q]) + sq(BEn[q] - BEh[q]) + sq(LAn[q] - LAh[q])
                      + sq(zn - Zh[q]) + sq(vn - Vh[q]) + sq((zn - vn) - (Zh[q] - Vh[q]));
                psum += sq(THn[q] - THh[q]) + sq(BEn[q] - BEh[q]) + sq(LAn[q] - LAh[q]);        /* ||Delta s||^2   */
                dsum += sq(zn - Zh[q]) + sq(vn - Vh[q]) + sq((zn - vn) - (Zh[q] - Vh[q]));      /* ||G Delta q||^2 */
            }
            if (has_du) {                                      /* R12 */
                for (int i = 0; i < nu; ++i) {
                    size_t q = (size_t)k * nu + i;
                    double dn = clip(DU[q] + DEh[q], du_lo[i], du_hi[i]);
                    Dn[q] = dn;
                    DEn[q] = DEh[q] + DU[q] - dn;
                    csum += sq(DEn[q] - DEh[q]) + sq(dn - Dh[q]);
                    psum += sq(DEn[q] - DEh[q]);
                    dsum += sq(dn - Dh[q]);
                }
            }
        }
        c = rho * csum;
        rp = rho * psum; rd = rho * dsum;
        iters = it + 1;
        if (c_hist) c_hist[it] = c;

        /* ---- step 5 (R11) ---- */
        if (c < tol) {
            memcpy(Z, Zn, szb * sizeof(double)); memcpy(V, Vn, szb * sizeof(double));
            memcpy(TH, THn, szb * sizeof(double)); memcpy(BE, BEn, szb * sizeof(double));
            memcpy(LA, LAn, szb * sizeof(double));
            if (has_du) { memcpy(D, Dn, szu * sizeof(double)); memcpy(DE, DEn, szu * sizeof(double)); }
            if (acc_hist) acc_hist[it] = 0;
            break;
        }
        /* ---- steps 6 / 7 (R5, R6) ---- */
        int accept = (c <= eta * c_prev);
        if (forced && it < n_forced) accept = forced[it] ? 1 : 0;
        if (acc_hist) acc_hist[it] = (unsigned char)accept;
        double kappa;
        if (accept) {
            double alpha_next = 0.5 + 0.5 * sqrt(1.0 + 4.0 * alpha * alpha);
            kappa = (alpha - 1.0) / alpha_next;
            alpha = alpha_next;
        } else {
            kappa = 0.0;
            alpha = 1.0;
            ++restarts;
        }
        for (size_t q = 0; q < szb; ++q) {
            Zh[q] = Zn[q] + kappa * (Zn[q] - Z[q]);
            Vh[q] = Vn[q] + kappa * (Vn[q] - V[q]);
            THh[q] = THn[q] + kappa * (THn[q] - TH[q]);
            BEh[q] = BEn[q] + kappa * (BEn[q] - BE[q]);
            LAh[q] = LAn[q] + kappa * (LAn[q] - LA[q]);
            Z[q] = Zn[q]; V[q] = Vn[q]; TH[q] = THn[q]; BE[q] = BEn[q]; LA[q] = LAn[q];
        }
        if (has_du)
            for (size_t q = 0; q < szu; ++q) {
                Dh[q] = Dn[q] + kappa * (Dn[q] - D[q]);
                DEh[q] = DEn[q] + kappa * (DEn[q] - DE[q]);
                D[q] = Dn[q]; DE[q] = DEn[q];
            }
        c_prev = c;
    }
    if (info) { info[0] = iters; info[1] = restarts; }
    if (c_last) *c_last = c;
    if (r_parts) { r_parts[0] = rp; r_parts[1] = rd; }

done:
    free(Abar); free(Bbar); free(ebar); free(Qbar); free(QbarN); free(qb); free(xbar0);
    free(M); free(H); free(S);
    free(Zh); free(Vh); free(THh); free(BEh); free(LAh); free(Dh); free(DEh);
    free(Zn); free(Vn); free(THn); free(BEn); free(LAn); free(Dn); free(DEn);
    free(t1); free(t2); free(t3); free(t4); free(va); free(vb); free(vt); free(vz);
    return rc;
}

/* The per-solve cache alone, exposed so that tests can pin it
 * against numpy.linalg.inv: M [N][nu][nu], H [N][nb][nb]. */
int pimpc_oracle_cache(
    int nx, int nu, int N, const double *A, const double *B,
    const double *Q, const double *R, const double *P, const double *Wdu,
    int has_du, double rho, double *M, double *H)
{
    if (nx <= 0 || nu <= 0 || N <= 0 || !(rho > 0.0)) return -1;
    const int nb = nx + nu;
    double *S = (double *)calloc((size_t)nb * nb, sizeof(double));
    double *Ab1 = (double *)calloc((size_t)nb * nb, sizeof(double));
    if (!S || !Ab1) { free(S); free(Ab1); return -2; }
    int rc = 0;
    for (int k = 0; k < N && rc == 0; ++k) {
        const double *Bk = B + (size_t)k * nx * nu;
        for (int i = 0; i < nu; ++i)
            for (int j = 0; j < nu; ++j) {
                double s = (i == j) ? 1.0 : 0.0;               /* I of Bbar^T Bbar = B^T B + I */
                for (int p = 0; p < nx; ++p) s += Bk[p * nu + i] * Bk[p * nu + j];
                if (Wdu) s += Wdu[i * nu + j] / rho;
                if (has_du && i == j) s += 1.0;
                S[i * nu + j] = s;
            }
        if (spd_inverse(nu, S, M + (size_t)k * nu * nu) != 0) { rc = -5; break; }
        if (k < N - 1) {
            memset(Ab1, 0, (size_t)nb * nb * sizeof(double));
            for (int i = 0; i < nx; ++i) {
                for (int j = 0; j < nx; ++j) Ab1[i * nb + j] = A[((size_t)(k + 1) * nx + i) * nx + j];
                for (int j = 0; j < nu; ++j) Ab1[i * nb + nx + j] = B[((size_t)(k + 1) * nx + i) * nu + j];
            }
            for (int i = 0; i < nu; ++i) Ab1[(nx + i) * nb + nx + i] = 1.0;
        }
        for (int i = 0; i < nb; ++i)
            for (int j = 0; j < nb; ++j) {
                double s = 0.0;
                if (i < nx && j < nx) s = (k == N - 1 && P) ? P[i * nx + j] : Q[i * nx + j];
                if (i >= nx && j >= nx) s = R[(i - nx) * nu + (j - nx)];
                if (i == j) s += rho;
                if (k < N - 1) {
                    double a = 0.0;
                    for (int p = 0; p < nb; ++p) a += Ab1[p * nb + i] * Ab1[p * nb + j];
                    s += rho * a;
                }
                S[i * nb + j] = s;
            }
        if (spd_inverse(nb, S, H + (size_t)k * nb * nb) != 0) { rc = -5; break; }
    }
    free(S); free(Ab1);
    return rc;
}
