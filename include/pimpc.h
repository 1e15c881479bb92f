/*
 * pimpc.h -- C ABI of libpimpc.so: the accelerated, restarted ADMM iteration of piMPC
 * (arxiv 2601.14414, Algorithm 1) over the velocity-form, construction-free
 * MPC-QP (Problem (11)) as hand-written sm_100a CUDA.
 *
 * Conventions (all entry points)
 *   - Plain C: opaque handle, plain pointers and sizes, no C++/torch types.
 *   - Every data pointer may be HOST or DEVICE memory (resolved with cudaPointerGetAttributes).
 *     Numeric arrays have the element type of the handle (`dtype`: double or float), row-major,
 *     innermost index contiguous.  Scalars in structs are always double/int.
 *   - Ownership: the library owns all device state.  Inputs are copied during the call: a host
 *     buffer may be reused when the call returns; a device buffer once the handle's stream reaches
 *     that point.  Outputs are caller-allocated.
 *   - Errors: every function returns PIMPC_OK (0) or a negative code and never throws or aborts.
 *     pimpc_last_error() gives a message.  A CUDA error poisons the handle (PIMPC_ESTATE later).
 *   - A handle is not thread-safe; distinct handles are independent.  All work of a handle is
 *     enqueued on its stream (opts.stream, a cudaStream_t; NULL = legacy default stream).
 *   - There is no CPU fallback: without a CUDA device pimpc_create returns PIMPC_ECUDA.
 *
 * Notation (stage-indexed, k = 0..N-1, nb = nx+nu), as in the paper:
 *   X[k] = xbar_{k+1}, Z[k] = z_{k+1}, V[k] = v_k, TH[k] = theta_k, BE[k] = beta_k,
 *   LA[k] = lambda_k, DU[k] = Delta u_k; D[k], DE[k] = copy / scaled dual of the optional
 *   Delta-u box (reading R12; active only when finite du bounds were supplied).
 */
#ifndef PIMPC_H
#define PIMPC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pimpc_s *pimpc_t;

enum { PIMPC_OK = 0, PIMPC_EINVAL = -1, PIMPC_ENOMEM = -2, PIMPC_ECUDA = -3, PIMPC_ESTATE = -4,
       PIMPC_ENOTPD = -5 };
enum { PIMPC_F64 = 0, PIMPC_F32 = 1 };

/* Iteration drivers.  AUTO picks by footprint. */
enum {
    PIMPC_ENGINE_AUTO = 0,
    PIMPC_ENGINE_STAGED = 1,   /* one launch per step of Alg. 1 per iteration; any nx,nu; the A/B baseline */
    PIMPC_ENGINE_RESIDENT = 2, /* one CTA per instance, all stage data on-chip for every iteration      */
    PIMPC_ENGINE_STREAM = 3,   /* persistent CTAs stream per-stage blobs HBM->smem (bulk async copies); nx <= 50, nu <= 15 */
    PIMPC_ENGINE_COOP = 4      /* cooperative grid, data resident in smem, one grid barrier per iteration */
};

/* which = selector of pimpc_get_state / pimpc_set_state */
enum { PIMPC_X = 0, PIMPC_Z = 1, PIMPC_V = 2, PIMPC_TH = 3, PIMPC_BE = 4, PIMPC_LA = 5, PIMPC_D = 6,
       PIMPC_DE = 7, PIMPC_DU = 8 };

/* Launch-shape overrides of the fused engines; 0 everywhere = automatic (what pimpc_default_opts sets).  They do not
 * change WHAT is computed, only how the stages are spread over CTAs / lanes; the parity tests use them to reach every
 * code path (ranges that split instances, ragged ranges, single-CTA runs) on small problems. */
typedef struct {
    int grid;             /* STREAM: at most this many CTAs; COOP: this many (<= N, <= SMs; fewer = longer ranges per CTA) */
    int ctas_per_sm;      /* STREAM: resident CTAs per SM                                                          */
    int ring_slots;       /* STREAM: at most this many slots in the bulk-copy ring                                 */
    int stages_per_group; /* COOP: stages per lane group (1 or 2)                                                  */
    int cluster;          /* COOP: -1 = never one thread-block cluster (exchange through L2), n > 0 = cluster of
                             n CTAs (<= 16), 0 = automatic (one cluster for short horizons)                       */
    int rows_per_lane;    /* RESIDENT: matrix rows per lane (1 or 2; 2 only where instantiated)                    */
    int lookahead;        /* COOP: >= 0 = run the next iteration's phases on the PREDICTED accept / restart decision
                             while the partial sums of c travel (same bits), -1 = wait for the decision */
    int reserved_;
} pimpc_tune;

typedef struct {
    int dtype;        /* PIMPC_F64 | PIMPC_F32: arithmetic and I/O element type                      */
    int engine;       /* PIMPC_ENGINE_*; AUTO = 0                                                     */
    double rho;       /* ADMM penalty, > 0; 0 -> 1.0                                   */
    double eta;       /* restart threshold; < 0 -> 0.999; 0 = plain ADMM           */
    double c0;        /* c^0; 0 -> 1.0                                             */
    int history;      /* > 0: keep (c^{i+1}, accept bit) of up to `history` iterations per instance   */
    void *stream;     /* cudaStream_t on which all work of the handle is enqueued                     */
    void *workspace;  /* DEVICE memory for the handle's problem data, cache and iterates, or NULL: the library
                         allocates.  256-byte aligned, at least pimpc_workspace_bytes() bytes, owned by the caller
                         and kept alive until pimpc_destroy.  Engine-private scratch that depends on the launch
                         plan (packed blobs, exchange words, result staging) is always allocated by the library. */
    size_t workspace_bytes; /* size of `workspace`; EINVAL if it is given and too small                */
    pimpc_tune tune;  /* launch-shape overrides, all 0 = automatic                                    */
} pimpc_opts;

/* Per-instance result record written by pimpc_get (always double/int, host or device). */
typedef struct {
    double c;         /* c^{i+1} of the last executed iteration                    */
    double alpha;     /* alpha after the last decision                             */
    double r_prim2;   /* rho ||F p + G q - h||^2 of the returned iterate: the primal-residual half of c
                         ((14a), (15c)), evaluated from its definition on X, DU, Z, V[, D]  */
    double r_dual2;   /* c - r_prim2 = rho ||G (q^{i+1} - qhat^i)||^2, the dual-residual half  */
    int iters;        /* iterations executed (i+1 at the break of step 5, else max_iters)             */
    int restarts;     /* number of times step 7 (restart) was taken                                   */
    int converged;    /* 1 if step 5 (c < tol) stopped the instance                                   */
    int pad_;
} pimpc_result;

typedef struct {
    int engine;               /* engine the last pimpc_solve used                                     */
    int launches;             /* kernels launched by the last pimpc_solve (incl. the cache kernel)    */
    long long total_launches; /* kernels launched by this handle since creation                       */
    size_t device_bytes;      /* device memory owned by the handle                                    */
    int sm_count;             /* SMs of the device                                                    */
    int grid, block;          /* launch shape of the iteration kernel of the last solve               */
    size_t smem_bytes;        /* dynamic shared memory of that kernel                                 */
    double setup_ms;          /* device time of the cache kernel of the last solve (0 if it did not run) */
    double iter_ms;           /* device time of the iteration kernel(s) of the last solve (CUDA events on
                                 the handle's stream; pimpc_get_info waits for them)                  */
} pimpc_info;

/* On-chip peaks of the current device, MEASURED by dependency-chain microbenchmarks (a few tens of milliseconds each):
 * the rooflines the register-resident engine is reported against ("measure both with an FMA-chain
 * microbenchmark ... declare which one binds").  TFLOP/s count 2 flops per FMA. */
typedef struct {
    double ffma_tflops;   /* scalar fma.rn.f32                                                          */
    double ffma2_tflops;  /* packed fma.rn.f32x2 (what the fp32 mat-vecs of the RESIDENT engine issue)  */
    double dfma_tflops;   /* fma.rn.f64                                                                 */
    double smem_gbs;      /* conflict-free 16-byte shared-memory loads, all SMs                         */
    int sm_count;
    int pad_;
    /* Latencies of one dependent instruction (SM cycles, one warp alone on an SM, clock64 around a chain): what an in-order
     * warp pays per step of a dependency chain -- the register-resident kernels run 3-4 warps per scheduler in lock-step
     * phases, so these, not the pipe rates above, set the length of a phase. */
    double lat_ffma2_cycles;  /* fma.rn.f32x2 -> fma.rn.f32x2                                               */
    double lat_dadd_cycles;   /* add.f64 -> add.f64                                                         */
    double lat_shfl_cycles;   /* shfl.sync.bfly -> shfl.sync.bfly                                           */
    double lat_lds_cycles;    /* ld.shared (pointer chase)                                                  */
    /* Shared-memory pipe cycles per warp-wide 16-byte load when groups of 8 lanes read the same 16 bytes (the broadcast
     * vector loads of the RESIDENT engine), 16 warps per SM, addresses moving every iteration; a load with 32 distinct
     * addresses takes 4 (smem_gbs above). */
    double lds128_bcast_cycles;
} pimpc_peaks;

const char *pimpc_version(void);

/* Run the microbenchmarks on the current device and `stream` (a cudaStream_t, NULL = default); synchronises.
 * EINVAL: out is NULL; ECUDA / ENOMEM on device errors. */
int pimpc_measure_peaks(pimpc_peaks *out, void *stream);

/* Fill `o` with defaults (f64, AUTO, rho=1, eta=0.999, c0=1, no history, default stream, no workspace, tune = 0). */
void pimpc_default_opts(pimpc_opts *o);

/* Device bytes pimpc_create allocates for these dimensions = the size a caller-provided opts.workspace must have
 * (0 on invalid arguments). */
size_t pimpc_workspace_bytes(int nx, int nu, int N, int batch, const pimpc_opts *opts);

/* Create a solver for `batch` independent MPC instances with nx states, nu inputs, horizon N
 * (Problem (1)).  Cold start (all iterates 0, reading R9), e_k = 0, qbar = 0,
 * u_prev = 0, no bounds (+-inf), Q = I, R = I until the setters are called.
 * opts may be NULL (defaults).  EINVAL: nx,nu,N,batch <= 0, nx+nu > 160, batch > 65535, rho <= 0, bad dtype,
 * workspace too small or misaligned. */
int pimpc_create(pimpc_t *out, int nx, int nu, int N, int batch, const pimpc_opts *opts);
int pimpc_destroy(pimpc_t h);

/* Per-stage setter (BASELINE.json north_star).  b = instance, k = stage.
 * A_k [nx][nx], B_k [nx][nu], e_k [nx] (dynamics (1b)); any may be NULL = unchanged.
 * Q [nx][nx], R [nu][nu]: shared stage cost (Qbar = diag(Q,R)), NULL = unchanged.
 * bounds [2][nx+nu] = (x_lo;u_lo) then (x_hi;u_hi) of the box Xbar = X x U, shared by
 * all stages and instances unless per-instance bounds were set, NULL = unchanged.
 * x0 [nx]: x(t) of instance b, NULL = unchanged. */
int pimpc_set_stage(pimpc_t h, int b, int k, const void *A_k, const void *B_k, const void *e_k,
                    const void *Q, const void *R, const void *bounds, const void *x0);

/* Bulk setter: A [batch][N][nx][nx], B [batch][N][nx][nu], e [batch][N][nx] or NULL (= keep). */
int pimpc_set_stages(pimpc_t h, const void *A, const void *B, const void *e);

/* Cost.  Q [nx][nx] = C'W_y C and R [nu][nu] = W_u symmetric PSD; so are P and Wdu.  The cache kernels
 * rely on the symmetry (they read the pivot row of each exchange step from the pivot column): a non-symmetric matrix is not
 * detected and gives a wrong cache.
 * P [nx][nx] or NULL: terminal weight used instead of Q at stage N-1 (R14; NULL = Q).
 * Wdu [nu][nu] or NULL: weight on Delta u (R13; NULL = 0).
 * qbar [nx+nu] or NULL: linear term col(C'W_y r_y, W_u r_u) (NULL = 0); replaces per-stage linear terms.
 * per_instance != 0: each array has a leading [batch] dimension. */
int pimpc_set_cost(pimpc_t h, const void *Q, const void *R, const void *P, const void *Wdu,
                   const void *qbar, int per_instance);

/* Box constraints.  lo, hi [nx+nu] = (x_lo;u_lo), (x_hi;u_hi); +-inf = unbounded.
 * du_lo, du_hi [nu] or both NULL: box on Delta u (R12).  Passing finite du bounds enables the
 * D/DE consensus block; passing NULL disables it (the iteration is then exactly Alg. 1).
 * per_instance != 0: leading [batch] dimension.  EINVAL if any lo > hi or a NaN. */
int pimpc_set_bounds(pimpc_t h, const void *lo, const void *hi, const void *du_lo, const void *du_hi,
                     int per_instance);

/* Tracking cost of problem (1a): 1/2 ||C x_{k+1} - r_y||^2_{W_y} + 1/2 ||u_k - r_u||^2_{W_u}.  Forms, on the
 * device and in double precision,  Q = C'W_y C,  R = W_u,  qbar = col(C'W_y r_y, W_u r_u) and installs them
 * as the (shared) cost of the handle, like pimpc_set_cost(Q, R, P = NULL, Wdu = unchanged, qbar).
 * C [ny][nx], Wy [ny][ny], Wu [nu][nu] symmetric PSD; ry, ru may be NULL (= 0).
 * per_stage == 0: ry [ny], ru [nu].  per_stage != 0: time-varying references ry [N][ny] (for x_1..x_N), ru [N][nu] (for
 * u_0..u_{N-1}); qbar then differs per stage (only the STAGED and STREAM engines take per-stage terms).
 * EINVAL: ny <= 0, ny > 160, C / Wy / Wu NULL, per-instance cost already set. */
int pimpc_set_tracking(pimpc_t h, int ny, const void *C, const void *Wy, const void *Wu, const void *ry, const void *ru,
                       int per_stage);

/* Per-stage boxes and linear terms (stage-dependent sets X_k, U_k and references; problem (1) with stage-dependent data):
 * lo, hi [N][nb] (row k bounds (x_{k+1}; u_k)) replace the shared box of pimpc_set_bounds; qbar [N][nb] replaces the
 * shared linear term.  lo and hi come together; any argument NULL = that item is not per-stage (back to the shared one).
 * per_instance != 0: leading [batch] dimension.  Only the STAGED and STREAM engines take per-stage terms (AUTO picks
 * among them).  EINVAL if any lo > hi or a NaN. */
int pimpc_set_stage_terms(pimpc_t h, const void *lo, const void *hi, const void *qbar, int per_instance);

/* General closed convex set for part of z_{k+1} (Theorem 1: the z-update is Proj of the same argument
 * for ANY closed convex set).  The components [i0, i0 + len) of every (x_{k+1}; u_k) are projected onto
 *   PIMPC_SET_HALFSPACE  {s : a's <= b}        PIMPC_SET_HYPERPLANE {s : a's = b}
 *   PIMPC_SET_SOC        {(s, r) : ||s||_2 <= r}, r = the last of the len components
 *   PIMPC_SET_L1BALL     {s : ||s||_1 <= b}
 * (closed forms of [22, Ch. 6]) instead of being clipped; the other components keep their box: the
 * constraint set is the product box x set.  a [len] (halfspace, hyperplane; element type of the handle; else NULL),
 * b = offset or radius.  PIMPC_SET_NONE removes the set.  Shared by all stages and instances.  Only the STAGED and STREAM
 * engines take a general set.  EINVAL: bad kind or range, a missing or all zero, b < 0 for the l1 ball, len < 2 for the cone. */
enum { PIMPC_SET_NONE = 0, PIMPC_SET_HALFSPACE = 1, PIMPC_SET_HYPERPLANE = 2, PIMPC_SET_SOC = 3, PIMPC_SET_L1BALL = 4 };
int pimpc_set_constraint(pimpc_t h, int kind, int i0, int len, const void *a, double b);

/* x0 [batch][nx] = x(t); u_prev [batch][nu] = u(t-1) or NULL (= 0)  (xbar_0, R10). */
int pimpc_set_x0(pimpc_t h, const void *x0, const void *u_prev);

/* One invocation of Algorithm 1 per instance from the current iterates (hats = iterates,
 * alpha_0 = 1, c^0 = c0): recomputes the cache {M_k, H_k} if stage
 * data, cost or rho changed, then runs up to max_iters iterations; an instance stops early when
 * c^{i+1} < tol (step 5); tol <= 0 runs exactly max_iters.  Asynchronous on the
 * handle's stream; errors detected on the device (non-finite input, matrix not positive definite)
 * are reported by the next pimpc_get / pimpc_sync.  max_iters == 0 only refreshes the cache. */
int pimpc_solve(pimpc_t h, int max_iters, double tol);

/* Results of the last solve (synchronises the stream).  Any pointer may be NULL.
 * x [batch][N][nx] = x_1..x_N and u [batch][N][nu] = u_0..u_{N-1} are read from Z (bound-feasible);
 * du [batch][N][nu] = Delta u_0..; res [batch] pimpc_result. */
int pimpc_get(pimpc_t h, void *x, void *u, void *du, pimpc_result *res);

/* Raw iterates, [batch][N][nx+nu] (X,Z,V,TH,BE,LA) or [batch][N][nu] (D,DE,DU), for parity checks and
 * warm starts.  get synchronises.  set replaces one array of the current iterate
 * (X and DU are outputs only: EINVAL). */
int pimpc_get_state(pimpc_t h, int which, void *out);
int pimpc_set_state(pimpc_t h, int which, const void *in);

/* History of the last solve: c [batch][cap] (double), accepted [batch][cap] (unsigned char),
 * cap = opts.history; entries beyond an instance's `iters` are 0.  Synchronises. */
int pimpc_get_history(pimpc_t h, double *c, unsigned char *accepted);

/* The cache of the last solve, for parity checks: M [batch][N][nu][nu], H [batch][N][nb][nb]. */
int pimpc_get_cache(pimpc_t h, void *M, void *H);

/* Cold start: all iterates = 0 (R9). */
int pimpc_reset(pimpc_t h);

/* Receding-horizon warm start (Alg. 1 takes its initial iterates "such as from warm-start" and returns them for the
 * next MPC step; reading R18): the current iterate of every instance is shifted by `steps` stages,
 * stage k takes the values of stage k + steps (Z, V, TH, BE, LA, D, DE); the last `steps` stages repeat the old last
 * stage.  0 <= steps < N, else EINVAL.  Asynchronous on the handle's stream.  X and DU (outputs of the last
 * iteration) are not touched. */
int pimpc_shift(pimpc_t h, int steps);

/* Wait for the handle's stream; returns a deferred device-side error if one was raised. */
int pimpc_sync(pimpc_t h);

/* Launch shape, launch counts and device timings of the last solve.  Synchronises the stream if a
 * solve is pending (the timings come from CUDA events recorded around the kernels). */
int pimpc_get_info(pimpc_t h, pimpc_info *info);
const char *pimpc_last_error(pimpc_t h);

/* ---- allocation-free entry point ----------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (stream capture, tight serving loops, harnesses that forbid it).
 * r_prim2[b] = rho ||F p + G q - h||^2 of an iterate the caller holds: the primal-residual half of c^{i+1}
 * (the consensus constraints of Problem (11)), the same definition, accumulation
 * type (double) and chunking as pimpc_result.r_prim2 of pimpc_get, without a handle.  No cudaMalloc / cudaFree / allocating
 * library call, no host synchronisation: two kernel launches on `stream` (a cudaStream_t of the CURRENT device, NULL =
 * default stream).
 *
 * Every pointer is a DEVICE pointer to a dense array of element type `dtype` (PIMPC_F64 | PIMPC_F32); r_prim2 is
 * double[batch] in device memory whatever the dtype.  Inputs are only read; the caller owns everything.
 *   A [batch][N][nx][nx], B [batch][N][nx][nu], e [batch][N][nx] or NULL (= 0)           stage data
 *   x0 [batch][nx], u_prev [batch][nu] or NULL (= 0)                                     xbar_0
 *   X, Z, V [batch][N][nx+nu], DU [batch][N][nu], D [batch][N][nu] or NULL (no Delta-u box)
 *                                                  the layouts pimpc_get_state(PIMPC_X / _Z / _V / _DU / _D) returns
 * The per-CTA partial sums live in a file-scope __device__ array of PIMPC_NOALLOC_MAX_PARTS doubles (256 KiB, held by
 * every GPU that loads the library until the process exits).  Limit: batch <= PIMPC_NOALLOC_MAX_PARTS (an instance
 * gets min(64, N (nx+nu) / 2048, PIMPC_NOALLOC_MAX_PARTS / batch) >= 1 partials); beyond it, or with a bad dtype /
 * shape / NULL required pointer: PIMPC_EINVAL, nothing launched.  PIMPC_ECUDA: the scratch address could not be
 * resolved or a launch failed.  pimpc_noalloc_last_error() returns the message of the calling thread's last failure.
 * ALL calls on a device share the array: calls that may overlap on the GPU (different streams, other host threads)
 * race and give wrong sums -- order them on one stream or with events.  The array keeps the previous call's contents;
 * nothing in it has to start at zero (every partial a call reads was written by that call's first kernel). */
#define PIMPC_NOALLOC_MAX_PARTS 32768
int pimpc_rprim2_noalloc(int dtype, int nx, int nu, int N, int batch, const void *A, const void *B, const void *e,
                         const void *x0, const void *u_prev, const void *X, const void *DU, const void *Z, const void *V,
                         const void *D, double rho, double *r_prim2, void *stream);
const char *pimpc_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PIMPC_H */
