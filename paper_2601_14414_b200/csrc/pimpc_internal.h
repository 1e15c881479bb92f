// Internal declarations of libpimpc.so (not part of the ABI; see include/pimpc.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/pimpc.h"

constexpr int PIMPC_MAX_NB = 160;        // nx + nu ceiling (the generic cache kernel keeps an nb x nb double matrix in shared memory)

// Per-instance control block of Algorithm 1 (device memory, one per instance).
// alpha, c_prev: state of the accept/restart test; kappa = (alpha_i-1)/alpha_{i+1}
// is the momentum used to form the hats of the NEXT iteration from (cur, prev).
// i_prev/i_cur/i_new: which of the three rotating state buffers hold the previous iterate, the
// current iterate and the one being written.  After a solve i_cur holds the returned iterate.
struct InstCtl {
    double alpha, c_prev, c_last, kappa;
    int i_prev, i_cur, i_new;
    int done, iters, restarts;
    int pad_[2];
};
static_assert(sizeof(InstCtl) == 64, "InstCtl must be 64 bytes");

// Device error flag bits (raised by kernels, reported by pimpc_sync / pimpc_get).
enum { PIMPC_DEVERR_NONFINITE = 1, PIMPC_DEVERR_NOTPD = 2 };

// Geometry and pointers handed to every kernel by value.  T = float or double.
// State record of one (instance, stage): [Z(nb) V(nb) TH(nb) BE(nb) LA(nb) D(nu) DE(nu) pad] = rec elements.
template <typename T>
struct Prob {
    int nx, nu, nb, N, batch, rec;
    int has_du, has_e, has_q;        // has_q: a linear cost term qbar was supplied
    const T *A, *B, *e;              // [batch][N][nx][nx], [batch][N][nx][nu], [batch][N][nx] or null
    const T *x0, *uprev;             // [batch][nx], [batch][nu]
    const T *Q, *R, *P, *Wdu, *qbar; // cost; P, Wdu may be null; stride 0 = shared by all instances
    int cost_stride_q, cost_stride_r, qbar_stride;
    const T *lo, *hi, *dlo, *dhi;    // bounds; strides 0 = shared
    int bnd_stride, dbnd_stride;
    // per-stage boxes / linear terms (pimpc_set_stage_terms, pimpc_set_tracking with per-stage references) or null;
    // element (b, k, i) at [b * *_bstride + k * nb + i]
    const T *lo_k, *hi_k, *qbar_k;
    size_t lok_bstride, qbk_bstride;
    // general convex set on the components [set_i0, set_i0 + set_len) of z (pimpc_set_constraint); set_kind = PIMPC_SET_*
    int set_kind, set_i0, set_len;
    const T *set_a;                  // [set_len] normal vector (halfspace, hyperplane)
    double set_b, set_inv_aa;        // offset / radius; 1 / ||a||^2
    T *H, *M;                        // cache: [batch][N][nb][nb] (symmetric), [batch][N][nu][nu]
    T *S;                            // 3 rotating buffers of [batch][N][rec]
    size_t buf_stride;               // elements between buffers
    T *X, *DU;                       // [batch][N][nb], [batch][N][nu]
    InstCtl *ctl;                    // [batch]
    double *partial;                 // [batch][nparts] partial sums of c (before the factor rho)
    int nparts;
    double *hist_c;                  // [batch][hist_cap] or null
    unsigned char *hist_a;
    int hist_cap;
    int *err;                        // device error flag
    double rho, eta, tol, c0;

    __host__ __device__ size_t st(int b, int k) const { return ((size_t)b * N + k) * rec; }
    __host__ __device__ int oZ() const { return 0; }
    __host__ __device__ int oV() const { return nb; }
    __host__ __device__ int oTH() const { return 2 * nb; }
    __host__ __device__ int oBE() const { return 3 * nb; }
    __host__ __device__ int oLA() const { return 4 * nb; }
    __host__ __device__ int oD() const { return 5 * nb; }
    __host__ __device__ int oDE() const { return 5 * nb + nu; }
    // box and linear term of row i of stage k of instance b
    __device__ T lo_at(int b, int k, int i) const { return lo_k ? lo_k[(size_t)b * lok_bstride + (size_t)k * nb + i] : lo[(size_t)b * bnd_stride + i]; }
    __device__ T hi_at(int b, int k, int i) const { return hi_k ? hi_k[(size_t)b * lok_bstride + (size_t)k * nb + i] : hi[(size_t)b * bnd_stride + i]; }
    __device__ T qbar_at(int b, int k, int i) const { return qbar_k ? qbar_k[(size_t)b * qbk_bstride + (size_t)k * nb + i] : qbar[(size_t)b * qbar_stride + i]; }
};

// Projection of the candidate vector t[0..len) (shared or global memory, read by every calling thread) onto the general
// set of the handle (closed forms of [22, Ch. 6]): returns component j of the projection.  Every thread
// evaluates the few scalars the closed form needs redundantly, in the same fixed order (deterministic, no atomics).
template <typename T>
__device__ inline T proj_set_component(const Prob<T> &p, const T *t, int j)
{
    const int n = p.set_len;
    const T tj = t[j];
    if (p.set_kind == PIMPC_SET_HALFSPACE || p.set_kind == PIMPC_SET_HYPERPLANE) {
        T at = (T)0;
        for (int i = 0; i < n; ++i) at += p.set_a[i] * t[i];
        T s = (at - (T)p.set_b) * (T)p.set_inv_aa;
        if (p.set_kind == PIMPC_SET_HALFSPACE && !(at > (T)p.set_b)) s = (T)0;
        return tj - s * p.set_a[j];
    }
    if (p.set_kind == PIMPC_SET_SOC) {                     // (x, r): inside -> t; ||x|| <= -r -> 0; else ((||x|| + r)/2)(x/||x||, 1)
        T n2 = (T)0;
        for (int i = 0; i < n - 1; ++i) n2 += t[i] * t[i];
        const T nx_ = sqrt(n2), r = t[n - 1];
        if (nx_ <= r) return tj;
        if (nx_ <= -r) return (T)0;
        const T s = (T)0.5 * (nx_ + r);
        return j == n - 1 ? s : s * tj / nx_;
    }
    if (p.set_kind == PIMPC_SET_L1BALL) {                  // soft threshold with tau = max_m (sum of the m largest |t| - r) / m
        T l1 = (T)0;
        for (int i = 0; i < n; ++i) l1 += fabs(t[i]);
        if (l1 <= (T)p.set_b) return tj;
        T tau = (T)0;
        for (int m = 0; m < n; ++m) {                      // candidate: the elements not smaller than |t_m|
            const T um = fabs(t[m]);
            T sum = (T)0; int cnt = 0;
            for (int i = 0; i < n; ++i) { const T ui = fabs(t[i]); if (ui >= um) { sum += ui; ++cnt; } }
            const T cand = (sum - (T)p.set_b) / (T)cnt;
            tau = cand > tau ? cand : tau;
        }
        const T mag = fabs(tj) - tau;
        return mag > (T)0 ? (tj > (T)0 ? mag : -mag) : (T)0;
    }
    return tj;
}

struct pimpc_s {
    int nx = 0, nu = 0, nb = 0, N = 0, batch = 0, rec = 0;
    int dtype = PIMPC_F64;
    size_t esz = 8;
    int engine_req = PIMPC_ENGINE_AUTO;
    double rho = 1.0, eta = 0.999, c0 = 1.0;
    int hist_cap = 0;
    cudaStream_t stream = nullptr;
    pimpc_tune tune{};                       // launch-shape overrides (opts.tune), all 0 = automatic
    unsigned char *ws = nullptr;             // caller-provided workspace (opts.workspace) or null
    size_t ws_bytes = 0, ws_used = 0;
    int device = 0, sm_count = 0;
    size_t smem_optin = 0;

    // device buffers (element type = dtype unless noted)
    void *A = nullptr, *B = nullptr, *e = nullptr, *x0 = nullptr, *uprev = nullptr;
    void *Q = nullptr, *R = nullptr, *P = nullptr, *Wdu = nullptr, *qbar = nullptr;
    int cost_per_instance = 0;
    void *lo = nullptr, *hi = nullptr, *dlo = nullptr, *dhi = nullptr;
    int bnd_per_instance = 0;
    int has_du = 0, has_e = 0, has_P = 0, has_wdu = 0, has_q = 0;
    void *lo_k = nullptr, *hi_k = nullptr, *qbar_k = nullptr;   // per-stage boxes / linear terms, [batch or 1][N][nb]
    size_t lok_cap = 0, hik_cap = 0, qbk_cap = 0;               // allocated bytes
    int has_lok = 0, has_qbk = 0, lok_per_instance = 0, qbk_per_instance = 0;
    int set_kind = 0, set_i0 = 0, set_len = 0;                  // general convex set (pimpc_set_constraint)
    void *set_a = nullptr;
    size_t set_a_cap = 0;
    double set_b = 0.0, set_inv_aa = 0.0;
    void *trk = nullptr;                                        // staging of pimpc_set_tracking's inputs
    size_t trk_cap = 0;
    void *H = nullptr, *M = nullptr, *S = nullptr, *X = nullptr, *DU = nullptr;
    InstCtl *ctl = nullptr;
    double *partial = nullptr;
    size_t partial_cap = 0;                  // bytes
    double *hist_c = nullptr;
    unsigned char *hist_a = nullptr;
    int *err = nullptr;
    // scratch of the STAGED engine (allocated on first use)
    void *hat = nullptr, *W = nullptr, *G = nullptr, *rhs = nullptr;
    // alpha_j / kappa_j tables of the fused engines (j consecutive accepted steps), [tab_cap] doubles
    double *alpha_tab = nullptr, *kappa_tab = nullptr;
    int tab_cap = 0;
    // engine-private storage (packed blobs of the STREAM engine etc.)
    void *blob = nullptr;
    size_t blob_bytes = 0;
    double *spartial = nullptr;              // [2][batch][span] partial sums of c of the STREAM engine
    size_t spartial_cap = 0;                 // bytes
    bool blob_dirty = true;
    void *stage_buf = nullptr;               // device staging of results bound for host memory (grown on demand, kept)
    size_t stage_bytes = 0;
    void *coop_buf = nullptr;                // tagged exchange words of the COOP engine (partials of c, boundary iterates)
    size_t coop_bytes = 0;

    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};   // before cache kernel, before iteration, after iteration
    bool ev_pending = false, ev_setup = false;

    bool cache_dirty = true;                 // every stage of the cache {M_k, H_k} must be recomputed
    std::vector<int> dirty_stages;           // else: flattened (b * N + k) cache entries touched by pimpc_set_stage
    double *res_part = nullptr;              // partial sums of r_prim2 (k_rprim), [batch][chunks]
    size_t res_part_cap = 0;
    int *dirty_dev = nullptr;                // device copy of dirty_stages
    size_t dirty_cap = 0;
    size_t device_bytes = 0;
    pimpc_info info{};
    std::string errmsg;
    int poisoned = 0;
};

// ---- kernels / engine entry points (each returns the number of kernels it launched, <0 on error) ----
template <typename T> Prob<T> make_prob(pimpc_s *h, double tol);

int launch_setup(pimpc_s *h, const int *list_dev, int nlist);   // a0: cache {M_k, H_k} of every stage (list_dev = null) or of the listed ones
int launch_begin(pimpc_s *h);                       // Alg. 1 input: alpha=1, c_prev=c0, hats=iterates
int run_staged(pimpc_s *h, int iters, double tol);  // v0 engine
int run_resident(pimpc_s *h, int iters, double tol);
bool resident_supported(const pimpc_s *h, std::string *why);
bool resident2_plan(const pimpc_s *h, int *nxp, int *nup, int *maxn);   // padded shape of the two-rows-per-lane kernel
int run_resident2(pimpc_s *h, int iters, double tol);
int ensure_alpha_table(pimpc_s *h, int iters);     // alpha_j / kappa_j tables cover `iters` accepted steps; returns launches
int run_coop(pimpc_s *h, int iters, double tol);
bool coop_supported(const pimpc_s *h, std::string *why);
int run_stream(pimpc_s *h, int iters, double tol);
bool stream_supported(const pimpc_s *h, std::string *why);
int launch_gather(pimpc_s *h, void *x, void *u, void *du, pimpc_result *res_dev);
int launch_state_io(pimpc_s *h, int which, void *buf_dev, int set);
int launch_zero_state(pimpc_s *h);
int launch_shift(pimpc_s *h, int steps);              // warm-start shift of the current iterate (reading R18)
// Q = C'W_y C, R = W_u, qbar[k] = (C'W_y r_y[k]; W_u r_u[k]) from the staged inputs (device, element type of the handle)
int launch_tracking(pimpc_s *h, int ny, const void *C, const void *Wy, const void *Wu, const void *ry, const void *ru,
                    int nref, void *qbar_out);
inline bool has_stage_terms(const pimpc_s *h);

inline bool has_stage_terms(const pimpc_s *h) { return h->has_lok || h->has_qbk || h->set_kind != 0; }

// (Re)allocate an engine-private device buffer of at least `bytes` (kept if large enough); accounts device_bytes; a failed
// cudaMalloc returns PIMPC_ENOMEM without poisoning the handle.
int pimpc_grow(pimpc_s *h, void **ptr, size_t *cap, size_t bytes);

#define PIMPC_CUDA_TRY(h, expr)                                                         \
    do {                                                                                \
        cudaError_t err__ = (expr);                                                     \
        if (err__ != cudaSuccess) {                                                     \
            (h)->errmsg = std::string(#expr) + ": " + cudaGetErrorString(err__);        \
            (h)->poisoned = 1;                                                          \
            return PIMPC_ECUDA;                                                         \
        }                                                                               \
    } while (0)
