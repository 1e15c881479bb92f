// STREAM engine: Algorithm 1 for problems whose stage data does not fit on chip
// (C5: nx=48, nu=12, N=2000, batch 64: 6 GB of stage matrices).  ONE cooperative launch per solve;
// persistent CTAs each own a contiguous range of (instance, stage) pairs and, every iteration,
// stream one packed blob per stage HBM -> shared memory with bulk asynchronous copies (TMA 1-D,
// cp.async.bulk + mbarrier ring), so HBM sees exactly the algorithmic bytes:
//   blob'_j = { H_j (symmetric, stored once: lower triangle of 4 x 4 blocks if nb % 4 == 0, else circulant order),
//               [A_{j+1} B_{j+1}], M_{j+1}, e_{j+1} }
//   + the (current, previous) iterate records of stage j+1 in, the new record of stage j out.
// The regrouping (H of stage j with A, B, M of stage j+1) makes every step need ONE blob:
//   step j:  g = Abar_{j+1}^T w_{j+1},  rhs/du/av of stage j+1          (Alg. 1 step 1)
//            xbar_{j+1} = H_j h_j                                       (step 1)
//            b_{j+1} = Abar_{j+1} xbar_{j+1} + ebar - lambdahat          (first half of step 2)
//            z, v, theta, beta, lambda, d, delta of stage j + its part of c   (steps 2-4)
// with b_j, av_j, du_j carried from step j-1.  A range that starts inside an instance recomputes the
// primal step of the stage before it (halo), so there is no intra-iteration exchange between CTAs.
// One grid barrier per iteration: partial sums of c -> every CTA takes the accept / restart decision
// (steps 5-7) of its instances from bit-identical numbers (fixed summation order).
// Hats (steps 6/7) are never stored: recomputed from (cur, prev, kappa) when a record arrives.
#include <cooperative_groups.h>

#include <algorithm>

#include "pimpc_internal.h"

namespace cg = cooperative_groups;

namespace {

constexpr int pow2ceil_s(int v) { int p = 1; while (p < v) p <<= 1; return p; }
constexpr int round4(int v) { return (v + 3) / 4 * 4; }

template <typename T, int NX, int NU>
struct SCfg {
    static constexpr int NB = NX + NU;
    static constexpr int NS = NB / 2 + 1;                 // circulant rows s = 0..NB/2:  C[s][i] = H[i][(i+s) % NB]
    // NB % 4 == 0: the symmetric H_j is stored as its lower triangle of 4 x 4 blocks instead (block t = I(I+1)/2 + J, J <= I;
    // row a of block t at [a][t][0..3] (fp64: [a][half][t][0..1]), so consecutive lanes read consecutive 16-byte words): one thread multiplies a block
    // and its transpose from registers -- 6 16-byte loads per 32 FMAs where the circulant order needs 64 4-byte loads
    static constexpr bool BLKH = NB % 4 == 0;
    static constexpr int NBK = NB / 4, NBLK = NBK * (NBK + 1) / 2;
    static constexpr int OC = 0, OAB = BLKH ? 16 * NBLK : NS * NB, OM = OAB + NX * NB, OE = OM + NU * NU;
    static constexpr int BLOB = round4(OE + NX);          // elements per blob'
    static constexpr int REC = round4(5 * NB + 2 * NU);   // iterate record (same as Prob<T>::rec)
    static constexpr int SLOT = BLOB + 2 * REC;           // ring slot: blob', cur record, prev record
    static constexpr int IP = pow2ceil_s(NB);             // padded column index
    static constexpr int NT = (4 * NX + IP + 31) / 32 * 32;   // threads: 4 per x-row (row products) + one per component (dual)
    static constexpr int NPART = NT / IP;                 // column-products are split into NPART row ranges
    static constexpr int NW = NT / 32;
    static constexpr int MAXI = 16;                       // instances a CTA's range may touch
    // the thread that issues the bulk copies: lane 0 of a warp with no work in phases A, C and E (the refill of a slot then
    // overlaps phase A of the next step instead of preceding it on warp 0)
    static constexpr int PROD = NT >= 128 ? 96 : (NT >= 64 ? 32 : 0);
    static_assert(PROD == 0 || PROD >= NB, "the producer's warp has no hats to form");
    // register budget: 64 per thread in fp32 (1024 resident threads: 4 CTAs of 256), 128 in fp64 (512 threads: shared memory
    // holds 2 CTAs of the wide shapes anyway).  Without a bound ptxas picks what it likes (124 registers once in fp32: -27 %)
    static constexpr int MINB = (sizeof(T) == 4 ? 1024 : 512) / NT > 2 ? (sizeof(T) == 4 ? 1024 : 512) / NT : 2;
    static_assert(NT >= 4 * NX + NB && NPART >= 1 && IP + NU <= NT, "thread mapping");
    static_assert(!BLKH || (NBLK <= NT - 32 && NU <= 32), "one thread per 4 x 4 block of H, the last warp for M rhs");
    // fixed shared-memory vectors (elements of T)
    static constexpr int V_HAT = 0;                       // [2][REC] hats of stages j, j+1 (ping-pong on stage parity)
    static constexpr int V_W = V_HAT + 2 * REC;           // [IP] w_{j+1}
    static constexpr int V_D = V_W + IP;                  // [IP] vhat - betahat of stage j+1
    static constexpr int V_H = V_D + IP;                  // [2 NB] h_j twice (circulant wrap)
    static constexpr int V_GP = V_H + 2 * NB;             // [NPART][IP] partial Abar^T w
    static constexpr int V_RP = V_GP + NPART * IP;        // [NPART][IP] partial Bbar^T d (u columns)
    static constexpr int V_XP = V_RP + NPART * IP;        // [NPART][IP] partial H h; BLKH: [NBK][NB] from V_GP on (gp, rp are dead by then)
    static constexpr int XP_LEN = BLKH && NBK * NB > 3 * NPART * IP ? NBK * NB - 2 * NPART * IP : NPART * IP;
    static constexpr int V_X = V_XP + XP_LEN;         // [IP] xbar_{j+1}
    static constexpr int V_RHS = V_X + IP;                // [IP] rhs of the Delta-u update
    static constexpr int V_DU = V_RHS + IP;               // [2][IP] Delta u carry
    static constexpr int V_B = V_DU + 2 * IP;             // [2][IP] b carry
    static constexpr int V_AV = V_B + 2 * IP;             // [2][IP] a carry
    static constexpr int V_END = round4(V_AV + 2 * IP);
};

// CTA-local copy of the control state of one instance (see InstCtl)
struct LInst {
    double alpha, c_prev, c_last;
    float kappa_f; int pad0;
    double kappa;
    int b, i_prev, i_cur, i_new, done, iters, restarts, owner;
    int c_lo, c_hi;                                        // first / last CTA whose range holds a dual step of the instance
};

struct Seg { int b, j0, nsteps, pstep, halo; };   // steps j0..: optional P step (state of stage j0 only), then S steps

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk asynchronous copy global -> shared (TMA), completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

template <typename T> __device__ __forceinline__ T clips(T v, T lo, T hi) { return fmin(fmax(v, lo), hi); }
__device__ __forceinline__ void ld4s(const float *p, float (&o)[4])
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ld4s(const double *p, double (&o)[4])
{
    const double2 a = *reinterpret_cast<const double2 *>(p), b = *reinterpret_cast<const double2 *>(p + 2);
    o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}

// row a of 4 x 4 block t of H (see SCfg::BLKH): consecutive lanes read consecutive 16-byte words in either precision
__device__ __forceinline__ void ldblk(const float *Cb, int a, int nblk, int t, float (&o)[4]) { ld4s(Cb + (a * nblk + t) * 4, o); }
__device__ __forceinline__ void ldblk(const double *Cb, int a, int nblk, int t, double (&o)[4])
{
    const double2 lo = *reinterpret_cast<const double2 *>(Cb + ((2 * a) * nblk + t) * 2);
    const double2 hi = *reinterpret_cast<const double2 *>(Cb + ((2 * a + 1) * nblk + t) * 2);
    o[0] = lo.x; o[1] = lo.y; o[2] = hi.x; o[3] = hi.y;
}
__device__ __forceinline__ void st4s(float *p, const float (&v)[4]) { *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], v[3]); }
__device__ __forceinline__ void st4s(double *p, const double (&v)[4])
{
    *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[1]); *reinterpret_cast<double2 *>(p + 2) = make_double2(v[2], v[3]);
}

// ---- pack: blob'_j of every (instance, j = -1..N-1), once per solve after the cache kernel ----------
template <typename T, int NX, int NU>
__global__ void __launch_bounds__(128) k_pack(const Prob<T> p, T *__restrict__ blob)
{
    using C = SCfg<T, NX, NU>;
    constexpr int NB = C::NB;
    const int j = (int)blockIdx.x - 1, b = blockIdx.y, N = p.N;
    T *out = blob + ((size_t)b * (N + 1) + (j + 1)) * C::BLOB;
    const bool hasH = j >= 0, hasN = j + 1 <= N - 1;
    const size_t sj = (size_t)b * N + (hasH ? j : 0), sn = (size_t)b * N + (hasN ? j + 1 : 0);
    // the caller's shape nx <= NX, nu <= NU sits inside the instantiated one: pad rows and columns are zero (and stay zero)
    const int nx = p.nx, nu = p.nu, nb = p.nb;
    auto gix = [&](int i) -> int { return i < NX ? (i < nx ? i : -1) : (i - NX < nu ? nx + (i - NX) : -1); };
    const T *H = p.H + sj * nb * nb, *A = p.A + sn * nx * nx, *B = p.B + sn * nx * nu, *M = p.M + sn * nu * nu;
    for (int idx = threadIdx.x; idx < C::BLOB; idx += blockDim.x) {
        T v = (T)0;
        if (idx < C::OAB) {
            int i, c;
            if constexpr (C::BLKH) {
                // 16-byte words of consecutive blocks are adjacent: [a][t][0..3] in fp32, [a][half][t][0..1] in fp64
                constexpr int EW = 16 / (int)sizeof(T), HW = 4 / EW;          // elements per word, words per block row
                const int wq = idx / EW, t = wq % C::NBLK, ah = wq / C::NBLK;
                const int a = ah / HW, bq = (ah % HW) * EW + idx % EW;
                int I = 0; while ((I + 1) * (I + 2) / 2 <= t) ++I;
                i = 4 * I + a; c = 4 * (t - I * (I + 1) / 2) + bq;
            } else {
                const int s = idx / NB;
                i = idx - s * NB;
                c = i + s; if (c >= NB) c -= NB;
            }
            const int gi = gix(i), gc = gix(c);
            if (hasH && gi >= 0 && gc >= 0) v = H[gi * nb + gc];
        } else if (idx < C::OM) {
            const int q = idx - C::OAB, r = q / NB, c = q - r * NB;
            if (hasN && r < nx) { if (c < NX) { if (c < nx) v = A[r * nx + c]; } else if (c - NX < nu) v = B[r * nu + (c - NX)]; }
        } else if (idx < C::OE) {
            const int q = idx - C::OM, r = q / NU, c = q - r * NU;
            if (hasN && r < nu && c < nu) v = M[r * nu + c];
        } else if (idx < C::OE + NX) {
            if (hasN && p.e && idx - C::OE < nx) v = p.e[sn * nx + (idx - C::OE)];
        }
        out[idx] = v;
    }
}

struct StreamSmem {
    static constexpr int MAXSLOT = 16;
    uint64_t bar[MAXSLOT];
    LInst inst[16];
    Seg seg[16];
    double red[32];
    int nseg, total, pad_[2];
};

struct Cursor {
    int sg, o;
    __device__ void next(const Seg *seg) { if (++o >= seg[sg].nsteps) { o = 0; ++sg; } }
};

// EXT: per-stage boxes / linear terms or a general convex set are present (pimpc_set_stage_terms, pimpc_set_tracking with
// per-stage references, pimpc_set_constraint); the plain variant carries none of their address arithmetic or barriers.
// PAD: the caller's shape nx <= NX, nu <= NU runs INSIDE this instantiation: blobs and the on-chip vectors are padded (pad
// rows / columns zero, zero boxes, zero iterates: they run the same instructions and stay exactly zero), the records and the
// caller's vectors in HBM keep the real shape and are indexed through gix().  The exact shapes compile without any of it.
template <typename T, int NX, int NU, bool EXT, bool PAD>
__global__ void __launch_bounds__(SCfg<T, NX, NU>::NT, SCfg<T, NX, NU>::MINB)
k_stream(const Prob<T> p, const T *__restrict__ blob, double *__restrict__ partial, const int iters, const int nslot, const int span)
{
    using C = SCfg<T, NX, NU>;
    constexpr int NB = C::NB, IP = C::IP, NPART = C::NPART, REC = C::REC, BLOB = C::BLOB, SLOT = C::SLOT;
    constexpr int RP = (NX + NPART - 1) / NPART;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    StreamSmem &sm = *reinterpret_cast<StreamSmem *>(smem_raw);
    T *vec = reinterpret_cast<T *>(smem_raw + ((sizeof(StreamSmem) + 127) / 128) * 128);
    T *ring = vec + C::V_END;
    T *hat = vec + C::V_HAT, *wv = vec + C::V_W, *dv = vec + C::V_D, *gp = vec + C::V_GP, *rp = vec + C::V_RP;
    T *hv = vec + C::V_H, *xp = vec + (C::BLKH ? C::V_GP : C::V_XP), *xv = vec + C::V_X, *rhs = vec + C::V_RHS, *duc = vec + C::V_DU;
    T *bc = vec + C::V_B, *avc = vec + C::V_AV;

    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = p.N, N1 = N + 1;
    const long long S_tot = (long long)p.batch * N1, G = gridDim.x, cta = blockIdx.x;
    const long long s0 = cta * S_tot / G, s1 = (cta + 1) * S_tot / G;
    const int b_first = (int)(s0 / N1), n_local = (int)((s1 - 1) / N1) - b_first + 1;
    const T rho = (T)p.rho;
    const bool has_du = p.has_du != 0, has_q = p.has_q != 0, gset = EXT && p.set_kind != PIMPC_SET_NONE;
    const int ci = tid % IP, prt = tid / IP;              // column index / row-range part of the column products
    const int di = tid - 4 * NX;                           // component of the dual update (threads >= 4 NX)
    static_assert(!(EXT && PAD), "padded shapes run the plain variant only");
    int bI = 0;                                            // BLKH: this thread's 4 x 4 block (bI, bJ) of the lower triangle of H
    if (C::BLKH && tid < C::NBLK) while ((bI + 1) * (bI + 2) / 2 <= tid) ++bI;
    const int bJ = tid - bI * (bI + 1) / 2;
    const int rnx = PAD ? p.nx : NX, rnu = PAD ? p.nu : NU, rnb = rnx + rnu, rrec = PAD ? p.rec : REC;    // the shape in HBM
    auto gix = [&](int i) -> int { return !PAD ? i : (i < NX ? (i < rnx ? i : -1) : (i - NX < rnu ? rnx + (i - NX) : -1)); };

    if (tid == 0) {
        for (int s = 0; s < nslot; ++s) mbar_init(&sm.bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < n_local) {
        const int b = b_first + tid;
        const InstCtl c = p.ctl[b];
        LInst &L = sm.inst[tid];
        L.alpha = c.alpha; L.c_prev = c.c_prev; L.c_last = c.c_last; L.kappa = 0.0; L.kappa_f = 0.f;
        L.b = b; L.i_prev = c.i_prev; L.i_cur = c.i_cur; L.i_new = c.i_new; L.done = c.done; L.iters = 0; L.restarts = 0;
        const long long first = (long long)b * N1;
        L.owner = first >= s0 && first < s1;
        L.c_lo = (int)(((first + 1) * G - 1) / S_tot); L.c_hi = (int)(((first + N1) * G - 1) / S_tot);
    }
    __syncthreads();
    uint32_t phase = 0;                                    // parity bit per ring slot

    for (int it = 0; it < iters; ++it) {
        const bool write_x = p.tol > 0.0 || it == iters - 1;
        // ---- this iteration's steps: one segment per active instance of the range ---------------------
        if (tid == 0) {
            int ns = 0, total = 0;
            for (int li = 0; li < n_local; ++li) {
                if (sm.inst[li].done) continue;
                const long long base = (long long)(b_first + li) * N1;
                const long long lo = s0 > base ? s0 : base, hi = s1 < base + N1 ? s1 : base + N1;
                const int jlo = (int)(lo - base) - 1, jhi = (int)(hi - base) - 1;     // steps with a dual update: jlo..jhi-1
                Seg sgm;
                sgm.b = li;
                sgm.halo = jlo >= 0;                       // range starts inside the instance: recompute step jlo-1
                sgm.j0 = sgm.halo ? jlo - 1 : -1;
                sgm.pstep = sgm.j0 >= 0;                   // the halo step needs the hats of its own stage first
                sgm.nsteps = (jhi - sgm.j0) + sgm.pstep;
                sm.seg[ns++] = sgm;
                total += sgm.nsteps;
            }
            sm.nseg = ns; sm.total = total;
        }
        __syncthreads();
        const int total = sm.total;

        // producer: thread PROD issues the bulk copies of step n into slot n % nslot
        auto issue = [&](const Cursor &cu, int slot) {
            const Seg sg = sm.seg[cu.sg];
            const LInst &L = sm.inst[sg.b];
            const bool isP = sg.pstep && cu.o == 0;
            const int j = isP ? sg.j0 : sg.j0 + cu.o - sg.pstep;
            T *dst = ring + (size_t)slot * SLOT;
            const int ks = isP ? j : j + 1;                // stage whose records are loaded
            const bool rec_ok = ks <= N - 1;
            const uint32_t bytes = (isP ? 0u : (uint32_t)(BLOB * sizeof(T))) + (rec_ok ? 2u * (uint32_t)rrec * sizeof(T) : 0u);
            mbar_expect_tx(&sm.bar[slot], bytes);
            if (!isP) bulk_g2s(dst, blob + ((size_t)L.b * N1 + (j + 1)) * BLOB, BLOB * sizeof(T), &sm.bar[slot]);
            if (rec_ok) {
                const size_t off = p.st(L.b, ks);
                bulk_g2s(dst + BLOB, p.S + (size_t)L.i_cur * p.buf_stride + off, rrec * sizeof(T), &sm.bar[slot]);
                bulk_g2s(dst + BLOB + REC, p.S + (size_t)L.i_prev * p.buf_stride + off, rrec * sizeof(T), &sm.bar[slot]);
            }
        };
        Cursor pc{0, 0}, cc{0, 0};
        int issued = 0;
        if (tid == C::PROD)
            for (; issued < nslot && issued < total; ++issued) { issue(pc, issued); pc.next(sm.seg); }

        double acc = 0.0;                                  // this thread's part of sum ||.||^2 of the current segment
        int slot = 0;
        // per-segment state, reloaded when a segment starts (uniform branch): the segment record, the instance, its momentum
        // and -- plain variant -- this thread's bounds and linear term, which are the same for every stage of the instance
        Seg sg = sm.seg[0];
        int li = 0, b = 0;
        T kap = (T)0, lo_c = (T)0, hi_c = (T)0, dlo_c = (T)0, dhi_c = (T)0, qb_c = (T)0;
        for (int n = 0; n < total; ++n) {
            if (cc.o == 0) {
                sg = sm.seg[cc.sg];
                li = sg.b;
                b = sm.inst[li].b;
                kap = (T)sm.inst[li].kappa;
                if constexpr (!EXT) {
                    if (di >= 0 && di < NB) {
                        const int gi = gix(di);
                        const bool real = !PAD || gi >= 0;
                        lo_c = real ? p.lo[(size_t)b * p.bnd_stride + gi] : (T)0;
                        hi_c = real ? p.hi[(size_t)b * p.bnd_stride + gi] : (T)0;
                        if (has_du && di >= NX) {
                            dlo_c = real ? p.dlo[(size_t)b * p.dbnd_stride + (di - NX)] : (T)0;
                            dhi_c = real ? p.dhi[(size_t)b * p.dbnd_stride + (di - NX)] : (T)0;
                        }
                    }
                    if (has_q && tid < NB) qb_c = (!PAD || gix(tid) >= 0) ? p.qbar[(size_t)b * p.qbar_stride + gix(tid)] : (T)0;
                }
            }
            const LInst &L = sm.inst[li];
            const bool isP = sg.pstep && cc.o == 0;
            const int so = cc.o - sg.pstep;                // index of the S step inside the segment
            const int j = isP ? sg.j0 : sg.j0 + so;
            const bool first = j == -1, has_next = j < N - 1;
            const bool do_dual = !isP && j >= 0 && !(sg.halo && so == 0);
            const bool last_of_seg = cc.o == sg.nsteps - 1;
            const bool do_next = has_next && !last_of_seg;
            const T *sl = ring + (size_t)slot * SLOT;
            const T *Cb = sl + C::OC, *AB = sl + C::OAB, *Mb = sl + C::OM, *Eb = sl + C::OE;
            const T *cu = sl + BLOB, *pv = cu + REC;
            const int ks = isP ? j : j + 1;
            T *hs = hat + (ks & 1) * REC;                  // hats of stage ks
            const T *hj = hat + (j & 1) * REC;             // hats of stage j
            const int pn = (j + 1) & 1, pj = j & 1;        // carry parity of stages j+1, j

            mbar_wait(&sm.bar[slot], (phase >> slot) & 1u);
            phase ^= 1u << slot;

            // ---- A: hats of stage ks from (cur, prev, kappa) (steps 6/7); w, v - beta ----
            if (tid < NB && ks <= N - 1) {
                const int i = tid, gi = gix(i);
                T h5[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    const T a = (!PAD || gi >= 0) ? cu[c * rnb + gi] : (T)0, q = (!PAD || gi >= 0) ? pv[c * rnb + gi] : (T)0;
                    h5[c] = a + kap * (a - q);
                    hs[c * NB + i] = h5[c];
                }
                if (has_du && i < NU) {
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const T a = (!PAD || i < rnu) ? cu[5 * rnb + c * rnu + i] : (T)0, q = (!PAD || i < rnu) ? pv[5 * rnb + c * rnu + i] : (T)0;
                        hs[5 * NB + c * NU + i] = a + kap * (a - q);
                    }
                }
                if (!isP) {
                    T w = h5[0] - h5[1] + h5[4];
                    if (i < NX) w -= Eb[i];
                    wv[i] = w;
                    dv[i] = h5[1] - h5[3];
                }
            }
            __syncthreads();
            if (!isP) {
                // ---- B: column products with [A_{j+1} B_{j+1}]: g = Abar^T w (all columns), Bbar^T (vhat - betahat) (u columns)
                if (has_next && ci < NB) {
                    const int r0 = prt * RP, r1 = r0 + RP < NX ? r0 + RP : NX;
                    T a0 = (T)0, a1 = (T)0;
                    if constexpr (NX % NPART == 0 && RP % 4 == 0) {        // compile-time trip count, 16-byte vector loads
                        const T *ABp = AB + r0 * NB + ci;
                        const bool ucol = ci >= NX;
#pragma unroll
                        for (int rr = 0; rr < RP; rr += 4) {
                            T w4[4], d4[4];
                            ld4s(wv + r0 + rr, w4);
                            ld4s(dv + r0 + rr, d4);
#pragma unroll
                            for (int q = 0; q < 4; ++q) {
                                const T a = ABp[(rr + q) * NB];
                                a0 += a * w4[q];
                                if (ucol) a1 += a * d4[q];
                            }
                        }
                    } else {
                        for (int r = r0; r < r1; ++r) {
                            const T a = AB[r * NB + ci];
                            a0 += a * wv[r];
                            if (ci >= NX) a1 += a * dv[r];
                        }
                    }
                    gp[prt * IP + ci] = a0;
                    if (ci >= NX) rp[prt * IP + ci - NX] = a1;
                }
                __syncthreads();
                // ---- C: h_j (reading R2) and the rhs of the Delta-u update of stage j+1 ----
                if (tid < NB && !first) {
                    const int i = tid;
                    T h = rho * (hj[i] - hj[2 * NB + i]);
                    if (has_next) {
                        T g = (T)0;
#pragma unroll
                        for (int q = 0; q < NPART; ++q) g += gp[q * IP + i];
                        if (i >= NX) g += wv[i];                                    // the [0 I] rows of Abar_{j+1}
                        h += rho * g;
                    }
                    if (has_q) h += EXT ? p.qbar_at(b, j, i) : qb_c;
                    hv[i] = h; hv[i + NB] = h;
                }
                if (tid >= IP && tid < IP + NU && do_next) {
                    const int q = tid - IP;
                    T r = dv[NX + q];
#pragma unroll
                    for (int k2 = 0; k2 < NPART; ++k2) r += rp[k2 * IP + q];
                    if (has_du) r += hs[5 * NB + q] - hs[5 * NB + NU + q];
                    rhs[q] = r;
                }
                __syncthreads();
                // ---- D: xbar_{j+1} = H_j h_j.  BLKH: H stored as the lower triangle of 4 x 4 blocks; the thread of block (I, J)
                // adds B h_J to segment I and B^T h_I to segment J, as partial xp[other block index][component] (each written once;
                // phase E sums them in ascending order: a fixed order that does not depend on the thread mapping); the last warp
                // forms Delta u_{j+1} = M rhs meanwhile.  Else: circulant order C[s][i] = H[i][(i+s) % NB] ----
                if constexpr (C::BLKH) {
                    if (tid < C::NBLK && !first) {
                        T m[4][4], hI[4], hJ[4], y[4];
#pragma unroll
                        for (int a = 0; a < 4; ++a) ldblk(Cb, a, C::NBLK, tid, m[a]);
                        ld4s(hv + 4 * bJ, hJ);
                        ld4s(hv + 4 * bI, hI);
#pragma unroll
                        for (int a = 0; a < 4; ++a) y[a] = ((m[a][0] * hJ[0] + m[a][1] * hJ[1]) + m[a][2] * hJ[2]) + m[a][3] * hJ[3];
                        st4s(xp + bJ * NB + 4 * bI, y);
                        if (bI != bJ) {
#pragma unroll
                            for (int c = 0; c < 4; ++c) y[c] = ((m[0][c] * hI[0] + m[1][c] * hI[1]) + m[2][c] * hI[2]) + m[3][c] * hI[3];
                            st4s(xp + bI * NB + 4 * bJ, y);
                        }
                    }
                    if (tid >= C::NT - 32 && tid - (C::NT - 32) < NU && do_next) {
                        const int q = tid - (C::NT - 32);
                        T d = (T)0;
#pragma unroll
                        for (int k2 = 0; k2 < NU; ++k2) d += Mb[q * NU + k2] * rhs[k2];
                        duc[pn * IP + q] = d;
                    }
                } else
                if (ci < NB && !first) {
                    T a0 = (T)0, a1 = (T)0;
                    constexpr int QD = (C::NS + NPART - 1) / NPART;
                    const T *Cp = Cb + prt * NB, *hp = hv + ci + prt;
                    const int im0 = ci - prt;
#pragma unroll
                    for (int q = 0; q < QD; ++q) {                         // s = prt + q NPART: same order as a rolled loop
                        const int s = prt + q * NPART;
                        if (s < C::NS) {
                            const T *Cs = Cp + q * NPART * NB;
                            a0 += Cs[ci] * hp[q * NPART];
                            if (s > 0 && 2 * s != NB) {
                                const int imw = im0 - q * NPART;           // (ci - s); h is stored twice, so hv[imw + NB] = h[(ci - s) mod NB]
                                a1 += Cs[imw < 0 ? imw + NB : imw] * hv[imw + NB];
                            }
                        }
                    }
                    xp[prt * IP + ci] = a0 + a1;
                }
                __syncthreads();
                // ---- E: xbar_{j+1}; Delta u_{j+1} = M rhs ----
                if (tid < NB) {
                    const int i = tid;
                    T x;
                    if (first) {                                                   // xbar_0
                        if (!PAD) x = i < NX ? p.x0[(size_t)b * NX + i] : p.uprev[(size_t)b * NU + (i - NX)];
                        else x = i < NX ? (i < rnx ? p.x0[(size_t)b * rnx + i] : (T)0) : (i - NX < rnu ? p.uprev[(size_t)b * rnu + (i - NX)] : (T)0);
                    }
                    else if constexpr (C::BLKH) {
                        T x0_ = xp[i], x1_ = C::NBK > 1 ? xp[NB + i] : (T)0;
#pragma unroll
                        for (int o = 2; o < C::NBK; ++o) { if (o & 1) x1_ += xp[o * NB + i]; else x0_ += xp[o * NB + i]; }
                        x = C::NBK > 1 ? x0_ + x1_ : x0_;
                    }
                    else {
                        x = (T)0;
#pragma unroll
                        for (int q = 0; q < NPART; ++q) x += xp[q * IP + i];
                    }
                    xv[i] = x;
                }
                if (!C::BLKH && tid >= IP && tid < IP + NU && do_next) {
                    const int q = tid - IP;
                    T d = (T)0;
#pragma unroll
                    for (int k2 = 0; k2 < NU; ++k2) d += Mb[q * NU + k2] * rhs[k2];
                    duc[pn * IP + q] = d;
                }
                __syncthreads();
                // ---- F: b_{j+1}, a_{j+1} (row products, 4 lanes per x-row) and steps 2-4 of stage j ----
                if (do_next) {                               // uniform branch: every lane takes part in the shuffles
                    const int r = tid >> 2, q = tid & 3;
                    T s0_ = (T)0, s1_ = (T)0;
                    if (tid < 4 * NX) {
#pragma unroll
                        for (int c = q; c < NB; c += 4) {
                            const T a = AB[r * NB + c];
                            s0_ += a * xv[c];
                            if (c >= NX) s1_ += a * duc[pn * IP + c - NX];
                        }
                    }
                    s0_ += __shfl_xor_sync(0xffffffffu, s0_, 1); s1_ += __shfl_xor_sync(0xffffffffu, s1_, 1);
                    s0_ += __shfl_xor_sync(0xffffffffu, s0_, 2); s1_ += __shfl_xor_sync(0xffffffffu, s1_, 2);
                    if (tid < 4 * NX && q == 0) {
                        bc[pn * IP + r] = s0_ + Eb[r] - hs[4 * NB + r];            // b = Abar xbar + ebar - lambdahat
                        avc[pn * IP + r] = s1_ + hs[3 * NB + r];                   // a = Bbar du + betahat
                    }
                }
                if constexpr (!EXT) {
                    if (di >= 0 && di < NB) {
                        const int i = di, gi = gix(i);
                        const bool real = !PAD || gi >= 0;                             // pad components: zero box, nothing stored
                        if (do_next && i >= NX) {
                            bc[pn * IP + i] = xv[i] - hs[4 * NB + i];
                            avc[pn * IP + i] = duc[pn * IP + i - NX] + hs[3 * NB + i];
                        }
                        if (do_dual) {
                            const T zh = hj[i], vh = hj[NB + i], thh = hj[2 * NB + i], beh = hj[3 * NB + i], lah = hj[4 * NB + i];
                            const T av = avc[pj * IP + i], bv = bc[pj * IP + i], x = xv[i];
                            const T lo = lo_c, hi = hi_c;
                            const T gam = av - bv;
                            const T zn = clips(((T)2 * (x + thh + bv) + gam) * (T)(1.0 / 3.0), lo, hi);   // Thm 1 (proof form, R1)
                            const T vn = (T)0.5 * (zn + gam);
                            const T thn = thh + x - zn, ben = av - vn, lan = zn - bv - vn;
                            const T d0 = thn - thh, d1 = ben - beh, d2 = lan - lah, d3 = zn - zh, d4 = vn - vh;
                            const T d5 = (zn - vn) - (zh - vh);
                            T a = d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5;
                            T *nw = p.S + (size_t)L.i_new * p.buf_stride + p.st(b, j);
                            if (real) { nw[gi] = zn; nw[rnb + gi] = vn; nw[2 * rnb + gi] = thn; nw[3 * rnb + gi] = ben; nw[4 * rnb + gi] = lan; }
                            if (has_du && i >= NX) {                                   // Delta-u box copy (reading R12)
                                const int q = i - NX;
                                const T duq = duc[pj * IP + q], dh = hj[5 * NB + q], deh = hj[5 * NB + NU + q];
                                const T dn = clips(duq + deh, dlo_c, dhi_c);
                                const T den = deh + duq - dn;
                                const T e0 = den - deh, e1 = dn - dh;
                                a += e0 * e0 + e1 * e1;
                                if (real) { nw[5 * rnb + q] = dn; nw[5 * rnb + rnu + q] = den; }
                            }
                            acc += (double)a;
                            if (write_x && real) {
                                p.X[((size_t)b * N + j) * rnb + gi] = x;
                                if (i >= NX) p.DU[((size_t)b * N + j) * rnu + (i - NX)] = duc[pj * IP + i - NX];
                            }
                        }
                    }
                } else {
                    const bool dthread = di >= 0 && di < NB;
                    if (dthread && do_next && di >= NX) {
                        bc[pn * IP + di] = xv[di] - hs[4 * NB + di];
                        avc[pn * IP + di] = duc[pn * IP + di - NX] + hs[3 * NB + di];
                    }
                    // argument of Proj of stage j (Thm 1, proof form, R1); with a general set (pimpc_set_constraint) the whole
                    // vector is staged in shared memory first (xp is free after phase E) -- a CTA-uniform extra barrier
                    if constexpr (EXT) {
                        if (gset && do_dual) {
                            if (dthread) {
                                const int i = di;
                                const T av = avc[pj * IP + i], bv = bc[pj * IP + i];
                                xp[i] = ((T)2 * (xv[i] + hj[2 * NB + i] + bv) + (av - bv)) * (T)(1.0 / 3.0);
                            }
                            __syncthreads();
                        }
                    }
                    if (dthread) {
                        const int i = di;
                        if (do_dual) {
                            const T zh = hj[i], vh = hj[NB + i], thh = hj[2 * NB + i], beh = hj[3 * NB + i], lah = hj[4 * NB + i];
                            const T av = avc[pj * IP + i], bv = bc[pj * IP + i], x = xv[i];
                            const T gam = av - bv;
                            const T zarg = ((T)2 * (x + thh + bv) + gam) * (T)(1.0 / 3.0);
                            T zn;
                            if (EXT && gset && i >= p.set_i0 && i < p.set_i0 + p.set_len) zn = proj_set_component(p, xp + p.set_i0, i - p.set_i0);
                            else if (EXT) zn = clips(zarg, p.lo_at(b, j, i), p.hi_at(b, j, i));
                            else zn = clips(zarg, p.lo[(size_t)b * p.bnd_stride + i], p.hi[(size_t)b * p.bnd_stride + i]);
                            const T vn = (T)0.5 * (zn + gam);
                            const T thn = thh + x - zn, ben = av - vn, lan = zn - bv - vn;
                            const T d0 = thn - thh, d1 = ben - beh, d2 = lan - lah, d3 = zn - zh, d4 = vn - vh;
                            const T d5 = (zn - vn) - (zh - vh);
                            T a = d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5;
                            T *nw = p.S + (size_t)L.i_new * p.buf_stride + p.st(b, j);
                            nw[i] = zn; nw[NB + i] = vn; nw[2 * NB + i] = thn; nw[3 * NB + i] = ben; nw[4 * NB + i] = lan;
                            if (has_du && i >= NX) {                                   // Delta-u box copy (reading R12)
                                const int q = i - NX;
                                const T duq = duc[pj * IP + q], dh = hj[5 * NB + q], deh = hj[5 * NB + NU + q];
                                const T dn = clips(duq + deh, p.dlo[(size_t)b * p.dbnd_stride + q], p.dhi[(size_t)b * p.dbnd_stride + q]);
                                const T den = deh + duq - dn;
                                const T e0 = den - deh, e1 = dn - dh;
                                a += e0 * e0 + e1 * e1;
                                nw[5 * NB + q] = dn; nw[5 * NB + NU + q] = den;
                            }
                            acc += (double)a;
                            if (write_x) {
                                p.X[((size_t)b * N + j) * NB + i] = x;
                                if (i >= NX) p.DU[((size_t)b * N + j) * NU + (i - NX)] = duc[pj * IP + i - NX];
                            }
                        }
                    }
                }
            }
            __syncthreads();                                 // slot and ping-pong vectors are free again
            if (tid == C::PROD && issued < total) { issue(pc, slot); pc.next(sm.seg); ++issued; }
            if (++slot == nslot) slot = 0;
            // ---- end of a segment: this CTA's part of c of the instance (fixed order) ----
            if (last_of_seg) {
                double s = acc;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                if (lane == 0) sm.red[warp] = s;
                __syncthreads();
                if (tid == 0) {
                    double t = 0.0;
                    for (int w = 0; w < C::NW; ++w) t += sm.red[w];
                    partial[(size_t)L.b * span + ((int)cta - L.c_lo)] = t;     // slot = position among the instance's CTAs
                }
                acc = 0.0;
            }
            if (++cc.o >= sg.nsteps) { cc.o = 0; ++cc.sg; }
        }
        // new records were written through the generic proxy and are read next iteration by bulk copies
        __threadfence();
        fence_proxy_async();
        grid.sync();
        // ---- steps 4-7: c of every instance of the range, same order in every CTA ----
        // one warp per instance: lanes stride over the instance's CTAs, then a fixed butterfly (bit-identical in every CTA)
        for (int li = warp; li < n_local; li += C::NW) {
            LInst &L = sm.inst[li];
            if (L.done) continue;
            const double *pp = partial + (size_t)L.b * span;
            double s = 0.0;
            for (int q = lane; q <= L.c_hi - L.c_lo; q += 32) s += __ldcg(&pp[q]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane != 0) continue;
            const double c = p.rho * s;
            L.c_last = c; L.iters = it + 1;
            int accept = 0;
            if (p.tol > 0.0 && c < p.tol) {                  // step 5: the returned iterate is the new one
                L.done = 1; L.i_cur = L.i_new;
            } else {
                accept = c <= p.eta * L.c_prev;              // steps 6 / 7 (R5, R6)
                if (accept) {
                    const double an = 0.5 + 0.5 * sqrt(1.0 + 4.0 * L.alpha * L.alpha);
                    L.kappa = (L.alpha - 1.0) / an; L.alpha = an;
                } else {
                    L.kappa = 0.0; L.alpha = 1.0; L.restarts += 1;
                }
                L.c_prev = c;
                const int fresh = 3 - L.i_cur - L.i_new;
                L.i_prev = L.i_cur; L.i_cur = L.i_new; L.i_new = fresh;
            }
            if (L.owner && p.hist_c && it < p.hist_cap) {
                p.hist_c[(size_t)L.b * p.hist_cap + it] = c;
                p.hist_a[(size_t)L.b * p.hist_cap + it] = (unsigned char)accept;
            }
        }
        __syncthreads();
        // partial[] is rewritten next iteration: every CTA must have read it first.  The next grid barrier
        // comes only after the next writes, so double-buffer by iteration parity instead of a second barrier.
        partial += (it & 1) ? -(ptrdiff_t)((size_t)p.batch * span) : (ptrdiff_t)((size_t)p.batch * span);
    }
    if (tid < n_local && sm.inst[tid].owner) {
        const LInst &L = sm.inst[tid];
        InstCtl c = p.ctl[L.b];
        c.alpha = L.alpha; c.c_prev = L.c_prev; c.c_last = L.c_last; c.kappa = L.kappa;
        c.i_prev = L.i_prev; c.i_cur = L.i_cur; c.i_new = L.i_new;
        c.done = L.done; c.iters = L.iters; c.restarts = L.restarts;
        p.ctl[L.b] = c;
    }
}

struct StreamPlan { int grid, nslot; size_t smem; };

template <typename T, int NX, int NU, bool EXT, bool PAD>
int plan_stream(pimpc_s *h, StreamPlan *pl)
{
    using C = SCfg<T, NX, NU>;
    auto kern = k_stream<T, NX, NU, EXT, PAD>;
    const size_t fixed = ((sizeof(StreamSmem) + 127) / 128) * 128 + (size_t)C::V_END * sizeof(T);
    const size_t slot = (size_t)C::SLOT * sizeof(T);
    // CTAs per SM: enough bytes in flight per SM to cover the HBM latency (>= 2 slots per CTA), several
    // CTAs so that one CTA's step barriers overlap another's math; opts.tune overrides.
    const size_t per_sm = 227 * 1024;
    int want = h->tune.ctas_per_sm;
    if (want <= 0) want = slot > 32 * 1024 ? 2 : (slot > 8 * 1024 ? 4 : 6);   // C5 fp32: 4 CTAs per SM 0.73 ms/it, 3: 0.82, 2: 1.04
    int nslot = 0, per = want;
    for (; per >= 1; --per) {
        const size_t budget = per_sm / per - 1024;
        if (budget < fixed + 2 * slot && per > 1) continue;
        nslot = (int)std::min<size_t>((budget - fixed) / slot, StreamSmem::MAXSLOT);
        if (nslot >= 2 || per == 1) break;
    }
    const int force = h->tune.ring_slots;
    if (force > 0) nslot = std::min(force, nslot);
    if (nslot < 1) { h->errmsg = "STREAM: a ring slot does not fit in shared memory"; return PIMPC_EINVAL; }
    const size_t smem = fixed + (size_t)nslot * slot;
    PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    PIMPC_CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, C::NT, smem));
    if (occ < 1) { h->errmsg = "STREAM kernel does not fit on an SM"; return PIMPC_EINVAL; }
    occ = std::min(occ, per);
    const long long S_tot = (long long)h->batch * (h->N + 1);
    long long grid = std::min<long long>(S_tot, (long long)h->sm_count * occ);
    const int gforce = h->tune.grid;                          // fewer CTAs = longer ranges per CTA
    if (gforce > 0) grid = std::min<long long>(grid, gforce);
    // a CTA's range may touch at most MAXI instances
    while (grid > 1 && (S_tot / grid + 1) / (h->N + 1) + 2 > C::MAXI) grid /= 2;   // never true for the shapes AUTO sends here
    if ((S_tot / grid + 1) / (h->N + 1) + 2 > C::MAXI) { h->errmsg = "STREAM: too many instances per CTA"; return PIMPC_EINVAL; }
    pl->grid = (int)grid; pl->nslot = nslot; pl->smem = smem;
    return PIMPC_OK;
}

template <typename T, int NX, int NU, bool EXT, bool PAD>
int run_stream_e(pimpc_s *h, int iters, double tol)
{
    using C = SCfg<T, NX, NU>;
    StreamPlan pl;
    int rc = plan_stream<T, NX, NU, EXT, PAD>(h, &pl);
    if (rc) return rc;
    int launches = 0;
    const size_t nblob = (size_t)h->batch * (h->N + 1);
    const size_t bbytes = nblob * C::BLOB * sizeof(T);
    if (!h->blob || h->blob_bytes < bbytes) {
        rc = pimpc_grow(h, &h->blob, &h->blob_bytes, bbytes); if (rc) return rc;
        h->blob_dirty = true;
    }
    int span = (pl.grid + h->batch - 1) / h->batch + 2;        // CTAs whose ranges can touch one instance
    const size_t pneed = 2 * (size_t)h->batch * span;
    rc = pimpc_grow(h, (void **)&h->spartial, &h->spartial_cap, pneed * sizeof(double)); if (rc) return rc;
    Prob<T> p = make_prob<T>(h, tol);
    if (h->blob_dirty) {
        k_pack<T, NX, NU><<<dim3(h->N + 1, h->batch), 128, 0, h->stream>>>(p, (T *)h->blob);
        PIMPC_CUDA_TRY(h, cudaGetLastError());
        h->blob_dirty = false;
        ++launches;
    }
    const T *blob = (const T *)h->blob;
    double *partial = h->spartial;
    int nslot = pl.nslot;
    void *args[] = {(void *)&p, (void *)&blob, (void *)&partial, (void *)&iters, (void *)&nslot, (void *)&span};
    PIMPC_CUDA_TRY(h, cudaLaunchCooperativeKernel((const void *)k_stream<T, NX, NU, EXT, PAD>, dim3(pl.grid), dim3(C::NT), args, pl.smem, h->stream));
    h->info.grid = pl.grid; h->info.block = C::NT; h->info.smem_bytes = pl.smem;
    return launches + 1;
}

template <typename T, int NX, int NU>
int run_stream_t(pimpc_s *h, int iters, double tol)
{
    return has_stage_terms(h) ? run_stream_e<T, NX, NU, true, false>(h, iters, tol) : run_stream_e<T, NX, NU, false, false>(h, iters, tol);
}

// (nx, nu) with a STREAM instantiation: the three BASELINE.json shapes and the paper's Table I shapes
#define PIMPC_STREAM_SHAPES(X) X(4, 2) X(12, 4) X(48, 12) X(10, 3) X(20, 6) X(30, 10) X(50, 15)
// containers of every other shape with nx <= 50, nu <= 15 (plain variant: no general set, no per-stage terms), smallest first:
// the caller's shape runs inside the first one that holds it (template flag PAD)
#define PIMPC_STREAM_CONTAINERS(X) X(12, 4) X(20, 6) X(30, 10) X(48, 12) X(50, 15)

bool stream_exact(const pimpc_s *h)
{
#define X(NX_, NU_) if (h->nx == NX_ && h->nu == NU_) return true;
    PIMPC_STREAM_SHAPES(X)
#undef X
    return false;
}
bool stream_container(const pimpc_s *h)
{
    if (has_stage_terms(h)) return false;
#define X(NX_, NU_) if (h->nx <= NX_ && h->nu <= NU_) return true;
    PIMPC_STREAM_CONTAINERS(X)
#undef X
    return false;
}
bool stream_shape(const pimpc_s *h) { return stream_exact(h) || stream_container(h); }

} // namespace

bool stream_supported(const pimpc_s *h, std::string *why)
{
    if (!stream_shape(h)) { if (why) *why = "no STREAM instantiation holds this (nx, nu) (nx <= 50, nu <= 15; general sets and per-stage terms: exact shapes only)"; return false; }
    const long long S_tot = (long long)h->batch * (h->N + 1);
    const long long grid = std::min<long long>(S_tot, h->sm_count);
    if ((S_tot / grid + 1) / (h->N + 1) + 2 > 16) { if (why) *why = "too many short instances per CTA"; return false; }
    return true;
}

int run_stream(pimpc_s *h, int iters, double tol)
{
    if (!stream_shape(h)) { h->errmsg = "STREAM engine not applicable"; return PIMPC_EINVAL; }
    const bool d = h->dtype == PIMPC_F64;
#define X(NX_, NU_) \
    if (h->nx == NX_ && h->nu == NU_) return d ? run_stream_t<double, NX_, NU_>(h, iters, tol) : run_stream_t<float, NX_, NU_>(h, iters, tol);
    PIMPC_STREAM_SHAPES(X)
#undef X
#define X(NX_, NU_) \
    if (h->nx <= NX_ && h->nu <= NU_) \
        return d ? run_stream_e<double, NX_, NU_, false, true>(h, iters, tol) : run_stream_e<float, NX_, NU_, false, true>(h, iters, tol);
    PIMPC_STREAM_CONTAINERS(X)
#undef X
    h->errmsg = "STREAM engine not applicable";
    return PIMPC_EINVAL;
}
