// RESIDENT engine, two rows per lane (the C4 kernel): Algorithm 1 with one CTA per MPC instance,
// ONE launch per solve and everything an instance needs on chip for all its iterations.
//
// Mapping.  A group of LPS = pow2(NBP / 2) lanes owns one stage, lane li owns rows 2 li, 2 li + 1 of that stage (both
// x-rows or both u-rows), a warp owns 32 / LPS consecutive stages, the CTA the whole horizon.  The shape is PADDED at
// compile time (NXP x-rows, NUP u-rows, multiples of 4) and the real nx <= NXP, nu <= NUP are run-time: pad rows and
// pad columns carry zero matrices, zero bounds and zero iterates, run the same instructions and stay exactly zero.
//
// Per-solve prologue (registers of the row owner, read from HBM once per solve):
//   Hrow  row of H_k
//   G     row of G_k = rho H_k [A_{k+1} B_{k+1}]^T  (nb x nx)                     -- step 1 re-associated:
//           xbar_{k+1} = H_k h_k,  h_k = qbar + rho (zhat - thetahat) + rho Abar_{k+1}^T w_{k+1}   (R2)
//                      = H_k (t_k + rho [0; w_u]) + G_k w_x,   t_k = qbar + rho (zhat - thetahat),
//         so the transposed product with Abar_{k+1} (columns in shared memory, a dependent second mat-vec in round 1)
//         becomes 12 more columns of the SAME row product: one exchange and one mat-vec less per iteration
//   U     x-rows: row of [A_k B_k];  u-rows: row of J_k = M_k Bbar_k^T = [M_k B_k^T | M_k] -- the paper's cached J_k
//         (PAPER.md:341):  Delta u_k = J_k (vhat - betahat) + M_k (dhat - deltahat) = [M B^T | M] (dv_x ; dv_u + dhat - deltahat)
// Iterates (z, v, theta, beta, lambda, d, delta; current and previous) are register PAIRS of the same lane; every
// element-wise step of Alg. 1 works on both rows at once with packed fp32 instructions (add/mul/fma.f32x2 on sm_100a).
// Per iteration only five 16-element vectors per stage go through shared memory (w, t, rr out; xbar, Delta u back),
// read with 16-byte broadcast loads; the slot stride makes those loads and the 8-byte own-row stores conflict-free.
// c (step 4) is reduced in a fixed order by a dedicated REDUCER warp (the CTA's last warp, which owns no stage): every lane of
// a stage warp stores its partial sum, the reducer adds its column over the warps (a balanced tree in T), then over the lanes
// (butterfly), promotes the total to double and takes the accept / restart decision (steps 5-7) for the whole CTA.
//
// The decision is PREDICTED (round 2): steps 5-7 gate the hats of the next iteration, and the reduce ->
// decide chain was 30 % of an iteration with nothing to overlap it.  Almost every step is accepted, so right after step 4 the
// stage warps form the next hats with the momentum of an accepted step (own registers only) and run phases A and B of the
// next iteration while the reducer sums and decides; they read the decision word before phase C, the first point that
// overwrites an iterate.  A restart repeats A and B with kappa = 0 (hat = new iterate needs `cur` only: the previous iterate
// is dead from phase A on); a stop returns the iterate phase C has not touched.  When a restart is DUE (the run of accepted
// steps has reached the length of the previous run, or the last two steps were restarts) the stage warps wait for the
// decision (~300 cycles) instead of betting a repeated A + B (~1100) on "accept".  Results are those of the unpredicted
// order, bit for bit.  Two CTA barriers per iteration (xbar / Delta u slots alternate by the parity of the iteration, so the
// stopped iteration's primal step survives the predicted phase B).
#include <algorithm>
#include <cstdio>

#include "pimpc_internal.h"

namespace {

constexpr int pow2ceil_r(int v) { int p = 1; while (p < v) p <<= 1; return p; }

// ---- register pairs and packed arithmetic ------------------------------------------------------------------------
template <typename T> struct Pr;
template <> struct Pr<float> { typedef float2 t; };
template <> struct Pr<double> { typedef double2 t; };

__device__ __forceinline__ float2 mk2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }   // a - b, one rounding
__device__ __forceinline__ double2 add2(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 mul2(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ double2 fma2(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ double2 sub2(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
template <typename P, typename T> __device__ __forceinline__ P clip2(P v, P lo, P hi)
{
    return mk2((T)fmin(fmax(v.x, lo.x), hi.x), (T)fmin(fmax(v.y, lo.y), hi.y));
}

// 4 consecutive elements as two pairs (one 16-byte load in fp32, two in fp64)
__device__ __forceinline__ void ld4p(const float *p, float2 &a, float2 &b)
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    a = make_float2(v.x, v.y); b = make_float2(v.z, v.w);
}
__device__ __forceinline__ void ld4p(const double *p, double2 &a, double2 &b)
{
    a = *reinterpret_cast<const double2 *>(p); b = *reinterpret_cast<const double2 *>(p + 2);
}
// 4 consecutive elements of global memory (16-byte aligned in fp32, 32-byte in fp64)
__device__ __forceinline__ void ldg4(const float *p, float (&o)[4])
{
    const float4 v = __ldg(reinterpret_cast<const float4 *>(p));
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ldg4(const double *p, double (&o)[4])
{
    const double2 a = __ldg(reinterpret_cast<const double2 *>(p)), b = __ldg(reinterpret_cast<const double2 *>(p + 2));
    o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}
__device__ __forceinline__ float2 ldp(const float *p) { return *reinterpret_cast<const float2 *>(p); }
__device__ __forceinline__ double2 ldp(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void stp(float *p, float2 v) { *reinterpret_cast<float2 *>(p) = v; }
__device__ __forceinline__ void stp(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }

template <typename T, int NXP, int NUP, bool GS>
struct R2Cfg {
    static constexpr int NBP = NXP + NUP;
    static constexpr int LPS = pow2ceil_r(NBP / 2);           // lanes per stage
    static constexpr int SPW = 32 / LPS;                      // stages per warp
    static constexpr int ROWP = 2 * LPS;                      // padded vector length of a stage
    static constexpr int WPE = sizeof(T) / 4;
    static constexpr int KAPN = 1024;                         // kappa table entries cached in smem
    // One block per stage slot s = k + 1 (slot 0 holds xbar_0, slot NS + 1 a zero w):
    //   W  w_k = zhat - vhat - ebar + lambdahat     T  t_k = qbar + rho (zhat - thetahat)
    //   RR (vhat - betahat) with (dhat - deltahat) added on the u rows      X  xbar_{k+1}      DU Delta u_k
    //   E  e_k per row (read only when present)
    // and once per CTA (the same for every stage): per-row constants B = qbar, du_lo, du_hi, lo, hi
    //   G  the lane's two rows of G_k, [2][NXP / 2][LPS][2] (8-byte pieces, lane-major: see ld4p on load widths):
    //      written by the prologue; read every iteration when the rows do not fit in registers (GS: more than 12 warps cap
    //      a thread at 128 registers), else copied to registers once
    // X and DU exist twice (parity of the iteration, see "speculated" above): OX + par * ROWP, ODU + par * NUP
    static constexpr int OW = 0, OT = ROWP, ORR = 2 * ROWP, OX = 3 * ROWP, ODU = 5 * ROWP, OE = ODU + 2 * NUP, OG = OE + ROWP,
                         SS0 = OG + NXP * ROWP;
    // slot stride == 64 / SPW words (mod 32): shared memory serves 8- and 16-byte accesses one half-warp at a time, and
    // the SPW / 2 groups of a half-warp then hit disjoint banks with their own-row accesses and their broadcast chunks
    // (measured on B200: 8-byte own-row stores 2 wavefronts instead of 4 with a stride of 32 / SPW)
    static constexpr int TGT = (64 / SPW) % 32;
    static constexpr int SSW0 = SS0 * WPE;
    static constexpr int SSW = SSW0 + ((TGT - SSW0 % 32) + 32) % 32;
    static constexpr int SS = SSW / WPE;
    static_assert(NXP % 4 == 0 && NUP % 4 == 0 && LPS >= 4 && LPS <= 32 && ROWP >= NBP && (SS * sizeof(T)) % 16 == 0 && SSW % WPE == 0, "bad row blocking");
    static size_t smem_bytes(int nmain)                       // nmain = warps that own stages (the CTA has one more: the reducer)
    {
        const size_t NS = (size_t)nmain * SPW;
        return ((NS + 2) * SS + KAPN + 10 * ROWP + 2 * (size_t)nmain * 32) * sizeof(T) + 8 * sizeof(double);
    }
};

template <typename P> struct R2State { P z, v, th, be, la, d, de; };

// Phase clock profile of CTA 0 (a -DR2_PROF build for profiles/, never shipped): cycles per phase, warps 0 and last.
#ifdef R2_PROF
__device__ long long g_r2prof[1024 * 16 * 8];
#define R2P(i) do { if (blockIdx.x == 0 && lane == 0 && pit < 1024) g_r2prof[(pit * 16 + warp) * 8 + (i)] = clock64(); } while (0)
#else
#define R2P(i) do { } while (0)
#endif

// GS: the rows of G_k live in shared memory instead of registers (CTAs of 13..16 warps: 4 warps share a sub-partition's
// 16 K registers, 128 per thread; up to 12 warps get 168).
template <typename T, int NXP, int NUP, int MAXT, bool DU, bool GS>
__global__ void __launch_bounds__(MAXT, 1)
k_res2(const Prob<T> p, const double *__restrict__ alpha_tab, const double *__restrict__ kappa_tab, const int iters)
{
    using C = R2Cfg<T, NXP, NUP, GS>;
    using P = typename Pr<T>::t;
    constexpr int NBP = C::NBP, LPS = C::LPS, SPW = C::SPW, SS = C::SS;
    constexpr int OW = C::OW, OT = C::OT, ORR = C::ORR, OX = C::OX, ODU = C::ODU, OE = C::OE, OG = C::OG, ROWP = C::ROWP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nmain = (blockDim.x >> 5) - 1;                  // warps 0..nmain-1 own stages, warp nmain is the reducer
    const int NS = nmain * SPW, N = p.N, nx = p.nx, nu = p.nu, nb = p.nb;
    int *sDec = reinterpret_cast<int *>(smem_raw);            // [0] decision of the reducer: 0 accept, 1 restart, 2 stop
    T *sKap = reinterpret_cast<T *>(smem_raw + 8 * sizeof(double));   // [KAPN]
    T *sBnd = sKap + C::KAPN;                                 // [5][ROWP] qbar, du_lo, du_hi, lo, hi by padded row, then
                                                              // [5][ROWP] zeros: the constants of the pad stages (k >= N)
    T *sAcc = sBnd + 10 * ROWP;                               // [2][nmain * 32] per-lane partial sums of c by parity of the iteration
    T *sBlk = sAcc + 2 * nmain * 32;                          // [NS + 2][SS]

    const int li = lane % LPS, k = warp * SPW + lane / LPS;
    const bool stage_ok = k < N;
    const int i0 = 2 * li;                                    // first padded row of the lane
    const bool isu = stage_ok && i0 >= NXP && i0 < NBP;       // the lane owns u rows
    const bool isx = !isu;                                    // x rows; pad lanes and pad stages take the same path with zeros
    const T rho = (T)p.rho;
    const P rho2 = mk2(rho, rho);
    T *const blk = sBlk + (size_t)(k + 1) * SS;               // block of the own stage
    T *const own = blk + i0;                                  // + own rows
    const T *const bnd = sBnd + (stage_ok ? 0 : 5 * ROWP) + i0;   // own rows of the per-CTA constants (pad stages: zeros)
    const bool has_e = p.e != nullptr, has_q = p.has_q != 0;
    // padded index -> index in the caller's arrays (-1: pad)
    auto gidx = [&](int i) -> int { return i < NXP ? (i < nx ? i : -1) : (i - NXP < nu ? nx + (i - NXP) : -1); };

    for (int i = tid; i < (NS + 2) * SS; i += blockDim.x) sBlk[i] = (T)0;      // pads must stay finite zeros
    for (int i = tid; i < min(iters + 1, C::KAPN); i += blockDim.x) sKap[i] = (T)kappa_tab[i];
    for (int i = tid; i < 5 * ROWP; i += blockDim.x) sBnd[5 * ROWP + i] = (T)0;
    __syncthreads();

#ifdef R2_PROF
    int pit = 0;
#endif
    for (int b = blockIdx.x; b < p.batch; b += gridDim.x) {
        // ---- [A_k B_k] of every stage of the instance -> the stage's slot (the area that later holds G_k), padded, by ONE
        // coalesced cooperative load of the whole CTA: the per-solve prologue then forms U, J_k and G_k from shared memory
        // (per-lane rolled loops over global memory made the prologue 0.67 ms of C4's 7.15 ms kernel)
        for (int e0 = tid; e0 < NS * NXP * ROWP; e0 += 4 * blockDim.x) {
            T v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {                      // four independent loads in flight per thread
                const int i = e0 + u * blockDim.x;
                const int ks = i / (NXP * ROWP), q = i - ks * (NXP * ROWP), r = q / ROWP, c = q - r * ROWP;
                v[u] = (T)0;
                if (ks < N && r < nx && c < NBP) {
                    const size_t st = (size_t)b * N + ks;
                    if (c < NXP) { if (c < nx) v[u] = p.A[st * nx * nx + r * nx + c]; }
                    else if (c - NXP < nu) v[u] = p.B[st * nx * nu + r * nu + (c - NXP)];
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = e0 + u * blockDim.x;
                if (i < NS * NXP * ROWP) { const int ks = i / (NXP * ROWP); sBlk[(size_t)(ks + 1) * SS + OG + (i - ks * (NXP * ROWP))] = v[u]; }
            }
        }
        __syncthreads();
        if (warp == nmain) {
            // ---- the reducer warp: step 4's sum and steps 5-7 for the whole CTA.  It follows the barrier
            // sequence of the stage warps: per iteration bar1 (phase A published | partial sums of the previous iteration
            // complete), bar2 (phase B done | decision published), two more after a restart.
            // the next instance of this CTA: its stage data and iterates -> L2 while this one iterates (the reducer warp has the
            // time), so that the next prologue pays L2 instead of HBM latencies
            if (b + (int)gridDim.x < p.batch) {
                const size_t bn = (size_t)b + gridDim.x;
                auto pf = [&](const void *base, size_t bytes) {
                    for (size_t o = (size_t)lane * 128; o < bytes; o += 32 * 128)
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(base) + o));
                };
                pf(p.A + bn * N * nx * nx, (size_t)N * nx * nx * sizeof(T));
                pf(p.B + bn * N * nx * nu, (size_t)N * nx * nu * sizeof(T));
                pf(p.H + bn * N * nb * nb, (size_t)N * nb * nb * sizeof(T));
                pf(p.M + bn * N * nu * nu, (size_t)N * nu * nu * sizeof(T));
                pf(p.S + (size_t)p.ctl[bn].i_cur * p.buf_stride + p.st((int)bn, 0), (size_t)N * p.rec * sizeof(T));
            }
            double c_last = p.c0, c_prev = p.c0, thr = p.eta * p.c0;   // thr = eta c^{i}: ready before c^{i+1} arrives
            int jacc = 0, nrest = 0, n_it = 0, lrun = 0;       // lrun: accepted steps before the last restart
            bool done = false;
            auto decide = [&](const int it) -> int {
                // fixed order: this lane's column over the stage warps (all loads in flight at once, zeros beyond nmain, a
                // balanced tree), then the butterfly over the lanes -- in T: for fp32 handles an fp32 tree of <= 512 partials
                // (relative error <= 9 * 2^-24, far below the error the partials already carry) keeps the chain at ~230
                // cycles (a double chain with its conversions took ~700: the stage warps waited for it at barrier 2)
                const T *a = sAcc + (it & 1) * nmain * 32 + lane;
                T v[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) v[j] = j < nmain ? a[j * 32] : (T)0;
#pragma unroll
                for (int w = 8; w > 0; w >>= 1)
#pragma unroll
                    for (int j = 0; j < w; ++j) v[j] += v[j + w];
                T sumT = v[0];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sumT += __shfl_xor_sync(0xffffffffu, sumT, o);
                const double sum = (double)sumT;
                const double c = p.rho * sum;
                const bool stop = p.tol > 0.0 && c < p.tol;
                const bool accept = !stop && c <= thr;
                const int dec = stop ? 2 : (accept ? 0 : 1);
                if (lane == 0) {
                    *reinterpret_cast<volatile int *>(sDec) = dec;
                    if (p.hist_c && it < p.hist_cap) {
                        p.hist_c[(size_t)b * p.hist_cap + it] = c; p.hist_a[(size_t)b * p.hist_cap + it] = (unsigned char)accept;
                    }
                }
                c_prev = c_last; c_last = c; thr = p.eta * c; n_it = it + 1;
                if (accept) ++jacc;
                else if (!stop) { lrun = jacc > 0 ? jacc : -1; jacc = 0; ++nrest; }      // -1: a restart right after a restart
                done = stop;
                return dec;
            };
            __syncthreads();
            // Mirror of the stage warps' schedule (see `iteration`): a decision is either PREDICTED as "accept" and taken between
            // barriers 1 and 2 of the next iteration (a restart then repeats A and B: two more barriers), or -- when the run of
            // accepted steps has reached the length of the previous run, i.e. a restart is due -- WAITED for right after phase C.
            int it = 0;
            bool resolved = true;                              // is the decision of iteration it-1 taken at the top of iteration it
#pragma unroll 1
            for (; it < iters; ++it) {
                __syncthreads();
                int dec = 0;
                if (!resolved) dec = decide(it - 1);
                __syncthreads();
                if (!resolved) {
                    if (dec == 2) break;
                    if (dec == 1) { __syncthreads(); __syncthreads(); }
                }
                resolved = (lrun > 0 && jacc >= lrun) || (lrun < 0 && jacc == 0);
                if (resolved) {
                    __syncthreads();
                    dec = decide(it);
                    __syncthreads();
                    if (dec == 2) break;
                }
            }
            if (!done && !resolved) { __syncthreads(); decide(iters - 1); __syncthreads(); }
            if (lane == 0) {
                InstCtl c = p.ctl[b];
                c.alpha = alpha_tab[jacc]; c.c_last = c_last;
                c.c_prev = done ? c_prev : c_last;
                c.kappa = jacc > 0 ? (double)(T)kappa_tab[jacc - 1] : 0.0;      // momentum of the last hats formed
                c.done = done ? 1 : 0; c.iters = n_it; c.restarts = nrest;
                p.ctl[b] = c;
            }
            __syncthreads();
            continue;
        }
        const int i_cur = p.ctl[b].i_cur;
        const size_t sk = (size_t)b * N + (stage_ok ? k : 0);
        const bool inner = stage_ok && k < N - 1;
        const bool native = nx == NXP && nu == NUP;            // no pad rows / columns: row-major H_k rows are NBP contiguous elements
        // ---- stage matrices -> registers (once per solve) ----------------------------------------------------------
        T Hrow[2][NBP], G[2][NXP], U[2][NBP];
        R2State<P> sa, sb;
        {
            const T *const ab = blk + OG, *const ab1 = blk + SS + OG;          // [A_k B_k], [A_{k+1} B_{k+1}] as [NXP][ROWP]
            T st_[7][2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int gi = gidx(i0 + r);
                const bool ok = stage_ok && gi >= 0;
                const bool oku = ok && i0 >= NXP;
                const T *Hk = p.H + sk * nb * nb + (size_t)(ok ? gi : 0) * nb;
                if (native) {                                          // unpadded shape: 16-byte loads of the row (a scalar load per
                                                                       // element touched 32 sectors per instruction, 16 times per row)
#pragma unroll
                    for (int j = 0; j < NBP; j += 4) {
                        T h4[4] = {(T)0, (T)0, (T)0, (T)0};
                        if (ok) ldg4(Hk + j, h4);
                        Hrow[r][j] = h4[0]; Hrow[r][j + 1] = h4[1]; Hrow[r][j + 2] = h4[2]; Hrow[r][j + 3] = h4[3];
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < NBP; ++j) { const int gj = gidx(j); Hrow[r][j] = (ok && gj >= 0) ? Hk[gj] : (T)0; }
                }
                if (i0 < NXP) {                                        // x rows: row of [A_k B_k] (pad rows and pad stages: zeros)
#pragma unroll
                    for (int j = 0; j < NBP; ++j) U[r][j] = ab[(i0 + r) * ROWP + j];
                } else {
                    // u rows: row of J_k = M_k Bbar_k^T = [M_k B_k^T | M_k], the paper's cached J_k
                    T mrow[NUP];
#pragma unroll
                    for (int c = 0; c < NUP; ++c) mrow[c] = (oku && c < nu) ? p.M[sk * nu * nu + (size_t)(gi - nx) * nu + c] : (T)0;
#pragma unroll
                    for (int j = 0; j < NXP; ++j) {
                        T acc = (T)0;
#pragma unroll
                        for (int c = 0; c < NUP; ++c) acc = fma(mrow[c], ab[j * ROWP + NXP + c], acc);
                        U[r][j] = acc;
                    }
#pragma unroll
                    for (int c = 0; c < NUP; ++c) U[r][NXP + c] = mrow[c];
                }
                own[OE + r] = (ok && i0 < NXP && has_e) ? p.e[sk * nx + gi] : (T)0;
                // G_k row = rho * Hrow . [A_{k+1} B_{k+1}]^T in the arithmetic of the handle (two accumulators per entry; in fp32 a
                // 16-term product sum is good to ~4e-7 relative, two orders below the iterate error the fp32 path carries anyway)
#pragma unroll
                for (int j = 0; j < NXP; ++j) {
                    T a0 = (T)0, a1 = (T)0;
                    if (inner) {
#pragma unroll
                        for (int c4 = 0; c4 < NBP; c4 += 4) {
                            const T *q = ab1 + j * ROWP + c4;
                            a0 = fma(Hrow[r][c4], q[0], a0); a1 = fma(Hrow[r][c4 + 1], q[1], a1);
                            a0 = fma(Hrow[r][c4 + 2], q[2], a0); a1 = fma(Hrow[r][c4 + 3], q[3], a1);
                        }
                    }
                    G[r][j] = rho * (a0 + a1);
                }
                // ---- iterate of the previous solve / cold start (hats = iterates: prev = cur) ----
                const T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(b, stage_ok ? k : 0);
                st_[0][r] = ok ? rec[p.oZ() + gi] : (T)0;
                st_[1][r] = ok ? rec[p.oV() + gi] : (T)0;
                st_[2][r] = ok ? rec[p.oTH() + gi] : (T)0;
                st_[3][r] = ok ? rec[p.oBE() + gi] : (T)0;
                st_[4][r] = ok ? rec[p.oLA() + gi] : (T)0;
                st_[5][r] = (oku && DU) ? rec[p.oD() + (gi - nx)] : (T)0;
                st_[6][r] = (oku && DU) ? rec[p.oDE() + (gi - nx)] : (T)0;
            }
            sa.z = mk2(st_[0][0], st_[0][1]); sa.v = mk2(st_[1][0], st_[1][1]); sa.th = mk2(st_[2][0], st_[2][1]);
            sa.be = mk2(st_[3][0], st_[3][1]); sa.la = mk2(st_[4][0], st_[4][1]);
            sa.d = mk2(st_[5][0], st_[5][1]); sa.de = mk2(st_[6][0], st_[6][1]);
        }
        sb = sa;
        if (tid < ROWP) {                                      // slot 0: xbar_0 = (x(t); u(t-1))
            const int g0 = gidx(tid);
            const bool okr = tid < NBP && g0 >= 0, oku0 = okr && tid >= NXP;
            sBnd[tid] = okr ? p.qbar[(size_t)b * p.qbar_stride + g0] : (T)0;
            sBnd[ROWP + tid] = (oku0 && DU) ? p.dlo[(size_t)b * p.dbnd_stride + (g0 - nx)] : (T)0;
            sBnd[2 * ROWP + tid] = (oku0 && DU) ? p.dhi[(size_t)b * p.dbnd_stride + (g0 - nx)] : (T)0;
            sBnd[3 * ROWP + tid] = okr ? p.lo[(size_t)b * p.bnd_stride + g0] : (T)0;
            sBnd[4 * ROWP + tid] = okr ? p.hi[(size_t)b * p.bnd_stride + g0] : (T)0;
            sBlk[OX + tid] = sBlk[OX + ROWP + tid] =
                (tid < NBP && g0 >= 0) ? (tid < NXP ? p.x0[(size_t)b * nx + g0] : p.uprev[(size_t)b * nu + (g0 - nx)]) : (T)0;
        }

        T kap = (T)0;                                          // momentum of the hats being formed
        int jacc = 0, lrun = 0;                                // accepted steps in a row (a pending one counted as accepted), and before the last restart
        bool pend = false;                                     // the decision of the previous iteration is still open
        P zh, vh, thh, beh, lah, dh, deh;                      // hats of the iteration in flight (A -> C)
        P xs, du;                                              // own rows of xbar_{k+1}, Delta u_k of the iteration in flight (B -> C)
        zh = vh = thh = beh = lah = dh = deh = xs = du = mk2((T)0, (T)0);

        // ---- A: steps 6/7 of the previous iteration: hats from (cur, prev, kappa); publish w, t, rr ----
        auto publish = [&]() {
            P wv = add2(sub2(zh, vh), lah);                                     // w_k = zhat - vhat - ebar + lambdahat
            if (has_e) wv = sub2(wv, ldp(own + OE));
            P tv = mul2(rho2, sub2(zh, thh));                                   // t_k = rho (zhat - thetahat) [+ qbar]
            if (has_q) tv = add2(tv, ldp(bnd));
            P rr = sub2(vh, beh);                                               // vhat - betahat [+ dhat - deltahat]
            if (DU) rr = add2(rr, sub2(dh, deh));
            stp(own + OW, wv); stp(own + OT, tv); stp(own + ORR, rr);
        };
        auto phaseA = [&](const R2State<P> &cur, const R2State<P> &prv) {
            const P kap2 = mk2(kap, kap);
            zh = fma2(kap2, sub2(cur.z, prv.z), cur.z);
            vh = fma2(kap2, sub2(cur.v, prv.v), cur.v);
            thh = fma2(kap2, sub2(cur.th, prv.th), cur.th);
            beh = fma2(kap2, sub2(cur.be, prv.be), cur.be);
            lah = fma2(kap2, sub2(cur.la, prv.la), cur.la);
            if (DU) {
                dh = fma2(kap2, sub2(cur.d, prv.d), cur.d);
                deh = fma2(kap2, sub2(cur.de, prv.de), cur.de);
            }
            publish();
        };
        // restart (step 7): kappa = 0, hat = the new iterate itself.  Written without the previous iterate ON PURPOSE: it is
        // then dead from phase A on, and its 14 registers serve phases B and C as load buffers.
        auto phaseA_restart = [&](const R2State<P> &cur) {
            zh = cur.z; vh = cur.v; thh = cur.th; beh = cur.be; lah = cur.la;
            if (DU) { dh = cur.d; deh = cur.de; }
            publish();
        };
        // ---- B: step 1: xbar_{k+1} = Hrow (t + rho [0; w_u]) + G w_x;  Delta u_k = [M B^T | M] rr ----
        auto phaseB = [&](const int par) {
            P xa[2], da[2];
            xa[0] = xa[1] = da[0] = da[1] = mk2((T)0, (T)0);
            // one vector at a time, all its chunks in flight before its products (with the three vectors interleaved chunk by
            // chunk ptxas sank every load next to its use, and the in-order warp paid the 29-cycle shared-memory latency
            // once per chunk: C4 kernel 7.37 -> 7.09 ms): t, then rr, then w -- the u part of w first, it joins t (the
            // [0 I] rows of Abar_{k+1})
            P tv[NBP / 2], wv[NBP / 2];
#pragma unroll
            for (int c4 = NXP; c4 < NBP; c4 += 4) ld4p(blk + SS + OW + c4, wv[c4 / 2], wv[c4 / 2 + 1]);
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) ld4p(blk + OT + c4, tv[c4 / 2], tv[c4 / 2 + 1]);
#pragma unroll
            for (int c2 = NXP / 2; c2 < NBP / 2; ++c2) tv[c2] = fma2(rho2, wv[c2], tv[c2]);
#pragma unroll
            for (int c2 = 0; c2 < NBP / 2; ++c2)
#pragma unroll
                for (int r = 0; r < 2; ++r) xa[r] = fma2(mk2(Hrow[r][2 * c2], Hrow[r][2 * c2 + 1]), tv[c2], xa[r]);
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) ld4p(blk + ORR + c4, tv[c4 / 2], tv[c4 / 2 + 1]);
#pragma unroll
            for (int c4 = 0; c4 < NXP; c4 += 4) ld4p(blk + SS + OW + c4, wv[c4 / 2], wv[c4 / 2 + 1]);
#pragma unroll
            for (int c2 = 0; c2 < NBP / 2; ++c2)
#pragma unroll
                for (int r = 0; r < 2; ++r) da[r] = fma2(mk2(U[r][2 * c2], U[r][2 * c2 + 1]), tv[c2], da[r]);
            if (GS) {                                          // the rows of G_k from shared memory, a row's pieces in flight together
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    P g[NXP / 2];
#pragma unroll
                    for (int c2 = 0; c2 < NXP / 2; ++c2) g[c2] = ldp(blk + OG + ((r * (NXP / 2) + c2) * LPS + li) * 2);
#pragma unroll
                    for (int c2 = 0; c2 < NXP / 2; ++c2) xa[r] = fma2(g[c2], wv[c2], xa[r]);
                }
            } else {
#pragma unroll
                for (int c2 = 0; c2 < NXP / 2; ++c2)
#pragma unroll
                    for (int r = 0; r < 2; ++r) xa[r] = fma2(mk2(G[r][2 * c2], G[r][2 * c2 + 1]), wv[c2], xa[r]);
            }
            xs = mk2(xa[0].x + xa[0].y, xa[1].x + xa[1].y);
            du = mk2(da[0].x + da[0].y, da[1].x + da[1].y);                      // meaningful on the u rows only
            stp(own + OX + par * ROWP, xs);
            if (isu) stp(own + ODU + par * NUP - NXP, du);
        };
        // ---- C: steps 2-4; the new iterate overwrites prv's registers; the lane's partial of c -> sAcc ----
        auto phaseC = [&](R2State<P> &prv, const int par) {
            P ba[2], aa[2], xu0 = mk2((T)0, (T)0), xu1 = xu0;
            ba[0] = ba[1] = aa[0] = aa[1] = mk2((T)0, (T)0);
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                P x0, x1;
                ld4p(blk - SS + OX + par * ROWP + c4, x0, x1);
                if (NUP == 4 && c4 == NXP) { xu0 = x0; xu1 = x1; }                           // the u part of xbar_k
#pragma unroll
                for (int r = 0; r < 2; ++r) {                                               // [A_k B_k] xbar_k (x rows)
                    ba[r] = fma2(mk2(U[r][c4], U[r][c4 + 1]), x0, ba[r]);
                    ba[r] = fma2(mk2(U[r][c4 + 2], U[r][c4 + 3]), x1, ba[r]);
                }
            }
#pragma unroll
            for (int c4 = 0; c4 < NUP; c4 += 4) {
                P u0, u1;
                ld4p(blk + ODU + par * NUP + c4, u0, u1);
#pragma unroll
                for (int r = 0; r < 2; ++r) {                                               // B_k Delta u_k (x rows)
                    aa[r] = fma2(mk2(U[r][NXP + c4], U[r][NXP + c4 + 1]), u0, aa[r]);
                    aa[r] = fma2(mk2(U[r][NXP + c4 + 2], U[r][NXP + c4 + 3]), u1, aa[r]);
                }
            }
            // own rows of xbar_k (u rows: the [0 I] rows of Abar_k): with four u rows they sit in the chunk just loaded
            const P xpi = NUP == 4 ? ((li & 1) ? xu1 : xu0) : ldp(own - SS + OX + par * ROWP);
            const P a_in = isx ? mk2(aa[0].x + aa[0].y, aa[1].x + aa[1].y) : du;
            P bx = mk2(ba[0].x + ba[0].y, ba[1].x + ba[1].y);
            if (has_e) bx = add2(bx, ldp(own + OE));                                        // pad / u rows hold e = 0
            const P b_in = isx ? bx : xpi;
            const P av = add2(a_in, beh);                                                   // a = Bbar du + betahat
            const P bv = sub2(b_in, lah);                                                   // b = Abar xbar_k + ebar - lambdahat
            const P gam = sub2(av, bv);
            const P s1 = add2(xs, thh);
            const P zc = mul2(fma2(add2(s1, bv), mk2((T)2, (T)2), gam), mk2((T)(1.0 / 3.0), (T)(1.0 / 3.0)));
            const P zn = clip2<P, T>(zc, ldp(bnd + 3 * ROWP), ldp(bnd + 4 * ROWP));          // Thm 1 (proof form, R1)
            const P vn = mul2(mk2((T)0.5, (T)0.5), add2(zn, gam));
            const P thn = sub2(s1, zn);
            const P ben = sub2(av, vn);
            const P lan = sub2(sub2(zn, bv), vn);
            const P d0 = sub2(thn, thh), d1 = sub2(ben, beh), d2 = sub2(lan, lah), d3 = sub2(zn, zh), d4 = sub2(vn, vh);
            const P d5 = sub2(sub2(zn, vn), sub2(zh, vh));
            P acc2 = mul2(d0, d0);
            acc2 = fma2(d1, d1, acc2); acc2 = fma2(d2, d2, acc2); acc2 = fma2(d3, d3, acc2);
            acc2 = fma2(d4, d4, acc2); acc2 = fma2(d5, d5, acc2);
            prv.z = zn; prv.v = vn; prv.th = thn; prv.be = ben; prv.la = lan;
            if (DU) {                                                          // Delta-u box copy (reading R12); x rows: zeros
                const P duu = isx ? mk2((T)0, (T)0) : du;
                const P t = add2(duu, deh);
                const P dn = clip2<P, T>(t, ldp(bnd + ROWP), ldp(bnd + 2 * ROWP));
                const P den = sub2(t, dn);
                const P e0 = sub2(den, deh), e1 = sub2(dn, dh);
                acc2 = fma2(e0, e0, acc2); acc2 = fma2(e1, e1, acc2);
                prv.d = dn; prv.de = den;
            }
            // step 4: the lane's partial sum goes to the reducer warp (no shuffles, no fp64 in the stage warps)
            sAcc[par * nmain * 32 + tid] = acc2.x + acc2.y;
        };
        // One iteration of Alg. 1 on (cur, prv) = iterates i, i-1; par = it & 1 (compile-time after unrolling by two).  On
        // entry phase A of this iteration has run (speculated momentum) and the decision of iteration it-1 is pending
        // (it > 0): the reducer warp takes it between the two barriers.  Returns true when iteration it-1 stopped (c < tol).
        auto iteration = [&](R2State<P> &cur, R2State<P> &prv, const int it, const int par) -> int {
#ifdef R2_PROF
            if (blockIdx.x == 0 && lane == 0 && pit < 1024) g_r2prof[(pit * 16 + warp) * 8 + 4] = 0;
#endif
            R2P(0);
            __syncthreads();
            R2P(1);
            phaseB(par);
            R2P(2);
            __syncthreads();
            R2P(3);
            if (pend) {
                const int dec = *reinterpret_cast<volatile int *>(sDec);       // steps 5-7 of iteration it-1 (the reducer warp)
                if (dec == 2) return 1;
                if (dec == 1) {                                // restart: A and B again with kappa = 0
                    lrun = jacc > 1 ? jacc - 1 : -1;           // (the pending step had been counted as accepted; -1: restart after restart)
                    kap = (T)0; jacc = 0;
                    phaseA_restart(cur);
                    __syncthreads();
                    phaseB(par);
                    __syncthreads();
                    R2P(4);
                }
            }
            phaseC(prv, par);
            if ((lrun > 0 && jacc >= lrun) || (lrun < 0 && jacc == 0)) {
                // the run of accepted steps has reached the length of the previous run, or the last two steps were restarts (the
                // slowly converging tail of C1 / C3 restarts every step): a restart is due (C4: right two times out of three).  Wait for the decision (~300 cycles) instead of betting a repeated A + B (~1100) on "accept".
                __syncthreads();
                __syncthreads();
                const int dec = *reinterpret_cast<volatile int *>(sDec);
                if (dec == 2) return 2;
                pend = false;
                if (dec == 0) {
                    T kg = (T)0;
                    if (jacc >= C::KAPN) kg = (T)kappa_tab[jacc];
                    kap = jacc < C::KAPN ? sKap[jacc] : kg;
                    ++jacc;
                    phaseA(prv, cur);
                } else {
                    lrun = jacc > 0 ? jacc : -1; kap = (T)0; jacc = 0;
                    phaseA_restart(prv);
                }
            } else {
                T kg = (T)0;
                if (jacc >= C::KAPN) kg = (T)kappa_tab[jacc];
                kap = jacc < C::KAPN ? sKap[jacc] : kg;        // predict: the step is accepted
                ++jacc;
                pend = true;
                phaseA(prv, cur);                              // hats of iteration it + 1: the new iterate sits in prv's registers
            }
            R2P(5);
#ifdef R2_PROF
            ++pit;
#endif
            return 0;
        };

        // ---- results: iterate -> S[i_cur], xbar and Delta u of the last iteration (called at each exit of the loop: the
        // two iterate sets never merge, so the unrolled-by-two loop carries them in place without register moves).
        // the last iteration had parity par; pending: its decision is still open (the reducer warp takes it between two barriers) ----
        auto finish = [&](const R2State<P> &fin, const bool pending, const int par) {
            if (pending) { __syncthreads(); __syncthreads(); }
            const size_t sk = (size_t)b * N + (stage_ok ? k : 0);
            const T fz[2] = {fin.z.x, fin.z.y}, fv[2] = {fin.v.x, fin.v.y}, fth[2] = {fin.th.x, fin.th.y};
            const T fbe[2] = {fin.be.x, fin.be.y}, fla[2] = {fin.la.x, fin.la.y}, fd[2] = {fin.d.x, fin.d.y}, fde[2] = {fin.de.x, fin.de.y};
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int gi = gidx(i0 + r);
                if (stage_ok && gi >= 0) {
                    T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(b, k);
                    rec[p.oZ() + gi] = fz[r]; rec[p.oV() + gi] = fv[r]; rec[p.oTH() + gi] = fth[r];
                    rec[p.oBE() + gi] = fbe[r]; rec[p.oLA() + gi] = fla[r];
                    p.X[sk * nb + gi] = own[OX + par * ROWP + r];
                    if (i0 >= NXP) {
                        p.DU[sk * nu + (gi - nx)] = own[ODU + par * NUP - NXP + r];
                        if (DU) { rec[p.oD() + (gi - nx)] = fd[r]; rec[p.oDE() + (gi - nx)] = fde[r]; }
                    }
                }
            }
        };

        __syncthreads();                                       // every stage has read its neighbour's [A B]; slot 0 and the boxes are in place
        if (GS) {                                              // G_k -> the slot (lane-major 8-byte pieces), over the staged [A_k B_k]
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int c2 = 0; c2 < NXP / 2; ++c2) stp(blk + OG + ((r * (NXP / 2) + c2) * LPS + li) * 2, mk2(G[r][2 * c2], G[r][2 * c2 + 1]));
        }
#ifdef R2_PROF
        pit = 0; R2P(5); pit = 1;
#endif
        phaseA(sa, sb);                                        // kappa = 0: hats = iterates (Alg. 1 input)
        {
            int it = 0;
#pragma unroll 1
            for (;;) {
                if (it >= iters) { finish(sa, pend, 1); break; }
                int r = iteration(sa, sb, it, 0);
                if (r == 1) { finish(sa, false, 1); break; }                             // iteration it-1 stopped
                if (r == 2) { finish(sb, false, 0); break; }                             // iteration it stopped
                if (it + 1 >= iters) { finish(sb, pend, 0); break; }
                r = iteration(sb, sa, it + 1, 1);
                if (r == 1) { finish(sb, false, 0); break; }
                if (r == 2) { finish(sa, false, 1); break; }
                it += 2;
            }
        }
        __syncthreads();
#ifdef R2_PROF
        if (blockIdx.x == 0 && b == 0 && lane == 0 && (warp == 0 || warp == nmain - 1 || warp == 5)) {
            // slots: 0 after A, 1 after bar1, 2 after B, 3 after bar2, 4 redo (A and B again), 5 after C; row pit-1 slot 5/4 = start
            // slots: 0 at entry (after C + A of the previous iteration), 1 after bar1, 2 after B, 3 after bar2, 4 after a redo, 5 end
            long long acc[6] = {0, 0, 0, 0, 0, 0};
            int nredo = 0;
            for (int r = 1; r < pit && r < 1024; ++r) {
                const long long *cur = g_r2prof + (r * 16 + warp) * 8, *prv = g_r2prof + ((r - 1) * 16 + warp) * 8;
                acc[0] += cur[0] - prv[5]; acc[1] += cur[1] - cur[0]; acc[2] += cur[2] - cur[1]; acc[3] += cur[3] - cur[2];
                long long t3 = cur[3];
                if (cur[4] > cur[3]) { acc[4] += cur[4] - cur[3]; t3 = cur[4]; ++nredo; }
                acc[5] += cur[5] - t3;
            }
            printf("R2_PROF warp %d iters %d redo %d: gap %lld bar1 %lld B %lld bar2 %lld redo(A,B) %lld C+A %lld  total %lld (cycles per iteration)\n",
                   warp, iters, nredo, acc[0] / iters, acc[1] / iters, acc[2] / iters, acc[3] / iters, acc[4] / iters, acc[5] / iters,
                   (acc[0] + acc[1] + acc[2] + acc[3] + acc[4] + acc[5]) / iters);
        }
#endif
    }
}

template <typename T, int NXP, int NUP, int MAXT, bool GS>
int launch_res2(pimpc_s *h, int iters, double tol)
{
    using C = R2Cfg<T, NXP, NUP, GS>;
    const int nmain = (h->N + C::SPW - 1) / C::SPW, nthr = (nmain + 1) * 32;   // stage warps + the reducer warp
    auto kern = h->has_du ? k_res2<T, NXP, NUP, MAXT, true, GS> : k_res2<T, NXP, NUP, MAXT, false, GS>;
    const size_t smem = C::smem_bytes(nmain);
    PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    PIMPC_CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nthr, smem));
    if (occ < 1 || nthr > MAXT) { h->errmsg = "RESIDENT kernel does not fit on an SM"; return PIMPC_EINVAL; }
    const int grid = std::min(h->batch, h->sm_count * occ);
    Prob<T> p = make_prob<T>(h, tol);
    kern<<<grid, nthr, smem, h->stream>>>(p, h->alpha_tab, h->kappa_tab, iters);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    h->info.grid = grid; h->info.block = nthr; h->info.smem_bytes = smem;
    return 1;
}

} // namespace

// Padded shapes with an instantiation, smallest first: {NXP, NUP, stages per warp, max STAGE warps}; the CTA has one more
// warp, the reducer.  fp32 keeps 2 * (2 NBP + NXP) matrix words per lane in registers (88 for (12, 4)) while the CTA has at
// most 12 warps (168 registers per thread); 13..16 warps (128 registers) move the 2 NXP words of G_k to shared memory.
// fp64 doubles the words: (4, 4) only.
bool resident2_plan(const pimpc_s *h, int *nxp, int *nup, int *maxn)
{
    struct S { int nxp, nup, spw, maxw; };
    static const S f32[] = {{4, 4, 8, 15}, {8, 4, 4, 15}, {8, 8, 4, 15}, {12, 4, 4, 15}};
    static const S f64[] = {{4, 4, 8, 7}};
    const S *tab = h->dtype == PIMPC_F32 ? f32 : f64;
    const int n = h->dtype == PIMPC_F32 ? 4 : 1;
    for (int i = 0; i < n; ++i)
        if (h->nx <= tab[i].nxp && h->nu <= tab[i].nup) {
            *nxp = tab[i].nxp; *nup = tab[i].nup; *maxn = tab[i].spw * tab[i].maxw;
            return true;
        }
    return false;
}

int run_resident2(pimpc_s *h, int iters, double tol)
{
    int nxp, nup, maxn;
    if (!resident2_plan(h, &nxp, &nup, &maxn) || h->N > maxn) { h->errmsg = "RESIDENT engine not applicable"; return PIMPC_EINVAL; }
    if (h->dtype == PIMPC_F64) return launch_res2<double, 4, 4, 256, false>(h, iters, tol);
    if (nxp == 4) return launch_res2<float, 4, 4, 512, false>(h, iters, tol);
    if (nxp == 8 && nup == 4) return launch_res2<float, 8, 4, 512, false>(h, iters, tol);
    const bool small = h->N <= 44;                             // <= 11 stage warps of 4 stages + the reducer: 12 warps
    if (nxp == 8) return small ? launch_res2<float, 8, 8, 384, false>(h, iters, tol) : launch_res2<float, 8, 8, 512, true>(h, iters, tol);
    return small ? launch_res2<float, 12, 4, 384, false>(h, iters, tol) : launch_res2<float, 12, 4, 512, true>(h, iters, tol);
}
