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
//   G     row of G_k = rho H_k [A_{k+1} B_{k+1}]^T  (nb x nx), formed in double   -- step 1 re-associated:
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
// Three CTA barriers per iteration.  c (step 4) is reduced in a fixed order: stage sums in T (xor butterfly over the
// group), warp sums and the sum over warps in double; every thread takes the same accept / restart decision (steps
// 5-7) from bit-identical numbers.
#include <algorithm>

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
    static constexpr int MAXW = 16;                           // warps per CTA (second reduction level reads 16 partials)
    // One block per stage slot s = k + 1 (slot 0 holds xbar_0, slot NS + 1 a zero w):
    //   W  w_k = zhat - vhat - ebar + lambdahat     T  t_k = qbar + rho (zhat - thetahat)
    //   RR (vhat - betahat) with (dhat - deltahat) added on the u rows      X  xbar_{k+1}      DU Delta u_k
    //   E  e_k per row (read only when present)
    // and once per CTA (the same for every stage): per-row constants B = qbar, du_lo, du_hi, lo, hi
    //   G  the lane's two rows of G_k, [2][NXP / 4][LPS][4] (a warp's 16-byte loads are contiguous per group, conflict-free):
    //      written by the prologue; read every iteration when the rows do not fit in registers (GS: more than 12 warps cap
    //      a thread at 128 registers), else copied to registers once
    static constexpr int OW = 0, OT = ROWP, ORR = 2 * ROWP, OX = 3 * ROWP, ODU = 4 * ROWP, OE = ODU + NUP, OG = OE + ROWP,
                         SS0 = OG + NXP * ROWP;
    // slot stride == 64 / SPW words (mod 32): shared memory serves 8- and 16-byte accesses one half-warp at a time, and
    // the SPW / 2 groups of a half-warp then hit disjoint banks with their own-row accesses and their broadcast chunks
    // (measured on B200: 8-byte own-row stores 2 wavefronts instead of 4 with a stride of 32 / SPW)
    static constexpr int TGT = (64 / SPW) % 32;
    static constexpr int SSW0 = SS0 * WPE;
    static constexpr int SSW = SSW0 + ((TGT - SSW0 % 32) + 32) % 32;
    static constexpr int SS = SSW / WPE;
    static_assert(NXP % 4 == 0 && NUP % 4 == 0 && LPS >= 4 && LPS <= 32 && ROWP >= NBP && (SS * sizeof(T)) % 16 == 0 && SSW % WPE == 0, "bad row blocking");
    static size_t smem_bytes(int nwarps)
    {
        const size_t NS = (size_t)nwarps * SPW;
        return ((NS + 2) * SS + KAPN + 10 * ROWP) * sizeof(T) + 40 * sizeof(double);
    }
};

template <typename P> struct R2State { P z, v, th, be, la, d, de; };

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
    constexpr int NG = GS ? 1 : NXP;                          // register copy of G only when it is not in shared memory
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int NS = nwarps * SPW, N = p.N, nx = p.nx, nu = p.nu, nb = p.nb;
    double *red = reinterpret_cast<double *>(smem_raw);       // [16] warp partials of c (zero beyond nwarps), [32..33] c of the last two iterations
    int *sCnt = reinterpret_cast<int *>(red + 34);            // [0] restarts
    T *sKap = reinterpret_cast<T *>(red + 40);                // [KAPN]
    T *sBnd = sKap + C::KAPN;                                 // [5][ROWP] qbar, du_lo, du_hi, lo, hi by padded row, then
                                                              // [5][ROWP] zeros: the constants of the pad stages (k >= N)
    T *sBlk = sBnd + 10 * ROWP;                               // [NS + 2][SS]

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
    if (tid < 16) red[tid] = 0.0;
    for (int i = tid; i < 5 * ROWP; i += blockDim.x) sBnd[5 * ROWP + i] = (T)0;
    __syncthreads();

    for (int b = blockIdx.x; b < p.batch; b += gridDim.x) {
        const int i_cur = p.ctl[b].i_cur;
        const size_t sk = (size_t)b * N + (stage_ok ? k : 0);
        const bool inner = stage_ok && k < N - 1;
        // ---- stage matrices -> registers (once per solve) ----------------------------------------------------------
        T Hrow[2][NBP], G[2][NG], U[2][NBP];
        R2State<P> sa, sb;
        {
            // J_k = M_k Bbar_k^T: its nu x nx block M_k B_k^T is formed by the whole lane group (rolled loops,
            // double accumulation) in the scratch that later holds G_k, then picked up by the u rows
            if (stage_ok) {
                const T *Bk = p.B + sk * nx * nu, *Mk = p.M + sk * nu * nu;
#pragma unroll 1
                for (int e = li; e < NUP * NXP; e += LPS) {
                    const int iu = e / NXP, j = e - iu * NXP;
                    double s = 0.0;
                    if (iu < nu && j < nx)
                        for (int c = 0; c < nu; ++c) s += (double)Mk[iu * nu + c] * (double)Bk[j * nu + c];
                    blk[OG + e] = (T)s;
                }
            }
            __syncwarp();
            T st_[7][2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int gi = gidx(i0 + r);
                const bool ok = stage_ok && gi >= 0;
                const bool okx = ok && i0 < NXP, oku = ok && i0 >= NXP;
                const T *Hk = p.H + sk * nb * nb + (size_t)(ok ? gi : 0) * nb;
#pragma unroll
                for (int j = 0; j < NBP; ++j) { const int gj = gidx(j); Hrow[r][j] = (ok && gj >= 0) ? Hk[gj] : (T)0; }
                const T *Ak = p.A + sk * nx * nx, *Bk = p.B + sk * nx * nu, *Mk = p.M + sk * nu * nu;
#pragma unroll
                for (int j = 0; j < NBP; ++j) {
                    const int gj = gidx(j);
                    T v = (T)0;
                    if (okx && gj >= 0) v = j < NXP ? Ak[gi * nx + gj] : Bk[gi * nu + (gj - nx)];          // row of [A_k B_k]
                    else if (oku && gj >= 0) v = j >= NXP ? Mk[(size_t)(gi - nx) * nu + (gj - nx)]        // row of M_k
                                                         : blk[OG + (i0 + r - NXP) * NXP + j];                // row of M_k B_k^T (staged below)
                    U[r][j] = v;
                }
                own[OE + r] = (okx && has_e) ? p.e[sk * nx + gi] : (T)0;
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
            __syncwarp();                                      // the scratch is reused
            // G_k rows = rho * Hrow . [A_{k+1} B_{k+1}]^T, accumulated in double (the factors are the rounded inputs); a
            // rolled loop over the nx rows of [A_{k+1} B_{k+1}], every element loaded once for both rows of the lane
            {
                const T *A1 = p.A + (sk + (inner ? 1 : 0)) * nx * nx, *B1 = p.B + (sk + (inner ? 1 : 0)) * nx * nu;
#pragma unroll 1
                for (int j = 0; j < NXP; ++j) {
                    double s0 = 0.0, s1 = 0.0;
                    if (inner && j < nx) {
#pragma unroll
                        for (int c = 0; c < NBP; ++c) {
                            const int gc = gidx(c);
                            if (gc >= 0) {
                                const double a = (double)(c < NXP ? A1[j * nx + gc] : B1[j * nu + (gc - nx)]);
                                s0 += (double)Hrow[0][c] * a; s1 += (double)Hrow[1][c] * a;
                            }
                        }
                    }
                    blk[OG + ((0 * (NXP / 4) + j / 4) * LPS + li) * 4 + (j & 3)] = (T)(p.rho * s0);
                    blk[OG + ((1 * (NXP / 4) + j / 4) * LPS + li) * 4 + (j & 3)] = (T)(p.rho * s1);
                }
                if (!GS) {
#pragma unroll
                    for (int r = 0; r < 2; ++r)
#pragma unroll
                        for (int j = 0; j < NXP; ++j) G[r][j % NG] = blk[OG + ((r * (NXP / 4) + j / 4) * LPS + li) * 4 + (j & 3)];
                }
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
            sBlk[OX + tid] = (tid < NBP && g0 >= 0) ? (tid < NXP ? p.x0[(size_t)b * nx + g0] : p.uprev[(size_t)b * nu + (g0 - nx)]) : (T)0;
        }
        if (tid == 0) { red[32] = p.c0; red[33] = p.c0; sCnt[0] = 0; }

        T kap = (T)0;
        int jacc = 0, it_done = 0;
        bool done = false;
        double *const hc = p.hist_c ? p.hist_c + (size_t)b * p.hist_cap : nullptr;
        unsigned char *const ha = p.hist_a ? p.hist_a + (size_t)b * p.hist_cap : nullptr;

        // One iteration of Alg. 1.  cur/prv: iterate i and i-1; the hats overwrite prv's registers, then the new iterate does.
        // par = it & 1 (compile-time after unrolling by two): c^{i} sits in red[32 + (par ^ 1)], c^{i+1} goes to red[32 + par].
        auto iteration = [&](R2State<P> &cur, R2State<P> &prv, const int it, const int par) -> bool {
            // ---- A: steps 6/7 of the previous iteration: hats from (cur, prev, kappa) ----
            const P kap2 = mk2(kap, kap);
            const P zh = fma2(kap2, sub2(cur.z, prv.z), cur.z);
            const P vh = fma2(kap2, sub2(cur.v, prv.v), cur.v);
            const P thh = fma2(kap2, sub2(cur.th, prv.th), cur.th);
            const P beh = fma2(kap2, sub2(cur.be, prv.be), cur.be);
            const P lah = fma2(kap2, sub2(cur.la, prv.la), cur.la);
            P dh = mk2((T)0, (T)0), deh = dh;
            if (DU) {
                dh = fma2(kap2, sub2(cur.d, prv.d), cur.d);
                deh = fma2(kap2, sub2(cur.de, prv.de), cur.de);
            }
            P wv = add2(sub2(zh, vh), lah);                                     // w_k = zhat - vhat - ebar + lambdahat
            if (has_e) wv = sub2(wv, ldp(own + OE));
            P tv = mul2(rho2, sub2(zh, thh));                                   // t_k = rho (zhat - thetahat) [+ qbar]
            if (has_q) tv = add2(tv, ldp(bnd));
            P rr = sub2(vh, beh);                                               // vhat - betahat [+ dhat - deltahat]
            if (DU) rr = add2(rr, sub2(dh, deh));
            stp(own + OW, wv); stp(own + OT, tv); stp(own + ORR, rr);
            // (neighbour-to-neighbour mbarrier hand-overs instead of this CTA barrier and the next were measured 12 % slower)
            __syncthreads();
            // ---- B: step 1: xbar_{k+1} = Hrow (t + rho [0; w_u]) + G w_x;  Delta u_k = [M B^T | M] rr ----
            P xa[2], da[2];
            xa[0] = xa[1] = da[0] = da[1] = mk2((T)0, (T)0);
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                P t0, t1, w0, w1, r0, r1;
                ld4p(blk + OT + c4, t0, t1);
                ld4p(blk + SS + OW + c4, w0, w1);
                ld4p(blk + ORR + c4, r0, r1);
                if (c4 >= NXP) { t0 = fma2(rho2, w0, t0); t1 = fma2(rho2, w1, t1); }       // the [0 I] rows of Abar_{k+1}
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    xa[r] = fma2(mk2(Hrow[r][c4], Hrow[r][c4 + 1]), t0, xa[r]);
                    xa[r] = fma2(mk2(Hrow[r][c4 + 2], Hrow[r][c4 + 3]), t1, xa[r]);
                    if (c4 < NXP) {
                        if (GS) {
                            P g0, g1;
                            ld4p(blk + OG + ((r * (NXP / 4) + c4 / 4) * LPS + li) * 4, g0, g1);
                            xa[r] = fma2(g0, w0, xa[r]);
                            xa[r] = fma2(g1, w1, xa[r]);
                        } else {
                            xa[r] = fma2(mk2(G[r][c4 % NG], G[r][(c4 + 1) % NG]), w0, xa[r]);
                            xa[r] = fma2(mk2(G[r][(c4 + 2) % NG], G[r][(c4 + 3) % NG]), w1, xa[r]);
                        }
                    }
                    da[r] = fma2(mk2(U[r][c4], U[r][c4 + 1]), r0, da[r]);
                    da[r] = fma2(mk2(U[r][c4 + 2], U[r][c4 + 3]), r1, da[r]);
                }
            }
            const P xs = mk2(xa[0].x + xa[0].y, xa[1].x + xa[1].y);
            const P du = mk2(da[0].x + da[0].y, da[1].x + da[1].y);              // meaningful on the u rows only
            stp(own + OX, xs);
            if (isu) stp(own + ODU - NXP, du);
            __syncthreads();
            // ---- C: steps 2-4 ----
            P ba[2], aa[2], xu0 = mk2((T)0, (T)0), xu1 = xu0;
            ba[0] = ba[1] = aa[0] = aa[1] = mk2((T)0, (T)0);
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                P x0, x1;
                ld4p(blk - SS + OX + c4, x0, x1);
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
                ld4p(blk + ODU + c4, u0, u1);
#pragma unroll
                for (int r = 0; r < 2; ++r) {                                               // B_k Delta u_k (x rows)
                    aa[r] = fma2(mk2(U[r][NXP + c4], U[r][NXP + c4 + 1]), u0, aa[r]);
                    aa[r] = fma2(mk2(U[r][NXP + c4 + 2], U[r][NXP + c4 + 3]), u1, aa[r]);
                }
            }
            // own rows of xbar_k (u rows: the [0 I] rows of Abar_k): with four u rows they sit in the chunk just loaded
            const P xpi = NUP == 4 ? ((li & 1) ? xu1 : xu0) : ldp(own - SS + OX);
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
            // step 4: c = rho * sum (fixed order: group butterfly in T, then double)
            T acc = acc2.x + acc2.y;
#pragma unroll
            for (int o = LPS / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            double s = (double)acc;
#pragma unroll
            for (int o = 16; o >= LPS; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) red[warp] = s;
            const T kap_acc = jacc < C::KAPN ? sKap[jacc] : (T)kappa_tab[jacc];     // momentum if the step is accepted: off the decision's path
            __syncthreads();
            const double c_prev = red[32 + (par ^ 1)];
            // second level, same bits in every thread: the 16 partials (zeros beyond the CTA's warps), one per lane of each
            // half-warp, then a four-level butterfly.  Measured on B200 (C4, kernel ms): this 7.95, four partials per lane
            // + two levels 8.07, sixteen same-address loads + a tree of DADDs 8.13
            s = red[lane & 15];
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            // steps 5-7; every thread decides from the same bits
            const double c = p.rho * s;
            it_done = it + 1;
            const bool stop = p.tol > 0.0 && c < p.tol;
            const bool accept = !stop && c <= p.eta * c_prev;
            if (tid == 0) {
                red[32 + par] = c;
                if (!accept && !stop) ++sCnt[0];
                if (hc && it < p.hist_cap) { hc[it] = c; ha[it] = (unsigned char)accept; }
            }
            if (stop) { done = true; return true; }
            if (accept) {
                kap = kap_acc;
                ++jacc;
            } else {
                kap = (T)0; jacc = 0;
            }
            return false;
        };

        // ---- results: iterate -> S[i_cur], xbar and Delta u of the last iteration (called at each exit of the loop: the
        // two iterate sets never merge, so the unrolled-by-two loop carries them in place without register moves) ----
        auto write_back = [&](const R2State<P> &fin) {
            const T fz[2] = {fin.z.x, fin.z.y}, fv[2] = {fin.v.x, fin.v.y}, fth[2] = {fin.th.x, fin.th.y};
            const T fbe[2] = {fin.be.x, fin.be.y}, fla[2] = {fin.la.x, fin.la.y}, fd[2] = {fin.d.x, fin.d.y}, fde[2] = {fin.de.x, fin.de.y};
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int gi = gidx(i0 + r);
                if (stage_ok && gi >= 0) {
                    T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(b, k);
                    rec[p.oZ() + gi] = fz[r]; rec[p.oV() + gi] = fv[r]; rec[p.oTH() + gi] = fth[r];
                    rec[p.oBE() + gi] = fbe[r]; rec[p.oLA() + gi] = fla[r];
                    p.X[sk * nb + gi] = own[OX + r];
                    if (i0 >= NXP) {
                        p.DU[sk * nu + (gi - nx)] = own[ODU - NXP + r];
                        if (DU) { rec[p.oD() + (gi - nx)] = fd[r]; rec[p.oDE() + (gi - nx)] = fde[r]; }
                    }
                }
            }
        };

        __syncthreads();
        {
            int it = 0;
            for (;;) {
                if (it >= iters) { write_back(sa); break; }
                if (iteration(sa, sb, it, 0) || it + 1 >= iters) { write_back(sb); break; }
                if (iteration(sb, sa, it + 1, 1)) { write_back(sa); break; }
                it += 2;
            }
        }
        __syncthreads();                         // red[], sCnt of the last iteration are visible to thread 0
        if (tid == 0) {
            InstCtl c = p.ctl[b];
            const int last = (it_done - 1) & 1;
            c.alpha = alpha_tab[jacc]; c.c_last = it_done ? red[32 + last] : p.c0;
            c.c_prev = done ? red[32 + (last ^ 1)] : c.c_last;
            c.kappa = (double)kap;
            c.done = done ? 1 : 0; c.iters = it_done; c.restarts = sCnt[0];
            p.ctl[b] = c;
        }
        __syncthreads();
    }
}

template <typename T, int NXP, int NUP, int MAXT, bool GS>
int launch_res2(pimpc_s *h, int iters, double tol)
{
    using C = R2Cfg<T, NXP, NUP, GS>;
    const int nwarps = (h->N + C::SPW - 1) / C::SPW;
    auto kern = h->has_du ? k_res2<T, NXP, NUP, MAXT, true, GS> : k_res2<T, NXP, NUP, MAXT, false, GS>;
    const size_t smem = C::smem_bytes(nwarps);
    PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    PIMPC_CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nwarps * 32, smem));
    if (occ < 1) { h->errmsg = "RESIDENT kernel does not fit on an SM"; return PIMPC_EINVAL; }
    const int grid = std::min(h->batch, h->sm_count * occ);
    Prob<T> p = make_prob<T>(h, tol);
    kern<<<grid, nwarps * 32, smem, h->stream>>>(p, h->alpha_tab, h->kappa_tab, iters);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    h->info.grid = grid; h->info.block = nwarps * 32; h->info.smem_bytes = smem;
    return 1;
}

} // namespace

// Padded shapes with an instantiation, smallest first: {NXP, NUP, stages per warp, max warps}.  fp32 keeps 2 * (2 NBP + NXP)
// matrix words per lane in registers (88 for (12, 4)) while the CTA has at most 12 warps (168 registers per thread);
// 13..16 warps (128 registers) move the 2 NXP words of G_k to shared memory.  fp64 doubles the words: (4, 4) only.
bool resident2_plan(const pimpc_s *h, int *nxp, int *nup, int *maxn)
{
    struct S { int nxp, nup, spw, maxw; };
    static const S f32[] = {{4, 4, 8, 16}, {8, 4, 4, 16}, {8, 8, 4, 16}, {12, 4, 4, 16}};
    static const S f64[] = {{4, 4, 8, 8}};
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
    const bool small = h->N <= 48;                             // <= 12 warps of 4 stages
    if (nxp == 8) return small ? launch_res2<float, 8, 8, 384, false>(h, iters, tol) : launch_res2<float, 8, 8, 512, true>(h, iters, tol);
    return small ? launch_res2<float, 12, 4, 384, false>(h, iters, tol) : launch_res2<float, 12, 4, 512, true>(h, iters, tol);
}
