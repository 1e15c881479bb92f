// RESIDENT engine: Algorithm 1 with one CTA per MPC instance and ONE launch per
// solve.  Everything an instance needs for all its iterations stays on chip:
//   * the stage matrices (rows of H_k, columns of Abar_{k+1}, rows of [A_k B_k], columns of B_k,
//     rows of M_k) live in REGISTERS of the lane that owns the row -- they are read from HBM once
//     per solve;
//   * the iterates (z, v, theta, beta, lambda, d, delta; current and previous) live in registers
//     of the same lane; the hats of steps 6/7 are recomputed from (cur, prev, kappa);
//   * only the vectors a mat-vec needs from other lanes (w, v-beta, h, xbar, rhs, du) go through
//     shared memory, read back with 16-byte broadcast loads.
// Mapping: a group of LPS = pow2(ceil(nb/R)) lanes owns one stage, lane li owns rows li*R..li*R+R-1
// of that stage; a warp owns 32/LPS consecutive stages; the CTA owns the whole horizon, so the
// neighbour coupling (stage k needs w_{k+1} and xbar_k) and the reduction of c (step 4) cost three
// CTA barriers per iteration and no global memory traffic.  The CTA loops over instances
// (grid-stride), so a launch covers any batch.
// c is reduced in a fixed order (xor butterflies; every warp repeats the second level), so every
// thread takes the same accept/restart decision (steps 5-7) from bit-identical numbers.
#include <algorithm>

#include "pimpc_internal.h"

namespace {

constexpr int pow2ceil_c(int v) { int p = 1; while (p < v) p <<= 1; return p; }

__device__ __forceinline__ void ld4(const float *p, float (&o)[4])
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ld4(const double *p, double (&o)[4])
{
    const double2 a = *reinterpret_cast<const double2 *>(p), b = *reinterpret_cast<const double2 *>(p + 2);
    o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}
template <typename T> __device__ __forceinline__ T clipv(T v, T lo, T hi) { return fmin(fmax(v, lo), hi); }

// own rows of a lane -> shared memory: one 8-byte store when a lane owns two fp32 rows
template <typename T, int R> __device__ __forceinline__ void st_rows(T *p, const T (&v)[R])
{
#pragma unroll
    for (int r = 0; r < R; ++r) p[r] = v[r];
}
template <> __device__ __forceinline__ void st_rows<float, 2>(float *p, const float (&v)[2])
{
    *reinterpret_cast<float2 *>(p) = make_float2(v[0], v[1]);
}

// (c0, c1) += (a0, a1) * (b0, b1): one packed FFMA2 on sm_100a (two IEEE fmas, half the issue slots); two DFMAs in fp64
__device__ __forceinline__ void fma2p(float &c0, float &c1, float a0, float a1, float b0, float b1)
{
    const float2 r = __ffma2_rn(make_float2(a0, a1), make_float2(b0, b1), make_float2(c0, c1));
    c0 = r.x; c1 = r.y;
}
__device__ __forceinline__ void fma2p(double &c0, double &c1, double a0, double a1, double b0, double b1)
{
    c0 = fma(a0, b0, c0); c1 = fma(a1, b1, c1);
}

// alpha_j and kappa_j after j consecutive accepted steps from alpha_0 = 1:
// alpha_{j+1} = 0.5 + 0.5 sqrt(1 + 4 alpha_j^2), kappa_j = (alpha_j - 1) / alpha_{j+1}.
__global__ void k_alpha_table(double *alpha, double *kappa, int n)
{
    if (blockIdx.x || threadIdx.x) return;
    double a = 1.0;
    for (int j = 0; j < n; ++j) {
        const double an = 0.5 + 0.5 * sqrt(1.0 + 4.0 * a * a);
        alpha[j] = a;
        kappa[j] = (a - 1.0) / an;
        a = an;
    }
}

template <typename T, int NX, int NU, int R>
struct RCfg {
    static constexpr int NB = NX + NU;
    static constexpr int LPS = pow2ceil_c((NB + R - 1) / R);   // lanes per stage
    static constexpr int SPW = 32 / LPS;                       // stages per warp
    static constexpr int ROWP = LPS * R;                       // padded vector length of a stage
    static constexpr int NBP = (NB + 3) / 4 * 4;
    static constexpr int NUP = (NU + 3) / 4 * 4;
    static constexpr int KAPN = 1024;                          // kappa table entries cached in smem
    // Shared memory: one block per stage slot s = k+1 (slot 0 holds xbar_0, slot NS+1 a zero w), so every
    // access of a lane is (one of three per-thread base registers) + a compile-time offset:
    //   W  w_k = zhat - vhat - ebar + lambdahat      X  xbar_{k+1}        D  vhat - betahat     H  h_k
    //   RH rhs of the Delta-u update    DU Delta u_k   AT columns of Abar_{k+1} (rows < nx), [R][NX/4][LPS][4]
    static constexpr int OW = 0, OX = ROWP, OD = 2 * ROWP, OH = 3 * ROWP, ORH = 4 * ROWP, ODU = ORH + NUP,
                         OC = ODU + NUP /* qbar, e, du_lo, du_hi rows */, OAT = OC + 4 * ROWP, SS0 = OAT + NX * ROWP;
    // stage stride == LPS (mod 32 words): the groups of a warp hit disjoint banks on own-element accesses
    // (two rows per lane: 16 words, so that the 8-byte own-row accesses of a half-warp hit disjoint banks)
    static constexpr int SST = (R == 2 && sizeof(T) == 4) ? 16 : LPS;
    static constexpr int SS = SS0 + ((SST - SS0 % 32) + 32) % 32;
    static_assert(NX % 4 == 0 && NX + NUP == NBP, "RESIDENT engine needs nx % 4 == 0");
    static_assert(NX % R == 0 && LPS <= 32 && LPS >= 4 && ROWP >= NBP && ROWP % 4 == 0 && SS % 4 == 0, "bad row blocking");
    static size_t smem_bytes(int nwarps)
    {
        const size_t NS = (size_t)nwarps * SPW;
        return ((NS + 2) * SS + KAPN) * sizeof(T) + 36 * sizeof(double);
    }
};

template <typename T, int R>
struct RState { T z[R], v[R], th[R], be[R], la[R], d[R], de[R]; };

// DU: the Delta-u box block (reading R12) is active.  Pad rows / pad stages carry zero matrices, zero
// bounds and zero iterates, so they run the same instructions and contribute exact zeros.
template <typename T, int NX, int NU, int R, int MAXT, bool DU>
__global__ void __launch_bounds__(MAXT, 1)      // the register file is split per SM sub-partition: 7 warps x 72 regs
k_resident(const Prob<T> p, const double *__restrict__ alpha_tab, const double *__restrict__ kappa_tab, const int iters)
{
    using C = RCfg<T, NX, NU, R>;
    constexpr int NB = C::NB, LPS = C::LPS, SPW = C::SPW, NBP = C::NBP, NUP = C::NUP, SS = C::SS;
    constexpr int OW = C::OW, OX = C::OX, OD = C::OD, OH = C::OH, ORH = C::ORH, ODU = C::ODU, OAT = C::OAT, OC = C::OC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int NS = nwarps * SPW, N = p.N;
    double *red = reinterpret_cast<double *>(smem_raw);       // [32] warp partials of c, [32..33] c of the last two iterations
    int *sCnt = reinterpret_cast<int *>(red + 34);            // [0] restarts
    T *sKap = reinterpret_cast<T *>(red + 36);                // [KAPN]
    T *sBlk = sKap + C::KAPN;                                 // [NS+2][SS]

    const int li = lane % LPS, k = warp * SPW + lane / LPS;
    const bool stage_ok = k < N;
    const T rho = (T)p.rho;
    T *const blk = sBlk + (size_t)(k + 1) * SS;               // block of the own stage
    T *const own = blk + li * R;                              // + own rows
    T *const atp = blk + OAT + li * 4;                        // + own lane slot of the Abar^T columns
    const bool has_e = p.e != nullptr, has_q = p.has_q != 0;

    for (int i = tid; i < (NS + 2) * SS; i += blockDim.x) sBlk[i] = (T)0;      // pads must stay finite zeros
    for (int i = tid; i < min(iters + 1, C::KAPN); i += blockDim.x) sKap[i] = (T)kappa_tab[i];
    __syncthreads();

    for (int b = blockIdx.x; b < p.batch; b += gridDim.x) {
        const int i_cur = p.ctl[b].i_cur;
        const size_t sk = (size_t)b * N + (stage_ok ? k : 0);
        // ---- stage matrices -> registers / smem (once per solve) ------------------------------
        T Hrow[R][NBP], U[R][NBP], lo[R], hi[R];
        bool isx[R];
        RState<T, R> sa, sb;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = li * R + r;
            const bool ok = stage_ok && i < NB;
            isx[r] = i < NX || !stage_ok;              // pad stages: every row takes the (all-zero) x-row path
            const bool okx = ok && i < NX, oku = ok && i >= NX;
            const bool inner = ok && k < N - 1;
            const T *Hk = p.H + sk * NB * NB + (size_t)(ok ? i : 0) * NB;
#pragma unroll
            for (int j = 0; j < NBP; ++j) Hrow[r][j] = (ok && j < NB) ? Hk[j] : (T)0;
            const T *A1 = p.A + (sk + (inner ? 1 : 0)) * NX * NX, *B1 = p.B + (sk + (inner ? 1 : 0)) * NX * NU;
#pragma unroll
            for (int q = 0; q < NX; ++q)                       // column i of Abar_{k+1} (rows < nx)
                atp[((r * (NX / 4) + q / 4) * LPS) * 4 + (q & 3)] =
                    !inner ? (T)0 : (i < NX ? A1[q * NX + i] : B1[q * NU + (i - NX)]);
            const T *Ak = p.A + sk * NX * NX, *Bk = p.B + sk * NX * NU, *Mk = p.M + sk * NU * NU;
#pragma unroll
            for (int j = 0; j < NBP; ++j) {
                T v = (T)0;
                if (okx) v = j < NX ? Ak[i * NX + j] : (j < NB ? Bk[i * NU + (j - NX)] : (T)0);    // row i of [A_k B_k]
                else if (oku) v = j < NX ? Bk[j * NU + (i - NX)] : (j < NB ? Mk[(i - NX) * NU + (j - NX)] : (T)0);
                U[r][j] = v;                                   // u-rows: column of B_k, then row of M_k
            }
            lo[r] = ok ? p.lo[(size_t)b * p.bnd_stride + i] : (T)0;
            hi[r] = ok ? p.hi[(size_t)b * p.bnd_stride + i] : (T)0;
            // per-row constants read back from smem only when present: qbar_i, e_i, du bounds
            own[OC + r] = ok ? p.qbar[(size_t)b * p.qbar_stride + i] : (T)0;
            own[OC + C::ROWP + r] = (okx && has_e) ? p.e[sk * NX + i] : (T)0;
            own[OC + 2 * C::ROWP + r] = (oku && DU) ? p.dlo[(size_t)b * p.dbnd_stride + (i - NX)] : (T)0;
            own[OC + 3 * C::ROWP + r] = (oku && DU) ? p.dhi[(size_t)b * p.dbnd_stride + (i - NX)] : (T)0;
            // ---- iterate of the previous solve / cold start (hats = iterates: prev = cur) --------
            const T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(b, stage_ok ? k : 0);
            sa.z[r] = ok ? rec[p.oZ() + i] : (T)0;
            sa.v[r] = ok ? rec[p.oV() + i] : (T)0;
            sa.th[r] = ok ? rec[p.oTH() + i] : (T)0;
            sa.be[r] = ok ? rec[p.oBE() + i] : (T)0;
            sa.la[r] = ok ? rec[p.oLA() + i] : (T)0;
            sa.d[r] = (oku && DU) ? rec[p.oD() + (i - NX)] : (T)0;
            sa.de[r] = (oku && DU) ? rec[p.oDE() + (i - NX)] : (T)0;
        }
        sb = sa;
        if (tid < C::ROWP)                                     // slot 0: xbar_0 = (x(t); u(t-1))
            sBlk[OX + tid] = tid < NX ? p.x0[(size_t)b * NX + tid] : (tid < NB ? p.uprev[(size_t)b * NU + (tid - NX)] : (T)0);
        if (tid == 0) { red[32] = p.c0; red[33] = p.c0; sCnt[0] = 0; }

        T kap = (T)0;
        int jacc = 0, it_done = 0;
        bool done = false;
        double *const hc = p.hist_c ? p.hist_c + (size_t)b * p.hist_cap : nullptr;
        unsigned char *const ha = p.hist_a ? p.hist_a + (size_t)b * p.hist_cap : nullptr;

        // One iteration of Alg. 1.  cur/prv: iterate i and i-1; the new iterate overwrites prv.
        // par = it & 1 (compile-time after unrolling by two): c^{i} sits in red[32 + (par ^ 1)], c^{i+1} goes to red[32 + par].
        auto iteration = [&](RState<T, R> &cur, RState<T, R> &prv, const int it, const int par) -> bool {
            T zh[R], vh[R], thh[R], beh[R], lah[R], dh[R], deh[R], dv[R], ev[R], wv[R];
            // steps 6/7 of the previous iteration: hats from (cur, prev, kappa)
#pragma unroll
            for (int r = 0; r < R; ++r) {
                zh[r] = cur.z[r] + kap * (cur.z[r] - prv.z[r]);
                vh[r] = cur.v[r] + kap * (cur.v[r] - prv.v[r]);
                thh[r] = cur.th[r] + kap * (cur.th[r] - prv.th[r]);
                beh[r] = cur.be[r] + kap * (cur.be[r] - prv.be[r]);
                lah[r] = cur.la[r] + kap * (cur.la[r] - prv.la[r]);
                if (DU) {
                    dh[r] = cur.d[r] + kap * (cur.d[r] - prv.d[r]);
                    deh[r] = cur.de[r] + kap * (cur.de[r] - prv.de[r]);
                }
                dv[r] = vh[r] - beh[r];
                T w = zh[r] - vh[r] + lah[r];
                ev[r] = (T)0;
                if (has_e) { ev[r] = own[OC + C::ROWP + r]; w -= ev[r]; }
                wv[r] = w;
            }
            st_rows<T, R>(own + OW, wv);
            st_rows<T, R>(own + OD, dv);
            __syncthreads();
            // step 1: g = Abar_{k+1}^T w_{k+1}, rhs = Bbar_k^T (vhat - betahat) [+ dhat - deltahat]
            T g[R][2], rd[R][2];
#pragma unroll
            for (int r = 0; r < R; ++r) { g[r][0] = g[r][1] = (T)0; rd[r][0] = rd[r][1] = (T)0; }
#pragma unroll
            for (int c4 = 0; c4 < NX; c4 += 4) {
                T w4[4], d4[4];
                ld4(blk + SS + OW + c4, w4);
                ld4(blk + OD + c4, d4);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    T a4[4];
                    ld4(atp + ((r * (NX / 4) + c4 / 4) * LPS) * 4, a4);
#pragma unroll
                    for (int q = 0; q < 4; q += 2) {
                    fma2p(g[r][0], g[r][1], a4[q], a4[q + 1], w4[q], w4[q + 1]);
                    fma2p(rd[r][0], rd[r][1], U[r][c4 + q], U[r][c4 + q + 1], d4[q], d4[q + 1]);
                }
                }
            }
            T hv[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                T gg = g[r][0] + g[r][1];
                if (!isx[r]) gg += own[SS + OW + r];                                // the [0 I] rows of Abar_{k+1}
                T hh = rho * (zh[r] - thh[r]) + rho * gg;                           // h_k (index reading R2)
                if (has_q) hh += own[OC + r];
                hv[r] = hh;
                T rr = rd[r][0] + rd[r][1] + dv[r];
                if (DU) rr += dh[r] - deh[r];
                if (!isx[r]) own[ORH - NX + r] = rr;
            }
            st_rows<T, R>(own + OH, hv);
            __syncwarp();
            T x[R][2], du2[R][2], du[R];
#pragma unroll
            for (int r = 0; r < R; ++r) { x[r][0] = x[r][1] = (T)0; du2[r][0] = du2[r][1] = (T)0; }
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                T h4[4];
                ld4(blk + OH + c4, h4);
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int q = 0; q < 4; q += 2)                                        // xbar_{k+1} = H_k h_k
                        fma2p(x[r][0], x[r][1], Hrow[r][c4 + q], Hrow[r][c4 + q + 1], h4[q], h4[q + 1]);
            }
#pragma unroll
            for (int c4 = 0; c4 < NUP; c4 += 4) {
                T r4[4];
                ld4(blk + ORH + c4, r4);
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int q = 0; q < 4; q += 2)                                        // Delta u_k = M_k rhs (u-rows)
                        fma2p(du2[r][0], du2[r][1], U[r][NX + c4 + q], U[r][NX + c4 + q + 1], r4[q], r4[q + 1]);
            }
            T xs[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                xs[r] = x[r][0] + x[r][1];
                du[r] = du2[r][0] + du2[r][1];
                if (!isx[r]) own[ODU - NX + r] = du[r];
            }
            st_rows<T, R>(own + OX, xs);
            __syncthreads();
            // steps 2-4
            T dot[R][2], av2[R][2], avx[R];
#pragma unroll
            for (int r = 0; r < R; ++r) { dot[r][0] = dot[r][1] = (T)0; av2[r][0] = av2[r][1] = (T)0; }
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                T x4[4];
                ld4(blk - SS + OX + c4, x4);
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int q = 0; q < 4; q += 2)                                        // [A_k B_k] xbar_k (x-rows)
                        fma2p(dot[r][0], dot[r][1], U[r][c4 + q], U[r][c4 + q + 1], x4[q], x4[q + 1]);
            }
#pragma unroll
            for (int c4 = 0; c4 < NUP; c4 += 4) {
                T u4[4];
                ld4(blk + ODU + c4, u4);
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int q = 0; q < 4; q += 2)                                        // B_k Delta u_k (x-rows)
                        fma2p(av2[r][0], av2[r][1], U[r][NX + c4 + q], U[r][NX + c4 + q + 1], u4[q], u4[q + 1]);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) avx[r] = av2[r][0] + av2[r][1];
            T acc = (T)0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T xpi = own[-SS + OX + r];
                const T duu = isx[r] ? (T)0 : du[r];
                const T av = (isx[r] ? avx[r] : du[r]) + beh[r];                 // a = Bbar du + betahat
                const T bv = (isx[r] ? dot[r][0] + dot[r][1] + ev[r] : xpi) - lah[r];   // b = Abar xbar_k + ebar - lambdahat
                const T gam = av - bv;
                const T zn = clipv(((T)2 * (xs[r] + thh[r] + bv) + gam) * (T)(1.0 / 3.0), lo[r], hi[r]);
                const T vn = (T)0.5 * (zn + gam);
                const T thn = thh[r] + xs[r] - zn;
                const T ben = av - vn;
                const T lan = zn - bv - vn;
                const T d0 = thn - thh[r], d1 = ben - beh[r], d2 = lan - lah[r], d3 = zn - zh[r], d4 = vn - vh[r];
                const T d5 = (zn - vn) - (zh[r] - vh[r]);
                acc += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5;
                prv.z[r] = zn; prv.v[r] = vn; prv.th[r] = thn; prv.be[r] = ben; prv.la[r] = lan;
                if (DU) {                                                      // Delta-u box copy (reading R12); x-rows: zeros
                    const T dn = clipv(duu + deh[r], own[OC + 2 * C::ROWP + r], own[OC + 3 * C::ROWP + r]);
                    const T den = deh[r] + duu - dn;
                    const T e0 = den - deh[r], e1 = dn - dh[r];
                    acc += e0 * e0 + e1 * e1;
                    prv.d[r] = dn; prv.de[r] = den;
                }
            }
            // step 4: c = rho * sum (fixed order: group butterfly in T, then double).  An all-fp32 butterfly was measured
            // only 1.7 % faster on C4 and would widen the near-tie band of the decision, so c stays in double.
#pragma unroll
            for (int o = LPS / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            double s = (double)acc;
#pragma unroll
            for (int o = 16; o >= LPS; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) red[warp] = s;
            __syncthreads();
            const double c_prev = red[32 + (par ^ 1)];
            // every warp repeats the second level (butterfly over the warp partials): same bits everywhere.  A shuffle-free
            // tree of 16 broadcast loads + DADDs per lane was measured 4 % slower on C4 (B200).
            s = lane < nwarps ? red[lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
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
                kap = jacc < C::KAPN ? sKap[jacc] : (T)kappa_tab[jacc];
                ++jacc;
            } else {
                kap = (T)0; jacc = 0;
            }
            return false;
        };

        __syncthreads();
        bool in_b = false;                       // which of (sa, sb) holds the current iterate
        for (int it = 0; it < iters; it += 2) {
            if (iteration(sa, sb, it, 0)) { in_b = true; break; }
            in_b = true;
            if (it + 1 >= iters) break;
            if (iteration(sb, sa, it + 1, 1)) { in_b = false; break; }
            in_b = false;
        }
        if (in_b) sa = sb;                       // register moves; a reference select would force local memory
        const RState<T, R> &fin = sa;

        // ---- results: iterate -> S[i_cur], xbar and Delta u of the last iteration, control block ----
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = li * R + r;
            if (stage_ok && i < NB) {
                T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(b, k);
                rec[p.oZ() + i] = fin.z[r]; rec[p.oV() + i] = fin.v[r]; rec[p.oTH() + i] = fin.th[r];
                rec[p.oBE() + i] = fin.be[r]; rec[p.oLA() + i] = fin.la[r];
                p.X[sk * NB + i] = own[OX + r];
                if (i >= NX) {
                    p.DU[sk * NU + (i - NX)] = own[ODU - NX + r];
                    if (DU) { rec[p.oD() + (i - NX)] = fin.d[r]; rec[p.oDE() + (i - NX)] = fin.de[r]; }
                }
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

template <typename T, int NX, int NU, int R, int MAXT>
int launch_resident(pimpc_s *h, int iters, double tol, int nwarps)
{
    using C = RCfg<T, NX, NU, R>;
    auto kern = h->has_du ? k_resident<T, NX, NU, R, MAXT, true> : k_resident<T, NX, NU, R, MAXT, false>;
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

// The one-row-per-lane kernel above serves fp32 (12, 4) horizons beyond the 13 warps of the two-rows-per-lane kernel
// (61 <= N <= 64: 15 stage warps + the reducer) and opts.tune.rows_per_lane = 1; every other RESIDENT solve runs k_res2 (k_resident2.cu).
static bool one_row_shape(const pimpc_s *h) { return h->dtype == PIMPC_F32 && h->nx == 12 && h->nu == 4 && h->N <= 64; }

bool resident_supported(const pimpc_s *h, std::string *why)
{
    int nxp, nup, maxn;
    if (resident2_plan(h, &nxp, &nup, &maxn) && h->N <= maxn) return true;
    if (one_row_shape(h)) return true;
    if (why) *why = "no register-resident instantiation for this (dtype, nx, nu, N)";
    return false;
}

int ensure_alpha_table(pimpc_s *h, int iters)
{
    int launches = 0;
    if (h->tab_cap < iters + 2) {
        const int cap = std::max(iters + 2, 1024);
        size_t ca = (size_t)h->tab_cap * sizeof(double), ck = ca;
        int rc = pimpc_grow(h, (void **)&h->alpha_tab, &ca, cap * sizeof(double));
        if (!rc) rc = pimpc_grow(h, (void **)&h->kappa_tab, &ck, cap * sizeof(double));
        if (rc) { h->tab_cap = 0; return rc; }
        k_alpha_table<<<1, 32, 0, h->stream>>>(h->alpha_tab, h->kappa_tab, cap);
        PIMPC_CUDA_TRY(h, cudaGetLastError());
        h->tab_cap = cap;
        ++launches;
    }
    return launches;
}

int run_resident(pimpc_s *h, int iters, double tol)
{
    if (!resident_supported(h, nullptr)) { h->errmsg = "RESIDENT engine not applicable"; return PIMPC_EINVAL; }
    const int launches = ensure_alpha_table(h, iters);
    if (launches < 0) return launches;
    int nxp, nup, maxn, n;
    const bool two = resident2_plan(h, &nxp, &nup, &maxn) && h->N <= maxn;
    if (two && !(h->tune.rows_per_lane == 1 && one_row_shape(h))) {
        n = run_resident2(h, iters, tol);
    } else {
        const int nwarps = (h->N + 1) / 2;                     // 16 lanes per stage, 2 stages per warp
        n = nwarps <= 25 ? launch_resident<float, 12, 4, 1, 800>(h, iters, tol, nwarps)
                         : launch_resident<float, 12, 4, 1, 1024>(h, iters, tol, nwarps);
    }
    return n < 0 ? n : n + launches;
}
