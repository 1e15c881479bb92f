// COOP engine: Algorithm 1 for ONE long-horizon instance (batch = 1; C2, C3) with
// the whole problem resident on chip, spread over the SMs, and ONE cooperative launch per solve.
//   * CTA c owns the contiguous stages [k0, k1) of the horizon.  Their matrices (H_k, [A_k B_k], M_k)
//     are read from HBM once per solve into shared memory; their iterates (current and previous) live in
//     registers; a group of LPS lanes owns a stage (lane = row), SPG stages per group.
//   * The neighbour coupling across a CTA boundary costs no extra barrier: the stage before the range
//     is a "ghost" whose xbar_{k0} = H_{k0-1} h_{k0-1} is recomputed here (its H is resident too), and the
//     stage after the range is a ghost that only supplies w_{k1}.  The ghosts' iterates (z, theta) /
//     (z, v, lambda) arrive from the neighbour CTA as tagged words in global memory.
//   * The ONLY global exchange per iteration is data-flow, not a barrier: every CTA publishes its boundary
//     iterates as {value, iteration tag} words (8-byte single-copy-atomic stores, no fences) and ADDS its
//     partial sum of c (step 4), split into three fixed-point limbs, to three L2 words with
//     relaxed 64-bit atomics; integer sums are exact and order-independent, each word counts its arrivals in
//     its top bits, and a communication warp per CTA spins until the three words are complete: bit-identical c
//     in every CTA, so every thread takes the same accept / restart decision (steps 5-7).
//     Buffers are double-buffered on the iteration parity: a CTA cannot run two iterations ahead of a
//     neighbour because it needs that neighbour's next contribution first.
// The shape is PADDED at compile time (NX x-rows, NU u-rows, multiples of 4); the real nx <= NX, nu <= NU are run-time:
// pad rows and columns carry zero matrices, zero bounds and zero iterates, run the same instructions and stay exactly 0.
// The launch is cooperative only to guarantee co-residency of the polling CTAs.  Short horizons run as ONE thread-block
// cluster instead (template flag CL): the same tagged words are pushed into the peers' shared memory (DSMEM) and polled locally.
#include <algorithm>

#include "pimpc_internal.h"

namespace {

__host__ __device__ constexpr int pow2ceil_o(int v) { int p = 1; while (p < v) p <<= 1; return p; }
__host__ __device__ constexpr int round4_o(int v) { return (v + 3) / 4 * 4; }

// ---- tagged words: {value bits, iteration tag} in ONE 64-bit scalar access --------------------------------------
// The PTX memory model makes a scalar .b64 access single-copy atomic, so a reader can never pair a new tag with old
// value bits (a .v2.u32 access is two independent 32-bit accesses by specification).  fp32: one word {value, tag};
// fp64: two such words {lo, tag}, {hi, tag}, each atomic on its own, both tags must match.
// Ordering: a word is self-validating (the tag travels with the value), so no fence orders it against other words.
// Reuse of a parity buffer two iterations later is safe because the writer of iteration i+2 has consumed the partial
// sum of c of iteration i+1 from every CTA, which each CTA publishes only after its own reads of iteration i are done
// (program order through the CTA barrier between the ghost reads and the next phase D).
__device__ __forceinline__ uint64_t tw_pack(uint32_t v, uint32_t tag) { return (uint64_t)v | ((uint64_t)tag << 32); }
template <typename T> struct Tagged;
template <> struct Tagged<float> {
    typedef uint64_t W;
    static __device__ __forceinline__ void st(W *p, float v, uint32_t tag)
    {
        asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(tw_pack(__float_as_uint(v), tag)) : "memory");
    }
    static __device__ __forceinline__ bool ld(const W *p, uint32_t tag, float &v)
    {
        uint64_t w;
        asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(p) : "memory");
        v = __uint_as_float((uint32_t)w);
        return (uint32_t)(w >> 32) == tag;
    }
    // the same word in distributed shared memory: store to a peer CTA of the cluster, poll the own CTA's copy
    static __device__ __forceinline__ void st_cl(uint32_t raddr, float v, uint32_t tag)
    {
        asm volatile("st.relaxed.cluster.shared::cluster.b64 [%0], %1;" ::"r"(raddr), "l"(tw_pack(__float_as_uint(v), tag)) : "memory");
    }
    static __device__ __forceinline__ bool ld_sm(const W *p, uint32_t tag, float &v)
    {
        uint64_t w;
        asm volatile("ld.relaxed.cluster.shared::cta.b64 %0, [%1];" : "=l"(w) : "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
        v = __uint_as_float((uint32_t)w);
        return (uint32_t)(w >> 32) == tag;
    }
};
template <> struct Tagged<double> {
    typedef ulonglong2 W;
    static __device__ __forceinline__ void st(W *p, double v, uint32_t tag)
    {
        const uint64_t lo = tw_pack((uint32_t)__double2loint(v), tag), hi = tw_pack((uint32_t)__double2hiint(v), tag);
        asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(p), "l"(lo), "l"(hi) : "memory");
    }
    static __device__ __forceinline__ bool ld(const W *p, uint32_t tag, double &v)
    {
        uint64_t lo, hi;
        asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(lo), "=l"(hi) : "l"(p) : "memory");
        v = __hiloint2double((int)(uint32_t)hi, (int)(uint32_t)lo);
        return (uint32_t)(lo >> 32) == tag && (uint32_t)(hi >> 32) == tag;
    }
    static __device__ __forceinline__ void st_cl(uint32_t raddr, double v, uint32_t tag)
    {
        const uint64_t lo = tw_pack((uint32_t)__double2loint(v), tag), hi = tw_pack((uint32_t)__double2hiint(v), tag);
        asm volatile("st.relaxed.cluster.shared::cluster.v2.b64 [%0], {%1, %2};" ::"r"(raddr), "l"(lo), "l"(hi) : "memory");
    }
    static __device__ __forceinline__ bool ld_sm(const W *p, uint32_t tag, double &v)
    {
        uint64_t lo, hi;
        asm volatile("ld.relaxed.cluster.shared::cta.v2.b64 {%0, %1}, [%2];" : "=l"(lo), "=l"(hi) : "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
        v = __hiloint2double((int)(uint32_t)hi, (int)(uint32_t)lo);
        return (uint32_t)(lo >> 32) == tag && (uint32_t)(hi >> 32) == tag;
    }
};

// ---- exact, order-independent sum of the CTAs' partials of c through L2 atomics, no fences --------------------------
// A non-negative double is split into three 47-bit limbs at fixed binary points 2^-7, 2^-54, 2^-101 (it has 53 significant
// bits, so the split is exact between 2^-101 and 2^40); integer additions are associative, so the 64-bit atomic sums of the
// limbs over up to 255 CTAs are EXACT and independent of the arrival order: every CTA reads the same integers and rounds
// them to the same double.  Each limb word carries its own arrival count in its top 8 bits, so a word validates itself
// (like the tagged words of the halo exchange) and relaxed accesses suffice.  The words are never reset: in a later use of
// the same parity slot a CTA adds (new limb - its old limb) + one count, so the payload stays the sum of the CURRENT
// contributions (< 2^56 even while old and new ones are mixed) and the count advances by the grid size per use, modulo 256.
// A borrow from a transiently negative payload can only make the count look one too SMALL, never complete too early.
// One relaxed reduction per limb and a spin on three adjacent words replace the all-to-all of tagged partials.
struct Limbs { unsigned long long l[3]; };
__device__ __forceinline__ Limbs to_limbs(double s)
{
    Limbs r;
    s = fmin(fmax(s, 0.0), 1.0e12);                            // 2^40 > 1e12: the top limb stays below 2^47
    const double a = s * 128.0, fa = floor(a);                 // binary point 2^-7
    const double b = (a - fa) * 140737488355328.0, fb = floor(b);      // 2^47: binary point 2^-54
    const double c = (b - fb) * 140737488355328.0;             // binary point 2^-101
    r.l[2] = (unsigned long long)fa; r.l[1] = (unsigned long long)fb; r.l[0] = (unsigned long long)floor(c);
    return r;
}
__device__ __forceinline__ double from_limbs(unsigned long long l0, unsigned long long l1, unsigned long long l2)
{
    return (double)l2 * (1.0 / 128.0) + ((double)l1 * 5.551115123125783e-17 /* 2^-54 */ + (double)l0 * 3.944304526105059e-31 /* 2^-101 */);
}
__device__ __forceinline__ void red_add_relaxed(unsigned long long *p, unsigned long long v)
{
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// shared-memory address of the same variable in the CTA of rank `rank` of the cluster
__device__ __forceinline__ uint32_t map_peer(const void *local, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"((uint32_t)__cvta_generic_to_shared(local)), "r"(rank));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__device__ __forceinline__ void ld4o(const float *p, float (&o)[4])
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ld4o(const double *p, double (&o)[4])
{
    const double2 a = *reinterpret_cast<const double2 *>(p), b = *reinterpret_cast<const double2 *>(p + 2);
    o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}
template <typename T> __device__ __forceinline__ T clipo(T v, T lo, T hi) { return fmin(fmax(v, lo), hi); }

template <typename T, int NX, int NU>
struct OCfg {
    static constexpr int NB = NX + NU;
    static constexpr int LPS = pow2ceil_o(NB);                 // lanes per stage (one row per lane)
    static constexpr int NBP = round4_o(NB), NUP = round4_o(NU);
    static constexpr int WPE = sizeof(T) / 4;                  // 32-bit words per element
    static constexpr int HS = NBP + 4 / WPE;                   // matrix row stride: 16-byte row reads of consecutive lanes hit disjoint banks
    static constexpr int KAPN = 1024;
    static constexpr int MAXJ = 5;                             // partials polled per lane of the communication warp: grid <= 160
    // one block per virtual slot v = 0..L+1 (stage k0 - 1 + v):
    //   W w_k = zhat - vhat - ebar + lambdahat   X xbar_{k+1}   D vhat - betahat   HH h_k   RH rhs of the Delta-u update
    //   DU Delta u_k   E e_k   HM H_k [NB][HS]   AB [A_k B_k] [NX][HS]   MM M_k [NU][NUP]
    // X and DU exist twice (parity of the iteration: the speculated phases B, C of the next iteration must not destroy the
    // primal step of an iteration that turns out to have stopped): OX + par * LPS, ODU + par * NUP
    static constexpr int OW = 0, OX = LPS, OD = 3 * LPS, OHH = 4 * LPS, ORH = 5 * LPS, ODU = ORH + NUP, OE = ODU + 2 * NUP,
                         OHM = OE + LPS, OAB = OHM + NB * HS, OMM = OAB + NX * HS, SS0 = OMM + NU * NUP;
    // slot stride == LPS words (mod 32): the groups of a warp work on consecutive slots and hit disjoint banks
    static constexpr int SSW0 = SS0 * WPE;
    static constexpr int SSW = SSW0 + ((LPS - SSW0 % 32) + 32) % 32;
    static constexpr int SS = SSW / WPE;
    static_assert(SSW % WPE == 0 && SS % 4 == 0 && LPS <= 32 && NX % 4 == 0, "slot layout");
    // cluster variant: inbound exchange words in the CTA's own shared memory, [2 parities][CLMAX] partials of c and
    // [2][HALO] boundary iterates ([0, 3 LPS) from the right neighbour, [3 LPS, 5 LPS) from the left one)
    static constexpr int CLMAX = 16;
    static constexpr size_t xpart_bytes = 2 * CLMAX * 16, xhalo_bytes = 2 * 5 * LPS * 4 * sizeof(T);
    static constexpr size_t head_bytes = 40 * sizeof(double) + xpart_bytes + xhalo_bytes + (KAPN + 2 * LPS + 2 * NUP) * sizeof(T);
    // + [2][threads] per-lane partial sums of c (by parity of the iteration), behind the slots
    static size_t smem_bytes(int slots, int threads) { return head_bytes + ((size_t)slots * SS + 2 * (size_t)threads) * sizeof(T); }
    // exchange buffers per CTA and parity (tagged words): to the left neighbour (z, v, lambda) of the first stage,
    // to the right neighbour (z, theta) of the last stage
    static constexpr int HALO = 5 * LPS;
    // L2 path: two parity slots of three limb words for the exact atomic sum of c, 256 bytes apart (see to_limbs)
    static constexpr int PSTRIDE = 16, NREP = 8;               // sizing of the exchange buffer, in 16-byte words
};

template <typename T> struct OState { T z, v, th, be, la, d, de; };

// CL: the grid is ONE thread-block cluster (<= 16 CTAs) and the tagged words travel through distributed shared memory
// (a remote store lands in ~200 cycles) instead of L2 (850-1000 cycles per hop, 2400+ for an all-to-all of 64 CTAs).
template <typename T, int NX, int NU, int SPG, int MAXT, bool DU, bool CL>
__global__ void __launch_bounds__(MAXT, 1)
k_coop(const Prob<T> p, const double *__restrict__ alpha_tab, const double *__restrict__ kappa_tab, const int iters,
       typename Tagged<double>::W *__restrict__ part, typename Tagged<T>::W *__restrict__ halo, const int spec)
{
    using C = OCfg<T, NX, NU>;
    using TW = Tagged<T>;
    using TD = Tagged<double>;
    constexpr int NB = C::NB, LPS = C::LPS, NBP = C::NBP, NUP = C::NUP, HS = C::HS, SS = C::SS;
    constexpr int OW = C::OW, OX = C::OX, OD = C::OD, OHH = C::OHH, ORH = C::ORH, ODU = C::ODU, OE = C::OE, OHM = C::OHM,
                  OAB = C::OAB, OMM = C::OMM;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *red = reinterpret_cast<double *>(smem_raw);        // [32] warp partials, [32..33] c of the last two iterations
    typename TD::W *xPart = reinterpret_cast<typename TD::W *>(red + 40);                         // [2][CLMAX]
    typename TW::W *xHalo = reinterpret_cast<typename TW::W *>(smem_raw + 320 + C::xpart_bytes);  // [2][HALO]
    T *sKap = reinterpret_cast<T *>(smem_raw + 320 + C::xpart_bytes + C::xhalo_bytes);            // [KAPN]
    T *sQ = sKap + C::KAPN;                                    // [LPS] qbar
    T *sDlo = sQ + LPS, *sDhi = sDlo + NUP;                    // [NUP] Delta-u box
    T *sBlk = sDhi + NUP + (LPS - 2 * NUP % LPS) % LPS;        // [L+2][SS]   (head_bytes reserves 2 LPS + 2 NUP)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int ncw = nwarps - 1;                                // compute warps; the last warp is the communication warp
    const bool comm = warp == ncw;
    const int ngroups = ncw * (32 / LPS);
    const int g = tid / LPS, li = tid % LPS;
    const int N = p.N, G = gridDim.x, cta = blockIdx.x, nx = p.nx, nu = p.nu, nb = p.nb;
    // padded row / column index -> index in the caller's arrays (-1: pad)
    auto gidx = [&](int i) -> int { return i < NX ? (i < nx ? i : -1) : (i - NX < nu ? nx + (i - NX) : -1); };
    const int gi = li < NB ? gidx(li) : -1;
    const int k0 = (int)((long long)cta * N / G), k1 = (int)((long long)(cta + 1) * N / G), L = k1 - k0;
    const bool has_left = k0 > 0, has_right = k1 < N;
    const T rho = (T)p.rho;
    const bool has_e = p.e != nullptr, has_q = p.has_q != 0;
    const bool rowok = gi >= 0, isx = li < NX || !rowok;       // pad lanes take the x-row path with zeros
    const int i_cur = p.ctl[0].i_cur;

    // ---- once per solve: stage matrices -> shared memory, iterates -> registers ----------------------------
    for (int i = tid; i < (L + 2) * SS; i += blockDim.x) sBlk[i] = (T)0;
    for (int i = tid; i < min(iters + 1, C::KAPN); i += blockDim.x) sKap[i] = (T)kappa_tab[i];
    if (tid < LPS) { const int g0 = tid < NB ? gidx(tid) : -1; sQ[tid] = g0 >= 0 ? p.qbar[g0] : (T)0; }
    if (tid < NUP) {
        sDlo[tid] = (DU && tid < nu) ? p.dlo[tid] : (T)0;
        sDhi[tid] = (DU && tid < nu) ? p.dhi[tid] : (T)0;
    }
    if (CL) {
        for (int i = tid; i < (int)((C::xpart_bytes + C::xhalo_bytes) / 4); i += blockDim.x) reinterpret_cast<uint32_t *>(xPart)[i] = 0u;
    }
    __syncthreads();
    for (int v = 0; v <= L + 1; ++v) {
        const int k = k0 - 1 + v;
        if (k < 0 || k >= N) continue;
        T *blk = sBlk + (size_t)v * SS;
        if (v <= L)                                            // H_k: real stages and the left ghost
            for (int i = tid; i < NB * NB; i += blockDim.x) {
                const int gr = gidx(i / NB), gc = gidx(i % NB);
                blk[OHM + (i / NB) * HS + i % NB] = (gr >= 0 && gc >= 0) ? p.H[(size_t)k * nb * nb + gr * nb + gc] : (T)0;
            }
        if (v >= 1) {                                          // [A_k B_k], e_k: real stages and the right ghost
            for (int i = tid; i < NX * NB; i += blockDim.x) {
                const int r = i / NB, c = i % NB, gc = gidx(c);
                T val = (T)0;
                if (r < nx && gc >= 0) val = c < NX ? p.A[(size_t)k * nx * nx + r * nx + gc] : p.B[(size_t)k * nx * nu + r * nu + (gc - nx)];
                blk[OAB + r * HS + c] = val;
            }
            if (has_e && tid < nx) blk[OE + tid] = p.e[(size_t)k * nx + tid];
        }
        if (v >= 1 && v <= L)
            for (int i = tid; i < NU * NU; i += blockDim.x) {
                const int r = i / NU, c = i % NU;
                blk[OMM + r * NUP + c] = (r < nu && c < nu) ? p.M[(size_t)k * nu * nu + r * nu + c] : (T)0;
            }
    }
    if (!has_left && tid < LPS) {                              // slot 0 of the first CTA: xbar_0 = (x(t); u(t-1))
        const int g0 = tid < NB ? gidx(tid) : -1;
        sBlk[OX + tid] = sBlk[OX + LPS + tid] = g0 < 0 ? (T)0 : (tid < NX ? p.x0[g0] : p.uprev[g0 - nx]);
    }

    OState<T> sa[SPG], sb[SPG];
    T lo[SPG], hi[SPG];
    bool exist[SPG], real[SPG], ghl[SPG], ghr[SPG];
    T *blkp[SPG];
#pragma unroll
    for (int s = 0; s < SPG; ++s) {
        const int v = s * ngroups + g, k = k0 - 1 + v;
        exist[s] = !comm && v <= L + 1;
        real[s] = exist[s] && v >= 1 && v <= L;
        ghl[s] = exist[s] && v == 0 && has_left;
        ghr[s] = exist[s] && v == L + 1 && has_right;
        blkp[s] = sBlk + (size_t)(exist[s] ? v : 0) * SS;
        const bool ok = (real[s] || ghl[s] || ghr[s]) && rowok;
        const T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(0, ok ? k : 0);
        const bool oku = ok && li >= NX;
        sa[s].z = ok ? rec[p.oZ() + gi] : (T)0;
        sa[s].v = ok ? rec[p.oV() + gi] : (T)0;
        sa[s].th = ok ? rec[p.oTH() + gi] : (T)0;
        sa[s].be = ok ? rec[p.oBE() + gi] : (T)0;
        sa[s].la = ok ? rec[p.oLA() + gi] : (T)0;
        sa[s].d = (oku && DU) ? rec[p.oD() + (gi - nx)] : (T)0;
        sa[s].de = (oku && DU) ? rec[p.oDE() + (gi - nx)] : (T)0;
        sb[s] = sa[s];
        lo[s] = (real[s] && rowok) ? p.lo[gi] : (T)0;
        hi[s] = (real[s] && rowok) ? p.hi[gi] : (T)0;
    }
    const int hrow = rowok ? li : NB - 1;                      // clamped row indices of pad / u lanes (results unused)
    const int xrow = li < NX ? li : NX - 1;
    const int mrow = (li >= NX && rowok) ? li - NX : 0;
    const bool ulane = li >= NX && rowok;

    T kap = (T)0;                                // momentum of the hats being formed
    int jacc = 0;                                // accepted steps in a row, a pending (speculated) one counted as accepted
    unsigned long long xold[2][3] = {{0ull, 0ull, 0ull}, {0ull, 0ull, 0ull}};     // this CTA's limbs still inside the two parity slots
    // the accept / restart state of Alg. 1 lives in shared memory (lane 0 of the communication warp reads and writes it):
    // red[32] = c of the last iteration, red[33] = c of the one before, red[38] = eta * red[32], red[39] = c of the decision whose
    // bookkeeping is pending; sCtl = {accepted steps in a row, restarts, iterations, done}
    int *sCtl = reinterpret_cast<int *>(red + 36);
    if (tid == 0) { red[32] = p.c0; red[33] = p.c0; red[38] = p.eta * p.c0; sCtl[0] = sCtl[1] = sCtl[2] = sCtl[3] = 0; }
    const int slots_max = (N + G - 1) / G + 2;
    T *sAcc = sBlk + (size_t)slots_max * SS;     // [2][blockDim.x] per-lane partial sums of c by parity of the iteration
    int *sDec = reinterpret_cast<int *>(red + 34);   // decision of the communication warp: 0 accept, 1 restart, 2 stop
    __syncthreads();
    if (CL) cluster_sync_all();                  // every CTA of the cluster has zeroed its inbound words

    T zh[SPG], vh[SPG], thh[SPG], beh[SPG], lah[SPG], dh[SPG], deh[SPG], dv[SPG], ev[SPG];   // hats of the iteration in flight
    T xs[SPG], du[SPG];                                                                    // its primal step (own rows)
#pragma unroll
    for (int s = 0; s < SPG; ++s) { zh[s] = vh[s] = thh[s] = beh[s] = lah[s] = dh[s] = deh[s] = dv[s] = ev[s] = xs[s] = du[s] = (T)0; }

    // ---- A: steps 6/7 of the previous iteration: hats from (cur, prev, kappa); publish w, vhat - betahat ----
    auto publish = [&]() {
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            dv[s] = vh[s] - beh[s];
            T w = zh[s] - vh[s] + lah[s];
            ev[s] = (T)0;
            if (has_e && exist[s]) { ev[s] = blkp[s][OE + li]; w -= ev[s]; }
            if (exist[s]) { blkp[s][OW + li] = w; blkp[s][OD + li] = dv[s]; }
        }
    };
    auto phaseA = [&](OState<T> (&cur)[SPG], OState<T> (&prv)[SPG]) {
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            zh[s] = cur[s].z + kap * (cur[s].z - prv[s].z);
            vh[s] = cur[s].v + kap * (cur[s].v - prv[s].v);
            thh[s] = cur[s].th + kap * (cur[s].th - prv[s].th);
            beh[s] = cur[s].be + kap * (cur[s].be - prv[s].be);
            lah[s] = cur[s].la + kap * (cur[s].la - prv[s].la);
            if (DU) {
                dh[s] = cur[s].d + kap * (cur[s].d - prv[s].d);
                deh[s] = cur[s].de + kap * (cur[s].de - prv[s].de);
            }
        }
        publish();
    };
    // restart (step 7): kappa = 0, hat = the new iterate itself (the previous iterate is not needed)
    auto phaseA_restart = [&](OState<T> (&cur)[SPG]) {
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            zh[s] = cur[s].z; vh[s] = cur[s].v; thh[s] = cur[s].th; beh[s] = cur[s].be; lah[s] = cur[s].la;
            if (DU) { dh[s] = cur[s].d; deh[s] = cur[s].de; }
        }
        publish();
    };
    // ---- B, C: step 1 ----
    auto phaseBC = [&](const int par) {
        // B: g = Abar_{k+1}^T w_{k+1}, h_k; rhs = Bbar_k^T (vhat - betahat) [+ dhat - deltahat]
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            if (!(real[s] || ghl[s])) continue;
            const T *blk = blkp[s], *nxt = blk + SS;
            T g0 = (T)0, g1 = (T)0, r0 = (T)0, r1 = (T)0;
#pragma unroll
            for (int c4 = 0; c4 < NX; c4 += 4) {
                T w4[4], d4[4];
                ld4o(nxt + OW + c4, w4);
                ld4o(blk + OD + c4, d4);
#pragma unroll
                for (int q = 0; q < 4; q += 2) {
                    g0 += nxt[OAB + (c4 + q) * HS + li] * w4[q];
                    g1 += nxt[OAB + (c4 + q + 1) * HS + li] * w4[q + 1];
                    r0 += blk[OAB + (c4 + q) * HS + li] * d4[q];
                    r1 += blk[OAB + (c4 + q + 1) * HS + li] * d4[q + 1];
                }
            }
            T gg = g0 + g1;
            if (!isx) gg += nxt[OW + li];                                    // the [0 I] rows of Abar_{k+1}
            T hh = rho * (zh[s] - thh[s]) + rho * gg;                        // h_k (index reading R2)
            if (has_q) hh += sQ[li];
            blkp[s][OHH + li] = hh;
            T rr = r0 + r1 + dv[s];
            if (DU) rr += dh[s] - deh[s];
            if (ulane) blkp[s][ORH + li - NX] = rr;
        }
        __syncwarp();
        // C: xbar_{k+1} = H_k h_k; Delta u_k = M_k rhs
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            xs[s] = (T)0; du[s] = (T)0;
            if (!(real[s] || ghl[s])) continue;
            const T *blk = blkp[s];
            T x0 = (T)0, x1 = (T)0;
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                T h4[4], m4[4];
                ld4o(blk + OHH + c4, h4);
                ld4o(blk + OHM + hrow * HS + c4, m4);
                x0 += m4[0] * h4[0]; x1 += m4[1] * h4[1]; x0 += m4[2] * h4[2]; x1 += m4[3] * h4[3];
            }
            xs[s] = rowok ? x0 + x1 : (T)0;
            blkp[s][OX + par * LPS + li] = xs[s];
            if (real[s]) {
                T d0 = (T)0;
#pragma unroll
                for (int c4 = 0; c4 < NUP; c4 += 4) {
                    T r4[4], m4[4];
                    ld4o(blk + ORH + c4, r4);
                    ld4o(blk + OMM + mrow * NUP + c4, m4);
#pragma unroll
                    for (int q = 0; q < 4; ++q) d0 += m4[q] * r4[q];
                }
                du[s] = ulane ? d0 : (T)0;
                if (ulane) blkp[s][ODU + par * NUP + li - NX] = du[s];
            }
        }
    };
    // ---- D: steps 2-4 of the real stages; the new iterate overwrites prv; boundary iterates to the
    // neighbours; this lane's partial sum of c to the communication warp ----
    auto phaseD = [&](OState<T> (&prv)[SPG], const int it, const int par) {
        const uint32_t tag = (uint32_t)it + 1u;
        T acc = (T)0;
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            if (!real[s]) continue;
            const T *blk = blkp[s], *prvb = blk - SS;
            T t0 = (T)0, t1 = (T)0, avx = (T)0;
#pragma unroll
            for (int c4 = 0; c4 < NBP; c4 += 4) {
                T x4[4], a4[4];
                ld4o(prvb + OX + par * LPS + c4, x4);
                ld4o(blk + OAB + xrow * HS + c4, a4);
                t0 += a4[0] * x4[0]; t1 += a4[1] * x4[1]; t0 += a4[2] * x4[2]; t1 += a4[3] * x4[3];   // [A_k B_k] xbar_k (x-rows)
                if (c4 >= NX) {
                    T u4[4];
                    ld4o(blk + ODU + par * NUP + (c4 - NX), u4);
#pragma unroll
                    for (int q = 0; q < 4; ++q) avx += a4[q] * u4[q];                                  // B_k Delta u_k (x-rows)
                }
            }
            const bool xr = li < NX;
            const T xpi = prvb[OX + par * LPS + li];
            const T duu = isx ? (T)0 : du[s];
            const T av = (isx ? (xr ? avx : (T)0) : du[s]) + beh[s];                    // a = Bbar du + betahat
            const T bv = (isx ? (xr ? t0 + t1 + ev[s] : (T)0) : xpi) - lah[s];          // b = Abar xbar_k + ebar - lambdahat
            const T gam = av - bv;
            const T zn = clipo(((T)2 * (xs[s] + thh[s] + bv) + gam) * (T)(1.0 / 3.0), lo[s], hi[s]);   // Thm 1 (proof form, R1)
            const T vn = (T)0.5 * (zn + gam);
            const T thn = thh[s] + xs[s] - zn;
            const T ben = av - vn;
            const T lan = zn - bv - vn;
            const T d0 = thn - thh[s], d1 = ben - beh[s], d2 = lan - lah[s], d3 = zn - zh[s], d4 = vn - vh[s];
            const T d5 = (zn - vn) - (zh[s] - vh[s]);
            acc += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5;
            prv[s].z = zn; prv[s].v = vn; prv[s].th = thn; prv[s].be = ben; prv[s].la = lan;
            if (DU) {                                                          // Delta-u box copy (reading R12); x-rows: zeros
                const T dn = clipo(duu + deh[s], isx ? (T)0 : sDlo[mrow], isx ? (T)0 : sDhi[mrow]);
                const T den = deh[s] + duu - dn;
                const T e0 = den - deh[s], e1 = dn - dh[s];
                acc += e0 * e0 + e1 * e1;
                prv[s].d = dn; prv[s].de = den;
            }
            // boundary iterates for the neighbour CTAs' ghosts (tagged words, parity-double-buffered)
            const int v = s * ngroups + g;
            if (v == 1 && has_left) {
                if (CL) {
                    const uint32_t o = map_peer(xHalo + par * C::HALO + li, cta - 1), w = sizeof(typename TW::W) * LPS;
                    TW::st_cl(o, zn, tag); TW::st_cl(o + w, vn, tag); TW::st_cl(o + 2 * w, lan, tag);
                } else {
                    typename TW::W *o = halo + ((size_t)par * G + cta) * C::HALO;
                    TW::st(o + li, zn, tag); TW::st(o + LPS + li, vn, tag); TW::st(o + 2 * LPS + li, lan, tag);
                }
            }
            if (v == L && has_right) {
                if (CL) {
                    const uint32_t o = map_peer(xHalo + par * C::HALO + 3 * LPS + li, cta + 1), w = sizeof(typename TW::W) * LPS;
                    TW::st_cl(o, zn, tag); TW::st_cl(o + w, thn, tag);
                } else {
                    typename TW::W *o = halo + ((size_t)par * G + cta) * C::HALO + 3 * LPS;
                    TW::st(o + li, zn, tag); TW::st(o + LPS + li, thn, tag);
                }
            }
        }
        sAcc[par * blockDim.x + tid] = acc;                                    // (communication warp: zero)
    };
    // ---- the ghosts' new iterates, published by the neighbours in their phase D of iteration `it` ----
    auto ghosts = [&](OState<T> (&prv)[SPG], const int it, const int par) {
        const uint32_t tag = (uint32_t)it + 1u;
#pragma unroll
        for (int s = 0; s < SPG; ++s) {
            if (ghl[s] && rowok) {
                const typename TW::W *o = CL ? xHalo + par * C::HALO + 3 * LPS : halo + ((size_t)par * G + cta - 1) * C::HALO + 3 * LPS;
                T a, b2;
                bool ga = false, gb = false;
                do {
                    if (!ga) ga = CL ? TW::ld_sm(o + li, tag, a) : TW::ld(o + li, tag, a);
                    if (!gb) gb = CL ? TW::ld_sm(o + LPS + li, tag, b2) : TW::ld(o + LPS + li, tag, b2);
                } while (!(ga && gb));
                prv[s].z = a; prv[s].th = b2;
            }
            if (ghr[s] && rowok) {
                const typename TW::W *o = CL ? xHalo + par * C::HALO : halo + ((size_t)par * G + cta + 1) * C::HALO;
                T a, b2, c2;
                bool ga = false, gb = false, gc = false;
                do {
                    if (!ga) ga = CL ? TW::ld_sm(o + li, tag, a) : TW::ld(o + li, tag, a);
                    if (!gb) gb = CL ? TW::ld_sm(o + LPS + li, tag, b2) : TW::ld(o + LPS + li, tag, b2);
                    if (!gc) gc = CL ? TW::ld_sm(o + 2 * LPS + li, tag, c2) : TW::ld(o + 2 * LPS + li, tag, c2);
                } while (!(ga && gb && gc));
                prv[s].z = a; prv[s].v = b2; prv[s].la = c2;
            }
        }
    };
    // ---- communication warp: step 4 (the sum over the CTA, then over the CTAs) and steps 5-7 of iteration
    // `it`; publishes the decision to the compute warps.  Called between two CTA barriers, after every lane's phase D ----
    auto decide = [&](const int it) {
        if (!comm) return;
        const int par = it & 1;
        const uint32_t tag = (uint32_t)it + 1u;
        // fixed order: this lane's column over the compute warps (loads in flight together, a balanced tree in T), the butterfly
        // over the lanes, then double
        const T *a = sAcc + par * blockDim.x + lane;
        const double thr = red[38];                            // eta c^{i}: fetched before the sums
        T sT = (T)0;
#pragma unroll 1
        for (int j0 = 0; j0 < ncw; j0 += 8) {                  // eight warps at a time (short ranges: one batch)
            T v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) v[j] = j0 + j < ncw ? a[(j0 + j) * 32] : (T)0;
#pragma unroll
            for (int w = 4; w > 0; w >>= 1)
#pragma unroll
                for (int j = 0; j < w; ++j) v[j] += v[j + w];
            sT += v[0];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sT += __shfl_xor_sync(0xffffffffu, sT, o);
        double sum = (double)sT;
        if (CL) {                                  // push the partial into every CTA of the cluster, poll the own copies
            if (lane < G) TD::st_cl(map_peer(xPart + par * C::CLMAX + cta, lane), sum, tag);
            double val = 0.0;
            if (lane < G) while (!TD::ld_sm(xPart + par * C::CLMAX + lane, tag, val)) {}
            sum = val;
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);       // a cluster has at most 16 CTAs
        } else {
            // exact fixed-point atomic sum (see to_limbs): parity slot, three adjacent words, never reset
            unsigned long long *acc = reinterpret_cast<unsigned long long *>(part) + (size_t)par * 32;
            if (lane == 0) {
                const Limbs Lm = to_limbs(sum);
                const unsigned expect = (unsigned)((it / 2 + 1) * G) & 255u;              // arrivals in this slot so far, mod 256
                const unsigned long long one = 1ull << 56, mask = one - 1;
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    red_add_relaxed(acc + q, Lm.l[q] - xold[par][q] + one);
                    xold[par][q] = Lm.l[q];
                }
                unsigned long long v0, v1, v2;
                do {
                    v0 = ld_relaxed(acc); v1 = ld_relaxed(acc + 1); v2 = ld_relaxed(acc + 2);
                } while ((unsigned)(v0 >> 56) != expect || (unsigned)(v1 >> 56) != expect || (unsigned)(v2 >> 56) != expect);
                sum = from_limbs(v0 & mask, v1 & mask, v2 & mask);
            }
            sum = __shfl_sync(0xffffffffu, sum, 0);
        }
        if (lane == 0) {                                       // the decision word first: the compute warps wait for it
            const double c = p.rho * sum;
            const bool stop = p.tol > 0.0 && c < p.tol;
            const bool accept = !stop && c <= thr;
            *reinterpret_cast<volatile int *>(sDec) = stop ? 2 : (accept ? 0 : 1);
            red[39] = c;
        }
    };
    // the bookkeeping of that decision, off the critical path (after the barrier that hands the decision word over)
    auto book = [&](const int it) {
        if (!(comm && lane == 0)) return;
        const double c = red[39];
        const int dec = *reinterpret_cast<volatile int *>(sDec);
        if (cta == 0 && p.hist_c && it < p.hist_cap) { p.hist_c[it] = c; p.hist_a[it] = (unsigned char)(dec == 0); }
        red[33] = red[32]; red[32] = c; red[38] = p.eta * c; sCtl[2] = it + 1; sCtl[3] = dec == 2;
        if (dec == 0) ++sCtl[0];
        else if (dec == 1) { sCtl[0] = 0; ++sCtl[1]; }
    };

    // Barriers: bar_all = every warp of the CTA; bar_cmp = the compute warps only (named barrier 1), so that the communication
    // warp can sit in the exchange while the compute warps hand phase A to phase B.
    auto bar_all = [&]() { __syncthreads(); };
    auto bar_cmp = [&]() { if (!comm) asm volatile("bar.sync 1, %0;" ::"r"(ncw * 32) : "memory"); };

    // One iteration of Alg. 1 on (cur, prv) = iterates i, i-1; par = it & 1.  On entry phase A of this iteration has run; with
    // `pending` the decision of iteration it-1 is still open: the hats were formed with the momentum of an ACCEPTED step
    // (speculation) and the communication warp is summing / exchanging the partials of c and deciding
    // while the compute warps fetch the ghosts and run phases A, B, C; everybody resolves it before phase D, the first point
    // that overwrites an iterate.  A restart repeats A, B, C with kappa = 0.  Returns 0: go on, 1: iteration it-1 stopped
    // (iterate = cur), 2: this iteration stopped (iterate = prv).
    // Prediction: restart after two restarts in a row, else accept -- the accelerated phase restarts once every few steps
    // (C4: every 7th), a slowly converging tail restarts EVERY step (C2 / C3 after ~300 iterations: c falls by less than
    // eta per step), and both are then predicted right.  jacc counts RESOLVED accepted steps.
    bool pending = false, pred_restart = false;
    unsigned hist = 0;                                         // resolved decisions, newest in bit 0 (1 = restart)
    auto kappa_of = [&](int j) -> T { return j < C::KAPN ? sKap[j] : (T)kappa_tab[j]; };
    auto iteration = [&](OState<T> (&cur)[SPG], OState<T> (&prv)[SPG], const int it, const int par) -> int {
        bar_cmp();                                             // w, vhat - betahat of the neighbour stages
        phaseBC(par);
        if (pending) {
            bar_all();                                         // the communication warp has published the decision of iteration it-1
            const int dec = *reinterpret_cast<volatile int *>(sDec);
            book(it - 1);
            if (dec == 2) return 1;
            hist = (hist << 1) | (unsigned)(dec == 1);
            bool redo = false;
            if (dec == 0) {
                const T kacc = kappa_of(jacc);
                ++jacc;
                if (pred_restart) { kap = kacc; phaseA(cur, prv); redo = true; }
            } else {
                jacc = 0;
                if (!pred_restart) { kap = (T)0; phaseA_restart(cur); redo = true; }
            }
            if (redo) {                                        // mis-predicted: A, B, C again with the right momentum
                bar_cmp();
                phaseBC(par);
                bar_cmp();
            }
            pending = false;
        } else {
            bar_cmp();                                         // xbar, Delta u of the neighbour stages
        }
        phaseD(prv, it, par);
        bar_all();                                             // every lane's partial of c is in shared memory
        decide(it);                                            // communication warp; the others go on
        ghosts(prv, it, par);
        if (!spec || it + 1 >= iters) {                        // wait for the decision
            bar_all();
            const int dec = *reinterpret_cast<volatile int *>(sDec);
            book(it);
            if (dec == 2) return 2;
            hist = (hist << 1) | (unsigned)(dec == 1);
            if (dec == 0) { kap = kappa_of(jacc); ++jacc; }
            else { kap = (T)0; jacc = 0; }
            if (it + 1 < iters) phaseA(prv, cur);              // the new iterate sits in prv's registers
        } else {
            pred_restart = (hist & 3u) == 3u;
            pending = true;
            if (pred_restart) { kap = (T)0; phaseA_restart(prv); }
            else { kap = kappa_of(jacc); phaseA(prv, cur); }
        }
        return 0;
    };

    int fin_b = 0, last_par = 1;                 // which of (sa, sb) holds the returned iterate; parity of the iteration that made it
    if (iters > 0) phaseA(sa, sb);               // kappa = 0: hats = iterates (Alg. 1 input)
    for (int it = 0;; it += 2) {
        if (it >= iters) { fin_b = 0; last_par = 1; break; }
        int r = iteration(sa, sb, it, 0);
        if (r == 1) { fin_b = 0; last_par = 1; break; }
        if (r == 2 || it + 1 >= iters) { fin_b = 1; last_par = 0; break; }
        r = iteration(sb, sa, it + 1, 1);
        if (r == 1) { fin_b = 1; last_par = 0; break; }
        if (r == 2 || it + 2 >= iters) { fin_b = 0; last_par = 1; break; }
    }
    // ---- results: iterate -> S[i_cur], xbar and Delta u of the iteration that made it, control block ----
#pragma unroll
    for (int s = 0; s < SPG; ++s) {
        if (fin_b) sa[s] = sb[s];                // register moves; a reference select would force local memory
        if (!(real[s] && rowok)) continue;
        const int k = k0 - 1 + s * ngroups + g;
        T *rec = p.S + (size_t)i_cur * p.buf_stride + p.st(0, k);
        rec[p.oZ() + gi] = sa[s].z; rec[p.oV() + gi] = sa[s].v; rec[p.oTH() + gi] = sa[s].th;
        rec[p.oBE() + gi] = sa[s].be; rec[p.oLA() + gi] = sa[s].la;
        p.X[(size_t)k * nb + gi] = blkp[s][OX + last_par * LPS + li];
        if (li >= NX) {
            p.DU[(size_t)k * nu + (gi - nx)] = blkp[s][ODU + last_par * NUP + li - NX];
            if (DU) { rec[p.oD() + (gi - nx)] = sa[s].d; rec[p.oDE() + (gi - nx)] = sa[s].de; }
        }
    }
    if (cta == 0 && comm && lane == 0) {
        InstCtl c = p.ctl[0];
        const int r_jacc = sCtl[0], r_done = sCtl[3];
        c.alpha = alpha_tab[r_jacc]; c.c_last = red[32];
        c.c_prev = r_done ? red[33] : red[32];
        c.kappa = r_jacc > 0 ? (double)(T)kappa_tab[r_jacc - 1] : 0.0;          // momentum of the last hats formed
        c.done = r_done ? 1 : 0; c.iters = sCtl[2]; c.restarts = sCtl[1];
        p.ctl[0] = c;
    }
    if (CL) cluster_sync_all();                  // no CTA leaves while a peer could still address its shared memory
}

struct CoopPlan { int grid, spg, threads, slots; size_t smem; int cluster; };

// Horizons up to this length run as ONE cluster of 16 CTAs (B200, C3 generator, us per iteration, cluster vs 64 CTAs over
// L2: fp32 N=100 1.24 / 2.34, 200 1.42 / 2.25, 400 1.83 / 2.58, 700 2.57 / 2.55; fp64 N=100 1.56 / 2.45, 200 1.91 / 2.57,
// 400 2.75 / 2.70); beyond it the ranges per CTA get too long and more CTAs exchanging through L2 win.  The (20, 8)
// instantiation never takes the cluster by itself: a stage costs about twice as much there and 16 CTAs are too few
// ((20, 6) fp64, cluster vs L2: N=20 2.19 / 1.85, 50 2.31 / 1.83, 100 2.78 / 1.94; fp32 N=200 4.53 / 2.37).
constexpr int CL_MAXN_F32 = 600, CL_MAXN_F64 = 350;

template <typename T, int NX, int NU>
bool plan_coop(const pimpc_s *h, CoopPlan *pl, std::string *why)
{
    using C = OCfg<T, NX, NU>;
    const int gmax = std::min(h->sm_count, 32 * C::MAXJ);
    // at least 64 CTAs, then ranges of >= 10 stages, then as many CTAs as SMs (measured: the exchange grows with the grid;
    // C3 generator N=1000, 64 / 100 / 125 / 148 CTAs: fp32 1.92 / 1.89 / 2.06 / 2.12, fp64 2.37 / 2.15 / 2.28 / 2.33 us)
    // (the (20, 8) instantiation: ranges of >= 4 stages, a stage costs more than the exchange there: (20, 6) fp64 N=500
    // 64 / 100 / 125 / 148 CTAs 3.02 / 2.51 / 2.34 / 2.40 us per iteration)
    constexpr int RMIN = NX <= 12 ? 10 : 4;
    int grid = std::min(gmax, std::max((h->N + RMIN - 1) / RMIN, std::min(h->N, 64)));
    // short horizons: ONE cluster of <= 16 CTAs exchanging through distributed shared memory (opts.tune.cluster = -1
    // disables, = n forces n CTAs; automatic: 16 while N <= CL_MAXN)
    const int cl_opt = h->tune.cluster;
    const int grid_l2 = grid;
    int cluster = cl_opt != 0 ? std::min(std::max(cl_opt, 0), C::CLMAX) : (NX <= 12 && h->N <= (sizeof(T) == 4 ? CL_MAXN_F32 : CL_MAXN_F64) ? C::CLMAX : 0);
    int spg = 1, ncw = 0, slots = 0;
    size_t smem = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
        grid = grid_l2;
        if (cluster > 0) { cluster = std::min(cluster, h->N); grid = cluster; }
        const int gforce = h->tune.grid;                       // fewer CTAs = longer ranges per CTA
        if (gforce > 0) { grid = cluster ? std::min(grid, gforce) : std::min(std::min(gmax, h->N), gforce); if (cluster) cluster = grid; }
        const int L = (h->N + grid - 1) / grid;                // longest range
        const int gpw = 32 / C::LPS;
        slots = L + 2;
        const int spg_max = sizeof(T) == 8 ? 1 : 2;
        spg = std::min(spg_max, std::max(1, h->tune.stages_per_group));         // stages per lane group
        while (spg <= spg_max && ((slots + spg - 1) / spg + gpw - 1) / gpw > 31) ++spg;
        const bool fits_regs = spg <= spg_max;
        ncw = fits_regs ? ((slots + spg - 1) / spg + gpw - 1) / gpw : 0;
        smem = fits_regs ? C::smem_bytes(slots, (ncw + 1) * 32) : 0;
        if (fits_regs && smem <= h->smem_optin) break;
        // an AUTOMATIC cluster of 16 whose ranges are too long for one CTA (wide shapes): more CTAs exchanging through L2
        if (attempt == 0 && cluster > 0 && cl_opt == 0 && h->tune.grid <= 0) { cluster = 0; continue; }
        if (why) *why = fits_regs ? "stage matrices of a CTA's range do not fit in shared memory"
                                  : "horizon too long for the register-resident iterates of the COOP engine";
        return false;
    }
    pl->grid = grid; pl->spg = spg; pl->threads = (ncw + 1) * 32; pl->slots = slots; pl->smem = smem; pl->cluster = cluster;
    return true;
}

template <typename T, int NX, int NU, int SPG, int MAXT>
int launch_coop(pimpc_s *h, int iters, double tol, const CoopPlan &pl)
{
    using C = OCfg<T, NX, NU>;
    typedef typename Tagged<double>::W PW;
    typedef typename Tagged<T>::W HW;
    int spec = h->tune.lookahead >= 0 ? 1 : 0;                 // speculate the accept / restart decision unless opts.tune.lookahead = -1
    if (pl.cluster > 0) {
        // one thread-block cluster: co-scheduled by the hardware, exchange through distributed shared memory
        auto kc = h->has_du ? k_coop<T, NX, NU, SPG, MAXT, true, true> : k_coop<T, NX, NU, SPG, MAXT, false, true>;
        PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem));
        if (pl.cluster > 8) PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kc, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(pl.grid); cfg.blockDim = dim3(pl.threads); cfg.dynamicSmemBytes = pl.smem; cfg.stream = h->stream;
        cudaLaunchAttribute at1[1];
        at1[0].id = cudaLaunchAttributeClusterDimension;
        at1[0].val.clusterDim.x = pl.grid; at1[0].val.clusterDim.y = 1; at1[0].val.clusterDim.z = 1;
        cfg.attrs = at1; cfg.numAttrs = 1;
        int ncl = 0;
        if (cudaOccupancyMaxActiveClusters(&ncl, kc, &cfg) == cudaSuccess && ncl >= 1) {
            Prob<T> pc = make_prob<T>(h, tol);
            const double *atc = h->alpha_tab, *ktc = h->kappa_tab;
            PIMPC_CUDA_TRY(h, cudaLaunchKernelEx(&cfg, kc, pc, atc, ktc, iters, (PW *)nullptr, (HW *)nullptr, spec));
            h->info.grid = pl.grid; h->info.block = pl.threads; h->info.smem_bytes = pl.smem;
            return 1;
        }
        cudaGetLastError();                      // no room for such a cluster: the L2 path below with the same plan
    }
    auto kern = h->has_du ? k_coop<T, NX, NU, SPG, MAXT, true, false> : k_coop<T, NX, NU, SPG, MAXT, false, false>;
    PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem));
    int occ = 0;
    PIMPC_CUDA_TRY(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, pl.threads, pl.smem));
    if (occ < 1) { h->errmsg = "COOP kernel does not fit on an SM"; return PIMPC_EINVAL; }
    const size_t pbytes = 2 * (size_t)(pl.grid + C::NREP) * C::PSTRIDE * sizeof(PW), hbytes = 2 * (size_t)pl.grid * C::HALO * sizeof(HW);
    const size_t need = pbytes + hbytes;
    { const int rc = pimpc_grow(h, &h->coop_buf, &h->coop_bytes, need); if (rc) return rc; }
    PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->coop_buf, 0, need, h->stream));       // tag 0 = nothing published yet
    Prob<T> p = make_prob<T>(h, tol);
    PW *part = (PW *)h->coop_buf;
    HW *halo = (HW *)((unsigned char *)h->coop_buf + pbytes);
    const double *at = h->alpha_tab, *kt = h->kappa_tab;
    void *args[] = {(void *)&p, (void *)&at, (void *)&kt, (void *)&iters, (void *)&part, (void *)&halo, (void *)&spec};
    PIMPC_CUDA_TRY(h, cudaLaunchCooperativeKernel((const void *)kern, dim3(pl.grid), dim3(pl.threads), args, pl.smem, h->stream));
    h->info.grid = pl.grid; h->info.block = pl.threads; h->info.smem_bytes = pl.smem;
    return 1;
}

template <typename T, int NX, int NU>
int run_coop_t(pimpc_s *h, int iters, double tol)
{
    CoopPlan pl;
    std::string why;
    if (!plan_coop<T, NX, NU>(h, &pl, &why)) { h->errmsg = "COOP engine not applicable: " + why; return PIMPC_EINVAL; }
    int launches = ensure_alpha_table(h, iters);
    if (launches < 0) return launches;
    int n;
    // thread ceilings: the register budget per thread follows from the block size actually needed
    if constexpr (sizeof(T) == 8) {
        n = pl.threads <= 384 ? launch_coop<T, NX, NU, 1, 384>(h, iters, tol, pl)
            : pl.threads <= 512 ? launch_coop<T, NX, NU, 1, 512>(h, iters, tol, pl)
                                : launch_coop<T, NX, NU, 1, 1024>(h, iters, tol, pl);
    } else if (pl.spg == 1) {
        n = pl.threads <= 512 ? launch_coop<T, NX, NU, 1, 512>(h, iters, tol, pl) : launch_coop<T, NX, NU, 1, 1024>(h, iters, tol, pl);
    } else {
        n = pl.threads <= 640 ? launch_coop<T, NX, NU, 2, 640>(h, iters, tol, pl) : launch_coop<T, NX, NU, 2, 1024>(h, iters, tol, pl);
    }
    return n < 0 ? n : n + launches;
}

// padded shapes with an instantiation, smallest first: (4, 4), (12, 4), (20, 8) (one row per lane: nx + nu <= 32)
bool coop_shape(const pimpc_s *h) { return h->nx <= 20 && h->nu <= 8; }
int coop_class(const pimpc_s *h) { return (h->nx <= 4 && h->nu <= 4) ? 0 : ((h->nx <= 12 && h->nu <= 4) ? 1 : 2); }

} // namespace

bool coop_supported(const pimpc_s *h, std::string *why)
{
    if (h->batch != 1) { if (why) *why = "COOP engine is for batch = 1"; return false; }
    if (!coop_shape(h)) { if (why) *why = "no COOP instantiation holds this (nx, nu) (nx <= 20, nu <= 8)"; return false; }
    if (h->bnd_per_instance || h->cost_per_instance) { /* batch = 1: strides are irrelevant */ }
    CoopPlan pl;
    const bool d = h->dtype == PIMPC_F64;
    const int cls = coop_class(h);
    if (cls == 2) return d ? plan_coop<double, 20, 8>(h, &pl, why) : plan_coop<float, 20, 8>(h, &pl, why);
    if (cls == 1) return d ? plan_coop<double, 12, 4>(h, &pl, why) : plan_coop<float, 12, 4>(h, &pl, why);
    return d ? plan_coop<double, 4, 4>(h, &pl, why) : plan_coop<float, 4, 4>(h, &pl, why);
}

int run_coop(pimpc_s *h, int iters, double tol)
{
    std::string why;
    if (!coop_supported(h, &why)) { h->errmsg = "COOP engine not applicable: " + why; return PIMPC_EINVAL; }
    const bool d = h->dtype == PIMPC_F64;
    const int cls = coop_class(h);
    if (cls == 2) return d ? run_coop_t<double, 20, 8>(h, iters, tol) : run_coop_t<float, 20, 8>(h, iters, tol);
    if (cls == 1) return d ? run_coop_t<double, 12, 4>(h, iters, tol) : run_coop_t<float, 12, 4>(h, iters, tol);
    return d ? run_coop_t<double, 4, 4>(h, iters, tol) : run_coop_t<float, 4, 4>(h, iters, tol);
}
