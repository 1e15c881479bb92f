// a0: the per-solve cache of Algorithm 1 (Remark 5), plus the small
// bookkeeping kernels (begin / gather / state I/O).  One CTA per (instance, stage); the SPD
// matrix lives in shared memory in double precision whatever the handle's dtype and is inverted
// in place by Gauss-Jordan exchange steps without pivoting (safe for SPD matrices).
#include <algorithm>

#include "pimpc_internal.h"

namespace {

// In-place inverse of the SPD n x n matrix S (shared memory, row-major).  All threads call.
// Returns false (uniformly) if a pivot is not positive / finite.
__device__ bool gj_invert(double *S, double *colb, double *rowb, int n)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    bool ok = true;
    for (int p = 0; p < n; ++p) {
        __syncthreads();
        const double piv = S[p * n + p];
        if (!(piv > 0.0) || !isfinite(piv)) ok = false;
        for (int t = tid; t < n; t += nt) { colb[t] = S[t * n + p]; rowb[t] = S[p * n + t]; }
        __syncthreads();
        const double inv = 1.0 / piv;
        for (int idx = tid; idx < n * n; idx += nt) {
            const int i = idx / n, j = idx - i * n;
            double v;
            if (i == p) v = (j == p) ? inv : rowb[j] * inv;
            else if (j == p) v = -colb[i] * inv;
            else v = S[idx] - colb[i] * rowb[j] * inv;
            S[idx] = v;
        }
    }
    __syncthreads();
    return ok;
}

// list != null: only the cache entries of the listed flattened stage indices (b * N + k) are recomputed.
template <typename T>
__global__ void __launch_bounds__(256) k_setup(Prob<T> p, const int *__restrict__ list)
{
    extern __shared__ double sm[];
    const int nx = p.nx, nu = p.nu, nb = p.nb, N = p.N;
    double *S = sm, *colb = S + nb * nb, *rowb = colb + nb;
    const int sflat = list ? list[blockIdx.x] : (int)blockIdx.x;
    const int b = sflat / N, k = sflat - b * N;
    const int tid = threadIdx.x, nt = blockDim.x;
    const bool last = (k == N - 1);
    const T *A1 = p.A + ((size_t)b * N + (last ? k : k + 1)) * nx * nx;
    const T *B1 = p.B + ((size_t)b * N + (last ? k : k + 1)) * nx * nu;
    const T *Qx = (last && p.P) ? p.P + (size_t)b * p.cost_stride_q : p.Q + (size_t)b * p.cost_stride_q;
    const T *Rx = p.R + (size_t)b * p.cost_stride_r;
    const double rho = p.rho;
    bool finite = true;

    // H_k = (Qbar + rho I + rho Abar_{k+1}^T Abar_{k+1})^-1, k < N-1;  (Qbar_N + rho I)^-1, k = N-1
    for (int idx = tid; idx < nb * nb; idx += nt) {
        const int i = idx / nb, j = idx - i * nb;
        double s = 0.0;
        if (i < nx && j < nx) s = (double)Qx[i * nx + j];
        else if (i >= nx && j >= nx) s = (double)Rx[(i - nx) * nu + (j - nx)];
        if (i == j) s += rho;
        if (!last) {
            double a = (i == j && i >= nx) ? 1.0 : 0.0;          // the [0 I] rows of Abar
            for (int r = 0; r < nx; ++r) {
                const double ai = (i < nx) ? (double)A1[r * nx + i] : (double)B1[r * nu + (i - nx)];
                const double aj = (j < nx) ? (double)A1[r * nx + j] : (double)B1[r * nu + (j - nx)];
                a += ai * aj;
            }
            s += rho * a;
        }
        if (!isfinite(s)) finite = false;
        S[idx] = s;
    }
    bool ok = gj_invert(S, colb, rowb, nb);
    T *Hk = p.H + ((size_t)b * N + k) * nb * nb;
    for (int idx = tid; idx < nb * nb; idx += nt) {
        const int i = idx / nb, j = idx - i * nb;
        Hk[idx] = (T)(0.5 * (S[idx] + S[j * nb + i]));            // exactly symmetric
    }
    __syncthreads();

    // M_k = (B_k^T B_k + I [+ Wdu/rho] [+ I])^-1  so that J_k = M_k Bbar_k^T  (R12, R13)
    const T *Bk = p.B + ((size_t)b * N + k) * nx * nu;
    const T *Ak = p.A + ((size_t)b * N + k) * nx * nx;
    for (int idx = tid; idx < nx * nx; idx += nt)
        if (!isfinite((double)Ak[idx])) finite = false;
    for (int idx = tid; idx < nu * nu; idx += nt) {
        const int i = idx / nu, j = idx - i * nu;
        double s = (i == j) ? 1.0 : 0.0;
        for (int r = 0; r < nx; ++r) s += (double)Bk[r * nu + i] * (double)Bk[r * nu + j];
        if (p.Wdu) s += (double)p.Wdu[(size_t)b * p.cost_stride_r + idx] / rho;
        if (p.has_du && i == j) s += 1.0;
        if (!isfinite(s)) finite = false;
        S[idx] = s;
    }
    ok = gj_invert(S, colb, rowb, nu) && ok;
    T *Mk = p.M + ((size_t)b * N + k) * nu * nu;
    for (int idx = tid; idx < nu * nu; idx += nt) {
        const int i = idx / nu, j = idx - i * nu;
        Mk[idx] = (T)(0.5 * (S[idx] + S[j * nu + i]));
    }
    if (!finite) atomicOr(p.err, PIMPC_DEVERR_NONFINITE);
    else if (!ok && tid == 0) atomicOr(p.err, PIMPC_DEVERR_NOTPD);
}

// ---- a0 for 8 < nb <= 64: FOUR threads per matrix row, LP / 4 columns of the row in the registers of each, one CTA of
// 4 LP threads per (instance, stage); the matrix is padded to LP x LP with identity rows.  The pivot row and the pivot column
// of each exchange step travel through a double-buffered shared-memory line (one CTA barrier per pivot).  k_setup above keeps
// the matrix in shared memory (three loads, an integer division and a store per FMA, two barriers per pivot): C5, 128 000
// stages of 60 x 60, took 70.9 ms there.  Same exchange steps as gj_rows (rank-1 update, column p overwritten).
template <typename T, int LP>
__global__ void __launch_bounds__(LP * 4) k_setup_rows(Prob<T> p, const int *__restrict__ list)
{
    // LPK: a row line with every quarter (the CPT columns of one thread) shifted by 16 bytes more than the one before: the four
    // 16-byte words a warp-wide load touches (one per quarter) then sit in different banks (unshifted they are 128 bytes apart:
    // ncu counted 73 % of the shared-memory wavefronts as bank conflicts)
    constexpr int CPT = LP / 4, TS = LP + 1, NT = LP * 4, LPK = LP + 8;
    static_assert(CPT % 2 == 0, "16-byte alignment of the exchange lines");
    extern __shared__ __align__(16) double sm[];
    double *Ssm = sm;                                          // [LP][TS] after the inversion; before: [nx][LPK] rows of [A_{k+1} B_{k+1}]
    double *rowb = sm + LP * LPK, *colb = rowb + 2 * LPK;      // [2][LPK], [2][LP] (parity of the pivot)
    const int nx = p.nx, nu = p.nu, nb = p.nb, N = p.N;
    const int sflat = list ? list[blockIdx.x] : (int)blockIdx.x;
    const int b = sflat / N, k = sflat - b * N;
    // a warp holds 8 rows; 8 consecutive lanes share a quarter, so each quarter-warp of a 16-byte load of a row line reads ONE word
    const int tid = threadIdx.x, i = (tid >> 5) * 8 + (tid & 7), q = (tid >> 3) & 3, j0 = q * CPT, j0k = q * (CPT + 2);
    const int ik = i + 2 * (i / CPT);                          // position of column i in a shifted line
    const bool last = (k == N - 1);
    const T *A1 = p.A + ((size_t)b * N + (last ? k : k + 1)) * nx * nx;
    const T *B1 = p.B + ((size_t)b * N + (last ? k : k + 1)) * nx * nu;
    const T *Qx = (last && p.P) ? p.P + (size_t)b * p.cost_stride_q : p.Q + (size_t)b * p.cost_stride_q;
    const T *Rx = p.R + (size_t)b * p.cost_stride_r;
    const double rho = p.rho;
    bool finite = true;

    // H_k = (Qbar + rho I + rho Abar_{k+1}^T Abar_{k+1})^-1, k < N-1;  (Qbar_N + rho I)^-1, k = N-1
#pragma unroll 4
    for (int idx = tid; idx < nx * LP; idx += NT) {            // rows of [A_{k+1} B_{k+1}] as doubles, zero-padded to LP columns
        const int r = idx / LP, c = idx - r * LP;
        const double v = c < nx ? (double)A1[r * nx + c] : (c < nb ? (double)B1[r * nu + (c - nx)] : 0.0);
        if (!isfinite(v)) finite = false;
        Ssm[r * LPK + c + 2 * (c / CPT)] = v;
    }
    __syncthreads();
    double S[CPT];
    const double rl = last ? 0.0 : rho;                        // the terminal stage has no Abar_{k+1} term
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
        const int j = j0 + c;
        double v = 0.0;
        if (i < nb && j < nb) {
            if (i < nx && j < nx) v = (double)Qx[i * nx + j];
            else if (i >= nx && j >= nx) v = (double)Rx[(i - nx) * nu + (j - nx)];
            if (i == j) v += rho + (i >= nx ? rl : 0.0);        // rho I and the [0 I] rows of rho Abar^T Abar
        } else if (i == j) v = 1.0;                             // pad rows: identity
        S[c] = v;
    }
    for (int r = 0; r < nx; ++r) {                              // + rho [A B]^T [A B]
        const double ai = rl * Ssm[r * LPK + ik];
#pragma unroll
        for (int c = 0; c < CPT; c += 2) {
            const double2 v = *reinterpret_cast<const double2 *>(Ssm + r * LPK + j0k + c);
            S[c] = fma(ai, v.x, S[c]); S[c + 1] = fma(ai, v.y, S[c + 1]);
        }
    }
#pragma unroll
    for (int c = 0; c < CPT; ++c)
        if (!isfinite(S[c])) finite = false;

    // exchange steps; the pivot loop is unrolled over a quarter so that column pv has a compile-time index in its owners' registers
    bool ok = true;
    for (int qq = 0; qq < 4; ++qq) {
#pragma unroll
        for (int c0 = 0; c0 < CPT; ++c0) {
            const int pv = qq * CPT + c0;
            if (pv < nb) {                                      // uniform over the CTA
                double *rb = rowb + (pv & 1) * LPK, *cb = colb + (pv & 1) * LP;
                // column pv from its owners; the pivot ROW is the same numbers up to the sign of the pivoted rows (see gj_rows)
                if (q == qq) { cb[i] = S[c0]; rb[ik] = (i < pv) ? -S[c0] : S[c0]; }
                __syncthreads();                                // the lines of the previous pivot have the other parity
                const double piv = rb[qq * (CPT + 2) + c0];
                if (!(piv > 0.0) || !isfinite(piv)) ok = false;
                const double inv = 1.0 / piv;
                const double f = (i == pv) ? 1.0 - inv : cb[i] * inv;
#pragma unroll
                for (int c = 0; c < CPT; c += 2) {
                    const double2 r2 = *reinterpret_cast<const double2 *>(rb + j0k + c);
                    S[c] = fma(-f, r2.x, S[c]); S[c + 1] = fma(-f, r2.y, S[c + 1]);
                }
                if (q == qq) S[c0] = (i == pv) ? inv : -f;
            }
        }
    }
    __syncthreads();                                            // everybody is done with the rows of [A B] (first pivot at the latest) and the lines
#pragma unroll
    for (int c = 0; c < CPT; ++c) Ssm[i * TS + j0 + c] = S[c];
    __syncthreads();
    T *Hk = p.H + ((size_t)b * N + k) * nb * nb;
    for (int idx = tid; idx < nb * nb; idx += NT) {
        const int i2 = idx / nb, j2 = idx - i2 * nb;
        Hk[idx] = (T)(0.5 * (Ssm[i2 * TS + j2] + Ssm[j2 * TS + i2]));   // exactly symmetric
    }
    __syncthreads();

    // M_k = (B_k^T B_k + I [+ Wdu/rho] [+ I])^-1  so that J_k = M_k Bbar_k^T  (R12, R13)
    const T *Bk = p.B + ((size_t)b * N + k) * nx * nu;
    const T *Ak = p.A + ((size_t)b * N + k) * nx * nx;
    for (int idx = tid; idx < nx * nx; idx += NT)
        if (!isfinite((double)Ak[idx])) finite = false;
    for (int idx = tid; idx < nu * nu; idx += NT) {
        const int i2 = idx / nu, j2 = idx - i2 * nu;
        double v = (i2 == j2) ? 1.0 : 0.0;
        for (int r = 0; r < nx; ++r) v += (double)Bk[r * nu + i2] * (double)Bk[r * nu + j2];
        if (p.Wdu) v += (double)p.Wdu[(size_t)b * p.cost_stride_r + idx] / rho;
        if (p.has_du && i2 == j2) v += 1.0;
        if (!isfinite(v)) finite = false;
        Ssm[idx] = v;
    }
    ok = gj_invert(Ssm, colb, rowb, nu) && ok;
    T *Mk = p.M + ((size_t)b * N + k) * nu * nu;
    for (int idx = tid; idx < nu * nu; idx += NT) {
        const int i2 = idx / nu, j2 = idx - i2 * nu;
        Mk[idx] = (T)(0.5 * (Ssm[idx] + Ssm[j2 * nu + i2]));
    }
    if (!finite) atomicOr(p.err, PIMPC_DEVERR_NONFINITE);
    else if (!ok) atomicOr(p.err, PIMPC_DEVERR_NOTPD);
}

// ---- a0 for small stages (nb <= 32): one lane per matrix row, a group of LPS lanes per (instance, stage) --------
// Row i of the SPD matrix lives in the registers of lane i (double precision whatever the dtype); the pivot
// row of each Gauss-Jordan exchange step is broadcast through a per-group shared-memory row.  Same arithmetic
// as gj_invert above (no pivoting; safe for SPD), ~40 x less time than one CTA per stage on 16 x 16 blocks.
__host__ __device__ constexpr int pow2ceil_k(int v) { int p = 1; while (p < v) p <<= 1; return p; }

template <int W, int NPIV>
__device__ __forceinline__ bool gj_rows(double (&S)[W], double *rowb, const int li)
{
    bool ok = true;
#pragma unroll
    for (int p = 0; p < NPIV; ++p) {
        __syncwarp();
        // The pivot row, from the pivot COLUMN every lane already holds at a compile-time index: the matrix is symmetric at
        // the start (Q, R, W_du symmetric: include/pimpc.h) and an exchange step keeps S[p][j] = S[j][p] for the rows j not yet
        // pivoted and S[p][j] = -S[j][p] for the pivoted ones (j < p).  One 8-byte store per lane instead of the owner lane's
        // W / 2 16-byte stores (ncu: the stores were a third of the shared-memory wavefronts of this kernel).
        rowb[li] = (li < p) ? -S[p] : S[p];
        __syncwarp();
        const double piv = rowb[p], colv = S[p];
        if (!(piv > 0.0) || !isfinite(piv)) ok = false;
        const double inv = 1.0 / piv;
        // one exchange step as a rank-1 update S[i][:] -= f_i * pivot_row with f_i = S[i][p] / piv for i != p and
        // f_p = 1 - 1/piv (so that the pivot row becomes pivot_row / piv); column p is then overwritten with -f_i
        // (1/piv in the pivot row).  One select per step instead of one per element.
        const double f = (li == p) ? 1.0 - inv : colv * inv;
        if constexpr (W % 2 == 0) {
#pragma unroll
            for (int j = 0; j < W; j += 2) {
                const double2 r2 = *reinterpret_cast<const double2 *>(rowb + j);
                S[j] = fma(-f, r2.x, S[j]); S[j + 1] = fma(-f, r2.y, S[j + 1]);
            }
        } else {
#pragma unroll
            for (int j = 0; j < W; ++j) S[j] = fma(-f, rowb[j], S[j]);
        }
        S[p] = (li == p) ? inv : -f;
    }
    __syncwarp();
    return ok;
}

template <typename T, int NX, int NU>
__global__ void __launch_bounds__(128) k_setup_small(Prob<T> p, const int *__restrict__ list, const long long nlist)
{
    constexpr int NB = NX + NU, LPS = pow2ceil_k(NB), SPW = 32 / LPS, GPB = 4 * SPW, TS = LPS + 1;
    constexpr int GSZ = (NX * LPS > LPS * TS ? NX * LPS : LPS * TS) + LPS;
    static_assert(GSZ % 2 == 0 && LPS % 2 == 0, "16-byte alignment of the per-group buffers");
    __shared__ __align__(16) double sm[GPB * GSZ];
    const int tid = threadIdx.x, g = tid / LPS, li = tid % LPS, N = p.N;
    const long long nst = list ? nlist : (long long)p.batch * N, sraw = (long long)blockIdx.x * GPB + g;
    const bool act = sraw < nst;
    const long long spos = act ? sraw : nst - 1;               // idle groups repeat the last stage and do not store
    const long long sidx = list ? (long long)list[spos] : spos;
    const int b = (int)(sidx / N), k = (int)(sidx - (long long)b * N);
    double *buf = sm + g * GSZ, *rowb = buf + (GSZ - LPS);
    const bool last = (k == N - 1), rowok = li < NB;
    const T *A1 = p.A + (sidx + (last ? 0 : 1)) * NX * NX, *B1 = p.B + (sidx + (last ? 0 : 1)) * NX * NU;
    const T *Ak = p.A + sidx * NX * NX, *Bk = p.B + sidx * NX * NU;
    const T *Qx = (last && p.P) ? p.P + (size_t)b * p.cost_stride_q : p.Q + (size_t)b * p.cost_stride_q;
    const T *Rx = p.R + (size_t)b * p.cost_stride_r;
    const double rho = p.rho;
    bool finite = true;

    // H_k = (Qbar + rho I + rho Abar_{k+1}^T Abar_{k+1})^-1, k < N-1;  (Qbar_N + rho I)^-1, k = N-1
#pragma unroll
    for (int r = 0; r < NX; ++r) {                             // [A_{k+1} B_{k+1}] as doubles, column li by lane li
        const double a1 = li < NX ? (double)A1[r * NX + li] : (rowok ? (double)B1[r * NU + (li - NX)] : 0.0);
        const double a0 = li < NX ? (double)Ak[r * NX + li] : (rowok ? (double)Bk[r * NU + (li - NX)] : 0.0);
        if (!isfinite(a1) || !isfinite(a0)) finite = false;
        buf[r * LPS + li] = a1;
    }
    __syncwarp();
    double S[LPS];
    const double rl = last ? 0.0 : rho;                        // the terminal stage has no Abar_{k+1} term
#pragma unroll
    for (int j = 0; j < LPS; ++j) {
        double s = 0.0;
        if (rowok && j < NB) {
            if (li < NX && j < NX) s = (double)Qx[li * NX + j];
            else if (li >= NX && j >= NX) s = (double)Rx[(li - NX) * NU + (j - NX)];
            if (j == li) s += rho + (li >= NX ? rl : 0.0);      // rho I and the [0 I] rows of rho Abar^T Abar
        } else if (j == li) s = 1.0;                            // pad rows: identity
        S[j] = s;
    }
#pragma unroll
    for (int r = 0; r < NX; ++r) {                              // + rho [A B]^T [A B], accumulated in place
        const double ai = rl * buf[r * LPS + li];
#pragma unroll
        for (int j = 0; j < LPS; j += 2) {
            const double2 v = *reinterpret_cast<const double2 *>(buf + r * LPS + j);
            S[j] = fma(ai, v.x, S[j]); S[j + 1] = fma(ai, v.y, S[j + 1]);
        }
    }
#pragma unroll
    for (int j = 0; j < LPS; ++j)
        if (!isfinite(S[j])) finite = false;
    bool ok = gj_rows<LPS, NB>(S, rowb, li);
#pragma unroll
    for (int j = 0; j < LPS; ++j) buf[li * TS + j] = S[j];
    __syncwarp();
    if (act && rowok) {
        // row i by the lanes of the group (coalesced: a lane-per-row store touched 32 sectors per instruction, and the LSU pipe
        // was 90 % busy): H[i][li] = (S_i[li] + S_li[i]) / 2, exactly symmetric
        T *Hs = p.H + (size_t)sidx * NB * NB + li;
#pragma unroll
        for (int i = 0; i < NB; ++i) Hs[i * NB] = (T)(0.5 * (buf[i * TS + li] + S[i]));
    }
    __syncwarp();

    // M_k = (B_k^T B_k + I [+ Wdu/rho] [+ I])^-1  so that J_k = M_k Bbar_k^T  (R12, R13)
    constexpr int MW = NU;
    for (int idx = li; idx < NX * NU; idx += LPS) buf[idx] = (double)Bk[idx];
    __syncwarp();
    double Mr[MW];
#pragma unroll
    for (int j = 0; j < MW; ++j) {
        double s = (j == li) ? 1.0 : 0.0;
        if (li < NU) {
            for (int r = 0; r < NX; ++r) s += buf[r * NU + li] * buf[r * NU + j];
            if (p.Wdu) s += (double)p.Wdu[(size_t)b * p.cost_stride_r + li * NU + j] / rho;
            if (p.has_du && j == li) s += 1.0;
        }
        if (!isfinite(s)) finite = false;
        Mr[j] = s;
    }
    ok = gj_rows<MW, NU>(Mr, rowb, li) && ok;
    __syncwarp();
    if (li < NU) {
#pragma unroll
        for (int j = 0; j < MW; ++j) buf[li * TS + j] = Mr[j];
    }
    __syncwarp();
    if (act && li < NU) {
        T *Ms = p.M + (size_t)sidx * NU * NU + li;
#pragma unroll
        for (int i = 0; i < MW; ++i) Ms[i * NU] = (T)(0.5 * (buf[i * TS + li] + Mr[i]));
    }
    if (!finite) atomicOr(p.err, PIMPC_DEVERR_NONFINITE);
    else if (!ok) atomicOr(p.err, PIMPC_DEVERR_NOTPD);
}

// Tracking cost (1a) -> the cost of problem (11): Q = C'W_y C, R = W_u, and for each of the nref
// reference pairs qbar[k] = col(C'W_y r_y[k], W_u r_u[k]).  One thread per output element, double accumulation.
template <typename T>
__global__ void k_tracking(int nx, int nu, int ny, const T *__restrict__ C, const T *__restrict__ Wy, const T *__restrict__ Wu,
                           const T *__restrict__ ry, const T *__restrict__ ru, int nref, T *__restrict__ Q, T *__restrict__ R,
                           T *__restrict__ qbar)
{
    const int nb = nx + nu, nq = nx * nx, nr = nu * nu, total = nq + nr + nref * nb;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        if (idx < nq) {                                        // Q[i][j] = sum_{p,q} C[p][i] Wy[p][q] C[q][j]
            const int i = idx / nx, j = idx - i * nx;
            double s = 0.0;
            for (int a = 0; a < ny; ++a) {
                double w = 0.0;
                for (int b = 0; b < ny; ++b) w += (double)Wy[a * ny + b] * (double)C[b * nx + j];
                s += (double)C[a * nx + i] * w;
            }
            Q[idx] = (T)s;
        } else if (idx < nq + nr) {
            R[idx - nq] = Wu[idx - nq];
        } else {
            const int q = idx - nq - nr, k = q / nb, i = q - k * nb;
            double s = 0.0;
            if (i < nx) {                                      // (C'W_y r_y)_i
                if (ry)
                    for (int a = 0; a < ny; ++a) {
                        double w = 0.0;
                        for (int b = 0; b < ny; ++b) w += (double)Wy[a * ny + b] * (double)ry[k * ny + b];
                        s += (double)C[a * nx + i] * w;
                    }
            } else if (ru) {                                   // (W_u r_u)_i
                for (int b = 0; b < nu; ++b) s += (double)Wu[(i - nx) * nu + b] * (double)ru[k * nu + b];
            }
            qbar[q] = (T)s;
        }
    }
}

// Input of Alg. 1: hats = iterates (i_prev = i_cur), alpha_0 = 1, c^0 = c0.
template <typename T>
__global__ void k_begin(Prob<T> p)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p.batch) return;
    InstCtl c = p.ctl[b];
    c.alpha = 1.0; c.c_prev = p.c0; c.c_last = p.c0; c.kappa = 0.0;
    c.i_prev = c.i_cur; c.i_new = (c.i_cur + 1) % 3;
    c.done = 0; c.iters = 0; c.restarts = 0;
    p.ctl[b] = c;
    bool finite = true;
    for (int i = 0; i < p.nx; ++i) if (!isfinite((double)p.x0[(size_t)b * p.nx + i])) finite = false;
    for (int i = 0; i < p.nu; ++i) if (!isfinite((double)p.uprev[(size_t)b * p.nu + i])) finite = false;
    if (!finite) atomicOr(p.err, PIMPC_DEVERR_NONFINITE);
    if (p.hist_c)
        for (int i = 0; i < p.hist_cap; ++i) { p.hist_c[(size_t)b * p.hist_cap + i] = 0.0; p.hist_a[(size_t)b * p.hist_cap + i] = 0; }
}

template <typename T>
__global__ void k_gather(Prob<T> p, T *x, T *u, T *du)
{
    const int b = blockIdx.y;
    const InstCtl c = p.ctl[b];
    const T *S = p.S + (size_t)c.i_cur * p.buf_stride;
    const int per = p.nb + p.nu;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < p.N * per; idx += gridDim.x * blockDim.x) {
        const int k = idx / per, i = idx - k * per;
        if (i < p.nb) {
            const T z = S[p.st(b, k) + i];
            if (i < p.nx) { if (x) x[((size_t)b * p.N + k) * p.nx + i] = z; }
            else if (u) u[((size_t)b * p.N + k) * p.nu + (i - p.nx)] = z;
        } else if (du) {
            du[((size_t)b * p.N + k) * p.nu + (i - p.nb)] = p.DU[((size_t)b * p.N + k) * p.nu + (i - p.nb)];
        }
    }
}

// Result record of one instance per CTA.  r_prim2 = rho ||F p + G q - h||^2 of the returned iterate, from the definition
// of the three (four with the Delta-u box) consensus constraints of Problem (11) ((14a), (15c)):
//   xbar_{k+1} - z_{k+1},   Bbar_k Delta u_k - v_k,   z_{k+1} - Abar_k xbar_k - v_k - ebar_k   [, Delta u_k - d_k]
// accumulated in double in a fixed order (thread-strided, then a fixed tree), r_dual2 = c - r_prim2.
template <typename T>
__global__ void __launch_bounds__(128) k_rprim(Prob<T> p, double *__restrict__ part, const int chunk)
{
    __shared__ double red[128];
    const int b = blockIdx.y, nx = p.nx, nu = p.nu, nb = p.nb, N = p.N;
    const InstCtl c = p.ctl[b];
    const T *S = p.S + (size_t)c.i_cur * p.buf_stride;
    double acc = 0.0;
    const int i0 = blockIdx.x * chunk, i1 = min(N * nb, i0 + chunk);
    for (int idx = i0 + threadIdx.x; idx < i1; idx += blockDim.x) {
        const int k = idx / nb, i = idx - k * nb;
        const size_t sk = (size_t)b * N + k;
        const T *rec = S + p.st(b, k);
        const double z = (double)rec[p.oZ() + i], v = (double)rec[p.oV() + i], xk1 = (double)p.X[sk * nb + i];
        const T *du = p.DU + sk * nu;
        double bdu, axk;                                       // (Bbar_k Delta u_k)_i, (Abar_k xbar_k + ebar_k)_i
        if (i < nx) {
            const T *Ak = p.A + sk * nx * nx + (size_t)i * nx, *Bk = p.B + sk * nx * nu + (size_t)i * nu;
            bdu = 0.0; axk = p.e ? (double)p.e[sk * nx + i] : 0.0;
            for (int j = 0; j < nu; ++j) bdu += (double)Bk[j] * (double)du[j];
            for (int j = 0; j < nx; ++j) axk += (double)Ak[j] * (double)(k == 0 ? p.x0[(size_t)b * nx + j] : p.X[(sk - 1) * nb + j]);
            for (int j = 0; j < nu; ++j) axk += (double)Bk[j] * (double)(k == 0 ? p.uprev[(size_t)b * nu + j] : p.X[(sk - 1) * nb + nx + j]);
        } else {
            bdu = (double)du[i - nx];
            axk = (double)(k == 0 ? p.uprev[(size_t)b * nu + (i - nx)] : p.X[(sk - 1) * nb + i]);
        }
        const double r1 = xk1 - z, r2 = bdu - v, r3 = z - axk - v;
        acc += r1 * r1 + r2 * r2 + r3 * r3;
        if (p.has_du && i >= nx) { const double r4 = (double)du[i - nx] - (double)rec[p.oD() + (i - nx)]; acc += r4 * r4; }
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[(size_t)b * gridDim.x + blockIdx.x] = red[0];
}

__global__ void k_result(const InstCtl *__restrict__ ctl, const double *__restrict__ part, const int nch, const int batch,
                         const double rho, pimpc_result *res)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const InstCtl c = ctl[b];
    double s = 0.0;
    for (int q = 0; q < nch; ++q) s += part[(size_t)b * nch + q];
    pimpc_result r;
    r.c = c.c_last; r.alpha = c.alpha; r.iters = c.iters; r.restarts = c.restarts;
    r.converged = c.done; r.pad_ = 0;
    r.r_prim2 = c.iters > 0 ? rho * s : 0.0;
    r.r_dual2 = c.iters > 0 ? c.c_last - r.r_prim2 : 0.0;
    res[b] = r;
}

// which: PIMPC_X.. ; set = 0: state -> dense buffer, 1: dense buffer -> state (current iterate).
template <typename T>
__global__ void k_state_io(Prob<T> p, int which, T *buf, int set)
{
    const int b = blockIdx.y;
    const InstCtl c = p.ctl[b];
    T *S = p.S + (size_t)c.i_cur * p.buf_stride;
    int w, off = 0;
    T *dense = nullptr;
    switch (which) {
    case PIMPC_X: w = p.nb; dense = p.X; break;
    case PIMPC_DU: w = p.nu; dense = p.DU; break;
    case PIMPC_Z: w = p.nb; off = p.oZ(); break;
    case PIMPC_V: w = p.nb; off = p.oV(); break;
    case PIMPC_TH: w = p.nb; off = p.oTH(); break;
    case PIMPC_BE: w = p.nb; off = p.oBE(); break;
    case PIMPC_LA: w = p.nb; off = p.oLA(); break;
    case PIMPC_D: w = p.nu; off = p.oD(); break;
    default: w = p.nu; off = p.oDE(); break;
    }
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < p.N * w; idx += gridDim.x * blockDim.x) {
        const int k = idx / w, i = idx - k * w;
        T *src = dense ? dense + ((size_t)b * p.N + k) * w + i : S + p.st(b, k) + off + i;
        T *ext = buf + ((size_t)b * p.N + k) * w + i;
        if (set) *src = *ext; else *ext = *src;
    }
}

// Warm-start shift (reading R18): record k of the next rotating buffer = record min(k + steps, N-1) of the current one.
template <typename T>
__global__ void k_shift(Prob<T> p, int steps)
{
    const int b = blockIdx.y;
    const InstCtl c = p.ctl[b];
    const int dst = (c.i_cur + 1) % 3;
    const T *src = p.S + (size_t)c.i_cur * p.buf_stride;
    T *out = p.S + (size_t)dst * p.buf_stride;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < p.N * p.rec; idx += gridDim.x * blockDim.x) {
        const int k = idx / p.rec, i = idx - k * p.rec;
        const int ks = k + steps < p.N ? k + steps : p.N - 1;
        out[p.st(b, k) + i] = src[p.st(b, ks) + i];
    }
}

// after k_shift: the shifted buffer becomes the current iterate
__global__ void k_advance_cur(InstCtl *ctl, int batch)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    ctl[b].i_cur = (ctl[b].i_cur + 1) % 3;
}

__global__ void k_zero_ctl(InstCtl *ctl, int batch, double c0)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    InstCtl c;
    c.alpha = 1.0; c.c_prev = c0; c.c_last = c0; c.kappa = 0.0;
    c.i_prev = 0; c.i_cur = 0; c.i_new = 1; c.done = 0; c.iters = 0; c.restarts = 0; c.pad_[0] = c.pad_[1] = 0;
    ctl[b] = c;
}

} // namespace

template <typename T>
Prob<T> make_prob(pimpc_s *h, double tol)
{
    Prob<T> p{};
    p.nx = h->nx; p.nu = h->nu; p.nb = h->nb; p.N = h->N; p.batch = h->batch; p.rec = h->rec;
    p.has_du = h->has_du; p.has_e = h->has_e; p.has_q = h->has_q;
    p.A = (const T *)h->A; p.B = (const T *)h->B; p.e = h->has_e ? (const T *)h->e : nullptr;
    p.x0 = (const T *)h->x0; p.uprev = (const T *)h->uprev;
    p.Q = (const T *)h->Q; p.R = (const T *)h->R;
    p.P = h->has_P ? (const T *)h->P : nullptr;
    p.Wdu = h->has_wdu ? (const T *)h->Wdu : nullptr;
    p.qbar = (const T *)h->qbar;
    p.cost_stride_q = h->cost_per_instance ? h->nx * h->nx : 0;
    p.cost_stride_r = h->cost_per_instance ? h->nu * h->nu : 0;
    p.qbar_stride = h->cost_per_instance ? h->nb : 0;
    p.lo = (const T *)h->lo; p.hi = (const T *)h->hi; p.dlo = (const T *)h->dlo; p.dhi = (const T *)h->dhi;
    p.bnd_stride = h->bnd_per_instance ? h->nb : 0;
    p.dbnd_stride = h->bnd_per_instance ? h->nu : 0;
    p.lo_k = h->has_lok ? (const T *)h->lo_k : nullptr; p.hi_k = h->has_lok ? (const T *)h->hi_k : nullptr;
    p.qbar_k = h->has_qbk ? (const T *)h->qbar_k : nullptr;
    p.lok_bstride = h->lok_per_instance ? (size_t)h->N * h->nb : 0;
    p.qbk_bstride = h->qbk_per_instance ? (size_t)h->N * h->nb : 0;
    p.set_kind = h->set_kind; p.set_i0 = h->set_i0; p.set_len = h->set_len;
    p.set_a = (const T *)h->set_a; p.set_b = h->set_b; p.set_inv_aa = h->set_inv_aa;
    if (h->has_qbk) p.has_q = 1;
    p.H = (T *)h->H; p.M = (T *)h->M; p.S = (T *)h->S;
    p.buf_stride = (size_t)h->batch * h->N * h->rec;
    p.X = (T *)h->X; p.DU = (T *)h->DU;
    p.ctl = h->ctl; p.partial = h->partial; p.nparts = 0;
    p.hist_c = h->hist_c; p.hist_a = h->hist_a; p.hist_cap = h->hist_cap;
    p.err = h->err;
    p.rho = h->rho; p.eta = h->eta; p.tol = tol; p.c0 = h->c0;
    return p;
}
template Prob<float> make_prob<float>(pimpc_s *, double);
template Prob<double> make_prob<double>(pimpc_s *, double);

template <typename T, int NX, int NU>
static int setup_small_t(pimpc_s *h, const int *list, int nlist)
{
    Prob<T> p = make_prob<T>(h, 0.0);
    constexpr int GPB = 4 * (32 / pow2ceil_k(NX + NU));
    const long long nst = list ? nlist : (long long)h->batch * h->N;
    k_setup_small<T, NX, NU><<<(unsigned)((nst + GPB - 1) / GPB), 128, 0, h->stream>>>(p, list, nst);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}

template <typename T>
static int setup_t(pimpc_s *h, const int *list, int nlist)
{
    if (h->nx == 12 && h->nu == 4) return setup_small_t<T, 12, 4>(h, list, nlist);
    if (h->nx == 4 && h->nu == 2) return setup_small_t<T, 4, 2>(h, list, nlist);
    Prob<T> p = make_prob<T>(h, 0.0);
    if (h->nb > 8 && h->nb <= 64 && h->nu <= 32) {             // rows in registers, four threads per row (tiny matrices: k_setup below)
        const long long nst = list ? nlist : (long long)h->batch * h->N;
        if (h->nb <= 32) k_setup_rows<T, 32><<<(unsigned)nst, 128, (32 * 40 + 2 * 40 + 2 * 32) * sizeof(double), h->stream>>>(p, list);
        else k_setup_rows<T, 64><<<(unsigned)nst, 256, (64 * 72 + 2 * 72 + 2 * 64) * sizeof(double), h->stream>>>(p, list);
        PIMPC_CUDA_TRY(h, cudaGetLastError());
        return 1;
    }
    const size_t smem = ((size_t)h->nb * h->nb + 2 * h->nb) * sizeof(double);
    if (smem > 48 * 1024)
        PIMPC_CUDA_TRY(h, cudaFuncSetAttribute(k_setup<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int threads = h->nb * h->nb >= 1024 ? 256 : 128;
    const long long nst = list ? nlist : (long long)h->batch * h->N;
    k_setup<T><<<(unsigned)nst, threads, smem, h->stream>>>(p, list);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}

int launch_setup(pimpc_s *h, const int *list_dev, int nlist)
{
    return h->dtype == PIMPC_F64 ? setup_t<double>(h, list_dev, nlist) : setup_t<float>(h, list_dev, nlist);
}

int launch_tracking(pimpc_s *h, int ny, const void *C, const void *Wy, const void *Wu, const void *ry, const void *ru,
                    int nref, void *qbar_out)
{
    const int total = h->nx * h->nx + h->nu * h->nu + nref * h->nb, th = 128, bl = std::min(1024, (total + th - 1) / th);
    if (h->dtype == PIMPC_F64)
        k_tracking<double><<<bl, th, 0, h->stream>>>(h->nx, h->nu, ny, (const double *)C, (const double *)Wy, (const double *)Wu,
                                                     (const double *)ry, (const double *)ru, nref, (double *)h->Q, (double *)h->R, (double *)qbar_out);
    else
        k_tracking<float><<<bl, th, 0, h->stream>>>(h->nx, h->nu, ny, (const float *)C, (const float *)Wy, (const float *)Wu,
                                                    (const float *)ry, (const float *)ru, nref, (float *)h->Q, (float *)h->R, (float *)qbar_out);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}

int launch_begin(pimpc_s *h)
{
    const int th = 128, bl = (h->batch + th - 1) / th;
    if (h->dtype == PIMPC_F64) k_begin<double><<<bl, th, 0, h->stream>>>(make_prob<double>(h, 0.0));
    else k_begin<float><<<bl, th, 0, h->stream>>>(make_prob<float>(h, 0.0));
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}

int launch_gather(pimpc_s *h, void *x, void *u, void *du, pimpc_result *res)
{
    const int work = h->N * (h->nb + h->nu);
    const int th = 256, bl = min(64, (work + th - 1) / th);
    int n = 0;
    if (x || u || du) {
        if (h->dtype == PIMPC_F64)
            k_gather<double><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<double>(h, 0.0), (double *)x, (double *)u, (double *)du);
        else
            k_gather<float><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<float>(h, 0.0), (float *)x, (float *)u, (float *)du);
        ++n;
    }
    if (res) {
        const int rows = h->N * h->nb;
        const int nch = std::max(1, std::min(64, rows / 2048)), chunk = (rows + nch - 1) / nch;
        const int rc = pimpc_grow(h, (void **)&h->res_part, &h->res_part_cap, (size_t)h->batch * nch * sizeof(double));
        if (rc) return rc;
        if (h->dtype == PIMPC_F64) k_rprim<double><<<dim3(nch, h->batch), 128, 0, h->stream>>>(make_prob<double>(h, 0.0), h->res_part, chunk);
        else k_rprim<float><<<dim3(nch, h->batch), 128, 0, h->stream>>>(make_prob<float>(h, 0.0), h->res_part, chunk);
        k_result<<<(h->batch + 127) / 128, 128, 0, h->stream>>>(h->ctl, h->res_part, nch, h->batch, h->rho, res);
        n += 2;
    }
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return n;
}

int launch_state_io(pimpc_s *h, int which, void *buf, int set)
{
    const int work = h->N * h->nb;
    const int th = 256, bl = min(64, (work + th - 1) / th);
    if (h->dtype == PIMPC_F64)
        k_state_io<double><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<double>(h, 0.0), which, (double *)buf, set);
    else
        k_state_io<float><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<float>(h, 0.0), which, (float *)buf, set);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}

int launch_shift(pimpc_s *h, int steps)
{
    const int work = h->N * h->rec;
    const int th = 256, bl = min(64, (work + th - 1) / th);
    if (h->dtype == PIMPC_F64) k_shift<double><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<double>(h, 0.0), steps);
    else k_shift<float><<<dim3(bl, h->batch), th, 0, h->stream>>>(make_prob<float>(h, 0.0), steps);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    k_advance_cur<<<(h->batch + 127) / 128, 128, 0, h->stream>>>(h->ctl, h->batch);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 2;
}

int launch_zero_state(pimpc_s *h)
{
    const size_t sbytes = 3 * (size_t)h->batch * h->N * h->rec * h->esz;
    PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->S, 0, sbytes, h->stream));
    PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->X, 0, (size_t)h->batch * h->N * h->nb * h->esz, h->stream));
    PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->DU, 0, (size_t)h->batch * h->N * h->nu * h->esz, h->stream));
    const int th = 128, bl = (h->batch + th - 1) / th;
    k_zero_ctl<<<bl, th, 0, h->stream>>>(h->ctl, h->batch, h->c0);
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    return 1;
}
