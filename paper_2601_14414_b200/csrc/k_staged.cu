// STAGED engine: Algorithm 1 with one kernel per step per iteration.
// Works for any nx, nu (nb <= 128) and either dtype; all operands come from global memory / L2.
// It is the simplest-correct device path, the generic fallback and the A/B baseline for the
// fused engines.  Five launches per iteration:
//   k_hat    : hats from (cur, prev, kappa) (steps 6/7 of the previous iteration),
//              w_k = zhat_{k+1} - vhat_k - ebar_k + lambdahat_k
//   k_adj    : g_k = Abar_k^T w_k  and  rhs_k = Bbar_k^T (vhat_k - betahat_k) [+ dhat_k - deltahat_k]
//   k_primal : step 1: DU[k] = M_k rhs_k, X[k] = H_k (qbar + rho (zhat - thetahat) + rho g_{k+1})
//   k_dual   : steps 2-4: gamma, z, v, theta, beta, lambda (+ d, delta), partial sums of c
//   k_decide : steps 5-7: c, stop / accept / restart, alpha, kappa, buffer rotation
// Thread mapping: one thread per (stage, row i < nb); a CTA covers `spb` consecutive stages of one instance.
#include "pimpc_internal.h"

namespace {

template <typename T>
struct StagedScratch {
    T *hat;   // [batch][N][rec]
    T *W;     // [batch][N][nb]
    T *G;     // [batch][N][nb]
    T *rhs;   // [batch][N][nu]
};

template <typename T>
__global__ void k_hat(Prob<T> p, StagedScratch<T> s, int spb)
{
    const int b = blockIdx.y;
    const InstCtl c = p.ctl[b];
    if (c.done) return;
    const int nb = p.nb, nu = p.nu;
    const int t = threadIdx.x, ks = t / nb, i = t - ks * nb;
    const int k = blockIdx.x * spb + ks;
    if (ks >= spb || k >= p.N) return;
    const T kap = (T)c.kappa;
    const T *cur = p.S + (size_t)c.i_cur * p.buf_stride + p.st(b, k);
    const T *prv = p.S + (size_t)c.i_prev * p.buf_stride + p.st(b, k);
    T *hat = s.hat + p.st(b, k);
    T h[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
        const T a = cur[f * nb + i], q = prv[f * nb + i];
        h[f] = a + kap * (a - q);
        hat[f * nb + i] = h[f];
    }
    if (p.has_du && i < nu) {
        for (int f = 0; f < 2; ++f) {
            const int o = 5 * nb + f * nu + i;
            const T a = cur[o], q = prv[o];
            hat[o] = a + kap * (a - q);
        }
    }
    const T ek = (p.e && i < p.nx) ? p.e[((size_t)b * p.N + k) * p.nx + i] : (T)0;
    s.W[((size_t)b * p.N + k) * nb + i] = h[0] - h[1] - ek + h[4];     // zhat - vhat - ebar + lambdahat
}

template <typename T>
__global__ void k_adj(Prob<T> p, StagedScratch<T> s, int spb)
{
    const int b = blockIdx.y;
    if (p.ctl[b].done) return;
    const int nb = p.nb, nu = p.nu, nx = p.nx;
    const int t = threadIdx.x, ks = t / nb, j = t - ks * nb;
    const int k = blockIdx.x * spb + ks;
    if (ks >= spb || k >= p.N) return;
    const size_t sk = (size_t)b * p.N + k;
    const T *Ak = p.A + sk * nx * nx, *Bk = p.B + sk * nx * nu;
    const T *w = s.W + sk * nb;
    const T *hat = s.hat + p.st(b, k);
    // g_k[j] = sum_i Abar_k[i][j] w[i],  Abar = [A B; 0 I]
    T g = (T)0;
    if (j < nx) {
        for (int i = 0; i < nx; ++i) g += Ak[i * nx + j] * w[i];
    } else {
        const int jj = j - nx;
        T r = (T)0;
        for (int i = 0; i < nx; ++i) {
            const T bij = Bk[i * nu + jj];
            g += bij * w[i];
            r += bij * (hat[p.oV() + i] - hat[p.oBE() + i]);
        }
        g += w[j];
        r += hat[p.oV() + j] - hat[p.oBE() + j];
        if (p.has_du) r += hat[p.oD() + jj] - hat[p.oDE() + jj];
        s.rhs[sk * nu + jj] = r;
    }
    s.G[sk * nb + j] = g;
}

template <typename T>
__global__ void k_primal(Prob<T> p, StagedScratch<T> s, int spb)
{
    const int b = blockIdx.y;
    if (p.ctl[b].done) return;
    const int nb = p.nb, nu = p.nu;
    const int t = threadIdx.x, ks = t / nb, i = t - ks * nb;
    const int k = blockIdx.x * spb + ks;
    if (ks >= spb || k >= p.N) return;
    const size_t sk = (size_t)b * p.N + k;
    const T *Hk = p.H + sk * nb * nb;
    const T *hat = s.hat + p.st(b, k);
    const T rho = (T)p.rho;
    const bool inner = (k < p.N - 1);
    const T *g1 = s.G + (sk + (inner ? 1 : 0)) * nb;
    T x = (T)0;
    for (int j = 0; j < nb; ++j) {
        T h = p.qbar_at(b, k, j) + rho * (hat[p.oZ() + j] - hat[p.oTH() + j]);
        if (inner) h += rho * g1[j];
        x += Hk[j * nb + i] * h;            // H symmetric: column i == row i, coalesced over i
    }
    p.X[sk * nb + i] = x;
    if (i < nu) {
        const T *Mk = p.M + sk * nu * nu;
        const T *r = s.rhs + sk * nu;
        T d = (T)0;
        for (int j = 0; j < nu; ++j) d += Mk[i * nu + j] * r[j];
        p.DU[sk * nu + i] = d;
    }
}

template <typename T>
__device__ __forceinline__ T clipT(T v, T lo, T hi) { return v < lo ? lo : (v > hi ? hi : v); }

template <typename T>
__global__ void k_dual(Prob<T> p, StagedScratch<T> s, int spb)
{
    __shared__ double red[32];
    extern __shared__ __align__(16) unsigned char cand_raw[];  // [spb][nb] arguments of Proj (only with a general set)
    T *cand = reinterpret_cast<T *>(cand_raw);
    const int b = blockIdx.y;
    const InstCtl c = p.ctl[b];
    if (c.done) return;
    const int nb = p.nb, nu = p.nu, nx = p.nx;
    const int t = threadIdx.x, ks = t / nb, i = t - ks * nb;
    const int k = blockIdx.x * spb + ks;
    T acc = (T)0;
    const bool act = ks < spb && k < p.N;
    const bool gset = p.set_kind != PIMPC_SET_NONE;            // uniform over the grid
    T av = (T)0, bv = (T)0, zarg = (T)0;
    if (act) {
        const size_t sk = (size_t)b * p.N + k;
        const T *Ak = p.A + sk * nx * nx, *Bk = p.B + sk * nx * nu;
        const T *hat = s.hat + p.st(b, k);
        const T *du = p.DU + sk * nu;
        // a = Bbar du + betahat ; b = Abar xbar_k + ebar - lambdahat, xbar_k = X[k-1] (new) or xbar_0
        if (i < nx) {
            av = (T)0;
            for (int j = 0; j < nu; ++j) av += Bk[i * nu + j] * du[j];
            bv = (T)0;
            if (k == 0) {
                for (int j = 0; j < nx; ++j) bv += Ak[i * nx + j] * p.x0[(size_t)b * nx + j];
                for (int j = 0; j < nu; ++j) bv += Bk[i * nu + j] * p.uprev[(size_t)b * nu + j];
            } else {
                const T *xp = p.X + (sk - 1) * nb;
                for (int j = 0; j < nx; ++j) bv += Ak[i * nx + j] * xp[j];
                for (int j = 0; j < nu; ++j) bv += Bk[i * nu + j] * xp[nx + j];
            }
            if (p.e) bv += p.e[sk * nx + i];
        } else {
            av = du[i - nx];
            bv = (k == 0) ? p.uprev[(size_t)b * nu + (i - nx)] : p.X[(sk - 1) * nb + i];
        }
        av += hat[p.oBE() + i];
        bv -= hat[p.oLA() + i];
        zarg = ((T)2 * (p.X[sk * nb + i] + hat[p.oTH() + i] + bv) + (av - bv)) / (T)3;       // argument of Proj
        if (gset) cand[ks * nb + i] = zarg;
    }
    if (gset) __syncthreads();
    if (act) {
        const size_t sk = (size_t)b * p.N + k;
        const T *hat = s.hat + p.st(b, k);
        const T *du = p.DU + sk * nu;
        T *nw = p.S + (size_t)c.i_new * p.buf_stride + p.st(b, k);
        const T zh = hat[p.oZ() + i], vh = hat[p.oV() + i], thh = hat[p.oTH() + i];
        const T beh = hat[p.oBE() + i], lah = hat[p.oLA() + i];
        const T gam = av - bv;
        const T x = p.X[sk * nb + i];
        // z_{k+1} = Proj_Xbar(.): the box on every component outside the general set, the set's closed form inside it
        T zn;
        if (gset && i >= p.set_i0 && i < p.set_i0 + p.set_len) zn = proj_set_component(p, cand + ks * nb + p.set_i0, i - p.set_i0);
        else zn = clipT(zarg, p.lo_at(b, k, i), p.hi_at(b, k, i));
        const T vn = (T)0.5 * (zn + gam);
        const T thn = thh + x - zn;
        const T ben = av - vn;
        const T lan = zn - bv - vn;
        nw[p.oZ() + i] = zn; nw[p.oV() + i] = vn; nw[p.oTH() + i] = thn; nw[p.oBE() + i] = ben; nw[p.oLA() + i] = lan;
        T d0 = thn - thh, d1 = ben - beh, d2 = lan - lah, d3 = zn - zh, d4 = vn - vh, d5 = (zn - vn) - (zh - vh);
        acc = d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5;
        if (p.has_du && i < nu) {
            const T dh = hat[p.oD() + i], deh = hat[p.oDE() + i];
            const T dlo = p.dlo[(size_t)b * p.dbnd_stride + i], dhi = p.dhi[(size_t)b * p.dbnd_stride + i];
            const T dn = clipT(du[i] + deh, dlo, dhi);
            const T den = deh + du[i] - dn;
            nw[p.oD() + i] = dn; nw[p.oDE() + i] = den;
            const T e0 = den - deh, e1 = dn - dh;
            acc += e0 * e0 + e1 * e1;
        }
    }
    // block reduction in double, fixed order
    double v = (double)acc;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = t >> 5, lane = t & 31, nw_ = (blockDim.x + 31) >> 5;
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (t == 0) {
        double sum = 0.0;
        for (int w = 0; w < nw_; ++w) sum += red[w];
        p.partial[(size_t)b * p.nparts + blockIdx.x] = sum;
    }
}

// steps 5-7 for one instance per warp
template <typename T>
__global__ void k_decide(Prob<T> p, int it)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (b >= p.batch) return;
    InstCtl c = p.ctl[b];
    if (c.done) return;
    double s = 0.0;
    for (int q = lane; q < p.nparts; q += 32) s += p.partial[(size_t)b * p.nparts + q];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane != 0) return;
    const double cc = p.rho * s;
    c.c_last = cc;
    c.iters = it + 1;
    int accept = 0;
    if (p.tol > 0.0 && cc < p.tol) {                 // step 5: returned iterate = the new one
        c.done = 1;
        c.i_cur = c.i_new;
    } else {
        accept = (cc <= p.eta * c.c_prev);           // step 6 / 7 (R6: <=)
        if (accept) {
            const double an = 0.5 + 0.5 * sqrt(1.0 + 4.0 * c.alpha * c.alpha);
            c.kappa = (c.alpha - 1.0) / an;
            c.alpha = an;
        } else {
            c.kappa = 0.0;
            c.alpha = 1.0;
            c.restarts += 1;
        }
        c.c_prev = cc;
        const int fresh = 3 - c.i_cur - c.i_new;
        c.i_prev = c.i_cur; c.i_cur = c.i_new; c.i_new = fresh;
    }
    if (p.hist_c && it < p.hist_cap) {
        p.hist_c[(size_t)b * p.hist_cap + it] = cc;
        p.hist_a[(size_t)b * p.hist_cap + it] = (unsigned char)accept;
    }
    p.ctl[b] = c;
}

template <typename T>
int run_staged_t(pimpc_s *h, int iters, double tol)
{
    const int nb = h->nb;
    const int spb = nb >= 128 ? 1 : (256 / nb);
    const int threads = ((spb * nb + 31) / 32) * 32;   // whole warps (idle lanes are masked by ks >= spb)
    const int gx = (h->N + spb - 1) / spb;
    const size_t nst = (size_t)h->batch * h->N;
    {
        size_t c0 = h->hat ? ~(size_t)0 : 0, c1 = c0, c2 = c0, c3 = c0;            // allocated once per handle (sizes are fixed)
        int rc = pimpc_grow(h, &h->hat, &c0, nst * h->rec * h->esz);
        if (!rc) rc = pimpc_grow(h, &h->W, &c1, nst * nb * h->esz);
        if (!rc) rc = pimpc_grow(h, &h->G, &c2, nst * nb * h->esz);
        if (!rc) rc = pimpc_grow(h, &h->rhs, &c3, nst * h->nu * h->esz);
        if (!rc) rc = pimpc_grow(h, (void **)&h->partial, &h->partial_cap, (size_t)h->batch * gx * sizeof(double));
        if (rc) return rc;
    }
    Prob<T> p = make_prob<T>(h, tol);
    p.nparts = gx;
    StagedScratch<T> s{(T *)h->hat, (T *)h->W, (T *)h->G, (T *)h->rhs};
    const dim3 grid(gx, h->batch);
    const int dth = 128, dgrid = (h->batch + (dth / 32) - 1) / (dth / 32);
    for (int it = 0; it < iters; ++it) {
        k_hat<T><<<grid, threads, 0, h->stream>>>(p, s, spb);
        k_adj<T><<<grid, threads, 0, h->stream>>>(p, s, spb);
        k_primal<T><<<grid, threads, 0, h->stream>>>(p, s, spb);
        k_dual<T><<<grid, threads, h->set_kind ? (size_t)spb * nb * sizeof(T) : 0, h->stream>>>(p, s, spb);
        k_decide<T><<<dgrid, dth, 0, h->stream>>>(p, it);
    }
    PIMPC_CUDA_TRY(h, cudaGetLastError());
    h->info.grid = gx * h->batch; h->info.block = threads; h->info.smem_bytes = 0;
    return 5 * iters;
}

} // namespace

int run_staged(pimpc_s *h, int iters, double tol)
{
    return h->dtype == PIMPC_F64 ? run_staged_t<double>(h, iters, tol) : run_staged_t<float>(h, iters, tol);
}
