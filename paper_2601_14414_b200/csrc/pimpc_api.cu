// C ABI of libpimpc.so (include/pimpc.h): handle lifetime, host/device marshalling, engine choice.
// Every arithmetic step of Algorithm 1 runs in the kernels of k_*.cu; nothing here computes.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

#include "pimpc_internal.h"

namespace {

thread_local std::string g_last_error;   // for calls without a (valid) handle

int fail(pimpc_s *h, int code, const std::string &msg)
{
    if (h) h->errmsg = msg;
    g_last_error = msg;
    return code;
}

bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// Copy `bytes` into device memory of the handle, asynchronously on the handle's stream.  A pageable host source has
// been staged by the CUDA runtime when cudaMemcpyAsync returns (it may be reused at once); a page-locked host source
// or a device source is read when the stream reaches the copy (lifetime rule of include/pimpc.h).  No stream
// synchronisation here: several uploads of one step queue back to back.
int copy_in(pimpc_s *h, void *dst, const void *src, size_t bytes)
{
    if (bytes == 0) return PIMPC_OK;
    PIMPC_CUDA_TRY(h, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, h->stream));
    return PIMPC_OK;
}

int copy_out(pimpc_s *h, void *dst, const void *src, size_t bytes)
{
    if (bytes == 0) return PIMPC_OK;
    const bool dev = is_device_ptr(dst);
    PIMPC_CUDA_TRY(h, cudaMemcpyAsync(dst, src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    return PIMPC_OK;
}

// Bring a small array to the host (for validation) as doubles.
int fetch_host(pimpc_s *h, const void *src, size_t n, std::vector<double> &out)
{
    std::vector<unsigned char> raw(n * h->esz);
    if (is_device_ptr(src)) {
        PIMPC_CUDA_TRY(h, cudaMemcpyAsync(raw.data(), src, raw.size(), cudaMemcpyDeviceToHost, h->stream));
        PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    } else {
        memcpy(raw.data(), src, raw.size());
    }
    out.resize(n);
    for (size_t i = 0; i < n; ++i)
        out[i] = h->dtype == PIMPC_F64 ? ((const double *)raw.data())[i] : (double)((const float *)raw.data())[i];
    return PIMPC_OK;
}

int fill_value(pimpc_s *h, void *dst, size_t n, double v)
{
    std::vector<unsigned char> raw(n * h->esz);
    for (size_t i = 0; i < n; ++i) {
        if (h->dtype == PIMPC_F64) ((double *)raw.data())[i] = v;
        else ((float *)raw.data())[i] = (float)v;
    }
    PIMPC_CUDA_TRY(h, cudaMemcpyAsync(dst, raw.data(), raw.size(), cudaMemcpyHostToDevice, h->stream));
    PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return PIMPC_OK;
}

int fill_identity(pimpc_s *h, void *dst, int n)
{
    std::vector<unsigned char> raw((size_t)n * n * h->esz, 0);
    for (int i = 0; i < n; ++i) {
        if (h->dtype == PIMPC_F64) ((double *)raw.data())[i * n + i] = 1.0;
        else ((float *)raw.data())[i * n + i] = 1.0f;
    }
    PIMPC_CUDA_TRY(h, cudaMemcpyAsync(dst, raw.data(), raw.size(), cudaMemcpyHostToDevice, h->stream));
    PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return PIMPC_OK;
}

// Device memory of the handle: carved from the caller's workspace (opts.workspace) while it lasts, else cudaMalloc.
int dalloc(pimpc_s *h, void **p, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    if (h->ws) {
        const size_t need = (bytes + 255) / 256 * 256;
        if (h->ws_used + need <= h->ws_bytes) { *p = h->ws + h->ws_used; h->ws_used += need; return PIMPC_OK; }
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(h, PIMPC_ENOMEM, std::string("cudaMalloc failed: ") + cudaGetErrorString(e));
    }
    h->device_bytes += bytes;
    return PIMPC_OK;
}

// Device staging area of at least `bytes` (kept in the handle: no cudaMalloc / cudaFree, which synchronise the
// whole device, on the result path).
int staging(pimpc_s *h, size_t bytes, void **out)
{
    const int rc = pimpc_grow(h, &h->stage_buf, &h->stage_bytes, bytes);
    *out = h->stage_buf;
    return rc;
}

int rec_len(int nb, int nu) { return ((5 * nb + 2 * nu + 3) / 4) * 4; }

struct Sizes {
    size_t A, B, e, x0, up, H, M, S, X, DU, cost, bnd, ctl;
};

Sizes sizes(int nx, int nu, int N, int batch, size_t esz)
{
    const size_t nb = nx + nu, nst = (size_t)batch * N;
    Sizes s;
    s.A = nst * nx * nx * esz; s.B = nst * nx * nu * esz; s.e = nst * nx * esz;
    s.x0 = (size_t)batch * nx * esz; s.up = (size_t)batch * nu * esz;
    s.H = nst * nb * nb * esz; s.M = nst * nu * nu * esz;
    s.S = 3 * nst * rec_len((int)nb, nu) * esz; s.X = nst * nb * esz; s.DU = nst * nu * esz;
    s.cost = (size_t)batch * (2 * nx * nx + 2 * nu * nu + nb) * esz;
    s.bnd = (size_t)batch * (2 * nb + 2 * nu) * esz;
    s.ctl = (size_t)batch * sizeof(InstCtl);
    return s;
}

int check_handle(pimpc_s *h)
{
    if (!h) return fail(nullptr, PIMPC_EINVAL, "null handle");
    if (h->poisoned) return PIMPC_ESTATE;
    return PIMPC_OK;
}

// Every entry point that touches CUDA runs on the device the handle was created on, whatever the caller's current
// device is (a single process may drive one handle per GPU), and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const pimpc_s *h)
    {
        if (!h) return;
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return; }
        if (prev != h->device) switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// pimpc_set_stage touched stage k of instance b: cache entries H_{k-1} (holds Abar_k) and M_k, H_k... of that instance
void mark_stage_dirty(pimpc_s *h, int b, int k, bool hk_prev, bool mk)
{
    if (h->cache_dirty) return;
    if (h->dirty_stages.size() > 4096) { h->cache_dirty = true; h->dirty_stages.clear(); return; }
    if (hk_prev && k > 0) h->dirty_stages.push_back(b * h->N + k - 1);
    if (mk) h->dirty_stages.push_back(b * h->N + k);
}

int deferred_error(pimpc_s *h)
{
    int flag = 0;
    PIMPC_CUDA_TRY(h, cudaMemcpyAsync(&flag, h->err, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (flag) {
        PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->err, 0, sizeof(int), h->stream));
        h->cache_dirty = true;
        if (flag & PIMPC_DEVERR_NONFINITE) return fail(h, PIMPC_EINVAL, "non-finite value in A, B, Q, R, x0 or u_prev");
        return fail(h, PIMPC_ENOTPD, "a cache matrix (H_k or M_k) is not positive definite");
    }
    return PIMPC_OK;
}

} // namespace

int pimpc_grow(pimpc_s *h, void **ptr, size_t *cap, size_t bytes)
{
    if (*ptr && *cap >= bytes) return PIMPC_OK;
    if (*ptr) {
        cudaStreamSynchronize(h->stream);        // the old buffer may still be in use by queued work
        cudaFree(*ptr);
        h->device_bytes -= *cap;
        *ptr = nullptr; *cap = 0;
    }
    if (bytes == 0) bytes = 16;
    if (cudaMalloc(ptr, bytes) != cudaSuccess) {
        cudaGetLastError();
        *ptr = nullptr;
        return fail(h, PIMPC_ENOMEM, "cudaMalloc (engine scratch) failed");
    }
    *cap = bytes; h->device_bytes += bytes;
    return PIMPC_OK;
}

extern "C" {

const char *pimpc_version(void) { return "pimpc-b200 0.1 (sm_100a)"; }

void pimpc_default_opts(pimpc_opts *o)
{
    if (!o) return;
    o->dtype = PIMPC_F64; o->engine = PIMPC_ENGINE_AUTO; o->rho = 1.0; o->eta = 0.999; o->c0 = 1.0;
    o->history = 0; o->stream = nullptr; o->workspace = nullptr; o->workspace_bytes = 0;
    memset(&o->tune, 0, sizeof(o->tune));
}

// The allocations of pimpc_create, in order (dalloc rounds each to 256 bytes inside a workspace).
static std::vector<size_t> create_allocs(int nx, int nu, int N, int batch, size_t esz, int history)
{
    const Sizes s = sizes(nx, nu, N, batch, esz);
    const size_t nb = nx + nu, b = batch;
    std::vector<size_t> v = {s.A, s.B, s.x0, s.up, s.H, s.M, s.S, s.X, s.DU,
                             b * nx * nx * esz, b * nx * nx * esz, b * nu * nu * esz, b * nu * nu * esz, b * nb * esz,
                             b * nb * esz, b * nb * esz, b * nu * esz, b * nu * esz, s.ctl, sizeof(int)};
    if (history > 0) { v.push_back(b * history * sizeof(double)); v.push_back(b * (size_t)history); }
    return v;
}

size_t pimpc_workspace_bytes(int nx, int nu, int N, int batch, const pimpc_opts *opts)
{
    if (nx <= 0 || nu <= 0 || N <= 0 || batch <= 0 || nx + nu > PIMPC_MAX_NB || batch > 65535) return 0;
    const size_t esz = (opts && opts->dtype == PIMPC_F32) ? 4 : 8;
    size_t tot = 0;
    for (size_t a : create_allocs(nx, nu, N, batch, esz, opts ? opts->history : 0)) tot += (std::max<size_t>(a, 16) + 255) / 256 * 256;
    return tot;
}

int pimpc_create(pimpc_t *out, int nx, int nu, int N, int batch, const pimpc_opts *opts)
{
    if (!out) return fail(nullptr, PIMPC_EINVAL, "out is NULL");
    *out = nullptr;
    pimpc_opts o;
    pimpc_default_opts(&o);
    if (opts) o = *opts;
    if (o.rho == 0.0) o.rho = 1.0;
    if (o.eta < 0.0) o.eta = 0.999;
    if (o.c0 == 0.0) o.c0 = 1.0;
    if (nx <= 0 || nu <= 0 || N <= 0 || batch <= 0) return fail(nullptr, PIMPC_EINVAL, "nx, nu, N, batch must be positive");
    if (nx + nu > PIMPC_MAX_NB) return fail(nullptr, PIMPC_EINVAL, "nx + nu > 160 is not supported");
    if (batch > 65535) return fail(nullptr, PIMPC_EINVAL, "batch > 65535 is not supported (one handle per 65535 instances)");
    if (o.workspace) {
        if (((uintptr_t)o.workspace & 255) || !is_device_ptr(o.workspace)) return fail(nullptr, PIMPC_EINVAL, "workspace must be 256-byte aligned device memory");
        if (o.workspace_bytes < pimpc_workspace_bytes(nx, nu, N, batch, &o)) return fail(nullptr, PIMPC_EINVAL, "workspace smaller than pimpc_workspace_bytes()");
    }
    const pimpc_tune &tu = o.tune;
    if (tu.grid < 0 || tu.ctas_per_sm < 0 || tu.ring_slots < 0 || tu.stages_per_group < 0 || tu.stages_per_group > 2 ||
        tu.cluster < -1 || tu.cluster > 16 || tu.rows_per_lane < 0 || tu.rows_per_lane > 2 || tu.lookahead < -1 || tu.lookahead > 1)
        return fail(nullptr, PIMPC_EINVAL, "bad opts.tune");
    if (!(o.rho > 0.0) || !std::isfinite(o.rho)) return fail(nullptr, PIMPC_EINVAL, "rho must be positive");
    if (o.dtype != PIMPC_F64 && o.dtype != PIMPC_F32) return fail(nullptr, PIMPC_EINVAL, "bad dtype");
    if (o.engine < PIMPC_ENGINE_AUTO || o.engine > PIMPC_ENGINE_COOP) return fail(nullptr, PIMPC_EINVAL, "bad engine");
    if (o.history < 0) return fail(nullptr, PIMPC_EINVAL, "history < 0");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, PIMPC_ECUDA, "no CUDA device (libpimpc has no CPU fallback)");
    }
    pimpc_s *h = new (std::nothrow) pimpc_s();
    if (!h) return fail(nullptr, PIMPC_ENOMEM, "out of host memory");
    h->nx = nx; h->nu = nu; h->nb = nx + nu; h->N = N; h->batch = batch;
    h->rec = rec_len(h->nb, nu);
    h->dtype = o.dtype; h->esz = o.dtype == PIMPC_F64 ? 8 : 4;
    h->engine_req = o.engine; h->rho = o.rho; h->eta = o.eta; h->c0 = o.c0; h->hist_cap = o.history;
    h->stream = (cudaStream_t)o.stream;
    h->tune = o.tune;
    h->ws = (unsigned char *)o.workspace; h->ws_bytes = o.workspace ? o.workspace_bytes : 0;
    cudaGetDevice(&h->device);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, h->device) != cudaSuccess) { delete h; return fail(nullptr, PIMPC_ECUDA, "cudaGetDeviceProperties failed"); }
    h->sm_count = prop.multiProcessorCount;
    h->smem_optin = prop.sharedMemPerBlockOptin;

    const Sizes s = sizes(nx, nu, N, batch, h->esz);
    int rc = PIMPC_OK;
    auto A_ = [&](void **p, size_t bytes) { if (rc == PIMPC_OK) rc = dalloc(h, p, bytes); };
    A_(&h->A, s.A); A_(&h->B, s.B); A_(&h->x0, s.x0); A_(&h->uprev, s.up);
    A_(&h->H, s.H); A_(&h->M, s.M); A_(&h->S, s.S); A_(&h->X, s.X); A_(&h->DU, s.DU);
    A_(&h->Q, (size_t)batch * nx * nx * h->esz); A_(&h->P, (size_t)batch * nx * nx * h->esz);
    A_(&h->R, (size_t)batch * nu * nu * h->esz); A_(&h->Wdu, (size_t)batch * nu * nu * h->esz);
    A_(&h->qbar, (size_t)batch * h->nb * h->esz);
    A_(&h->lo, (size_t)batch * h->nb * h->esz); A_(&h->hi, (size_t)batch * h->nb * h->esz);
    A_(&h->dlo, (size_t)batch * nu * h->esz); A_(&h->dhi, (size_t)batch * nu * h->esz);
    A_((void **)&h->ctl, s.ctl); A_((void **)&h->err, sizeof(int));
    if (h->hist_cap > 0) {
        A_((void **)&h->hist_c, (size_t)batch * h->hist_cap * sizeof(double));
        A_((void **)&h->hist_a, (size_t)batch * h->hist_cap);
    }
    if (rc != PIMPC_OK) { std::string m = h->errmsg; pimpc_destroy(h); return fail(nullptr, rc, m); }

    // defaults: A = B = 0, x0 = u_prev = 0, Q = I, R = I, qbar = 0, bounds = +-inf, cold start
    auto ok = [&](cudaError_t e) { if (e != cudaSuccess && rc == PIMPC_OK) { rc = PIMPC_ECUDA; h->errmsg = cudaGetErrorString(e); } };
    ok(cudaMemsetAsync(h->A, 0, s.A, h->stream)); ok(cudaMemsetAsync(h->B, 0, s.B, h->stream));
    ok(cudaMemsetAsync(h->x0, 0, s.x0, h->stream)); ok(cudaMemsetAsync(h->uprev, 0, s.up, h->stream));
    ok(cudaMemsetAsync(h->qbar, 0, (size_t)batch * h->nb * h->esz, h->stream));
    ok(cudaMemsetAsync(h->err, 0, sizeof(int), h->stream));
    if (rc == PIMPC_OK) rc = fill_identity(h, h->Q, nx);
    if (rc == PIMPC_OK) rc = fill_identity(h, h->R, nu);
    const double inf = INFINITY;
    if (rc == PIMPC_OK) rc = fill_value(h, h->lo, h->nb, -inf);
    if (rc == PIMPC_OK) rc = fill_value(h, h->hi, h->nb, inf);
    if (rc == PIMPC_OK) rc = fill_value(h, h->dlo, nu, -inf);
    if (rc == PIMPC_OK) rc = fill_value(h, h->dhi, nu, inf);
    if (rc == PIMPC_OK) rc = launch_zero_state(h) < 0 ? PIMPC_ECUDA : PIMPC_OK;
    if (rc != PIMPC_OK) { std::string m = h->errmsg; pimpc_destroy(h); return fail(nullptr, rc, m); }
    h->info.sm_count = h->sm_count;
    for (auto &e : h->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { pimpc_destroy(h); return fail(nullptr, PIMPC_ECUDA, "cudaEventCreate failed"); }
    *out = h;
    return PIMPC_OK;
}

int pimpc_destroy(pimpc_t h)
{
    if (!h) return PIMPC_OK;
    DeviceGuard guard(h);
    if (!h->poisoned) cudaStreamSynchronize(h->stream);
    void *ptrs[] = {h->A, h->B, h->e, h->x0, h->uprev, h->Q, h->R, h->P, h->Wdu, h->qbar, h->lo, h->hi, h->dlo, h->dhi,
                    h->H, h->M, h->S, h->X, h->DU, h->ctl, h->partial, h->hist_c, h->hist_a, h->err,
                    h->hat, h->W, h->G, h->rhs, h->blob, h->alpha_tab, h->kappa_tab, h->spartial, h->coop_buf, h->stage_buf,
                    h->dirty_dev, h->res_part, h->lo_k, h->hi_k, h->qbar_k, h->set_a, h->trk};
    for (void *p : ptrs)                         // memory carved from the caller's workspace is the caller's
        if (p && !(h->ws && (unsigned char *)p >= h->ws && (unsigned char *)p < h->ws + h->ws_bytes)) cudaFree(p);
    for (auto &e : h->ev) if (e) cudaEventDestroy(e);
    cudaGetLastError();
    delete h;
    return PIMPC_OK;
}

int pimpc_set_stage(pimpc_t h, int b, int k, const void *A_k, const void *B_k, const void *e_k,
                    const void *Q, const void *R, const void *bounds, const void *x0)
{
    int rc = check_handle(h);
    if (rc) return rc;
    if (b < 0 || b >= h->batch || k < 0 || k >= h->N) return fail(h, PIMPC_EINVAL, "instance or stage index out of range");
    DeviceGuard guard(h);
    const size_t sk = (size_t)b * h->N + k, esz = h->esz;
    const int nx = h->nx, nu = h->nu, nb = h->nb;
    // H_{k-1} holds Abar_k = [A_k B_k; 0 I], M_k holds B_k: only those cache entries are recomputed
    if (A_k) { rc = copy_in(h, (char *)h->A + sk * nx * nx * esz, A_k, (size_t)nx * nx * esz); if (rc) return rc; mark_stage_dirty(h, b, k, true, false); h->blob_dirty = true; }
    if (B_k) { rc = copy_in(h, (char *)h->B + sk * nx * nu * esz, B_k, (size_t)nx * nu * esz); if (rc) return rc; mark_stage_dirty(h, b, k, true, true); h->blob_dirty = true; }
    if (e_k) {
        if (!h->e) {
            rc = dalloc(h, &h->e, (size_t)h->batch * h->N * nx * esz); if (rc) return rc;
            PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->e, 0, (size_t)h->batch * h->N * nx * esz, h->stream));
        }
        rc = copy_in(h, (char *)h->e + sk * nx * esz, e_k, (size_t)nx * esz); if (rc) return rc;
        h->has_e = 1;
        h->blob_dirty = true;                  // the STREAM engine reads e_k from its packed blobs
    }
    if (Q || R) {
        if (h->cost_per_instance) return fail(h, PIMPC_EINVAL, "per-instance cost is set; use pimpc_set_cost");
        if (Q) { rc = copy_in(h, h->Q, Q, (size_t)nx * nx * esz); if (rc) return rc; }
        if (R) { rc = copy_in(h, h->R, R, (size_t)nu * nu * esz); if (rc) return rc; }
        h->cache_dirty = true;
    }
    if (bounds) {
        if (h->bnd_per_instance) return fail(h, PIMPC_EINVAL, "per-instance bounds are set; use pimpc_set_bounds");
        std::vector<double> v;
        rc = fetch_host(h, bounds, 2 * (size_t)nb, v); if (rc) return rc;
        for (int i = 0; i < nb; ++i)
            if (std::isnan(v[i]) || std::isnan(v[nb + i]) || v[i] > v[nb + i]) return fail(h, PIMPC_EINVAL, "bounds: lo > hi or NaN");
        rc = copy_in(h, h->lo, bounds, (size_t)nb * esz); if (rc) return rc;
        rc = copy_in(h, h->hi, (const char *)bounds + (size_t)nb * esz, (size_t)nb * esz); if (rc) return rc;
    }
    if (x0) { rc = copy_in(h, (char *)h->x0 + (size_t)b * nx * esz, x0, (size_t)nx * esz); if (rc) return rc; }
    return PIMPC_OK;
}

int pimpc_set_stages(pimpc_t h, const void *A, const void *B, const void *e)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    const size_t nst = (size_t)h->batch * h->N, esz = h->esz;
    if (A) { rc = copy_in(h, h->A, A, nst * h->nx * h->nx * esz); if (rc) return rc; h->cache_dirty = true; }
    if (B) { rc = copy_in(h, h->B, B, nst * h->nx * h->nu * esz); if (rc) return rc; h->cache_dirty = true; }
    if (e) {
        if (!h->e) { rc = dalloc(h, &h->e, nst * h->nx * esz); if (rc) return rc; }
        rc = copy_in(h, h->e, e, nst * h->nx * esz); if (rc) return rc;
        h->has_e = 1;
        h->blob_dirty = true;                  // the STREAM engine reads e_k from its packed blobs
    }
    return PIMPC_OK;
}

int pimpc_set_cost(pimpc_t h, const void *Q, const void *R, const void *P, const void *Wdu, const void *qbar,
                   int per_instance)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (!Q || !R) return fail(h, PIMPC_EINVAL, "Q and R are required");
    const size_t rep = per_instance ? h->batch : 1, esz = h->esz;
    const size_t nq = (size_t)h->nx * h->nx, nr = (size_t)h->nu * h->nu;
    rc = copy_in(h, h->Q, Q, rep * nq * esz); if (rc) return rc;
    rc = copy_in(h, h->R, R, rep * nr * esz); if (rc) return rc;
    if (P) { rc = copy_in(h, h->P, P, rep * nq * esz); if (rc) return rc; }
    if (Wdu) { rc = copy_in(h, h->Wdu, Wdu, rep * nr * esz); if (rc) return rc; }
    if (qbar) { rc = copy_in(h, h->qbar, qbar, rep * h->nb * esz); if (rc) return rc; }
    else PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->qbar, 0, (size_t)h->batch * h->nb * esz, h->stream));
    h->has_P = P != nullptr; h->has_wdu = Wdu != nullptr; h->has_q = qbar != nullptr;
    h->has_qbk = 0;                                       // a per-stage linear term of an earlier call is replaced too
    h->cost_per_instance = per_instance ? 1 : 0;
    h->cache_dirty = true;
    return PIMPC_OK;
}

int pimpc_set_bounds(pimpc_t h, const void *lo, const void *hi, const void *du_lo, const void *du_hi, int per_instance)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (!lo || !hi) return fail(h, PIMPC_EINVAL, "lo and hi are required (use +-inf for no bound)");
    if ((du_lo == nullptr) != (du_hi == nullptr)) return fail(h, PIMPC_EINVAL, "du_lo and du_hi must be given together");
    const size_t rep = per_instance ? h->batch : 1, esz = h->esz;
    std::vector<double> a, b;
    rc = fetch_host(h, lo, rep * h->nb, a); if (rc) return rc;
    rc = fetch_host(h, hi, rep * h->nb, b); if (rc) return rc;
    for (size_t i = 0; i < a.size(); ++i)
        if (std::isnan(a[i]) || std::isnan(b[i]) || a[i] > b[i]) return fail(h, PIMPC_EINVAL, "bounds: lo > hi or NaN");
    if (du_lo) {
        rc = fetch_host(h, du_lo, rep * h->nu, a); if (rc) return rc;
        rc = fetch_host(h, du_hi, rep * h->nu, b); if (rc) return rc;
        for (size_t i = 0; i < a.size(); ++i)
            if (std::isnan(a[i]) || std::isnan(b[i]) || a[i] > b[i]) return fail(h, PIMPC_EINVAL, "du bounds: lo > hi or NaN");
    }
    rc = copy_in(h, h->lo, lo, rep * h->nb * esz); if (rc) return rc;
    rc = copy_in(h, h->hi, hi, rep * h->nb * esz); if (rc) return rc;
    const int had_du = h->has_du;
    if (du_lo) {
        rc = copy_in(h, h->dlo, du_lo, rep * h->nu * esz); if (rc) return rc;
        rc = copy_in(h, h->dhi, du_hi, rep * h->nu * esz); if (rc) return rc;
        h->has_du = 1;
    } else {
        h->has_du = 0;
    }
    if (had_du != h->has_du) h->cache_dirty = true;       // M_k contains the +I of the du block (R12)
    h->bnd_per_instance = per_instance ? 1 : 0;
    return PIMPC_OK;
}

int pimpc_set_tracking(pimpc_t h, int ny, const void *C, const void *Wy, const void *Wu, const void *ry, const void *ru,
                       int per_stage)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (ny <= 0 || ny > PIMPC_MAX_NB || !C || !Wy || !Wu) return fail(h, PIMPC_EINVAL, "set_tracking: ny, C, Wy, Wu are required");
    if (h->cost_per_instance) return fail(h, PIMPC_EINVAL, "set_tracking: a per-instance cost is set; use pimpc_set_cost");
    const size_t esz = h->esz, nref = per_stage ? h->N : 1;
    const size_t bC = (size_t)ny * h->nx * esz, bWy = (size_t)ny * ny * esz, bWu = (size_t)h->nu * h->nu * esz;
    const size_t bry = nref * ny * esz, bru = nref * h->nu * esz;
    auto al = [](size_t v) { return (v + 255) / 256 * 256; };
    rc = pimpc_grow(h, &h->trk, &h->trk_cap, al(bC) + al(bWy) + al(bWu) + al(bry) + al(bru)); if (rc) return rc;
    unsigned char *base = (unsigned char *)h->trk;
    void *dC = base, *dWy = base + al(bC), *dWu = (unsigned char *)dWy + al(bWy);
    void *dry = (unsigned char *)dWu + al(bWu), *dru = (unsigned char *)dry + al(bry);
    rc = copy_in(h, dC, C, bC); if (rc) return rc;
    rc = copy_in(h, dWy, Wy, bWy); if (rc) return rc;
    rc = copy_in(h, dWu, Wu, bWu); if (rc) return rc;
    if (ry) { rc = copy_in(h, dry, ry, bry); if (rc) return rc; }
    if (ru) { rc = copy_in(h, dru, ru, bru); if (rc) return rc; }
    void *qout = h->qbar;
    if (per_stage) {
        rc = pimpc_grow(h, &h->qbar_k, &h->qbk_cap, (size_t)h->N * h->nb * esz); if (rc) return rc;
        qout = h->qbar_k;
    }
    const int n = launch_tracking(h, ny, dC, dWy, dWu, ry ? dry : nullptr, ru ? dru : nullptr, (int)nref, qout);
    if (n < 0) return n;
    h->info.total_launches += n;
    h->has_P = 0; h->has_q = 1;
    h->has_qbk = per_stage ? 1 : 0; h->qbk_per_instance = 0;
    if (per_stage) h->blob_dirty = true;
    h->cache_dirty = true;
    return PIMPC_OK;
}

int pimpc_set_stage_terms(pimpc_t h, const void *lo, const void *hi, const void *qbar, int per_instance)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if ((lo == nullptr) != (hi == nullptr)) return fail(h, PIMPC_EINVAL, "set_stage_terms: lo and hi must be given together");
    const size_t rep = per_instance ? h->batch : 1, n = rep * h->N * h->nb, bytes = n * h->esz;
    if (lo) {
        std::vector<double> a, b;
        rc = fetch_host(h, lo, n, a); if (rc) return rc;
        rc = fetch_host(h, hi, n, b); if (rc) return rc;
        for (size_t i = 0; i < n; ++i)
            if (std::isnan(a[i]) || std::isnan(b[i]) || a[i] > b[i]) return fail(h, PIMPC_EINVAL, "stage bounds: lo > hi or NaN");
        rc = pimpc_grow(h, &h->lo_k, &h->lok_cap, bytes); if (rc) return rc;
        rc = pimpc_grow(h, &h->hi_k, &h->hik_cap, bytes); if (rc) return rc;
        rc = copy_in(h, h->lo_k, lo, bytes); if (rc) return rc;
        rc = copy_in(h, h->hi_k, hi, bytes); if (rc) return rc;
    }
    h->has_lok = lo != nullptr; h->lok_per_instance = per_instance ? 1 : 0;
    if (qbar) {
        rc = pimpc_grow(h, &h->qbar_k, &h->qbk_cap, bytes); if (rc) return rc;
        rc = copy_in(h, h->qbar_k, qbar, bytes); if (rc) return rc;
    }
    h->has_qbk = qbar != nullptr; h->qbk_per_instance = per_instance ? 1 : 0;
    return PIMPC_OK;
}

int pimpc_set_constraint(pimpc_t h, int kind, int i0, int len, const void *a, double b)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (kind == PIMPC_SET_NONE) { h->set_kind = PIMPC_SET_NONE; return PIMPC_OK; }
    if (kind < PIMPC_SET_NONE || kind > PIMPC_SET_L1BALL) return fail(h, PIMPC_EINVAL, "set_constraint: bad kind");
    if (i0 < 0 || len <= 0 || i0 + len > h->nb) return fail(h, PIMPC_EINVAL, "set_constraint: component range out of [0, nx + nu)");
    if (!std::isfinite(b)) return fail(h, PIMPC_EINVAL, "set_constraint: b is not finite");
    const bool lin = kind == PIMPC_SET_HALFSPACE || kind == PIMPC_SET_HYPERPLANE;
    if (kind == PIMPC_SET_SOC && len < 2) return fail(h, PIMPC_EINVAL, "set_constraint: a second-order cone needs len >= 2");
    if (kind == PIMPC_SET_L1BALL && b < 0.0) return fail(h, PIMPC_EINVAL, "set_constraint: negative radius");
    double inv_aa = 0.0;
    if (lin) {
        if (!a) return fail(h, PIMPC_EINVAL, "set_constraint: a is required for a halfspace / hyperplane");
        std::vector<double> v;
        rc = fetch_host(h, a, (size_t)len, v); if (rc) return rc;
        double aa = 0.0;
        for (double x : v) { if (!std::isfinite(x)) return fail(h, PIMPC_EINVAL, "set_constraint: a is not finite"); aa += x * x; }
        if (!(aa > 0.0)) return fail(h, PIMPC_EINVAL, "set_constraint: a is zero");
        inv_aa = 1.0 / aa;
        rc = pimpc_grow(h, &h->set_a, &h->set_a_cap, (size_t)len * h->esz); if (rc) return rc;
        rc = copy_in(h, h->set_a, a, (size_t)len * h->esz); if (rc) return rc;
    }
    h->set_kind = kind; h->set_i0 = i0; h->set_len = len; h->set_b = b; h->set_inv_aa = inv_aa;
    return PIMPC_OK;
}

int pimpc_set_x0(pimpc_t h, const void *x0, const void *u_prev)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (!x0) return fail(h, PIMPC_EINVAL, "x0 is NULL");
    rc = copy_in(h, h->x0, x0, (size_t)h->batch * h->nx * h->esz); if (rc) return rc;
    if (u_prev) { rc = copy_in(h, h->uprev, u_prev, (size_t)h->batch * h->nu * h->esz); if (rc) return rc; }
    else PIMPC_CUDA_TRY(h, cudaMemsetAsync(h->uprev, 0, (size_t)h->batch * h->nu * h->esz, h->stream));
    return PIMPC_OK;
}

int pimpc_solve(pimpc_t h, int max_iters, double tol)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (max_iters < 0) return fail(h, PIMPC_EINVAL, "max_iters < 0");
    if (h->hist_cap > 0 && max_iters > h->hist_cap) return fail(h, PIMPC_EINVAL, "max_iters exceeds opts.history");
    int launches = 0, n;
    PIMPC_CUDA_TRY(h, cudaEventRecord(h->ev[0], h->stream));
    h->ev_setup = h->cache_dirty || !h->dirty_stages.empty();
    if (h->cache_dirty) {
        n = launch_setup(h, nullptr, 0); if (n < 0) return n;
        launches += n;
        h->cache_dirty = false;
        h->dirty_stages.clear();
        h->blob_dirty = true;
    } else if (!h->dirty_stages.empty()) {
        // pimpc_set_stage touched a few stages: only their cache entries are re-inverted
        std::vector<int> &v = h->dirty_stages;
        std::sort(v.begin(), v.end());
        v.erase(std::unique(v.begin(), v.end()), v.end());
        rc = pimpc_grow(h, (void **)&h->dirty_dev, &h->dirty_cap, v.size() * sizeof(int)); if (rc) return rc;
        PIMPC_CUDA_TRY(h, cudaMemcpyAsync(h->dirty_dev, v.data(), v.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream));
        PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));          // v is host memory that is cleared below
        n = launch_setup(h, h->dirty_dev, (int)v.size()); if (n < 0) return n;
        launches += n;
        v.clear();
        h->blob_dirty = true;
    }
    n = launch_begin(h); if (n < 0) return n;
    launches += n;
    PIMPC_CUDA_TRY(h, cudaEventRecord(h->ev[1], h->stream));

    int engine = h->engine_req;
    std::string why;
    // per-stage boxes / linear terms and a general convex set are implemented by the STAGED and STREAM engines
    const bool ext = has_stage_terms(h);
    if (ext && (engine == PIMPC_ENGINE_RESIDENT || engine == PIMPC_ENGINE_COOP))
        return fail(h, PIMPC_EINVAL, "per-stage terms / a general set need the STREAM or STAGED engine");
    if (engine == PIMPC_ENGINE_AUTO && ext)
        engine = stream_supported(h, &why) ? PIMPC_ENGINE_STREAM : PIMPC_ENGINE_STAGED;
    if (engine == PIMPC_ENGINE_AUTO)
        engine = resident_supported(h, &why) ? PIMPC_ENGINE_RESIDENT
                 : coop_supported(h, &why) ? PIMPC_ENGINE_COOP
                 : (stream_supported(h, &why) ? PIMPC_ENGINE_STREAM : PIMPC_ENGINE_STAGED);
    if (engine == PIMPC_ENGINE_RESIDENT && !resident_supported(h, &why))
        return fail(h, PIMPC_EINVAL, "RESIDENT engine not applicable: " + why);
    if (engine == PIMPC_ENGINE_STREAM && !stream_supported(h, &why))
        return fail(h, PIMPC_EINVAL, "STREAM engine not applicable: " + why);
    if (engine == PIMPC_ENGINE_COOP && !coop_supported(h, &why))
        return fail(h, PIMPC_EINVAL, "COOP engine not applicable: " + why);
    if (max_iters > 0) {
        if (engine == PIMPC_ENGINE_RESIDENT) n = run_resident(h, max_iters, tol);
        else if (engine == PIMPC_ENGINE_STREAM) n = run_stream(h, max_iters, tol);
        else if (engine == PIMPC_ENGINE_COOP) n = run_coop(h, max_iters, tol);
        else n = run_staged(h, max_iters, tol);
        if (n < 0) return n;
        launches += n;
    }
    PIMPC_CUDA_TRY(h, cudaEventRecord(h->ev[2], h->stream));
    h->ev_pending = true;
    h->info.engine = engine;
    h->info.launches = launches;
    h->info.total_launches += launches;
    return PIMPC_OK;
}

int pimpc_get(pimpc_t h, void *x, void *u, void *du, pimpc_result *res)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    const size_t nst = (size_t)h->batch * h->N, esz = h->esz;
    // gather into device staging when the destination is host memory
    void *dx = nullptr, *du_ = nullptr, *ddu = nullptr;
    pimpc_result *dres = nullptr;
    const size_t bx = nst * h->nx * esz, bu = nst * h->nu * esz, br = (size_t)h->batch * sizeof(pimpc_result);
    auto al = [](size_t v) { return (v + 255) / 256 * 256; };
    const bool hx = x && !is_device_ptr(x), hu = u && !is_device_ptr(u), hd = du && !is_device_ptr(du), hr = res && !is_device_ptr(res);
    const size_t need = (hx ? al(bx) : 0) + (hu ? al(bu) : 0) + (hd ? al(bu) : 0) + (hr ? al(br) : 0);
    unsigned char *sb = nullptr;
    if (need) { rc = staging(h, need, (void **)&sb); if (rc) return rc; }
    size_t off = 0;
    dx = hx ? sb + off : x; off += hx ? al(bx) : 0;
    du_ = hu ? sb + off : u; off += hu ? al(bu) : 0;
    ddu = hd ? sb + off : du; off += hd ? al(bu) : 0;
    dres = hr ? (pimpc_result *)(sb + off) : res;
    int ng = 0;
    if (!rc) { ng = launch_gather(h, dx, du_, ddu, dres); if (ng < 0) rc = PIMPC_ECUDA; }
    if (!rc && x && dx != x) rc = copy_out(h, x, dx, nst * h->nx * esz);
    if (!rc && u && du_ != u) rc = copy_out(h, u, du_, nst * h->nu * esz);
    if (!rc && du && ddu != du) rc = copy_out(h, du, ddu, nst * h->nu * esz);
    if (!rc && res && (void *)dres != (void *)res) rc = copy_out(h, res, dres, (size_t)h->batch * sizeof(pimpc_result));
    h->info.total_launches += ng > 0 ? ng : 0;
    return rc ? rc : deferred_error(h);        // synchronises
}

static int state_width(pimpc_s *h, int which)
{
    switch (which) {
    case PIMPC_X: case PIMPC_Z: case PIMPC_V: case PIMPC_TH: case PIMPC_BE: case PIMPC_LA: return h->nb;
    case PIMPC_D: case PIMPC_DE: case PIMPC_DU: return h->nu;
    default: return -1;
    }
}

int pimpc_get_state(pimpc_t h, int which, void *out)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    const int w = state_width(h, which);
    if (w < 0 || !out) return fail(h, PIMPC_EINVAL, "bad selector or NULL buffer");
    const size_t bytes = (size_t)h->batch * h->N * w * h->esz;
    void *dev = out;
    const bool host = !is_device_ptr(out);
    if (host) { rc = staging(h, bytes, &dev); if (rc) return rc; }
    rc = launch_state_io(h, which, dev, 0) < 0 ? PIMPC_ECUDA : PIMPC_OK;
    if (!rc && host) rc = copy_out(h, out, dev, bytes);
    if (!rc) { cudaError_t e = cudaStreamSynchronize(h->stream); if (e != cudaSuccess) { h->poisoned = 1; rc = fail(h, PIMPC_ECUDA, cudaGetErrorString(e)); } }
    return rc;
}

int pimpc_set_state(pimpc_t h, int which, const void *in)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    const int w = state_width(h, which);
    if (w < 0 || !in || which == PIMPC_X || which == PIMPC_DU) return fail(h, PIMPC_EINVAL, "bad selector (X, DU are outputs) or NULL buffer");
    const size_t bytes = (size_t)h->batch * h->N * w * h->esz;
    void *dev = const_cast<void *>(in);
    const bool host = !is_device_ptr(in);
    if (host) {
        rc = staging(h, bytes, &dev); if (rc) return rc;
        rc = copy_in(h, dev, in, bytes);
    }
    if (!rc) rc = launch_state_io(h, which, dev, 1) < 0 ? PIMPC_ECUDA : PIMPC_OK;
    if (host) cudaStreamSynchronize(h->stream);
    return rc;
}

int pimpc_get_history(pimpc_t h, double *c, unsigned char *accepted)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (h->hist_cap <= 0) return fail(h, PIMPC_EINVAL, "handle was created with history = 0");
    if (c) { rc = copy_out(h, c, h->hist_c, (size_t)h->batch * h->hist_cap * sizeof(double)); if (rc) return rc; }
    if (accepted) { rc = copy_out(h, accepted, h->hist_a, (size_t)h->batch * h->hist_cap); if (rc) return rc; }
    PIMPC_CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return PIMPC_OK;
}

int pimpc_get_cache(pimpc_t h, void *M, void *H)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (h->cache_dirty) return fail(h, PIMPC_ESTATE, "cache not computed yet (call pimpc_solve first)");
    const size_t nst = (size_t)h->batch * h->N;
    if (M) { rc = copy_out(h, M, h->M, nst * h->nu * h->nu * h->esz); if (rc) return rc; }
    if (H) { rc = copy_out(h, H, h->H, nst * h->nb * h->nb * h->esz); if (rc) return rc; }
    return deferred_error(h);
}

int pimpc_reset(pimpc_t h)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    const int n = launch_zero_state(h);
    if (n < 0) return PIMPC_ECUDA;
    h->info.total_launches += n;
    return PIMPC_OK;
}

int pimpc_shift(pimpc_t h, int steps)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    if (steps < 0 || steps >= h->N) return fail(h, PIMPC_EINVAL, "shift: steps must be in [0, N)");
    if (steps == 0) return PIMPC_OK;
    const int n = launch_shift(h, steps);
    if (n < 0) return PIMPC_ECUDA;
    h->info.total_launches += n;
    return PIMPC_OK;
}

int pimpc_sync(pimpc_t h)
{
    int rc = check_handle(h);
    if (rc) return rc;
    DeviceGuard guard(h);
    return deferred_error(h);
}

int pimpc_get_info(pimpc_t h, pimpc_info *info)
{
    if (!h || !info) return fail(h, PIMPC_EINVAL, "null argument");
    DeviceGuard guard(h);
    if (h->ev_pending && !h->poisoned) {
        PIMPC_CUDA_TRY(h, cudaEventSynchronize(h->ev[2]));
        float a = 0.f, b = 0.f;
        PIMPC_CUDA_TRY(h, cudaEventElapsedTime(&a, h->ev[0], h->ev[1]));
        PIMPC_CUDA_TRY(h, cudaEventElapsedTime(&b, h->ev[1], h->ev[2]));
        h->info.setup_ms = h->ev_setup ? a : 0.0;
        h->info.iter_ms = b;
        h->ev_pending = false;
    }
    h->info.device_bytes = h->device_bytes;
    h->info.sm_count = h->sm_count;
    *info = h->info;
    return PIMPC_OK;
}

const char *pimpc_last_error(pimpc_t h)
{
    if (h) return h->errmsg.c_str();
    return g_last_error.c_str();
}

} // extern "C"
