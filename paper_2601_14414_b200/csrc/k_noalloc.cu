// Allocation-free entry point pimpc_rprim2_noalloc (include/pimpc.h): r_prim2 = rho ||F p + G q - h||^2 of an iterate the
// caller holds (consensus constraints of Problem (11)), for callers that cannot call
// cudaMalloc.  A variant of k_rprim / k_result (k_setup.cu: the result kernels of pimpc_get) that reads the caller's dense
// arrays instead of a handle's records and keeps its per-CTA partial sums in a file-scope __device__ array instead of an
// engine buffer.  Same residuals, same accumulation type (double), same order (thread-strided, fixed tree per CTA, CTAs
// in ascending order), so the result equals pimpc_result.r_prim2 bit for bit whenever the chunk count is the same.
//
// The array's name is a host-side stand-in in host code, not a device address: the address every launch passes to the
// kernels comes from cudaGetSymbolAddress, resolved once per device with that device current.
// Every call on a device shares the array; overlapping calls race (see the header).  Nothing in it must start at zero.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "pimpc.h"

namespace {

__device__ __align__(256) double g_noalloc_part[PIMPC_NOALLOC_MAX_PARTS];   // 256 KiB per GPU, until the process exits

constexpr int NA_MAXDEV = 64;
double *g_part_addr[NA_MAXDEV];          // device address of g_noalloc_part on device d (nullptr = not resolved yet)
std::mutex g_part_mutex;
thread_local char g_na_error[256];

int na_fail(int code, const char *msg, const char *detail = nullptr)
{
    if (detail) snprintf(g_na_error, sizeof(g_na_error), "pimpc_rprim2_noalloc: %s: %s", msg, detail);
    else snprintf(g_na_error, sizeof(g_na_error), "pimpc_rprim2_noalloc: %s", msg);
    return code;
}

// Partial sums of the squared consensus residuals of one chunk of (stage, component) pairs of instance blockIdx.y:
//   xbar_{k+1} - z_{k+1},   Bbar_k Delta u_k - v_k,   z_{k+1} - Abar_k xbar_k - v_k - ebar_k   [, Delta u_k - d_k]
template <typename T>
__global__ void __launch_bounds__(128)
k_rprim_noalloc(const int nx, const int nu, const int N, const T *__restrict__ A, const T *__restrict__ B, const T *__restrict__ e,
                const T *__restrict__ x0, const T *__restrict__ uprev, const T *__restrict__ X, const T *__restrict__ DU,
                const T *__restrict__ Z, const T *__restrict__ V, const T *__restrict__ D, double *__restrict__ part, const int chunk)
{
    __shared__ double red[128];
    const int b = blockIdx.y, nb = nx + nu;
    double acc = 0.0;
    const int i0 = blockIdx.x * chunk, i1 = min(N * nb, i0 + chunk);
    for (int idx = i0 + threadIdx.x; idx < i1; idx += blockDim.x) {
        const int k = idx / nb, i = idx - k * nb;
        const size_t sk = (size_t)b * N + k;
        const double z = (double)Z[sk * nb + i], v = (double)V[sk * nb + i], xk1 = (double)X[sk * nb + i];
        const T *du = DU + sk * nu;
        double bdu, axk;                                       // (Bbar_k Delta u_k)_i, (Abar_k xbar_k + ebar_k)_i
        if (i < nx) {
            const T *Ak = A + sk * nx * nx + (size_t)i * nx, *Bk = B + sk * nx * nu + (size_t)i * nu;
            bdu = 0.0; axk = e ? (double)e[sk * nx + i] : 0.0;
            for (int j = 0; j < nu; ++j) bdu += (double)Bk[j] * (double)du[j];
            for (int j = 0; j < nx; ++j) axk += (double)Ak[j] * (double)(k == 0 ? x0[(size_t)b * nx + j] : X[(sk - 1) * nb + j]);
            for (int j = 0; j < nu; ++j)
                axk += (double)Bk[j] * (double)(k == 0 ? (uprev ? uprev[(size_t)b * nu + j] : (T)0) : X[(sk - 1) * nb + nx + j]);
        } else {
            bdu = (double)du[i - nx];
            axk = (double)(k == 0 ? (uprev ? uprev[(size_t)b * nu + (i - nx)] : (T)0) : X[(sk - 1) * nb + i]);
        }
        const double r1 = xk1 - z, r2 = bdu - v, r3 = z - axk - v;
        acc += r1 * r1 + r2 * r2 + r3 * r3;
        if (D && i >= nx) { const double r4 = (double)du[i - nx] - (double)D[sk * nu + (i - nx)]; acc += r4 * r4; }
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[(size_t)b * gridDim.x + blockIdx.x] = red[0];
}

// r_prim2[b] = rho * (partials of instance b in ascending order)
__global__ void k_rprim_noalloc_sum(const double *__restrict__ part, const int nch, const int batch, const double rho,
                                    double *__restrict__ out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double s = 0.0;
    for (int q = 0; q < nch; ++q) s += part[(size_t)b * nch + q];
    out[b] = rho * s;
}

// Device address of the scratch array on the current device: cudaGetSymbolAddress once per device, with it current.
int scratch_address(double **out)
{
    int dev = -1;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) { cudaGetLastError(); return na_fail(PIMPC_ECUDA, "cudaGetDevice failed", cudaGetErrorString(ce)); }
    if (dev < 0 || dev >= NA_MAXDEV) return na_fail(PIMPC_EINVAL, "device ordinal beyond the 64 this entry point keeps addresses for");
    std::lock_guard<std::mutex> lock(g_part_mutex);
    if (!g_part_addr[dev]) {
        double *ptr = nullptr;
        ce = cudaGetSymbolAddress((void **)&ptr, g_noalloc_part);
        if (ce != cudaSuccess || !ptr) {
            cudaGetLastError();
            return na_fail(PIMPC_ECUDA, "cudaGetSymbolAddress(scratch) failed", cudaGetErrorString(ce));
        }
        g_part_addr[dev] = ptr;
    }
    *out = g_part_addr[dev];
    return PIMPC_OK;
}

template <typename T>
void launch_noalloc(int nx, int nu, int N, int batch, const void *A, const void *B, const void *e, const void *x0, const void *u_prev,
                    const void *X, const void *DU, const void *Z, const void *V, const void *D, double rho, double *part, int nch,
                    int chunk, double *out, cudaStream_t st)
{
    k_rprim_noalloc<T><<<dim3(nch, batch), 128, 0, st>>>(nx, nu, N, (const T *)A, (const T *)B, (const T *)e, (const T *)x0,
                                                         (const T *)u_prev, (const T *)X, (const T *)DU, (const T *)Z, (const T *)V,
                                                         (const T *)D, part, chunk);
    k_rprim_noalloc_sum<<<(batch + 127) / 128, 128, 0, st>>>(part, nch, batch, rho, out);
}

} // namespace

extern "C" {

int pimpc_rprim2_noalloc(int dtype, int nx, int nu, int N, int batch, const void *A, const void *B, const void *e,
                         const void *x0, const void *u_prev, const void *X, const void *DU, const void *Z, const void *V,
                         const void *D, double rho, double *r_prim2, void *stream)
{
    if (dtype != PIMPC_F64 && dtype != PIMPC_F32) return na_fail(PIMPC_EINVAL, "dtype must be PIMPC_F64 or PIMPC_F32");
    if (nx < 1 || nu < 1 || N < 1 || batch < 1) return na_fail(PIMPC_EINVAL, "nx, nu, N and batch must be >= 1");
    if (!A || !B || !x0 || !X || !DU || !Z || !V || !r_prim2)
        return na_fail(PIMPC_EINVAL, "A, B, x0, X, DU, Z, V and r_prim2 must not be NULL");
    if (batch > PIMPC_NOALLOC_MAX_PARTS) {
        char d[96];
        snprintf(d, sizeof(d), "batch = %d, limit PIMPC_NOALLOC_MAX_PARTS = %d", batch, PIMPC_NOALLOC_MAX_PARTS);
        return na_fail(PIMPC_EINVAL, "batch exceeds the static scratch (one partial sum per instance at least)", d);
    }
    if (batch > 65535) return na_fail(PIMPC_EINVAL, "batch exceeds gridDim.y");
    const long long rows = (long long)N * (nx + nu);
    if (rows > 0x7fffffffLL) return na_fail(PIMPC_EINVAL, "N (nx + nu) exceeds 2^31 - 1");
    int nch = (int)(rows / 2048 < 1 ? 1 : (rows / 2048 > 64 ? 64 : rows / 2048));      // pimpc_get's chunking ...
    if (nch > PIMPC_NOALLOC_MAX_PARTS / batch) nch = PIMPC_NOALLOC_MAX_PARTS / batch;   // ... while the scratch lasts
    const int chunk = (int)((rows + nch - 1) / nch);
    double *part = nullptr;
    const int rc = scratch_address(&part);
    if (rc != PIMPC_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == PIMPC_F64) launch_noalloc<double>(nx, nu, N, batch, A, B, e, x0, u_prev, X, DU, Z, V, D, rho, part, nch, chunk, r_prim2, st);
    else launch_noalloc<float>(nx, nu, N, batch, A, B, e, x0, u_prev, X, DU, Z, V, D, rho, part, nch, chunk, r_prim2, st);
    const cudaError_t ce = cudaGetLastError();
    if (ce != cudaSuccess) return na_fail(PIMPC_ECUDA, "kernel launch failed", cudaGetErrorString(ce));
    return PIMPC_OK;
}

const char *pimpc_noalloc_last_error(void) { return g_na_error; }

} // extern "C"
