// Measured on-chip peaks of the device the library runs on (SURVEY 8(d) "which roofline binds": "measure both with
// an FMA-chain microbenchmark"): FP32 FMA (scalar FFMA and packed FFMA2), FP64 FMA and shared-memory load bandwidth, plus
// what an in-order warp pays per dependent instruction (FFMA2, DADD, SHFL, LDS latencies) and per broadcast 16-byte load.
// bench.py reports the RESIDENT engine (C4) against these numbers, not against a nominal lanes x clock product.
// Each kernel keeps every SM sub-partition busy with independent dependency chains (8 accumulators per thread,
// 16 warps per SM), so the number is the pipe's sustained issue rate at the clocks of a tens-of-milliseconds run.
#include <algorithm>

#include "pimpc_internal.h"

namespace {

// MODE 0: fma.rn.f32, 1: fma.rn.f32x2 (two FMAs per instruction), 2: fma.rn.f64
template <int MODE>
__global__ void __launch_bounds__(512) k_probe_fma(float *out, const int reps, const float seed)
{
    if constexpr (MODE == 2) {
        double a[8], m = 1.0 + 1e-9 * seed, c = 1e-9 * seed;
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = seed + i + threadIdx.x;
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = fma(a[i], m, c);
        }
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += a[i];
        if (s == 12345.678) out[0] = (float)s;
    } else if constexpr (MODE == 1) {
        float2 a[8];
        const float2 m = make_float2(1.0f + 1e-7f * seed, 1.0f - 1e-7f * seed), c = make_float2(1e-7f * seed, -1e-7f * seed);
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = make_float2(seed + i + threadIdx.x, seed - i);
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = __ffma2_rn(a[i], m, c);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
        if (s == 12345.678f) out[0] = s;
    } else {
        float a[8], m = 1.0f + 1e-7f * seed, c = 1e-7f * seed;
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = seed + i + threadIdx.x;
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = fmaf(a[i], m, c);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += a[i];
        if (s == 12345.678f) out[0] = s;
    }
}

// Conflict-free 16-byte shared-memory loads: every lane its own 16 bytes, 512 bytes per warp instruction = 4 wavefronts.
__global__ void __launch_bounds__(512) k_probe_smem(float *out, const int reps)
{
    __shared__ float4 buf[2048];                               // 32 KB
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int idx = threadIdx.x;
    for (int r = 0; r < reps; ++r) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const float4 v = buf[(idx + u * 128) & 2047];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        idx = (idx + 17) & 2047;
    }
    if (acc.x + acc.y + acc.z + acc.w == 12345.678f) out[0] = acc.x;
}

// Dependent-chain latencies, one warp on one SM: cycles[m] = clock64 around 32 x reps dependent instructions.
// MODE 0: fma.rn.f32x2, 1: add.f64, 2: shfl.sync.bfly, 3: ld.shared pointer chase
template <int MODE>
__global__ void __launch_bounds__(32) k_probe_lat(long long *cycles, float *out, const int reps, const float seed)
{
    __shared__ int chase[1024];
    for (int i = threadIdx.x; i < 1024; i += 32) chase[i] = (i * 7 + 3) & 1023;
    __syncwarp();
    float2 a2 = make_float2(seed + threadIdx.x, seed);
    const float2 m2 = make_float2(1.0f + 1e-7f * seed, 1.0f - 1e-7f * seed), c2 = make_float2(1e-7f * seed, -1e-7f * seed);
    double d = seed + threadIdx.x;
    const double dc = 1e-9 * seed;
    float f = seed + threadIdx.x;
    int idx = threadIdx.x;
    const long long t0 = clock64();
#pragma unroll 1
    for (int r = 0; r < reps; ++r) {
#pragma unroll
        for (int u = 0; u < 32; ++u) {
            if constexpr (MODE == 0) a2 = __ffma2_rn(a2, m2, c2);
            else if constexpr (MODE == 1) d = d + dc;
            else if constexpr (MODE == 2) f = __shfl_xor_sync(0xffffffffu, f, 1);
            else idx = chase[idx];
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[MODE] = t1 - t0;
    out[1 + threadIdx.x] = a2.x + a2.y + (float)d + f + (float)idx;
}

// Broadcast 16-byte loads: groups of 8 lanes read the same 16 bytes (4 distinct addresses per warp), the pattern of the
// RESIDENT engine's vector loads; the address moves every iteration, so nothing can be hoisted out of the loop.
__global__ void __launch_bounds__(512) k_probe_smem_bcast(float *out, const int reps)
{
    __shared__ float4 buf[2048];                               // 32 KB
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int idx = ((threadIdx.x & 31) >> 3) * 5 + (threadIdx.x >> 5) * 64;
    for (int r = 0; r < reps; ++r) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const float4 v = buf[(idx + u * 128) & 2047];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        idx = (idx + 17) & 2047;
    }
    if (acc.x + acc.y + acc.z + acc.w == 12345.678f) out[0] = acc.x;
}

template <typename F>
int time_kernel(cudaStream_t st, F launch, double *ms_best)
{
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return PIMPC_ECUDA;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {                        // first pass warms up the clocks
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return PIMPC_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::min(best, ms);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *ms_best = best;
    return cudaGetLastError() == cudaSuccess ? PIMPC_OK : PIMPC_ECUDA;
}

} // namespace

extern "C" int pimpc_measure_peaks(pimpc_peaks *out, void *stream)
{
    if (!out) return PIMPC_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return PIMPC_ECUDA;
    }
    cudaStream_t st = (cudaStream_t)stream;
    float *sink = nullptr;
    if (cudaMalloc(&sink, 256) != cudaSuccess) { cudaGetLastError(); return PIMPC_ENOMEM; }
    *out = pimpc_peaks{};
    const int grid = sms * 2, block = 512, reps = 4096;       // 2 CTAs x 16 warps per SM
    const double threads = (double)grid * block, fma_per_thread = (double)reps * 64;
    double ms = 0.0;
    int rc = time_kernel(st, [&] { k_probe_fma<0><<<grid, block, 0, st>>>(sink, reps, 1.0f); }, &ms);
    if (!rc) { out->ffma_tflops = 2.0 * threads * fma_per_thread / (ms * 1e-3) / 1e12; }
    if (!rc) rc = time_kernel(st, [&] { k_probe_fma<1><<<grid, block, 0, st>>>(sink, reps, 1.0f); }, &ms);
    if (!rc) { out->ffma2_tflops = 4.0 * threads * fma_per_thread / (ms * 1e-3) / 1e12; }
    if (!rc) rc = time_kernel(st, [&] { k_probe_fma<2><<<grid, block, 0, st>>>(sink, reps / 4, 1.0f); }, &ms);
    if (!rc) { out->dfma_tflops = 2.0 * threads * (fma_per_thread / 4) / (ms * 1e-3) / 1e12; }
    if (!rc) rc = time_kernel(st, [&] { k_probe_smem<<<grid, block, 0, st>>>(sink, reps); }, &ms);
    if (!rc) { out->smem_gbs = threads * (double)reps * 16 * 16 / (ms * 1e-3) / 1e9; }
    out->sm_count = sms;
    // cycles per warp-wide broadcast load: 16 warps per SM (two 16-warp CTAs share an SM), at the clock of the FMA probes
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    if (!rc) rc = time_kernel(st, [&] { k_probe_smem_bcast<<<grid, block, 0, st>>>(sink, reps); }, &ms);
    if (!rc) out->lds128_bcast_cycles = ms * 1e-3 * (double)khz * 1e3 / ((double)reps * 16 * 32);     // 32 warps per SM issue 16 loads per rep
    // dependent-instruction latencies (one warp)
    long long *cyc = nullptr;
    if (!rc && cudaMalloc(&cyc, 4 * sizeof(long long)) != cudaSuccess) { cudaGetLastError(); rc = PIMPC_ENOMEM; }
    if (!rc) {
        const int lreps = 256;
        k_probe_lat<0><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f); k_probe_lat<0><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f);
        k_probe_lat<1><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f); k_probe_lat<1><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f);
        k_probe_lat<2><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f); k_probe_lat<2><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f);
        k_probe_lat<3><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f); k_probe_lat<3><<<1, 32, 0, st>>>(cyc, sink, lreps, 1.0f);
        long long hc[4] = {0, 0, 0, 0};
        if (cudaMemcpyAsync(hc, cyc, sizeof(hc), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
            cudaGetLastError(); rc = PIMPC_ECUDA;
        } else {
            const double n = 32.0 * lreps;
            out->lat_ffma2_cycles = hc[0] / n; out->lat_dadd_cycles = hc[1] / n; out->lat_shfl_cycles = hc[2] / n; out->lat_lds_cycles = hc[3] / n;
        }
    }
    if (cyc) cudaFree(cyc);
    cudaFree(sink);
    return rc;
}
