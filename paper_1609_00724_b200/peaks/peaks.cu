// Roofline denominators measured on the device (SURVEY.md 8(d) "Which roofline binds"): MEASURED_PEAKS.json carries
// only the HBM copy bandwidth and the bf16 GEMM rate, so the two peaks that bound the tracer are measured here:
//   qsl_peak_fma     issue rate of the plain FP pipe (DFMA or FFMA), independent chains, no memory traffic
//   qsl_peak_gather  rate of divergent 16-byte / 32-byte sample gathers (the tracer's load shape) over a footprint
//                    that is L1-, L2- or HBM-resident
// Both time themselves with CUDA events (warm-up + best of `reps`) and synchronise.  They are bench utilities, not
// part of the method: a library of their own (libqsl_peaks.so, include/qsl_peaks.h) that shares nothing with libqsl.
#include <cuda_runtime.h>

#include "qsl_peaks.h"

namespace qsl_peaks {

static int sm_count()
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1)
        return 1;
    return n;
}

#define PEAK_CUDA(call)                                   \
    do {                                                  \
        if ((call) != cudaSuccess) return QSL_PEAKS_ECUDA; \
    } while (0)

template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(int iters, T seed, T *out)
{
    // 8 independent chains per thread: enough ILP to cover the pipe latency at any occupancy
    T a0 = seed + (T)threadIdx.x, a1 = a0 + (T)1, a2 = a0 + (T)2, a3 = a0 + (T)3, a4 = a0 + (T)4, a5 = a0 + (T)5,
      a6 = a0 + (T)6, a7 = a0 + (T)7;
    const T m = (T)0.999999, c = (T)1e-6;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const T r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == (T)123.456) out[0] = r;     // never true; keeps the chains alive
}

__device__ __forceinline__ float4 peak_load(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ double4 peak_load(const double4 *p)
{
    double4 r;                                                      // one 256-bit LDG, as in the tracer
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// Each thread walks `iters` pseudo-random sample indices (LCG, different per thread) and sums what it loads.
template <typename S4>
__global__ void __launch_bounds__(256) gather_peak_kernel(const S4 *__restrict__ buf, unsigned long long mask,
                                                          int iters, double *out)
{
    unsigned long long s = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) * 0x9E3779B97F4A7C15ull + 12345ull;
    double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
#pragma unroll 1
    for (int i = 0; i < iters; i += 4) {
        unsigned long long i0, i1, i2, i3;
        s = s * 6364136223846793005ull + 1442695040888963407ull; i0 = (s >> 20) & mask;
        s = s * 6364136223846793005ull + 1442695040888963407ull; i1 = (s >> 20) & mask;
        s = s * 6364136223846793005ull + 1442695040888963407ull; i2 = (s >> 20) & mask;
        s = s * 6364136223846793005ull + 1442695040888963407ull; i3 = (s >> 20) & mask;
        const S4 v0 = peak_load(buf + i0), v1 = peak_load(buf + i1), v2 = peak_load(buf + i2), v3 = peak_load(buf + i3);
        acc0 += (double)v0.x + (double)v0.w; acc1 += (double)v1.y + (double)v1.w;
        acc2 += (double)v2.z + (double)v2.w; acc3 += (double)v3.x + (double)v3.w;
    }
    const double r = (acc0 + acc1) + (acc2 + acc3);
    if (r == 123.456) out[0] = r;
}

template <typename F>
static int time_best(int reps, double *best_ms, cudaStream_t s, F launch)
{
    cudaEvent_t e0, e1;
    PEAK_CUDA(cudaEventCreate(&e0));
    PEAK_CUDA(cudaEventCreate(&e1));
    double best = 1e300;
    cudaError_t e = cudaSuccess;
    for (int r = 0; r < reps + 2 && e == cudaSuccess; ++r) {       // 2 warm-up launches
        cudaEventRecord(e0, s);
        launch();
        cudaEventRecord(e1, s);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (r >= 2 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return QSL_PEAKS_ECUDA;
    *best_ms = best;
    return 0;
}

}  // namespace qsl_peaks

using namespace qsl_peaks;

extern "C" int qsl_peak_fma(int fp64, int reps, double *fma_per_s, void *stream)
{
    if (!fma_per_s || reps < 1) return QSL_PEAKS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    void *out = nullptr;
    if (cudaMalloc(&out, 16) != cudaSuccess) return QSL_PEAKS_ENOMEM;
    int rc = 0;
    const int iters = fp64 ? 2048 : 4096, threads = 256, blocks = sm_count() * 8;
    double ms = 0.0;
    rc = time_best(reps, &ms, s, [&] {
        if (fp64) fma_peak_kernel<double><<<blocks, threads, 0, s>>>(iters, 1.0, (double *)out);
        else fma_peak_kernel<float><<<blocks, threads, 0, s>>>(iters, 1.0f, (float *)out);
    });
    cudaFree(out);
    if (rc != 0) return rc;
    *fma_per_s = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
    return 0;
}

extern "C" int qsl_peak_gather(int bytes_per_sample, long long footprint_bytes, int reps, double *samples_per_s,
                               void *stream)
{
    if (!samples_per_s || reps < 1 || (bytes_per_sample != 16 && bytes_per_sample != 32) ||
        footprint_bytes < 4096) return QSL_PEAKS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    void *buf = nullptr, *out = nullptr;
    if (cudaMalloc(&buf, (size_t)footprint_bytes) != cudaSuccess) { cudaGetLastError(); return QSL_PEAKS_ENOMEM; }
    if (cudaMalloc(&out, 16) != cudaSuccess) { cudaGetLastError(); cudaFree(buf); return QSL_PEAKS_ENOMEM; }
    int rc = 0;
    cudaMemsetAsync(buf, 0, (size_t)footprint_bytes, s);
    unsigned long long n_samples = 1;                               // largest power of two that fits the footprint
    while (n_samples * 2 * (unsigned)bytes_per_sample <= (unsigned long long)footprint_bytes) n_samples *= 2;
    const unsigned long long mask = n_samples - 1;
    const int iters = 1024, threads = 256, blocks = sm_count() * 8;
    double ms = 0.0;
    rc = time_best(reps, &ms, s, [&] {
        if (bytes_per_sample == 16) gather_peak_kernel<float4><<<blocks, threads, 0, s>>>((const float4 *)buf, mask, iters, (double *)out);
        else gather_peak_kernel<double4><<<blocks, threads, 0, s>>>((const double4 *)buf, mask, iters, (double *)out);
    });
    cudaFree(buf); cudaFree(out);
    if (rc != 0) return rc;
    *samples_per_s = (double)blocks * threads * (double)iters / (ms * 1e-3);
    return 0;
}
