// Host-side dispatch of the trace / epilogue kernels for one sample type (instantiated in trace_f32.cu, trace_f64.cu).
#pragma once
#include "trace_kernels.cuh"

namespace qsl {

template <typename S, bool DEV, bool STRETCHED, bool INTERP>
static cudaError_t launch_trace_variant(const TraceArgs &A, bool refill, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    if (!refill) {
        const long long blocks = (n_items + threads - 1) / threads;
        count_launch();
        trace_kernel<S, DEV, STRETCHED, INTERP, false><<<(unsigned)blocks, threads, 0, s>>>(A);
    } else {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<S, DEV, STRETCHED, INTERP, true>, threads, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) per_sm = 1;
        long long blocks = (long long)sm_count() * per_sm;          // persistent: every CTA resident, grid = SMs x occupancy
        const long long need = (n_items + threads - 1) / threads;
        if (blocks > need) blocks = need;
        count_launch();
        trace_kernel<S, DEV, STRETCHED, INTERP, true><<<(unsigned)blocks, threads, 0, s>>>(A);
    }
    return cudaGetLastError();
}

template <typename S, bool STRETCHED, bool INTERP>
static cudaError_t launch_epilogue_variant(const EpilogueArgs &E, cudaStream_t s)
{
    const int threads = 128;
    const long long blocks = (E.T.n + threads - 1) / threads;
    count_launch();
    epilogue_kernel<S, STRETCHED, INTERP><<<(unsigned)blocks, threads, 0, s>>>(E);
    return cudaGetLastError();
}

// Higher-order interpolation (ORDER 2 / 3; paper mode NORMALIZE_FIRST only): always the persistent work-queue launch.
template <typename S, bool DEV, bool STRETCHED, int ORDER>
static cudaError_t launch_trace_ho_variant(const TraceArgs &A, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<S, DEV, STRETCHED, false, true, ORDER>, threads, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)sm_count() * per_sm;
    const long long need = (n_items + threads - 1) / threads;
    if (blocks > need) blocks = need;
    count_launch();
    trace_kernel<S, DEV, STRETCHED, false, true, ORDER><<<(unsigned)blocks, threads, 0, s>>>(A);
    return cudaGetLastError();
}

template <typename S, int ORDER>
static cudaError_t launch_trace_ho(const TraceArgs &A, bool dev, cudaStream_t s)
{
    const bool st = A.fv.stretched != 0;
    if (dev) return st ? launch_trace_ho_variant<S, true, true, ORDER>(A, s) : launch_trace_ho_variant<S, true, false, ORDER>(A, s);
    return st ? launch_trace_ho_variant<S, false, true, ORDER>(A, s) : launch_trace_ho_variant<S, false, false, ORDER>(A, s);
}

template <typename S, int ORDER>
static cudaError_t launch_epilogue_ho(const EpilogueArgs &E, cudaStream_t s)
{
    const int threads = 128;
    const long long blocks = (E.T.n + threads - 1) / threads;
    count_launch();
    if (E.T.fv.stretched) epilogue_kernel<S, true, false, ORDER><<<(unsigned)blocks, threads, 0, s>>>(E);
    else epilogue_kernel<S, false, false, ORDER><<<(unsigned)blocks, threads, 0, s>>>(E);
    return cudaGetLastError();
}

// Spherical geometry (uniform axes, paper mode, trilinear): always the persistent work-queue launch.
template <typename S, bool DEV>
static cudaError_t launch_trace_sph_variant(const TraceArgs &A, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_kernel<S, DEV, false, false, true, 1, true>, threads, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)sm_count() * per_sm;
    const long long need = (n_items + threads - 1) / threads;
    if (blocks > need) blocks = need;
    count_launch();
    trace_kernel<S, DEV, false, false, true, 1, true><<<(unsigned)blocks, threads, 0, s>>>(A);
    return cudaGetLastError();
}

template <typename S>
cudaError_t launch_trace(const TraceArgs &A, bool dev, bool refill, cudaStream_t s)
{
    if (A.fv.spherical) return dev ? launch_trace_sph_variant<S, true>(A, s) : launch_trace_sph_variant<S, false>(A, s);
    if (A.fv.order == 2) return launch_trace_ho<S, 2>(A, dev, s);
    if (A.fv.order == 3) return launch_trace_ho<S, 3>(A, dev, s);
    const bool st = A.fv.stretched != 0, in = A.fv.interp_mode == QSL_INTERP_FIRST;
#define QSL_DISPATCH(D, ST, IN) \
    if (dev == D && st == ST && in == IN) return launch_trace_variant<S, D, ST, IN>(A, refill, s);
    QSL_DISPATCH(false, false, false) QSL_DISPATCH(false, false, true) QSL_DISPATCH(false, true, false) QSL_DISPATCH(false, true, true)
    QSL_DISPATCH(true, false, false) QSL_DISPATCH(true, false, true) QSL_DISPATCH(true, true, false) QSL_DISPATCH(true, true, true)
#undef QSL_DISPATCH
    return cudaErrorInvalidValue;
}

template <typename S>
cudaError_t launch_epilogue(const EpilogueArgs &E, cudaStream_t s)
{
    if (E.T.fv.spherical) {
        const int threads = 128;
        const long long blocks = (E.T.n + threads - 1) / threads;
        count_launch();
        epilogue_kernel<S, false, false, 1, true><<<(unsigned)blocks, threads, 0, s>>>(E);
        return cudaGetLastError();
    }
    if (E.T.fv.order == 2) return launch_epilogue_ho<S, 2>(E, s);
    if (E.T.fv.order == 3) return launch_epilogue_ho<S, 3>(E, s);
    const bool st = E.T.fv.stretched != 0, in = E.T.fv.interp_mode == QSL_INTERP_FIRST;
    if (!st && !in) return launch_epilogue_variant<S, false, false>(E, s);
    if (!st && in) return launch_epilogue_variant<S, false, true>(E, s);
    if (st && !in) return launch_epilogue_variant<S, true, false>(E, s);
    return launch_epilogue_variant<S, true, true>(E, s);
}

}  // namespace qsl
