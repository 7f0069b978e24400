// V2 trace kernels (per-cell polynomial table, fp64 arithmetic; independent of the sample storage type).
#include "trace2_kernels.cuh"

namespace qsl {

template <bool DEV, bool STRETCHED, bool INTERP>
static cudaError_t launch_trace2_variant(const TraceArgs &A, bool refill, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    if (!refill) {
        const long long blocks = (n_items + threads - 1) / threads;
        count_launch();
        trace2_kernel<DEV, STRETCHED, INTERP, false><<<(unsigned)blocks, threads, 0, s>>>(A);
    } else {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace2_kernel<DEV, STRETCHED, INTERP, true>, threads, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) per_sm = 1;
        long long blocks = (long long)sm_count() * per_sm;          // persistent: every CTA resident, grid = SMs x occupancy
        const long long need = (n_items + threads - 1) / threads;
        if (blocks > need) blocks = need;
        count_launch();
        trace2_kernel<DEV, STRETCHED, INTERP, true><<<(unsigned)blocks, threads, 0, s>>>(A);
    }
    return cudaGetLastError();
}

cudaError_t launch_trace2(const TraceArgs &A, bool dev, bool refill, cudaStream_t s)
{
    const bool st = A.fv.stretched != 0, in = A.fv.interp_mode == QSL_INTERP_FIRST;
#define QSL_DISPATCH(D, ST, IN) \
    if (dev == D && st == ST && in == IN) return launch_trace2_variant<D, ST, IN>(A, refill, s);
    QSL_DISPATCH(false, false, false) QSL_DISPATCH(false, false, true) QSL_DISPATCH(false, true, false) QSL_DISPATCH(false, true, true)
    QSL_DISPATCH(true, false, false) QSL_DISPATCH(true, false, true) QSL_DISPATCH(true, true, false) QSL_DISPATCH(true, true, true)
#undef QSL_DISPATCH
    return cudaErrorInvalidValue;
}

}  // namespace qsl
