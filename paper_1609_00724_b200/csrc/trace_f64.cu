// Trace / epilogue kernels for fp64 field samples (double4 gathers), fp64 arithmetic.
#include "trace_launch.cuh"
namespace qsl {
cudaError_t launch_trace_f64(const TraceArgs &A, bool dev, bool refill, cudaStream_t s) { return launch_trace<double>(A, dev, refill, s); }
cudaError_t launch_epilogue_f64(const EpilogueArgs &E, cudaStream_t s) { return launch_epilogue<double>(E, s); }
}  // namespace qsl
