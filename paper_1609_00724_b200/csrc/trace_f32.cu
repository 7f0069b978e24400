// Trace / epilogue kernels for fp32 field samples (float4 gathers), fp64 arithmetic.
#include "trace_launch.cuh"
namespace qsl {
cudaError_t launch_trace_f32(const TraceArgs &A, bool dev, bool refill, cudaStream_t s) { return launch_trace<float>(A, dev, refill, s); }
cudaError_t launch_epilogue_f32(const EpilogueArgs &E, cudaStream_t s) { return launch_epilogue<float>(E, s); }
}  // namespace qsl
