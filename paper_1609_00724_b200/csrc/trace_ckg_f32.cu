// Cash-Karp in the stencil-gather kernel, fp32 field samples (float4 gathers), fp64 arithmetic.
#include "trace_ckg_kernels.cuh"
namespace qsl {
cudaError_t launch_trace_ckg_f32(const TraceArgs &A, double tol, bool dev, cudaStream_t s) { return launch_trace_ckg<float>(A, tol, dev, s); }
}  // namespace qsl
