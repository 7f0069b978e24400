// Cash-Karp in the stencil-gather kernel, fp64 field samples (double4 gathers).
#include "trace_ckg_kernels.cuh"
namespace qsl {
cudaError_t launch_trace_ckg_f64(const TraceArgs &A, double tol, bool dev, cudaStream_t s) { return launch_trace_ckg<double>(A, tol, dev, s); }
}  // namespace qsl
