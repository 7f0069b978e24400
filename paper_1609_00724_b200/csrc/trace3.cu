// Host side of the fp32-arithmetic trace kernel (QSL_ARITH_F32): trace box in cell coordinates, launch.
#include "trace3_kernels.cuh"

namespace qsl {

template <bool DEV, bool INTERP>
static int launch_trace3_variant(Trace3Args &A, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s)
{
    const long long n_items = 2 * A.T.n;
    const int threads = QSL_T3_THREADS;
    long long blocks = (n_items + threads - 1) / threads;
    if (refill) {
        int per_sm = 0;
        QSL_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace3_kernel<DEV, INTERP, true>, threads, 0));
        if (per_sm < 1) per_sm = 1;
        const long long resident = (long long)sm_count() * per_sm;   // persistent: grid = SMs x resident CTAs
        if (blocks > resident) blocks = resident;
    }
    void *basis = nullptr, *stash = nullptr;
    int rc = scratch_alloc(&stash, sizeof(float) * STASH3_FLOATS * (size_t)blocks * threads, s);
    if (rc == QSL_OK && DEV) rc = scratch_alloc(&basis, sizeof(double) * 6 * (size_t)A.T.n, s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        A.stash = (float *)stash;
        if (DEV) {
            count_launch();
            seed_basis3_kernel<INTERP><<<(unsigned)((A.T.n + 127) / 128), 128, 0, s>>>(A.T, (double *)basis);
            A.T.basis = (const double *)basis;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev0) e = cudaEventRecord(ev0, s);
        if (e == cudaSuccess) {
            count_launch();
            if (refill) trace3_kernel<DEV, INTERP, true><<<(unsigned)blocks, threads, 0, s>>>(A);
            else trace3_kernel<DEV, INTERP, false><<<(unsigned)blocks, threads, 0, s>>>(A);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev1) e = cudaEventRecord(ev1, s);
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(basis, s); scratch_free(stash, s);
    return rc;
}

// T: the arguments qsl_trace prepared for the fp64 kernels (uniform grid).  Adds the fp32 view: cell edges, step,
// and the trace box as (cell, offset) per face - box_lo[d] = origin(cl[d]) + off_lo[d] with 0 <= off_lo < h, and
// box_hi[d] = origin(ch[d]) + off_hi[d] with 0 < off_hi <= h (a face on a node belongs to the cell below it).
int launch_trace3(const TraceArgs &T, const void *cells32, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1,
                  cudaStream_t s)
{
    if (!cells32 || T.fv.stretched) return QSL_EINVAL;
    Trace3Args A;
    A.T = T;
    A.cells32 = (const float4 *)cells32;
    const int dims[3] = { T.fv.nx, T.fv.ny, T.fv.nz };
    for (int d = 0; d < 3; ++d) {
        const double h = T.fv.h[d], lo = T.fv.lo[d];
        A.hf[d] = (float)h;
        A.cmax[d] = dims[d] - 2;
        int cl = (int)floor((T.box_lo[d] - lo) / h);
        cl = cl < 0 ? 0 : (cl > dims[d] - 2 ? dims[d] - 2 : cl);
        if (T.box_lo[d] - fma((double)cl, h, lo) < 0.0 && cl > 0) --cl;           // rounding of the quotient
        if (T.box_lo[d] - fma((double)cl, h, lo) >= h && cl < dims[d] - 2) ++cl;
        int ch = (int)ceil((T.box_hi[d] - lo) / h) - 1;
        ch = ch < 0 ? 0 : (ch > dims[d] - 2 ? dims[d] - 2 : ch);
        if (T.box_hi[d] - fma((double)ch, h, lo) <= 0.0 && ch > 0) --ch;
        if (T.box_hi[d] - fma((double)ch, h, lo) > h && ch < dims[d] - 2) ++ch;
        A.cl[d] = cl; A.ch[d] = ch;
        A.cw[d] = ch - cl - 1 > 0 ? (unsigned)(ch - cl - 1) : 0u;
        A.off_lo[d] = (float)(T.box_lo[d] - fma((double)cl, h, lo));
        A.off_hi[d] = (float)(T.box_hi[d] - fma((double)ch, h, lo));
    }
    A.h_step = (float)T.h_uniform;
    A.cell_sy = dims[0] - 1;
    A.cell_sz = (dims[0] - 1) * (dims[1] - 1);
    A.null_eps = (float)T.null_eps;
    A.stash = nullptr;
    const bool in = T.fv.interp_mode == QSL_INTERP_FIRST;
    if (dev) return in ? launch_trace3_variant<true, true>(A, refill, ev0, ev1, s) : launch_trace3_variant<true, false>(A, refill, ev0, ev1, s);
    return in ? launch_trace3_variant<false, true>(A, refill, ev0, ev1, s) : launch_trace3_variant<false, false>(A, refill, ev0, ev1, s);
}

}  // namespace qsl
