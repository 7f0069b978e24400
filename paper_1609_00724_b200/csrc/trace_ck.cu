// Host side of the adaptive Cash-Karp trace kernel (QSL_CK45): launch on the fp64 cell table.
#include "trace_ck_kernels.cuh"

namespace qsl {

template <bool DEV, bool STRETCHED, bool INTERP, bool SPH = false>
static int launch_trace_ck_variant(TraceArgs &A, double tol, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    long long blocks = (n_items + threads - 1) / threads;
    if (refill) {
        int per_sm = 0;
        QSL_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_ck_kernel<DEV, STRETCHED, INTERP, true, SPH>, threads, 0));
        if (per_sm < 1) per_sm = 1;
        const long long resident = (long long)sm_count() * per_sm;   // persistent: grid = SMs x resident CTAs
        if (blocks > resident) blocks = resident;
    }
    void *basis = nullptr;
    int rc = QSL_OK;
    if (DEV) rc = scratch_alloc(&basis, sizeof(double) * 6 * (size_t)A.n, s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        if (DEV) {
            count_launch();
            seed_basis_kernel<STRETCHED, INTERP><<<(unsigned)((A.n + 127) / 128), 128, 0, s>>>(A, (double *)basis);
            A.basis = (const double *)basis;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev0) e = cudaEventRecord(ev0, s);
        if (e == cudaSuccess) {
            count_launch();
            if (refill) trace_ck_kernel<DEV, STRETCHED, INTERP, true, SPH><<<(unsigned)blocks, threads, 0, s>>>(A, tol);
            else trace_ck_kernel<DEV, STRETCHED, INTERP, false, SPH><<<(unsigned)blocks, threads, 0, s>>>(A, tol);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) {
            // the landings (reading A4) of all lines at once; part of the trace time
            count_launch();
            landing_ck_kernel<DEV, STRETCHED, INTERP, SPH><<<(unsigned)((n_items + 127) / 128), 128, 0, s>>>(A);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev1) e = cudaEventRecord(ev1, s);
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(basis, s);
    return rc;
}

int launch_trace_ck(TraceArgs &A, double tol, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s)
{
    const bool st = A.fv.stretched != 0, in = A.fv.interp_mode == QSL_INTERP_FIRST;
    if (A.fv.spherical)   // uniform axes, paper mode (qsl_field_create guarantees it)
        return dev ? launch_trace_ck_variant<true, false, false, true>(A, tol, refill, ev0, ev1, s)
                   : launch_trace_ck_variant<false, false, false, true>(A, tol, refill, ev0, ev1, s);
#define QSL_DISPATCH(D, ST, IN) \
    if (dev == D && st == ST && in == IN) return launch_trace_ck_variant<D, ST, IN>(A, tol, refill, ev0, ev1, s);
    QSL_DISPATCH(false, false, false) QSL_DISPATCH(false, false, true) QSL_DISPATCH(false, true, false) QSL_DISPATCH(false, true, true)
    QSL_DISPATCH(true, false, false) QSL_DISPATCH(true, false, true) QSL_DISPATCH(true, true, false) QSL_DISPATCH(true, true, true)
#undef QSL_DISPATCH
    return QSL_EINVAL;
}

}  // namespace qsl
