// Host side of the cell-frame trace kernel (trace3_kernels.cuh): trace box in cell coordinates, launch.  T = float is
// QSL_ARITH_F32 on the fp32 coefficient table; T = double runs the same kernel on the fp64 table (uniform grids).
#include <string.h>

#include "trace3_kernels.cuh"

namespace qsl {

template <typename T, typename S, bool DEV, bool INTERP, bool SPH = false>
static int launch_trace3_variant(Trace3Args<T> &A, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s)
{
    const long long n_items = 2 * A.T0.n;
    const int threads = QSL_T3_THREADS;
    long long blocks = (n_items + threads - 1) / threads;
    if (refill) {
        int per_sm = 0;
        QSL_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace3_kernel<T, DEV, INTERP, true, SPH>, threads, 0));
        if (per_sm < 1) per_sm = 1;
        const long long resident = (long long)sm_count() * per_sm;   // persistent: grid = SMs x resident CTAs
        if (blocks > resident) blocks = resident;
    }
    void *basis = nullptr;
    int rc = QSL_OK;
    if (DEV) rc = scratch_alloc(&basis, sizeof(double) * 6 * (size_t)A.T0.n, s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        if (DEV) {
            count_launch();
            seed_basis3_kernel<S, INTERP><<<(unsigned)((A.T0.n + 127) / 128), 128, 0, s>>>(A.T0, (double *)basis);
            A.T0.basis = (const double *)basis;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev0) e = cudaEventRecord(ev0, s);
        if (e == cudaSuccess) {
            count_launch();
            if (refill) trace3_kernel<T, DEV, INTERP, true, SPH><<<(unsigned)blocks, threads, 0, s>>>(A);
            else trace3_kernel<T, DEV, INTERP, false, SPH><<<(unsigned)blocks, threads, 0, s>>>(A);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) {
            // the landings (reading A4) of all lines at once; part of the trace time
            count_launch();
            landing3_kernel<T, DEV, INTERP, SPH><<<(unsigned)((n_items + 127) / 128), 128, 0, s>>>(A);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && ev1) e = cudaEventRecord(ev1, s);
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(basis, s);
    return rc;
}

static unsigned bits_of(float v) { unsigned u; memcpy(&u, &v, 4); return u; }
static unsigned bits_of(double v) { unsigned long long u; memcpy(&u, &v, 8); return (unsigned)(u >> 32); }

// G: the arguments qsl_trace prepared (uniform grid).  Adds the cell-frame view: cell edges, step, and the trace box as
// (cell, offset) per face - box_lo[d] = origin(cl[d]) + off_lo[d] with 0 <= off_lo < h, and box_hi[d] = origin(ch[d]) +
// off_hi[d] with 0 < off_hi <= h (a face on a node belongs to the cell below it).
template <typename T, typename S>
static int launch_trace3_t(const TraceArgs &G, const void *cells, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1,
                           cudaStream_t s)
{
    if (!cells || G.fv.stretched) return QSL_EINVAL;
    Trace3Args<T> A;
    A.T0 = G;
    A.cells = (const typename Real3<T>::V4 *)cells;
    const int dims[3] = { G.fv.nx, G.fv.ny, G.fv.nz };
    for (int d = 0; d < 3; ++d) {
        const double h = G.fv.h[d], lo = G.fv.lo[d];
        A.hf[d] = (T)h;
        A.hbits[d] = bits_of(A.hf[d]);
        A.cmax[d] = dims[d] - 2;
        int cl = (int)floor((G.box_lo[d] - lo) / h);
        cl = cl < 0 ? 0 : (cl > dims[d] - 2 ? dims[d] - 2 : cl);
        if (G.box_lo[d] - fma((double)cl, h, lo) < 0.0 && cl > 0) --cl;           // rounding of the quotient
        if (G.box_lo[d] - fma((double)cl, h, lo) >= h && cl < dims[d] - 2) ++cl;
        int ch = (int)ceil((G.box_hi[d] - lo) / h) - 1;
        ch = ch < 0 ? 0 : (ch > dims[d] - 2 ? dims[d] - 2 : ch);
        if (G.box_hi[d] - fma((double)ch, h, lo) <= 0.0 && ch > 0) --ch;
        if (G.box_hi[d] - fma((double)ch, h, lo) > h && ch < dims[d] - 2) ++ch;
        A.cl[d] = cl; A.ch[d] = ch;
        A.cw[d] = ch - cl - 1 > 0 ? (unsigned)(ch - cl - 1) : 0u;
        A.off_lo[d] = (T)(G.box_lo[d] - fma((double)cl, h, lo));
        A.off_hi[d] = (T)(G.box_hi[d] - fma((double)ch, h, lo));
    }
    A.h_step = (T)G.h_uniform;
    A.cell_sy = dims[0] - 1;
    A.cell_sz = (dims[0] - 1) * (dims[1] - 1);
    A.null_eps = (T)G.null_eps;
    A.row_sc = G.fv.row_sc;
    A.step_frac = (T)G.step_frac;
    const bool in = G.fv.interp_mode == QSL_INTERP_FIRST;
    if (G.fv.spherical) {       // fp32 arithmetic only (uniform axes, paper mode: qsl_field_create guarantees both)
        if constexpr (sizeof(T) == 4) {
            if (!G.fv.row_sc || in) return QSL_EINVAL;
            return dev ? launch_trace3_variant<T, S, true, false, true>(A, refill, ev0, ev1, s)
                       : launch_trace3_variant<T, S, false, false, true>(A, refill, ev0, ev1, s);
        } else {
            return QSL_EINVAL;
        }
    }
    if (dev) return in ? launch_trace3_variant<T, S, true, true>(A, refill, ev0, ev1, s) : launch_trace3_variant<T, S, true, false>(A, refill, ev0, ev1, s);
    return in ? launch_trace3_variant<T, S, false, true>(A, refill, ev0, ev1, s) : launch_trace3_variant<T, S, false, false>(A, refill, ev0, ev1, s);
}

// fp32 arithmetic on the fp32 table (fp32 samples)
int launch_trace3(const TraceArgs &G, const void *cells32, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1,
                  cudaStream_t s)
{
    return launch_trace3_t<float, float>(G, cells32, dev, refill, ev0, ev1, s);
}

// fp64 arithmetic on the fp64 table; samples_f32 = storage type of the node samples (seed basis pre-pass)
int launch_trace3_f64(const TraceArgs &G, bool samples_f32, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1,
                      cudaStream_t s)
{
    const long long nc = (long long)(G.fv.nx - 1) * (G.fv.ny - 1) * (G.fv.nz - 1);
    if (nc >= (1ll << 31)) return QSL_ERANGE;
    return samples_f32 ? launch_trace3_t<double, float>(G, G.fv.cells, dev, refill, ev0, ev1, s)
                       : launch_trace3_t<double, double>(G, G.fv.cells, dev, refill, ev0, ev1, s);
}

}  // namespace qsl
