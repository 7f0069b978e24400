// qsl_trace: host entry point.  Orders the seeds, runs the trace kernel over 2n work items
// (one per direction), then the Q/L epilogue, all asynchronously on the caller's stream.
#include <math.h>
#include <string.h>

#include "trace_kernels.cuh"

namespace qsl {
cudaError_t launch_trace_f32(const TraceArgs &A, bool dev, bool refill, cudaStream_t s);
cudaError_t launch_trace_f64(const TraceArgs &A, bool dev, bool refill, cudaStream_t s);
int launch_trace2(TraceArgs &A, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s);
int launch_trace_ck(TraceArgs &A, double tol, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s);
cudaError_t launch_trace_ckg_f32(const TraceArgs &A, double tol, bool dev, cudaStream_t s);
cudaError_t launch_trace_ckg_f64(const TraceArgs &A, double tol, bool dev, cudaStream_t s);
int launch_trace3(const TraceArgs &T, const void *cells32, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s);
int launch_trace3_f64(const TraceArgs &T, bool samples_f32, bool dev, bool refill, cudaEvent_t ev0, cudaEvent_t ev1, cudaStream_t s);
cudaError_t launch_epilogue_f32(const EpilogueArgs &E, cudaStream_t s);
cudaError_t launch_epilogue_f64(const EpilogueArgs &E, cudaStream_t s);
}  // namespace qsl

using namespace qsl;

// Measurement hook: an event pair around every trace-kernel launch (qsl_profile_enable / qsl_profile_trace_kernel_ms).
constexpr int PROF_MAX = 256;
static int g_profile = 0, g_prof_n = 0;
static cudaEvent_t g_ev0[PROF_MAX], g_ev1[PROF_MAX];
static int g_prof_mode[PROF_MAX], g_prof_made = 0;

extern "C" int qsl_profile_enable(int on)
{
    g_profile = on ? 1 : 0;
    g_prof_n = 0;
    return QSL_OK;
}

// Next free event pair (created on first use), or -1 when the pool is full (the launch is then not timed).
static int prof_slot(int mode)
{
    if (!g_profile || g_prof_n >= PROF_MAX) return -1;
    if (g_prof_n >= g_prof_made) {
        if (cudaEventCreate(&g_ev0[g_prof_made]) != cudaSuccess || cudaEventCreate(&g_ev1[g_prof_made]) != cudaSuccess) return -1;
        ++g_prof_made;
    }
    g_prof_mode[g_prof_n] = mode;
    return g_prof_n++;
}

extern "C" int qsl_profile_trace_kernel_ms(double ms[2], long long launches[2])
{
    if (!ms || !launches || g_prof_n == 0) return QSL_EINVAL;
    ms[0] = ms[1] = 0.0; launches[0] = launches[1] = 0;
    for (int i = 0; i < g_prof_n; ++i) {
        QSL_CUDA(cudaEventSynchronize(g_ev1[i]));
        float t = 0.f;
        QSL_CUDA(cudaEventElapsedTime(&t, g_ev0[i], g_ev1[i]));
        ms[g_prof_mode[i]] += (double)t; ++launches[g_prof_mode[i]];
    }
    g_prof_n = 0;
    return QSL_OK;
}

extern "C" int qsl_trace(const qsl_field *f, const qsl_trace_params *p, long long n, const double *seeds,
                         const qsl_trace_out *out, unsigned long long *total_steps, void *stream)
{
    if (!f || !p || !out || n < 0 || (n > 0 && !seeds)) return QSL_EINVAL;
    if (p->method != QSL_RK4 && p->method != QSL_EULER && p->method != QSL_CK45) return QSL_EINVAL;
    // the adaptive stepper runs in fp64 arithmetic, with a positive tolerance
    if (p->method == QSL_CK45 && (p->arith != QSL_ARITH_F64 || !(p->tol > 0.0))) return QSL_EINVAL;
    if (p->mode != QSL_TRACE_L && p->mode != QSL_TRACE_LQ) return QSL_EINVAL;
    if (p->arith != QSL_ARITH_F64 && p->arith != QSL_ARITH_F32) return QSL_EINVAL;
    // fp32 arithmetic (reading A6): needs the fp32 coefficient table (QSL_LAYOUT_CELL_TABLE_F32 / _BOTH), which
    // qsl_field_create only builds for fp32 samples on a uniform grid
    if (p->arith == QSL_ARITH_F32 && !f->d_cells32) return QSL_EINVAL;
    if (!(p->step_frac > 0.0) || p->max_steps < 1 || !(p->max_length > 0.0) || !(p->null_eps >= 0.0)) return QSL_EINVAL;
    for (int d = 0; d < 3; ++d)
        if (!(p->box_hi[d] >= p->box_lo[d])) return QSL_EINVAL;
    if (n >= (1ll << 31)) return QSL_ERANGE;
    cudaStream_t s = (cudaStream_t)stream;
    if (total_steps) QSL_CUDA(cudaMemsetAsync(total_steps, 0, sizeof(unsigned long long), s));
    if (n == 0) return QSL_OK;

    TraceArgs A;
    A.fv = f->view;
    for (int d = 0; d < 3; ++d) {
        A.inv_h[d] = 1.0 / f->view.h[d];
        A.box_lo[d] = p->box_lo[d]; A.box_hi[d] = p->box_hi[d];
        { unsigned long long bits; memcpy(&bits, &f->view.h[d], 8); A.h_hi[d] = (unsigned)(bits >> 32); }
    }
    A.h_uniform = p->step_frac * fmin(f->view.h[0], fmin(f->view.h[1], f->view.h[2]));
    A.step_frac = p->step_frac; A.max_length = p->max_length; A.null_eps = p->null_eps;
    A.max_steps = p->max_steps > 0xffffffffll ? 0xffffffffll : p->max_steps;
    A.method = p->method;
    const bool refill = !(p->flags & QSL_FLAG_NO_REFILL);
    A.interleave = refill ? 1 : 0;
    A.n = n; A.seeds = seeds; A.total_steps = total_steps;
    A.basis = nullptr; A.tie_zero = 0;

    void *perm = nullptr, *rec = nullptr, *queue = nullptr;
    int rc = scratch_alloc(&perm, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&rec, sizeof(double) * REC_DOUBLES * 2 * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&queue, sizeof(unsigned long long), s);
    if (rc == QSL_OK) rc = morton_order(f->view, n, seeds, (uint32_t *)perm, !(p->flags & QSL_FLAG_NO_SORT), s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        A.perm = (const uint32_t *)perm; A.rec = (double *)rec; A.queue = (unsigned long long *)queue;
        e = cudaMemsetAsync(queue, 0, sizeof(unsigned long long), s);
        const bool dev = p->mode == QSL_TRACE_LQ;
        const bool v2 = f->view.cells != nullptr && !(p->flags & QSL_FLAG_KERNEL_V1);
        if (e == cudaSuccess && p->method == QSL_CK45 && v2) {
            const int ps = prof_slot(p->mode);
            rc = launch_trace_ck(A, p->tol, dev, refill, ps >= 0 ? g_ev0[ps] : nullptr, ps >= 0 ? g_ev1[ps] : nullptr, s);
        } else if (e == cudaSuccess && p->method == QSL_CK45) {
            // no per-cell table (nodes-only layout, higher-order interpolation) or QSL_FLAG_KERNEL_V1: the gather kernel
            const int ps = prof_slot(p->mode);
            if (ps >= 0) e = cudaEventRecord(g_ev0[ps], s);
            if (e == cudaSuccess)
                e = f->sample_type == QSL_F32 ? launch_trace_ckg_f32(A, p->tol, dev, s) : launch_trace_ckg_f64(A, p->tol, dev, s);
            if (e == cudaSuccess && ps >= 0) e = cudaEventRecord(g_ev1[ps], s);
        } else if (e == cudaSuccess && p->arith == QSL_ARITH_F32) {
            const int ps = prof_slot(p->mode);
            rc = launch_trace3(A, f->d_cells32, dev, refill, ps >= 0 ? g_ev0[ps] : nullptr, ps >= 0 ? g_ev1[ps] : nullptr, s);
        } else if (e == cudaSuccess && v2 && !f->view.stretched && !f->view.spherical && (p->flags & QSL_FLAG_KERNEL_FRAME)) {
            const int ps = prof_slot(p->mode);
            rc = launch_trace3_f64(A, f->sample_type == QSL_F32, dev, refill, ps >= 0 ? g_ev0[ps] : nullptr, ps >= 0 ? g_ev1[ps] : nullptr, s);
        } else if (e == cudaSuccess && v2) {
            // the cell-table kernel allocates its own scratch and brackets its launch with the profiling events
            const int ps = prof_slot(p->mode);
            rc = launch_trace2(A, dev, refill, ps >= 0 ? g_ev0[ps] : nullptr, ps >= 0 ? g_ev1[ps] : nullptr, s);
        } else if (e == cudaSuccess) {
            const int ps = prof_slot(p->mode);
            if (ps >= 0) e = cudaEventRecord(g_ev0[ps], s);
            if (e == cudaSuccess)
                e = f->sample_type == QSL_F32 ? launch_trace_f32(A, dev, refill, s) : launch_trace_f64(A, dev, refill, s);
            if (e == cudaSuccess && ps >= 0) e = cudaEventRecord(g_ev1[ps], s);
        }
        if (rc != QSL_OK) e = cudaErrorUnknown;
        if (e == cudaSuccess) {
            EpilogueArgs E;
            E.T = A; E.with_dev = dev ? 1 : 0; E.out = *out;
            e = f->sample_type == QSL_F32 ? launch_epilogue_f32(E, s) : launch_epilogue_f64(E, s);
        }
        if (e != cudaSuccess && rc == QSL_OK) rc = record_cuda(e);
    }
    scratch_free(perm, s); scratch_free(rec, s); scratch_free(queue, s);
    return rc;
}
