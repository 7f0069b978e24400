// Adaptive Cash-Karp 5(4) in the stencil-gather kernel (QSL_CK45 on fields without a per-cell table: QSL_LAYOUT_NODES_ONLY,
// triquadratic / tricubic interpolation, QSL_FLAG_KERNEL_V1; Cartesian uniform / stretched and spherical).
// (Cash & Karp 1990 through Boost's stepper), :143 (tolerance 1e-2, the convergence check of the fixed-step rule); the
// controller is reading A16 of DESIGN.md, the landing reading A4 - as in trace_ck_kernels.cuh, which runs the same scheme on
// the cell table.  This is the convergence-check integrator, not the throughput path: the six stages run through ONE
// evaluate call site (the tricubic evaluation is ~2000 instructions) and the stage derivatives live in a per-thread array
// indexed by the stage number (local memory, L1-resident).
#pragma once
#include "trace_kernels.cuh"

namespace qsl {

// Cash & Karp (1990): coupling coefficients a[s][j], 5th-order weights, and (5th - 4th)-order weight differences
__constant__ double CKG_A[6][5] = {
    { 0.0, 0.0, 0.0, 0.0, 0.0 },
    { 1.0 / 5.0, 0.0, 0.0, 0.0, 0.0 },
    { 3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0 },
    { 3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0.0, 0.0 },
    { -11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0.0 },
    { 1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0 } };
__constant__ double CKG_B5[6] = { 37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0 };
__constant__ double CKG_E[6] = { 37.0 / 378.0 - 2825.0 / 27648.0, 0.0, 250.0 / 621.0 - 18575.0 / 48384.0,
                                 125.0 / 594.0 - 13525.0 / 55296.0, -277.0 / 14336.0, 512.0 / 1771.0 - 1.0 / 4.0 };

template <typename S, bool DEV, bool STRETCHED, bool INTERP, int ORDER = 1, bool SPH = false>
struct LineStateCKG : LineState<S, DEV, STRETCHED, INTERP, ORDER, SPH> {
    using Base = LineState<S, DEV, STRETCHED, INTERP, ORDER, SPH>;
    static constexpr int NV = Base::NV;
    int j;                     // controller state: h = h0 2^j

    // One attempt: six evaluations (seven in the landing phases 1..3: the last one, at the trial end, is the Newton update
    // of the landing step).  Returns true when the line has ended.
    __device__ bool advance_ck(const TraceArgs &A, double tol)
    {
        double kk[6][NV], nn[6];
        double ys[NV], yn[NV];
        double hs = this->phase == 0 ? 0.0 : this->hp, h = 0.0, hunit = 0.0, sh = 0.0;
#pragma unroll
        for (int c = 0; c < NV; ++c) { ys[c] = this->y[c]; yn[c] = this->y[c]; }
#pragma unroll 1
        for (int st = 0; st < 7; ++st) {
            double b[3], J[9], m, hmin, mf[3];
            evaluate<S, STRETCHED, INTERP, DEV, false, ORDER>(A, ys, b, J, m, hmin);
            const double bn = norm3(b);
            metric<SPH>(ys, mf);
            if (st == 6) {
                // landing: field at the trial end -> one Newton update of hp, clamped to [0, h_full] (reading A4)
                const int ax = this->axis;
                const double bd = ax == 0 ? b[0] : (ax == 1 ? b[1] : b[2]);
                const double xd = ax == 0 ? yn[0] : (ax == 1 ? yn[1] : yn[2]);
                const double g = this->sgn * bd * (ax == 0 ? mf[0] : (ax == 1 ? mf[1] : mf[2])), r = xd - this->bound;
                if (g != 0.0) {
                    const double hn = this->hp - r / g;
                    if (hn == hn) this->hp = fmin(fmax(hn, 0.0), this->hfull_);
                }
                ++this->phase;
                return false;
            }
            if (st == 0) {
                if (this->phase == 0) {
                    if (!(bn >= A.null_eps)) { this->finish(A, REC_STALL); return true; }
                    if ((long long)this->nsteps >= A.max_steps || this->lam >= A.max_length) { this->finish(A, REC_CAP); return true; }
                    hunit = STRETCHED ? hmin : fmin(A.fv.h[0], fmin(A.fv.h[1], A.fv.h[2]));
                    if (SPH) hunit = fmin(ys[2] * cos(ys[1]) * A.fv.h[0], fmin(ys[2] * A.fv.h[1], A.fv.h[2]));
                    h = (A.step_frac * hunit) * __hiloint2double((1023 + j) << 20, 0);      // exact scaling by 2^j
                    if (this->lam + h > A.max_length) h = A.max_length - this->lam;
                    hs = h;
                }
                sh = this->sgn * hs;
            }
            // stage derivative (b, J d1, J d2) in coordinate rates; the direction sign rides in sh
#pragma unroll
            for (int c = 0; c < 3; ++c) kk[st][c] = SPH ? b[c] * mf[c] : b[c];
            if (DEV) {
#pragma unroll
                for (int v = 0; v < 2; ++v)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const double jd = fma(J[c * 3 + 2], ys[(3 + 3 * v + 2) % NV],
                                              fma(J[c * 3 + 1], ys[(3 + 3 * v + 1) % NV], J[c * 3] * ys[(3 + 3 * v) % NV]));
                        kk[st][(3 + 3 * v + c) % NV] = SPH ? jd * mf[c] : jd;
                    }
            }
            nn[st] = bn;
            if (st < 5) {
                // next stage point: y + sh sum_j a[st+1][j] k_j
#pragma unroll
                for (int c = 0; c < NV; ++c) {
                    double acc = 0.0;
                    for (int q = 0; q <= st; ++q) acc = fma(CKG_A[st + 1][q], kk[q][c], acc);
                    ys[c] = fma(sh, acc, this->y[c]);
                }
                continue;
            }
            // st == 5: 5th-order result; in the landing phases 1..3 one more evaluation at the trial end follows
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                double acc = 0.0;
                for (int q = 0; q < 6; ++q) acc = fma(CKG_B5[q], kk[q][c], acc);
                yn[c] = fma(sh, acc, this->y[c]);
            }
            if (this->phase >= 1 && this->phase <= 3) {
#pragma unroll
                for (int c = 0; c < NV; ++c) ys[c] = yn[c];
                continue;
            }
            break;
        }
        double accL = 0.0;
        for (int q = 0; q < 6; ++q) accL = fma(CKG_B5[q], nn[q], accL);
        const double Ln = fma(hs, accL, this->L);
        if (this->phase == 0) {
            double emax = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double e = 0.0;
                for (int q = 0; q < 6; ++q) e = fma(CKG_E[q], kk[q][c], e);
                emax = fmax(emax, fabs(hs * e));
            }
            const double en = emax / (tol * hunit);
            if (en > 1.0 && j > -20) { --j; return false; }                 // reject: halve, retry from y
            if (inside_box(A, yn)) {
#pragma unroll
                for (int c = 0; c < NV; ++c) this->y[c] = yn[c];
                this->L = Ln; this->lam += h; ++this->nsteps;
                if (en < 1.0 / 64.0 && j < 2) ++j;
                return false;
            }
            // first face crossed by the chord: smallest fraction, tie -> lowest axis (reading A4)
            double phi = INFINITY; int ax = -1, fc = 255; double bd = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (yn[d] < A.box_lo[d]) {
                    const double f = (A.box_lo[d] - this->y[d]) / (yn[d] - this->y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d; bd = A.box_lo[d]; }
                } else if (yn[d] > A.box_hi[d]) {
                    const double f = (A.box_hi[d] - this->y[d]) / (yn[d] - this->y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d + 1; bd = A.box_hi[d]; }
                }
            }
            if (ax < 0) { this->finish(A, REC_STALL); return true; }   // non-finite trial point
            this->axis = ax; this->face_pending = fc; this->bound = bd; this->hp = phi * h; this->hfull_ = h; this->phase = 1;
            return false;
        }
        // phase 4: final landing step, snapped onto the face
#pragma unroll
        for (int c = 0; c < NV; ++c) this->y[c] = yn[c];
        if (this->axis == 0) this->y[0] = this->bound; else if (this->axis == 1) this->y[1] = this->bound; else this->y[2] = this->bound;
        this->L = Ln; this->lam += this->hp; ++this->nsteps; this->face = this->face_pending;
        this->finish(A, 0);
        return true;
    }
};

// Persistent grid with the work queue of trace_kernel.
template <typename S, bool DEV, bool STRETCHED, bool INTERP, int ORDER = 1, bool SPH = false>
__global__ void __launch_bounds__(128) trace_ckg_kernel(const TraceArgs A, const double tol)
{
    LineStateCKG<S, DEV, STRETCHED, INTERP, ORDER, SPH> ls;
    const long long n_items = 2 * A.n;
    unsigned long long my_steps = 0;
    const unsigned lane = threadIdx.x & 31u;
    bool have = false, drained = false;
    while (true) {
        if (!have && !drained) {
            const unsigned m = __activemask();
            const int leader = __ffs(m) - 1;
            unsigned long long base = 0;
            if ((int)lane == leader) base = atomicAdd(A.queue, (unsigned long long)__popc(m));
            base = __shfl_sync(m, base, leader);
            const long long q = (long long)base + __popc(m & ((1u << lane) - 1u));
            if (q >= n_items) drained = true;
            else { ls.j = 0; have = ls.init(A, q); }
        }
        if (__all_sync(0xffffffffu, drained && !have)) break;
        if (have) {
            if (ls.advance_ck(A, tol)) { my_steps += ls.nsteps; have = false; }
        }
    }
    if (A.total_steps) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_steps += __shfl_xor_sync(0xffffffffu, my_steps, o);
        if ((threadIdx.x & 31) == 0 && my_steps) atomicAdd(A.total_steps, my_steps);
    }
}

template <typename S, bool DEV, bool STRETCHED, bool INTERP, int ORDER, bool SPH>
static cudaError_t launch_trace_ckg_variant(const TraceArgs &A, double tol, cudaStream_t s)
{
    const long long n_items = 2 * A.n;
    const int threads = 128;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_ckg_kernel<S, DEV, STRETCHED, INTERP, ORDER, SPH>, threads, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)sm_count() * per_sm;
    const long long need = (n_items + threads - 1) / threads;
    if (blocks > need) blocks = need;
    count_launch();
    trace_ckg_kernel<S, DEV, STRETCHED, INTERP, ORDER, SPH><<<(unsigned)blocks, threads, 0, s>>>(A, tol);
    return cudaGetLastError();
}

template <typename S, bool DEV>
static cudaError_t launch_trace_ckg_dev(const TraceArgs &A, double tol, cudaStream_t s)
{
    const bool st = A.fv.stretched != 0, in = A.fv.interp_mode == QSL_INTERP_FIRST;
    if (A.fv.spherical) return launch_trace_ckg_variant<S, DEV, false, false, 1, true>(A, tol, s);
    if (A.fv.order == 2) return st ? launch_trace_ckg_variant<S, DEV, true, false, 2, false>(A, tol, s) : launch_trace_ckg_variant<S, DEV, false, false, 2, false>(A, tol, s);
    if (A.fv.order == 3) return st ? launch_trace_ckg_variant<S, DEV, true, false, 3, false>(A, tol, s) : launch_trace_ckg_variant<S, DEV, false, false, 3, false>(A, tol, s);
    if (!st && !in) return launch_trace_ckg_variant<S, DEV, false, false, 1, false>(A, tol, s);
    if (!st && in) return launch_trace_ckg_variant<S, DEV, false, true, 1, false>(A, tol, s);
    if (st && !in) return launch_trace_ckg_variant<S, DEV, true, false, 1, false>(A, tol, s);
    return launch_trace_ckg_variant<S, DEV, true, true, 1, false>(A, tol, s);
}

template <typename S>
cudaError_t launch_trace_ckg(const TraceArgs &A, double tol, bool dev, cudaStream_t s)
{
    return dev ? launch_trace_ckg_dev<S, true>(A, tol, s) : launch_trace_ckg_dev<S, false>(A, tol, s);
}

}  // namespace qsl
