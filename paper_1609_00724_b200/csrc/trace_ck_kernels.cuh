// Adaptive Cash-Karp 5(4) trace kernel (QSL_CK45).  PAPER.md:141: "an adaptive Runge-Kutta
// Cash-Karp method (Cash & Karp 1990)"; tolerance 1e-2, used "for testing the convergence properties" of
// the fixed-step scheme.  Reading A16 of DESIGN.md fixes the controller: h = step_frac * min_d h_c,d * 2^j with the
// integer j in [-20, +2] as per-line state; after a trial step e = max_d |x5_d - x4_d| / (tol * min_d h_c,d); e > 1
// (and j > -20) rejects and halves; an accepted step with e < 1/64 doubles the next one.  Only the position is
// controlled, so x, L and the step counts do not depend on the trace mode.
//
// The field evaluation, the cached per-cell polynomial, the records and the landing rule (reading A4) are those of
// the cell-table kernel (LineState2); an attempt is six evaluations; as there, the landings of all lines run in their
// own kernel (landing_ck_kernel) on the state the trace kernel recorded.  This is the convergence-check integrator, not the throughput path: the five stage
// derivatives of the 9-component state are held per thread and the kernel runs at two CTAs per SM.
#pragma once
#include "trace2_kernels.cuh"

namespace qsl {

// SPH: spherical geometry (reading A19) exactly as in the fixed-step kernel: coordinate rates = orthonormal components x
// metric factors; the step unit and the error unit hmin are the physical cell edges at the start of the step.
template <bool DEV, bool STRETCHED, bool INTERP, bool SPH = false>
struct LineStateCK : LineState2<DEV, STRETCHED, INTERP, SPH> {
    using Base = LineState2<DEV, STRETCHED, INTERP, SPH>;
    static constexpr int NV = Base::NV;
    int j;                     // controller state: h = h0 2^j

    // unsigned derivative (b, J d1, J d2) and |b| at the state ys; the direction sign is folded into the step
    __device__ __forceinline__ void eval(const TraceArgs &A, const double *ys, double *k, double &bn)
    {
        double d[3], b[3];
        this->enter_cell(A, ys, d);
        this->stage(d, ys, b, k);
        bn = SPH ? this->to_rates(ys, b, k) : norm3_fast(b);
#pragma unroll
        for (int c = 0; c < 3; ++c) k[c] = b[c];
    }

    // Step unit hmin (smallest cell edge at the line's point; physical edges in spherical geometry) and the step of the
    // controller state j, capped by the length left (reading A16)
    __device__ __forceinline__ double step_ck(const TraceArgs &A, double &hmin) const
    {
        hmin = STRETCHED ? fmin(this->hc[0], fmin(this->hc[1], this->hc[2])) : fmin(A.fv.h[0], fmin(A.fv.h[1], A.fv.h[2]));
        if (SPH) hmin = fmin(this->y[2] * this->cth * A.fv.h[0], fmin(this->y[2] * A.fv.h[1], A.fv.h[2]));
        double h = (A.step_frac * hmin) * __hiloint2double((1023 + j) << 20, 0);      // exact scaling by 2^j
        if (this->lam + h > A.max_length) h = A.max_length - this->lam;
        return h;
    }

    // One Cash-Karp step of size hs from y given k1 and n1 = |b| at y: 5th-order end ys, length Ln, and the largest
    // component emax of the position error estimate (5th - 4th order).  Five more evaluations.
    __device__ __forceinline__ void ck_step(const TraceArgs &A, double hs, const double *k1, double n1, double *ys, double &Ln,
                                            double &emax)
    {
        // Cash & Karp (1990): coupling coefficients, 5th-order weights, and (5th - 4th)-order weight differences
        constexpr double a21 = 1.0 / 5.0;
        constexpr double a31 = 3.0 / 40.0, a32 = 9.0 / 40.0;
        constexpr double a41 = 3.0 / 10.0, a42 = -9.0 / 10.0, a43 = 6.0 / 5.0;
        constexpr double a51 = -11.0 / 54.0, a52 = 5.0 / 2.0, a53 = -70.0 / 27.0, a54 = 35.0 / 27.0;
        constexpr double a61 = 1631.0 / 55296.0, a62 = 175.0 / 512.0, a63 = 575.0 / 13824.0, a64 = 44275.0 / 110592.0,
                         a65 = 253.0 / 4096.0;
        constexpr double b1 = 37.0 / 378.0, b3 = 250.0 / 621.0, b4 = 125.0 / 594.0, b6 = 512.0 / 1771.0;
        constexpr double e1 = b1 - 2825.0 / 27648.0, e3 = b3 - 18575.0 / 48384.0, e4 = b4 - 13525.0 / 55296.0,
                         e5 = -277.0 / 14336.0, e6 = b6 - 1.0 / 4.0;
        double k2[NV], k3[NV], k4[NV], k5[NV], k6[NV];
        double n2, n3, n4, n5, n6;
        const double sh = this->back ? -hs : hs;
#define QSL_CK_STAGE(EXPR, KOUT, NOUT)                                                   \
        {                                                                                \
            _Pragma("unroll") for (int c = 0; c < NV; ++c) ys[c] = fma(sh, (EXPR), this->y[c]); \
            eval(A, ys, KOUT, NOUT);                                                     \
        }
        QSL_CK_STAGE(a21 * k1[c], k2, n2)
        QSL_CK_STAGE(fma(a32, k2[c], a31 * k1[c]), k3, n3)
        QSL_CK_STAGE(fma(a43, k3[c], fma(a42, k2[c], a41 * k1[c])), k4, n4)
        QSL_CK_STAGE(fma(a54, k4[c], fma(a53, k3[c], fma(a52, k2[c], a51 * k1[c]))), k5, n5)
        QSL_CK_STAGE(fma(a65, k5[c], fma(a64, k4[c], fma(a63, k3[c], fma(a62, k2[c], a61 * k1[c])))), k6, n6)
#undef QSL_CK_STAGE
#pragma unroll
        for (int c = 0; c < NV; ++c) ys[c] = fma(sh, fma(b6, k6[c], fma(b4, k4[c], fma(b3, k3[c], b1 * k1[c]))), this->y[c]);
        Ln = fma(hs, fma(b6, n6, fma(b4, n4, fma(b3, n3, b1 * n1))), this->L);
        emax = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double e = hs * fma(e6, k6[c], fma(e5, k5[c], fma(e4, k4[c], fma(e3, k3[c], e1 * k1[c]))));
            emax = fmax(emax, fabs(e));
        }
    }

    // One attempt of the trace kernel: a trial step of the controller's size; rejected (halve, retry), accepted and
    // committed, or - accepted but ending outside the trace box - recorded as it stands with REC_LANDING and the
    // controller state in bits 16..23 of the flag word, for landing_ck_kernel.  Returns true when the line left the kernel.
    __device__ bool advance_ck(const TraceArgs &A, double tol)
    {
        double k1[NV], ys[NV], n1, hmin, Ln, emax;
        eval(A, this->y, k1, n1);
        if (!(n1 >= A.null_eps)) { this->finish(A, 255, this->nsteps == 0 ? REC_NULL_AT_SEED : REC_STALL); return true; }
        if ((long long)this->nsteps >= A.max_steps || this->lam >= A.max_length) { this->finish(A, 255, REC_CAP); return true; }
        const double h = step_ck(A, hmin);
        ck_step(A, h, k1, n1, ys, Ln, emax);
        const double en = emax / (tol * hmin);
        if (en > 1.0 && j > -20) { --j; return false; }                 // reject: halve, retry from y
        if (inside_box(A, ys)) {
            if (SPH) this->move_anchor(ys[1] - this->y[1]);
#pragma unroll
            for (int c = 0; c < NV; ++c) this->y[c] = ys[c];
            this->L = Ln; this->lam += h; ++this->nsteps;
            if (en < 1.0 / 64.0 && j < 2) ++j;
            return false;
        }
        this->finish(A, 255, REC_LANDING | ((uint32_t)(j + 32) << 16));
        return true;
    }

    // The landing of one line (reading A4) from the recorded state: the accepted trial step again, the chord, then
    // step(hp), Newton, step(hp), Newton, step(hp), Newton, step(hp) -> snap, every step a Cash-Karp step, k1 once.
    __device__ unsigned land_ck(const TraceArgs &A)
    {
        double k1[NV], ys[NV], n1, hmin, Ln, emax;
        eval(A, this->y, k1, n1);
        const double h = step_ck(A, hmin);
        ck_step(A, h, k1, n1, ys, Ln, emax);
        // first face crossed by the chord: smallest fraction, tie -> lowest axis (reading A4)
        double phi = INFINITY; int ax = -1, fc = 255; double bound = 0.0;
#pragma unroll
        for (int dd = 0; dd < 3; ++dd) {
            if (ys[dd] < A.box_lo[dd]) {
                const double f = (A.box_lo[dd] - this->y[dd]) / (ys[dd] - this->y[dd]);
                if (f < phi) { phi = f; ax = dd; fc = 2 * dd; bound = A.box_lo[dd]; }
            } else if (ys[dd] > A.box_hi[dd]) {
                const double f = (A.box_hi[dd] - this->y[dd]) / (ys[dd] - this->y[dd]);
                if (f < phi) { phi = f; ax = dd; fc = 2 * dd + 1; bound = A.box_hi[dd]; }
            }
        }
        if (ax < 0) { this->finish(A, 255, REC_STALL); return 0; }   // non-finite trial point
        double hp = phi * h;
        for (int it = 0; it < 4; ++it) {
            ck_step(A, hp, k1, n1, ys, Ln, emax);
            if (it == 3) break;
            // one Newton update of the landing step from the field at the trial end, clamped to [0, h]
            double kt[NV], nt, p[NV];
#pragma unroll
            for (int c = 0; c < NV; ++c) p[c] = c < 3 ? ys[c] : this->y[c];
            eval(A, p, kt, nt);
            const double bd = ax == 0 ? kt[0] : (ax == 1 ? kt[1] : kt[2]);
            const double xd = ax == 0 ? ys[0] : (ax == 1 ? ys[1] : ys[2]);
            const double gg = this->back ? -bd : bd, r = xd - bound;
            if (gg != 0.0) {
                const double hn = hp - r / gg;
                if (hn == hn) hp = fmin(fmax(hn, 0.0), h);
            }
        }
#pragma unroll
        for (int c = 0; c < NV; ++c) this->y[c] = ys[c];
        if (ax == 0) this->y[0] = bound; else if (ax == 1) this->y[1] = bound; else this->y[2] = bound;
        this->L = Ln; this->lam += hp; ++this->nsteps;
        this->finish(A, fc, 0);
        return 1;
    }
};

template <bool DEV, bool STRETCHED, bool INTERP, bool REFILL, bool SPH = false>
__global__ void __launch_bounds__(128, 2) trace_ck_kernel(const TraceArgs A, const double tol)
{
    LineStateCK<DEV, STRETCHED, INTERP, SPH> ls;
    const long long n_items = 2 * A.n;
    unsigned long long my_steps = 0;
    if (!REFILL) {
        const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (q < n_items) {
            ls.j = 0;
            if (ls.init(A, q)) { while (!ls.advance_ck(A, tol)) {} }
            my_steps = ls.nsteps;
        }
    } else {
        staged_queue<DEV, 128, QSL_T2_CHUNK>(
            A, [&](const double *x, const double *bs, uint32_t sl) { ls.j = 0; return ls.start(A, x, bs, sl); },
            [&]() { if (!ls.advance_ck(A, tol)) return false; my_steps += ls.nsteps; return true; });
    }
    if (A.total_steps) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_steps += __shfl_xor_sync(0xffffffffu, my_steps, o);
        if ((threadIdx.x & 31) == 0 && my_steps) atomicAdd(A.total_steps, my_steps);
    }
}

// The landings of all lines of a launch (reading A4), one thread per per-direction record flagged REC_LANDING (see
// landing_kernel); the controller state of the accepted trial step that left the box comes back from the flag word.
template <bool DEV, bool STRETCHED, bool INTERP, bool SPH = false>
__global__ void __launch_bounds__(128) landing_ck_kernel(const TraceArgs A)
{
    const long long sl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned added = 0;
    if (sl < 2 * A.n) {
        const double2 *__restrict__ r2 = reinterpret_cast<const double2 *>(A.rec + (size_t)sl * REC_DOUBLES);
        const double2 w5 = r2[5];
        const uint32_t fl = (uint32_t)__double2hiint(w5.x);
        if (fl & REC_LANDING) {
            LineStateCK<DEV, STRETCHED, INTERP, SPH> ls;
            constexpr int NV = LineStateCK<DEV, STRETCHED, INTERP, SPH>::NV;
            double v[10];
#pragma unroll
            for (int c = 0; c < 5; ++c) { const double2 t = r2[c]; v[2 * c] = t.x; v[2 * c + 1] = t.y; }
#pragma unroll
            for (int c = 0; c < NV; ++c) ls.y[c] = v[c];
            ls.L = v[9]; ls.lam = w5.y; ls.nsteps = (uint32_t)__double2loint(w5.x);
            ls.slot = (uint32_t)sl; ls.back = sl >= A.n; ls.phase = 0;
            ls.j = (int)((fl >> 16) & 255u) - 32;
            if (SPH) sincos(ls.y[1], &ls.sth, &ls.cth); else { ls.sth = 0.0; ls.cth = 1.0; }
            ls.x0[0] = ls.x0[1] = ls.x0[2] = __longlong_as_double(0x7ff8000000000000ll);
            ls.hc[0] = ls.hc[1] = ls.hc[2] = 0.0;
            added = ls.land_ck(A);
        }
    }
    if (A.total_steps) {
        const unsigned m = __ballot_sync(0xffffffffu, added != 0);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(A.total_steps, (unsigned long long)__popc(m));
    }
}

}  // namespace qsl
