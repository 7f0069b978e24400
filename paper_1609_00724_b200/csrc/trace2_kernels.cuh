// V2 trace kernel (the default): the same integration as trace_kernels.cuh (same state machine, same landing rule, same
// per-direction records and epilogue), but the field is read from the per-cell polynomial table built by
// qsl_field_create (field.cu, cell_table_kernel) and the current cell's 24 coefficients stay in registers for as long as
// the line stays inside that cell.  At h = 0.25 cell a line enters a new cell every ~2.5 steps = ~10 stage evaluations,
// so the gathers drop from 8 x 32 B per stage to 192 B per ~10 stages, and value + analytic gradient of the three
// components cost 33 FMAs instead of 75 FP64 instructions: the kernel moves from the L1 gather limit (profiles/r1a) to
// the FP64 pipe.
//
//  PAPER.md:95 (eq. 3), :101-107 (eq. 4)  trilinear kernels f_v;  :123, :137  gradient taken analytically on the kernels:
//  inside one cell the interpolant is the polynomial sum_m a_m dx^m0 dy^m1 dz^m2, whose x-derivative is the coefficient
//  of dx collected in Horner form (E below), etc.
#pragma once
#include "trace_kernels.cuh"

namespace qsl {

__device__ __forceinline__ double4 load_cell4(const double4 *p)
{
    double4 r;   // one 256-bit LDG (sm_100)
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// 0 <= a < b for b > 0, as one unsigned 64-bit integer compare of the bit patterns (runs on the integer pipe, not on
// the FP64 pipe).  False for negative a (sign bit set), -0.0 and NaN.
__device__ __forceinline__ bool in_range_bits(double a, double b)
{
    return (unsigned long long)__double_as_longlong(a) < (unsigned long long)__double_as_longlong(b);
}

template <bool DEV, bool STRETCHED, bool INTERP>
struct LineState2 {
    static constexpr int NV = DEV ? 9 : 3;
    // cached cell: monomial coefficients a[8 c + m], origin, edges (edges only needed on stretched grids)
    double a[24];
    double x0[3];
    double hc[3];
    // line state (as LineState)
    double y[NV];
    double L, lam, hp, bound, hfull;
    uint32_t nsteps;
    int phase, axis, face, face_pending;
    double sgn;
    long long slot;

    __device__ __forceinline__ void relocate(const TraceArgs &A, const double x[3])
    {
        int i, j, k; double t, ih;
        locate<STRETCHED>(A, 0, A.fv.nx, x[0], i, t, ih, hc[0]);
        locate<STRETCHED>(A, 1, A.fv.ny, x[1], j, t, ih, hc[1]);
        locate<STRETCHED>(A, 2, A.fv.nz, x[2], k, t, ih, hc[2]);
        if (STRETCHED) {
            x0[0] = __ldg(A.fv.axis[0] + i); x0[1] = __ldg(A.fv.axis[1] + j); x0[2] = __ldg(A.fv.axis[2] + k);
        } else {
            x0[0] = fma((double)i, A.fv.h[0], A.fv.lo[0]);
            x0[1] = fma((double)j, A.fv.h[1], A.fv.lo[1]);
            x0[2] = fma((double)k, A.fv.h[2], A.fv.lo[2]);
        }
        const double4 *__restrict__ p = (const double4 *)A.fv.cells + (((size_t)k * (A.fv.ny - 1) + j) * (A.fv.nx - 1) + i) * 6;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const double4 v = load_cell4(p + q);
            a[4 * q] = v.x; a[4 * q + 1] = v.y; a[4 * q + 2] = v.z; a[4 * q + 3] = v.w;
        }
    }

    // Evaluate(x) -> b[3], J[9] (J[3 c + d] = d b_c / d x_d); O1 of DESIGN.md.
    template <bool WITH_J>
    __device__ __forceinline__ void evaluate(const TraceArgs &A, const double x[3], double b[3], double J[9])
    {
        double dx = x[0] - x0[0], dy = x[1] - x0[1], dz = x[2] - x0[2];
        const double hx = STRETCHED ? hc[0] : A.fv.h[0], hy = STRETCHED ? hc[1] : A.fv.h[1], hz = STRETCHED ? hc[2] : A.fv.h[2];
        if (!(in_range_bits(dx, hx) && in_range_bits(dy, hy) && in_range_bits(dz, hz))) {
            relocate(A, x);
            dx = x[0] - x0[0]; dy = x[1] - x0[1]; dz = x[2] - x0[2];
        }
        double v[3], g[9];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double *q = a + 8 * c;
            const double P = fma(q[7], dz, q[3]);      // coefficient of dx dy
            const double Q = fma(q[5], dz, q[1]);      // coefficient of dx
            const double R = fma(q[6], dz, q[2]);      // coefficient of dy
            const double S = fma(q[4], dz, q[0]);
            const double E = fma(P, dy, Q);            // d/dx
            const double F = fma(R, dy, S);
            v[c] = fma(E, dx, F);
            if (WITH_J) {
                g[3 * c] = E;
                g[3 * c + 1] = fma(P, dx, R);
                g[3 * c + 2] = fma(fma(q[7], dy, q[5]), dx, fma(q[6], dy, q[4]));
            }
        }
        if (!INTERP) {
#pragma unroll
            for (int c = 0; c < 3; ++c) b[c] = v[c];
            if (WITH_J) {
#pragma unroll
                for (int q = 0; q < 9; ++q) J[q] = g[q];
            }
        } else {
            // reading A2: interpolate B, then normalise: b = B/|B|, J = (G - u (u^T G))/|B|
            const double nn = sqrt(fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0])));
            if (nn < 1e-300) {
#pragma unroll
                for (int c = 0; c < 3; ++c) b[c] = 0.0;
                if (WITH_J) {
#pragma unroll
                    for (int q = 0; q < 9; ++q) J[q] = 0.0;
                }
            } else {
                const double inv = 1.0 / nn;
                const double u0 = v[0] * inv, u1 = v[1] * inv, u2 = v[2] * inv;
                b[0] = u0; b[1] = u1; b[2] = u2;
                if (WITH_J) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        const double uG = fma(u2, g[6 + d], fma(u1, g[3 + d], u0 * g[d]));
                        J[d] = (g[d] - u0 * uG) * inv;
                        J[3 + d] = (g[3 + d] - u1 * uG) * inv;
                        J[6 + d] = (g[6 + d] - u2 * uG) * inv;
                    }
                }
            }
        }
    }

    __device__ bool init(const TraceArgs &A, long long q)
    {
        long long pos; int dir;
        if (A.interleave) { pos = q >> 1; dir = (int)(q & 1); } else { dir = q >= A.n ? 1 : 0; pos = q - (long long)dir * A.n; }
        slot = (long long)dir * A.n + pos;
        sgn = dir ? -1.0 : 1.0;
        const uint32_t si = A.perm[pos];
        double x[3] = { A.seeds[3 * (size_t)si], A.seeds[3 * (size_t)si + 1], A.seeds[3 * (size_t)si + 2] };
        L = 0.0; lam = 0.0; nsteps = 0; phase = 0; axis = 0; face = 255; face_pending = 255; hp = 0.0; bound = 0.0; hfull = 0.0;
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = c < 3 ? x[c] : 0.0;
        if (!inside_box(A, x)) { finish(A, REC_SEED_OUTSIDE); return false; }
        x0[0] = x0[1] = x0[2] = __longlong_as_double(0x7ff8000000000000ll);    // no cell cached yet
        double b[3], J[9];
        evaluate<false>(A, x, b, J);
        const double nb = norm3(b);
        if (!(nb >= A.null_eps)) { finish(A, REC_NULL_AT_SEED); return false; }
        if (DEV) {
            // O2 (PAPER.md:160 eq. 9, :163): a^, b^ orthonormal with B^(x0); reading A7: e = axis of smallest |u_d|
            const double inv = 1.0 / nb;
            const double u[3] = { b[0] * inv, b[1] * inv, b[2] * inv };
            int e = 0;
            if (fabs(u[1]) < fabs(u[e])) e = 1;
            if (fabs(u[2]) < fabs(u[e == 1 ? 1 : 0])) e = 2;
            const double ue = e == 0 ? u[0] : (e == 1 ? u[1] : u[2]);
            double av[3] = { -u[0] * ue, -u[1] * ue, -u[2] * ue };
            if (e == 0) av[0] += 1.0; else if (e == 1) av[1] += 1.0; else av[2] += 1.0;
            const double ia = 1.0 / norm3(av);
            av[0] *= ia; av[1] *= ia; av[2] *= ia;
            y[3 % NV] = av[0]; y[4 % NV] = av[1]; y[5 % NV] = av[2];
            y[6 % NV] = u[1] * av[2] - u[2] * av[1];
            y[7 % NV] = u[2] * av[0] - u[0] * av[2];
            y[8 % NV] = u[0] * av[1] - u[1] * av[0];
        }
        return true;
    }

    __device__ void finish(const TraceArgs &A, uint32_t flags)
    {
        double out[REC_DOUBLES];
#pragma unroll
        for (int c = 0; c < 9; ++c) out[c] = c < NV ? y[c % NV] : 0.0;
        out[9] = L;
        const uint32_t w1 = (uint32_t)face | flags;
        out[10] = __hiloint2double((int)w1, (int)nsteps);
        out[11] = lam;
        double2 *r2 = reinterpret_cast<double2 *>(A.rec + (size_t)slot * REC_DOUBLES);
#pragma unroll
        for (int c = 0; c < REC_DOUBLES / 2; ++c) r2[c] = make_double2(out[2 * c], out[2 * c + 1]);
    }

    // One attempt: a trial step (phase 0), a landing iteration (1..3) or the final landing step (4).  True when the
    // line has ended.  The sign of the direction is folded into the step (hs = sgn h), so the stage derivative is
    // (b, J d1, J d2, |b|) without the three + six multiplications by sgn; the rounding is unchanged (sgn = +-1).
    __device__ bool advance(const TraceArgs &A)
    {
        double acc[NV], accL = 0.0, ys[NV];
        double hs = phase == 0 ? 0.0 : hp, h = 0.0;
        const int last = A.method == QSL_EULER ? 0 : 3;
#pragma unroll
        for (int c = 0; c < NV; ++c) { acc[c] = 0.0; ys[c] = y[c]; }
        double Ln = L;
#pragma unroll 1
        for (int st = 0;; ++st) {
            double b[3], J[9];
            evaluate<DEV>(A, ys, b, J);
            const double bn = norm3(b);
            if (st == 0 && phase == 0) {
                // O4: stall / caps are tested on k1 before the step; h from the cell containing x
                if (!(bn >= A.null_eps)) { finish(A, REC_STALL); return true; }
                if ((long long)nsteps >= A.max_steps || lam >= A.max_length) { finish(A, REC_CAP); return true; }
                h = STRETCHED ? A.step_frac * fmin(hc[0], fmin(hc[1], hc[2])) : A.h_uniform;
                if (lam + h > A.max_length) h = A.max_length - lam;
                hs = h;
            }
            if (st > last) {
                // landing, "5th stage": b at the trial end -> one Newton update of hp (clamped to [0, h_full])
                const double bd = axis == 0 ? b[0] : (axis == 1 ? b[1] : b[2]);
                const double xd = axis == 0 ? ys[0] : (axis == 1 ? ys[1] : ys[2]);
                const double gg = sgn * bd, r = xd - bound;
                if (gg != 0.0) {
                    const double hn = hp - r / gg;
                    if (hn == hn) hp = fmin(fmax(hn, 0.0), hfull);
                }
                ++phase;
                return false;
            }
            // stage derivative k = (b, J d1, J d2, |b|)  (PAPER.md:79 eq. 1, :119 eq. 5; reading A3 for L)
            double k[NV];
#pragma unroll
            for (int c = 0; c < 3; ++c) k[c] = b[c];
            if (DEV) {
#pragma unroll
                for (int v = 0; v < 2; ++v)
#pragma unroll
                    for (int c = 0; c < 3; ++c)
                        k[(3 + 3 * v + c) % NV] = fma(J[c * 3 + 2], ys[(3 + 3 * v + 2) % NV],
                                                      fma(J[c * 3 + 1], ys[(3 + 3 * v + 1) % NV], J[c * 3] * ys[(3 + 3 * v) % NV]));
            }
            const double w = (st == 0 || st == last) ? 1.0 : 2.0;
#pragma unroll
            for (int c = 0; c < NV; ++c) acc[c] = fma(w, k[c], acc[c]);
            accL = fma(w, bn, accL);
            if (st == last) {
                const double fL = A.method == QSL_EULER ? hs : hs * (1.0 / 6.0), f = sgn * fL;
                // the trial end goes into ys (it is the "5th stage" point of the landing iterations)
#pragma unroll
                for (int c = 0; c < NV; ++c) ys[c] = fma(f, acc[c], y[c]);
                Ln = fma(fL, accL, L);
                if (phase >= 1 && phase <= 3) continue;
                break;
            }
            const double ch = sgn * (st == 2 ? hs : 0.5 * hs);
#pragma unroll
            for (int c = 0; c < NV; ++c) ys[c] = fma(ch, k[c], y[c]);
        }
        if (phase == 0) {
            if (inside_box(A, ys)) {
#pragma unroll
                for (int c = 0; c < NV; ++c) y[c] = ys[c];
                L = Ln; lam += h; ++nsteps;
                return false;
            }
            // first face crossed by the chord: smallest fraction, tie -> lowest axis (reading A4)
            double phi = INFINITY; int ax = -1, fc = 255; double bd = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (ys[d] < A.box_lo[d]) {
                    const double f = (A.box_lo[d] - y[d]) / (ys[d] - y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d; bd = A.box_lo[d]; }
                } else if (ys[d] > A.box_hi[d]) {
                    const double f = (A.box_hi[d] - y[d]) / (ys[d] - y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d + 1; bd = A.box_hi[d]; }
                }
            }
            if (ax < 0) { finish(A, REC_STALL); return true; }   // non-finite trial point
            axis = ax; face_pending = fc; bound = bd; hp = phi * h; hfull = h; phase = 1;
            return false;
        }
        // phase 4: final landing step
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = ys[c];
        if (axis == 0) y[0] = bound; else if (axis == 1) y[1] = bound; else y[2] = bound;
        L = Ln; lam += hp; ++nsteps; face = face_pending;
        finish(A, 0);
        return true;
    }
};

template <bool DEV, bool STRETCHED, bool INTERP, bool REFILL>
__global__ void __launch_bounds__(128) trace2_kernel(const TraceArgs A)
{
    LineState2<DEV, STRETCHED, INTERP> ls;
    const long long n_items = 2 * A.n;
    unsigned long long my_steps = 0;
    if (!REFILL) {
        const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (q < n_items && ls.init(A, q)) {
            while (!ls.advance(A)) {}
        }
        if (q < n_items) my_steps = ls.nsteps;
    } else {
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
                else have = ls.init(A, q);
            }
            if (__all_sync(0xffffffffu, drained && !have)) break;
            if (have) {
                if (ls.advance(A)) { my_steps += ls.nsteps; have = false; }
            }
        }
    }
    if (A.total_steps) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_steps += __shfl_xor_sync(0xffffffffu, my_steps, o);
        if ((threadIdx.x & 31) == 0 && my_steps) atomicAdd(A.total_steps, my_steps);
    }
}

}  // namespace qsl
