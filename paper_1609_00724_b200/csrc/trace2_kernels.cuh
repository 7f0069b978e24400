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

// Build-time switches of the measured variants (QSL_NVCC_EXTRA="-D..."; the defaults are what profiles/r2d measured best):
//   QSL_T2_HEADTEST  1: in-cell test at the head of an attempt as well (0: the cell of y is the cached one by construction)
//   QSL_T2_CHUNK     work items a warp stages per pop of the global counter
//   QSL_T2_TIE       scheduling fence between the work behind enter_cell() and the next polynomial (LineState2::tie)
//   QSL_T2_DEFER     deviation products behind enter_cell(): 0 never, 1 all stages, 2 stage 1, 3 stages 1 and 3
#ifndef QSL_T2_HEADTEST
#define QSL_T2_HEADTEST 0
#endif
#ifndef QSL_T2_CHUNK
#define QSL_T2_CHUNK 8
#endif
#ifndef QSL_T2_TIE
#define QSL_T2_TIE 1
#endif
#ifndef QSL_T2_DEFER
#define QSL_T2_DEFER 3
#endif

__device__ __forceinline__ double4 load_cell4(const double4 *p)
{
    double4 r;   // one 256-bit LDG (sm_100)
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// |v| for the length integrand (reading A3) and the stall test, branch-free: hardware reciprocal-square-root seed of
// max(|v|^2, 2^-600) and one coupled Newton step (relative error ~1e-13, five orders below the parity gate on L) instead
// of the IEEE sqrt sequence with its fix-up branch.  |v|^2 = 0 gives exactly 0, NaN and overflow propagate (the stall
// test then ends the line); |v| < 2^-300 comes out too small by at most 2^-300, far below any stall threshold.
__device__ __forceinline__ double norm3_fast(const double v[3])
{
    const double n2 = fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0]));
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(fmax(n2, 0x1p-600)));
    const double s = n2 * r, hr = 0.5 * r;
    const double e = fma(-s, hr, 0.5);                 // 0.5 (1 - n2 r^2)
    const double s1 = fma(s, e, s), h1 = fma(hr, e, hr);
    return fma(fma(-s1, s1, n2), h1, s1);
}

// SPH: spherical geometry (reading A19): the coordinate rates are the orthonormal components times the metric factors
// (1/(r cos theta), 1/r, 1) of the evaluation point; |b| for L and the stall test is taken before the scaling.
template <bool DEV, bool STRETCHED, bool INTERP, bool SPH = false>
struct LineState2 {
    static constexpr int NV = DEV ? 9 : 3;
    static constexpr int NJ = DEV ? 9 : 1;
    // cached cell: monomial coefficients a[8 c + m], origin (edges only on stretched grids)
    double a[24];
    double x0[3];
    double hc[3];
    // line state
    double y[NV];
    double L, lam;
    uint32_t nsteps, slot;
    int phase;
    bool back;
    double sth, cth;      // SPH: (sin, cos) of the latitude y[1] of the line's current point (metric_shift)

    // Cell search (reading A8: index clamped, offsets not) and load of the cell's 24 coefficients (six 256-bit loads).
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
        // the cell count is below 2^31 (qsl_field_create): the index in 32-bit arithmetic, one wide multiply for the address
        const unsigned lin = ((unsigned)k * (unsigned)(A.fv.ny - 1) + (unsigned)j) * (unsigned)(A.fv.nx - 1) + (unsigned)i;
        const double4 *__restrict__ p = (const double4 *)A.fv.cells + (size_t)lin * 6;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const double4 v = load_cell4(p + q);
            a[4 * q] = v.x; a[4 * q + 1] = v.y; a[4 * q + 2] = v.z; a[4 * q + 3] = v.w;
        }
    }

    // Makes the cached cell the one containing x and returns the offsets d = x - x_cell.  Called for the NEXT stage
    // point as soon as its position is known, so the table loads of a cell change are in flight while the ~50 FP64
    // instructions of the current stage that no longer need the old coefficients execute.  The "still inside" test is a
    // sufficient one on the high words of the bit patterns, 0 <= d < h: one unsigned integer compare per axis on the
    // integer pipe instead of two DSETP on the FP64 pipe.  It is false for negative d (sign bit), -0.0, NaN and for d
    // within 2^-20 (relative) below h: a false negative only costs a redundant search, which finds the right cell.
    // (A branch-free variant with predicated neighbour loads was slower in round 1; its numbers were not kept.  What was
    // measured on this path since - look-ahead staging in shared memory, register caps - is in profiles/r2b.)
    __device__ __forceinline__ void enter_cell(const TraceArgs &A, const double x[3], double d[3])
    {
        d[0] = x[0] - x0[0]; d[1] = x[1] - x0[1]; d[2] = x[2] - x0[2];
        const unsigned hx = STRETCHED ? (unsigned)__double2hiint(hc[0]) : A.h_hi[0], hy = STRETCHED ? (unsigned)__double2hiint(hc[1]) : A.h_hi[1],
                       hz = STRETCHED ? (unsigned)__double2hiint(hc[2]) : A.h_hi[2];
        if (!((unsigned)__double2hiint(d[0]) < hx && (unsigned)__double2hiint(d[1]) < hy && (unsigned)__double2hiint(d[2]) < hz)) {
            relocate(A, x);
            d[0] = x[0] - x0[0]; d[1] = x[1] - x0[1]; d[2] = x[2] - x0[2];
        }
    }

    // Field evaluation at offsets d inside the cached cell (O1 of DESIGN.md) fused with the deviation products:
    // b[3] and, with DEV, k[3 + 3 v + c] = sum_e J[c][e] dl_v[e] for the two deviation vectors dl = ys[3..8]
    // (eq. 5), component by component so that only one row of J is live at a time.
    __device__ __forceinline__ void stage(const double d[3], const double *ys, double b[3], double *k)
    {
        const double dx = d[0], dy = d[1], dz = d[2];
        if (!INTERP) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double *q = a + 8 * c;
                const double P = fma(q[7], dz, q[3]);      // coefficient of dx dy
                const double Q = fma(q[5], dz, q[1]);      // coefficient of dx
                const double R = fma(q[6], dz, q[2]);      // coefficient of dy
                const double S = fma(q[4], dz, q[0]);
                const double E = fma(P, dy, Q);            // d/dx
                const double F = fma(R, dy, S);
                b[c] = fma(E, dx, F);
                if (DEV) {
                    const double gy = fma(P, dx, R);
                    const double gz = fma(fma(q[7], dy, q[5]), dx, fma(q[6], dy, q[4]));
                    k[(3 + c) % NV] = fma(gz, ys[5 % NV], fma(gy, ys[4 % NV], E * ys[3 % NV]));
                    k[(6 + c) % NV] = fma(gz, ys[8 % NV], fma(gy, ys[7 % NV], E * ys[6 % NV]));
                }
            }
        } else {
            // reading A2: interpolate B, then normalise: b = B/|B|, J = (G - u (u^T G))/|B|
            double v[3], g[9], J[9];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double *q = a + 8 * c;
                const double P = fma(q[7], dz, q[3]), Q = fma(q[5], dz, q[1]), R = fma(q[6], dz, q[2]), S = fma(q[4], dz, q[0]);
                const double E = fma(P, dy, Q), F = fma(R, dy, S);
                v[c] = fma(E, dx, F);
                g[3 * c] = E;
                g[3 * c + 1] = fma(P, dx, R);
                g[3 * c + 2] = fma(fma(q[7], dy, q[5]), dx, fma(q[6], dy, q[4]));
            }
            const double nn = sqrt(fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0])));
            if (nn < 1e-300) {
#pragma unroll
                for (int c = 0; c < 3; ++c) b[c] = 0.0;
#pragma unroll
                for (int q = 0; q < 9; ++q) J[q] = 0.0;
            } else {
                const double inv = 1.0 / nn;
                const double u0 = v[0] * inv, u1 = v[1] * inv, u2 = v[2] * inv;
                b[0] = u0; b[1] = u1; b[2] = u2;
#pragma unroll
                for (int e = 0; e < 3; ++e) {
                    const double uG = fma(u2, g[6 + e], fma(u1, g[3 + e], u0 * g[e]));
                    J[e] = (g[e] - u0 * uG) * inv;
                    J[3 + e] = (g[3 + e] - u1 * uG) * inv;
                    J[6 + e] = (g[6 + e] - u2 * uG) * inv;
                }
            }
            if (DEV) {
#pragma unroll
                for (int w = 0; w < 2; ++w)
#pragma unroll
                    for (int c = 0; c < 3; ++c)
                        k[(3 + 3 * w + c) % NV] = fma(J[c * 3 + 2], ys[(3 + 3 * w + 2) % NV],
                                                      fma(J[c * 3 + 1], ys[(3 + 3 * w + 1) % NV], J[c * 3] * ys[(3 + 3 * w) % NV]));
            }
        }
    }

    // The same evaluation in two parts, for the fixed-step kernel: poly() needs the cached coefficients and gives b and
    // the nine entries J[3 c + e] = d b_c / d x_e; products() needs only J.  Between the two the kernel computes the next
    // stage point and enters its cell, so that the table loads of a cell change overwrite the coefficients while the
    // deviation products, |b| and the RK accumulators of this stage are still to be executed (see trial()).
    __device__ __forceinline__ void poly(const double d[3], double b[3], double *J)
    {
        const double dx = d[0], dy = d[1], dz = d[2];
        double g[9];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double *q = a + 8 * c;
            const double P = fma(q[7], dz, q[3]), Q = fma(q[5], dz, q[1]), R = fma(q[6], dz, q[2]), S = fma(q[4], dz, q[0]);
            const double E = fma(P, dy, Q), F = fma(R, dy, S);
            b[c] = fma(E, dx, F);
            if (DEV) {
                g[3 * c] = E;
                g[3 * c + 1] = fma(P, dx, R);
                g[3 * c + 2] = fma(fma(q[7], dy, q[5]), dx, fma(q[6], dy, q[4]));
            }
        }
        if (!INTERP) {
            if (DEV) {
#pragma unroll
                for (int q = 0; q < 9; ++q) J[q] = g[q];
            }
        } else {
            // reading A2: interpolate B, then normalise: b = B/|B|, J = (G - u (u^T G))/|B|
            const double v[3] = { b[0], b[1], b[2] };
            const double nn = sqrt(fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0])));
            if (nn < 1e-300) {
#pragma unroll
                for (int c = 0; c < 3; ++c) b[c] = 0.0;
                if (DEV) {
#pragma unroll
                    for (int q = 0; q < 9; ++q) J[q] = 0.0;
                }
            } else {
                const double inv = 1.0 / nn;
                const double u0 = v[0] * inv, u1 = v[1] * inv, u2 = v[2] * inv;
                b[0] = u0; b[1] = u1; b[2] = u2;
                if (DEV) {
#pragma unroll
                    for (int e = 0; e < 3; ++e) {
                        const double uG = fma(u2, g[6 + e], fma(u1, g[3 + e], u0 * g[e]));
                        J[e] = (g[e] - u0 * uG) * inv;
                        J[3 + e] = (g[3 + e] - u1 * uG) * inv;
                        J[6 + e] = (g[6 + e] - u2 * uG) * inv;
                    }
                }
            }
        }
    }
    __device__ __forceinline__ void products(const double *J, const double *ys, double *k)
    {
        if (DEV) {
#pragma unroll
            for (int w = 0; w < 2; ++w)
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    k[(3 + 3 * w + c) % NV] = fma(J[(c * 3 + 2) % NJ], ys[(3 + 3 * w + 2) % NV],
                                                  fma(J[(c * 3 + 1) % NJ], ys[(3 + 3 * w + 1) % NV], J[(c * 3) % NJ] * ys[(3 + 3 * w) % NV]));
        }
    }

    // SPH: the line's point moves by dt in latitude: rotate (sth, cth) and pull it back onto the unit circle (one Newton
    // step of 1/sqrt), so that rounding never accumulates in the modulus; the phase error grows like sqrt(steps) ulp.
    __device__ __forceinline__ void move_anchor(double dt)
    {
        double s, c;
        sincos_shift(sth, cth, dt, s, c);
        const double f = fma(-0.5, fma(s, s, fma(c, c, -1.0)), 1.0);
        sth = s * f; cth = c * f;
    }

    // b -> coordinate rates (and |b| of the unscaled vector), k -> coordinate deviation rates, at the point pt
    __device__ __forceinline__ double to_rates(const double *pt, double b[3], double *k)
    {
        const double bn = norm3_fast(b);
        if (SPH) {
            double mf[3];
            metric_shift(pt[2], sth, cth, pt[1] - y[1], mf);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                b[c] *= mf[c];
                if (DEV) { k[(3 + c) % NV] *= mf[c]; k[(6 + c) % NV] *= mf[c]; }
            }
        }
        return bn;
    }

    // Starts a line at the seed x with the orthonormal pair bs (a^, b^; unused without DEV) for record slot sl.
    // Returns false if the item ended at once (seed outside the trace box).
    // FIRST_CELL: the cell of the seed is cached on return (the fixed-step kernel's advance() relies on it)
    template <bool FIRST_CELL = false>
    __device__ __forceinline__ bool start(const TraceArgs &A, const double x[3], const double *bs, uint32_t sl)
    {
        slot = sl;
        back = (long long)sl >= A.n;
        L = 0.0; lam = 0.0; nsteps = 0; phase = 0;
        if (SPH) sincos(x[1], &sth, &cth); else { sth = 0.0; cth = 1.0; }
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = c < 3 ? x[c] : bs[(c - 3) % 6];
        if (!inside_box(A, x)) { finish(A, 255, REC_SEED_OUTSIDE); return false; }
        x0[0] = x0[1] = x0[2] = __longlong_as_double(0x7ff8000000000000ll);    // no cell cached yet
        hc[0] = hc[1] = hc[2] = 0.0;
        if (FIRST_CELL) relocate(A, x);
        if (DEV && SPH) {   // orthonormal pair -> coordinate deviations (eq. 8 inverted)
            double mf[3];
            metric_shift(x[2], sth, cth, 0.0, mf);
#pragma unroll
            for (int c = 0; c < 3; ++c) { y[(3 + c) % NV] *= mf[c]; y[(6 + c) % NV] *= mf[c]; }
        }
        return true;
    }

    // Starts work item q.  Returns false if the item ended at once (seed outside the trace box).  The orthonormal pair
    // a^, b^ of O2 comes from seed_basis_kernel (one thread per seed, all lanes busy) instead of being built here by
    // the one or two lanes of a warp that happen to be refilling; a null at the seed is caught by the first attempt.
    template <bool FIRST_CELL = false>
    __device__ bool init(const TraceArgs &A, long long q)
    {
        long long pos; int dir;
        if (A.interleave) { pos = q >> 1; dir = (int)(q & 1); } else { dir = q >= A.n ? 1 : 0; pos = q - (long long)dir * A.n; }
        const uint32_t si = A.perm[pos];
        const double x[3] = { A.seeds[3 * (size_t)si], A.seeds[3 * (size_t)si + 1], A.seeds[3 * (size_t)si + 2] };
        double bs[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
        if (DEV) {
            const double2 *__restrict__ bp = reinterpret_cast<const double2 *>(A.basis + 6 * (size_t)pos);
            const double2 b0 = bp[0], b1 = bp[1], b2 = bp[2];
            bs[0] = b0.x; bs[1] = b0.y; bs[2] = b1.x; bs[3] = b1.y; bs[4] = b2.x; bs[5] = b2.y;
        }
        return start<FIRST_CELL>(A, x, bs, (uint32_t)((long long)dir * A.n + pos));
    }

    __device__ void finish(const TraceArgs &A, int face, uint32_t flags)
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

    // Step size of a trial step from the current state (reading A5; spherical: physical cell edges, reading A19)
    __device__ __forceinline__ double step_size(const TraceArgs &A) const
    {
        double h = STRETCHED ? A.step_frac * fmin(hc[0], fmin(hc[1], hc[2])) : A.h_uniform;
        if (SPH) h = A.step_frac * fmin(y[2] * cth * A.fv.h[0], fmin(y[2] * A.fv.h[1], A.fv.h[2]));
        if (lam + h > A.max_length) h = A.max_length - lam;
        return h;
    }

    // Scheduling fence (not arithmetic): makes the offsets d of the next evaluation depend on `after` through an integer
    // OR with (bits of after & A.tie_zero), where tie_zero is a kernel argument that is always 0.  ptxas schedules a
    // basic block by critical path and would otherwise start the next stage's polynomial - whose first instruction
    // waits for the table loads of a cell change, and with it the whole in-order warp - ahead of the ~45 independent
    // FP64 instructions placed after enter_cell() to cover that latency (profiles/r2d: 14 % of the issue cycles of cfg2
    // were spent on the first instruction after the two cell-change sites that take nearly all the changes).
    __device__ __forceinline__ static void tie(const TraceArgs &A, double d[3], double after)
    {
        const int t = __double2loint(after) & (int)A.tie_zero;
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] = __hiloint2double(__double2hiint(d[c]), __double2loint(d[c]) | t);
    }

    // One step of size hs from y given b1 = b(y) and J1 = grad b(y) (poly() at y): trial end xn, the deviation
    // increments inc (trial end of component c >= 3 is y[c] + fc inc[c], formed only when the step is committed), the
    // trial length accL and bn1 = |b(y)|.  Four field evaluations per RK4 step in all; the cached cell on return is that
    // of xn.  Per stage: polynomial (value + gradient) -> position of the next stage point -> enter_cell for it (table
    // loads of a cell change in flight) -> deviation products, |b|, accumulators of this stage -> next polynomial.
    // Nearly all cell changes happen on the two half-step moves (stage 1 -> 2 and stage 3 -> 4: some lane of a warp
    // changes cell there in 94 % of the attempts, against 14 % at the other two); those two sites get the fence.
    // Spherical geometry needs the metric factors of the stage point before the next point: there the deviation
    // products and |b| come first.  The direction sign is folded into the step size.
    __device__ __forceinline__ void trial(const TraceArgs &A, double hs, const double b1[3], const double *J1, double xn[3],
                                          double *inc, double &fc, double &accL, double &bn1)
    {
        // deviation products before the next stage point (else after its enter_cell); per stage
        constexpr bool EARLY1 = SPH || !(QSL_T2_DEFER == 1 || QSL_T2_DEFER == 2 || QSL_T2_DEFER == 3);
        constexpr bool EARLY3 = SPH || !(QSL_T2_DEFER == 1 || QSL_T2_DEFER == 3);
        constexpr bool EARLY = SPH || QSL_T2_DEFER != 1;
        constexpr bool TIE = QSL_T2_TIE;
        double b[3], J[NJ], k[NV], d[3], acc[NV], ys[NV], bn;
        const double shs = back ? -hs : hs;
#pragma unroll
        for (int c = 0; c < 3; ++c) b[c] = b1[c];
        if (A.method == QSL_EULER) {
            products(J1, y, k);
            bn1 = SPH ? to_rates(y, b, k) : norm3_fast(b);
#pragma unroll
            for (int c = 0; c < 3; ++c) xn[c] = fma(shs, b[c], y[c]);
#pragma unroll
            for (int c = 3; c < NV; ++c) inc[c] = k[c];
            fc = shs;
            accL = fma(hs, bn1, L);
            enter_cell(A, xn, d);
            return;
        }
        // RK4 (reading A5): k2 = f(y + h/2 k1), k3 = f(y + h/2 k2), k4 = f(y + h k3), y+ = y + h/6 (k1 + 2 k2 + 2 k3 + k4)
        const double half = 0.5 * shs;
        // ---- stage 1 (polynomial done by the caller)
        if (EARLY1) { products(J1, y, k); if (SPH) bn = to_rates(y, b, k); }
#pragma unroll
        for (int c = 0; c < 3; ++c) ys[c] = fma(half, b[c], y[c]);
        enter_cell(A, ys, d);
        if (!EARLY1) products(J1, y, k);
        if (!SPH) bn = norm3_fast(b);
        bn1 = bn;
#pragma unroll
        for (int c = 0; c < NV; ++c) { acc[c] = c < 3 ? b[c] : k[c]; if (c >= 3) ys[c] = fma(half, k[c], y[c]); }
        accL = bn;
        if (TIE) tie(A, d, bn);
        // ---- stage 2
        poly(d, b, J);
        {
            double xs[3];
            if (EARLY) { products(J, ys, k); if (SPH) bn = to_rates(ys, b, k); }
#pragma unroll
            for (int c = 0; c < 3; ++c) xs[c] = fma(half, b[c], y[c]);
            enter_cell(A, xs, d);
            if (!EARLY) products(J, ys, k);
            if (!SPH) bn = norm3_fast(b);
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                const double kc = c < 3 ? b[c] : k[c];
                acc[c] = fma(2.0, kc, acc[c]); ys[c] = c < 3 ? xs[c] : fma(half, kc, y[c]);
            }
            accL = fma(2.0, bn, accL);
        }
        // ---- stage 3
        poly(d, b, J);
        {
            double xs[3];
            if (EARLY3) { products(J, ys, k); if (SPH) bn = to_rates(ys, b, k); }
#pragma unroll
            for (int c = 0; c < 3; ++c) xs[c] = fma(shs, b[c], y[c]);
            enter_cell(A, xs, d);
            if (!EARLY3) products(J, ys, k);
            if (!SPH) bn = norm3_fast(b);
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                const double kc = c < 3 ? b[c] : k[c];
                acc[c] = fma(2.0, kc, acc[c]); ys[c] = c < 3 ? xs[c] : fma(shs, kc, y[c]);
            }
            accL = fma(2.0, bn, accL);
            if (TIE) tie(A, d, accL);
        }
        // ---- stage 4
        poly(d, b, J);
        {
            const double fL = hs * (1.0 / 6.0), f = back ? -fL : fL;
            if (EARLY) { products(J, ys, k); if (SPH) bn = to_rates(ys, b, k); }
#pragma unroll
            for (int c = 0; c < 3; ++c) xn[c] = fma(f, fma(1.0, b[c], acc[c]), y[c]);
            // the trial end is where the next attempt starts if it is accepted: enter its cell now
            enter_cell(A, xn, d);
            if (!EARLY) products(J, ys, k);
            if (!SPH) bn = norm3_fast(b);
#pragma unroll
            for (int c = 3; c < NV; ++c) inc[c] = fma(1.0, k[c], acc[c]);
            fc = f;
            accL = fma(fL, fma(1.0, bn, accL), L);
        }
    }

    // One attempt of the trace kernel proper: a trial step from y, committed if its end is inside the closed trace box.
    // A line whose trial step leaves the box is written to its record as it stands, flagged REC_LANDING, and the lane is
    // free for the next work item: the landing of reading A4 (chord + three Newton updates + snap: five more steps'
    // worth of evaluations, a state machine of its own) is done for all lines at once by landing_kernel, where every
    // lane is in the same phase, instead of by one lane of a warp here while the other 31 wait.
    // Returns true when the line has left this kernel (landing pending, stall, cap).
    __device__ __forceinline__ bool advance(const TraceArgs &A)
    {
        double b[3], J[NJ], d[3], xn[3], inc[NV], fc, accL, bn;
        if (QSL_T2_HEADTEST) enter_cell(A, y, d);
        else {
            // the cell of y is the cached one: entered by the last stage of the previous attempt (y = its trial end) or,
            // for a line that has just started, by start_cell()
            d[0] = y[0] - x0[0]; d[1] = y[1] - x0[1]; d[2] = y[2] - x0[2];
        }
        poly(d, b, J);
        const double h = step_size(A);
        trial(A, h, b, J, xn, inc, fc, accL, bn);
        // O4: stall / caps are tested on k1 before the step is taken (here: before it is committed; the trial step of a
        // line that ends this way is discarded); h from the cell containing x
        if (!(bn >= A.null_eps) || (long long)nsteps >= A.max_steps || lam >= A.max_length) {
            finish(A, 255, !(bn >= A.null_eps) ? (nsteps == 0 ? REC_NULL_AT_SEED : REC_STALL) : REC_CAP);
            return true;
        }
        if (inside_box(A, xn)) {
            if (SPH) move_anchor(xn[1] - y[1]);
#pragma unroll
            for (int c = 0; c < NV; ++c) y[c] = c < 3 ? xn[c] : fma(fc, inc[c], y[c]);
            L = accL; lam += h; ++nsteps;
            return false;
        }
        finish(A, 255, REC_LANDING);
        return true;
    }

    // The landing of one line (reading A4), from the state the trace kernel recorded: the trial step is taken again
    // (same arithmetic, same end), the chord gives the first landing step hp, then
    //    step(hp), Newton, step(hp), Newton, step(hp), Newton, step(hp) -> snap onto the face
    // with the polynomial at y evaluated once.  Returns the number of steps added to the line (1, or 0 if the trial
    // point is not finite).
    __device__ unsigned land(const TraceArgs &A)
    {
        double b1[3], J1[NJ], b[3], J[NJ], k[NV], d[3], xn[3], inc[NV], fc, accL, bn1;
        enter_cell(A, y, d);
        poly(d, b1, J1);
        const double h = step_size(A);
        trial(A, h, b1, J1, xn, inc, fc, accL, bn1);
        // first face crossed by the chord: smallest fraction, tie -> lowest axis (reading A4)
        double phi = INFINITY; int ax = -1, face = 255; double bound = 0.0;
#pragma unroll
        for (int dd = 0; dd < 3; ++dd) {
            if (xn[dd] < A.box_lo[dd]) {
                const double f = (A.box_lo[dd] - y[dd]) / (xn[dd] - y[dd]);
                if (f < phi) { phi = f; ax = dd; face = 2 * dd; bound = A.box_lo[dd]; }
            } else if (xn[dd] > A.box_hi[dd]) {
                const double f = (A.box_hi[dd] - y[dd]) / (xn[dd] - y[dd]);
                if (f < phi) { phi = f; ax = dd; face = 2 * dd + 1; bound = A.box_hi[dd]; }
            }
        }
        if (ax < 0) { finish(A, 255, REC_STALL); return 0; }   // non-finite trial point
        const double yd = ax == 0 ? y[0] : (ax == 1 ? y[1] : y[2]);
        if (yd == bound) {
            // the line starts on the face it leaves through (photospheric seeds): hp = 0, every Newton residual is
            // exactly 0, so the landing of O4 ends where it started: one zero-length step
            ++nsteps;
            finish(A, face, 0);
            return 1;
        }
        double hp = phi * h;
        for (int it = 0; it < 4; ++it) {
            trial(A, hp, b1, J1, xn, inc, fc, accL, bn1);
            if (it == 3) break;
            // Newton update of hp from the field at the trial end (clamped to [0, h]); the cell of xn is cached
            d[0] = xn[0] - x0[0]; d[1] = xn[1] - x0[1]; d[2] = xn[2] - x0[2];
            poly(d, b, J);
            if (SPH) { products(J, y, k); to_rates(xn, b, k); }
            const double bd = ax == 0 ? b[0] : (ax == 1 ? b[1] : b[2]);
            const double xd = ax == 0 ? xn[0] : (ax == 1 ? xn[1] : xn[2]);
            const double gg = back ? -bd : bd, r = xd - bound;
            if (gg != 0.0) {
                const double hn = hp - r / gg;
                if (hn == hn) hp = fmin(fmax(hn, 0.0), h);
            }
        }
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = c < 3 ? xn[c] : fma(fc, inc[c], y[c]);
        if (ax == 0) y[0] = bound; else if (ax == 1) y[1] = bound; else y[2] = bound;
        L = accL; lam += hp; ++nsteps;
        finish(A, face, 0);
        return 1;
    }
};

// O2 (PAPER.md:160 eq. 9, :163): a^, b^ orthonormal with B^(x0); reading A7: e = axis of the smallest |u_d|.  One thread
// per seed in sorted order; writes (a^, b^) = 6 doubles per seed for the init of the trace kernel.
template <bool STRETCHED, bool INTERP>
__global__ void __launch_bounds__(128) seed_basis_kernel(const TraceArgs A, double *__restrict__ basis)
{
    const long long pos = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= A.n) return;
    const uint32_t si = A.perm[pos];
    const double x[3] = { A.seeds[3 * (size_t)si], A.seeds[3 * (size_t)si + 1], A.seeds[3 * (size_t)si + 2] };
    double o[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    if (inside_box(A, x)) {
        LineState2<false, STRETCHED, INTERP> ls;
        ls.relocate(A, x);
        const double d[3] = { x[0] - ls.x0[0], x[1] - ls.x0[1], x[2] - ls.x0[2] };
        double b[3];
        ls.stage(d, nullptr, b, nullptr);
        const double nb = norm3(b);
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
        o[0] = av[0]; o[1] = av[1]; o[2] = av[2];
        o[3] = u[1] * av[2] - u[2] * av[1];
        o[4] = u[2] * av[0] - u[0] * av[2];
        o[5] = u[0] * av[1] - u[1] * av[0];
    }
    double2 *w = reinterpret_cast<double2 *>(basis + 6 * (size_t)pos);
    w[0] = make_double2(o[0], o[1]); w[1] = make_double2(o[2], o[3]); w[2] = make_double2(o[4], o[5]);
}

// Resident CTAs per SM the register allocation is capped for: 3 x 128 threads (<= 168 registers) with the deviation
// vectors, 4 x 128 (<= 128 registers) without; the FP64 dependency chains need the extra warps more than the registers.
#ifndef QSL_T2_THREADS
#define QSL_T2_THREADS 128
#endif
#ifndef QSL_T2_MIN_BLOCKS_LQ
#define QSL_T2_MIN_BLOCKS_LQ 3
#endif
#ifndef QSL_T2_MIN_BLOCKS_L
#define QSL_T2_MIN_BLOCKS_L 4
#endif
// The persistent kernel (REFILL) takes its work items through staged_queue (trace_kernels.cuh).
template <bool DEV, bool STRETCHED, bool INTERP, bool REFILL, bool SPH = false>
__global__ void __launch_bounds__(QSL_T2_THREADS, DEV ? QSL_T2_MIN_BLOCKS_LQ : QSL_T2_MIN_BLOCKS_L) trace2_kernel(const TraceArgs A)
{
    LineState2<DEV, STRETCHED, INTERP, SPH> ls;
    const long long n_items = 2 * A.n;
    unsigned long long my_steps = 0;
    if (!REFILL) {
        const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (q < n_items && ls.template init<!QSL_T2_HEADTEST>(A, q)) {
            while (!ls.advance(A)) {}
        }
        if (q < n_items) my_steps = ls.nsteps;
    } else {
        staged_queue<DEV, QSL_T2_THREADS, QSL_T2_CHUNK>(
            A, [&](const double *x, const double *bs, uint32_t sl) { return ls.template start<!QSL_T2_HEADTEST>(A, x, bs, sl); },
            [&]() { if (!ls.advance(A)) return false; my_steps += ls.nsteps; return true; });
    }
    if (A.total_steps) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_steps += __shfl_xor_sync(0xffffffffu, my_steps, o);
        if ((threadIdx.x & 31) == 0 && my_steps) atomicAdd(A.total_steps, my_steps);
    }
}

// The landings of all lines of a launch (reading A4): one thread per per-direction record, in the Morton order of the
// seeds; a record without REC_LANDING (stall, cap, seed outside) is left as it is.  Every lane runs the same five steps.
template <bool DEV, bool STRETCHED, bool INTERP, bool SPH = false>
__global__ void __launch_bounds__(128) landing_kernel(const TraceArgs A)
{
    const long long sl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned added = 0;
    if (sl < 2 * A.n) {
        const double2 *__restrict__ r2 = reinterpret_cast<const double2 *>(A.rec + (size_t)sl * REC_DOUBLES);
        const double2 w5 = r2[5];
        if ((uint32_t)__double2hiint(w5.x) & REC_LANDING) {
            LineState2<DEV, STRETCHED, INTERP, SPH> ls;
            constexpr int NV = LineState2<DEV, STRETCHED, INTERP, SPH>::NV;
            double v[10];
#pragma unroll
            for (int c = 0; c < 5; ++c) { const double2 t = r2[c]; v[2 * c] = t.x; v[2 * c + 1] = t.y; }
#pragma unroll
            for (int c = 0; c < NV; ++c) ls.y[c] = v[c];
            ls.L = v[9]; ls.lam = w5.y; ls.nsteps = (uint32_t)__double2loint(w5.x);
            ls.slot = (uint32_t)sl; ls.back = sl >= A.n; ls.phase = 0;
            if (SPH) sincos(ls.y[1], &ls.sth, &ls.cth); else { ls.sth = 0.0; ls.cth = 1.0; }
            ls.x0[0] = ls.x0[1] = ls.x0[2] = __longlong_as_double(0x7ff8000000000000ll);
            ls.hc[0] = ls.hc[1] = ls.hc[2] = 0.0;
            added = ls.land(A);
        }
    }
    if (A.total_steps) {
        const unsigned m = __ballot_sync(0xffffffffu, added != 0);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(A.total_steps, (unsigned long long)__popc(m));
    }
}

}  // namespace qsl
