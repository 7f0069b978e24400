// fp32-arithmetic trace kernel (QSL_ARITH_F32, reading A6 of DESIGN.md: the throughput mode for fp32-sampled fields).
// The same method and state machine as trace2_kernels.cuh (PAPER.md:79 eq. 1, :119 eq. 5, :141, :163; readings A3-A5),
// re-designed for single precision instead of re-typed:
//
//  * the position is never held as an absolute fp32 coordinate (ulp(1.0f) = 6e-8 is 1.5e-5 of a 1/255 cell): a line
//    carries the integer index C of the cell whose polynomial is cached and the fp32 offset of its point from that
//    cell's origin.  Offsets are < 2 h, so their rounding is ~1e-10 of the box, and a cell change is an integer
//    neighbour step plus one subtraction of h - no floating-point search;
//  * the per-cell table holds the 24 monomial coefficients as fp32 (96 B = 3 sectors per cell, half the fp64 table);
//  * the trace box is given in cell coordinates (cell index + offset per face), so the "inside the box" test is an
//    integer compare for every cell that does not touch a face of the box;
//  * L and lambda are accumulated in fp64 (two DADD per step): summing ~1e3 increments of ~1e-3 in fp32 would by itself
//    cost 1e-6 of L.
// End records are written in fp64 (origin of the cell + offset), so the epilogue (eq. 11) is shared.
#pragma once
#include "trace_kernels.cuh"

namespace qsl {

// Scalar-type traits of the kernel: T = float (QSL_ARITH_F32, 96 B table entries) or double (the fp64 table).
template <typename T> struct Real3;
template <> struct Real3<float> {
    using V4 = float4;
    static __device__ __forceinline__ float4 load(const float4 *p) { return __ldg(p); }
    // bit pattern for the "0 <= p < h" test (one unsigned compare per axis): exact in fp32
    static __device__ __forceinline__ unsigned bits(float v) { return (unsigned)__float_as_int(v); }
    static __device__ __forceinline__ float rsqrt_seed(float n2) { return rsqrtf(fmaxf(n2, 7.8886e-31f)); }
    static __device__ __forceinline__ float rcp(float v) { return __frcp_rn(v); }
};
template <> struct Real3<double> {
    using V4 = double4;
    static __device__ __forceinline__ double4 load(const double4 *p)
    {
        double4 r;   // one 256-bit LDG (sm_100)
        asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
        return r;
    }
    // high word only: sufficient, not necessary (false for p within 2^-20 relative below h: a redundant reload)
    static __device__ __forceinline__ unsigned bits(double v) { return (unsigned)__double2hiint(v); }
    static __device__ __forceinline__ double rsqrt_seed(double n2)
    {
        double r;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(fmax(n2, 0x1p-600)));
        return r;
    }
    static __device__ __forceinline__ double rcp(double v) { return 1.0 / v; }
};

template <typename T>
struct Trace3Args {
    TraceArgs T0;                // the arguments of qsl_trace common to all kernels
    const typename Real3<T>::V4 *cells;   // 6 V4 per cell: monomial coefficients a[8 c + m] of the trilinear interpolant
    T hf[3];                     // cell edges
    unsigned hbits[3];           // Real3<T>::bits(hf)
    T h_step;                    // step_frac * min_d h_d
    int cmax[3];                 // n_d - 2: last cell index per axis
    int cell_sy, cell_sz;        // table strides in cells
    int cl[3], ch[3];            // cells containing box_lo / box_hi (box_hi on a node belongs to the cell below it)
    unsigned cw[3];              // max(ch - cl - 1, 0): number of cells strictly between them
    T off_lo[3], off_hi[3];      // offsets of box_lo / box_hi from the origins of cells cl / ch
    T null_eps;
    // spherical geometry (reading A19; SPH instantiations): (sin, cos) of the latitude of every row of cells (fp64
    // sincos rounded to fp32, built by qsl_field_create), and the step fraction (the step is sized per attempt)
    const float2 *row_sc;
    T step_frac;
};


// |v|, branch-free: hardware reciprocal square root of max(|v|^2, tiny) and one coupled Newton step (relative error
// ~1e-7 in fp32, ~1e-13 in fp64).  |v|^2 = 0 gives exactly 0; NaN and overflow propagate (and then stop the line through
// the stall test); |v| below 2^-50 (fp32) / 2^-300 (fp64) comes out too small, far under any stall threshold.
template <typename T>
__device__ __forceinline__ T norm3r_fast(const T v[3])
{
    const T n2 = fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0]));
    const T r = Real3<T>::rsqrt_seed(n2);
    const T s = n2 * r, hr = T(0.5) * r;
    if (sizeof(T) == 4) return fma(fma(-s, s, n2), hr, s);
    const T e = fma(-s, hr, T(0.5));                   // 0.5 (1 - n2 r^2)
    const T s1 = fma(s, e, s), h1 = fma(hr, e, hr);
    return fma(fma(-s1, s1, n2), h1, s1);
}

// SPH: spherical geometry (reading A19) in the cell frame.  The frame carries the radius of the cell's origin and
// (sin, cos) of its latitude; a point at offsets p has r = rc + p_r and cos(theta) = cc cos(p_theta) - sc sin(p_theta)
// with short polynomials of the offset (|p_theta| < 2 h_theta; terms through p^6 / p^5: below the fp32 ulp for cell
// edges up to 0.3 rad), so no evaluation calls a trigonometric function.
template <typename T, bool DEV, bool INTERP, bool SPH = false>
struct LineState3 {
    using Args = Trace3Args<T>;
    static constexpr int NV = DEV ? 9 : 3;
    T a[24];             // cached cell: monomial coefficients
    T rc, sc, cc;        // SPH: radius and (sin, cos) of the latitude of the origin of cell C
    int C[3];                // its index = the frame of every offset below
    T y[NV];             // y[0..2]: offset of the line's point from the origin of cell C; delta1, delta2
    double L, lam;
    uint32_t nsteps, slot;
    int phase;
    bool back;

    __device__ __forceinline__ void load_cell(const Args &A)
    {
        const typename Real3<T>::V4 *__restrict__ p = A.cells + ((size_t)((unsigned)C[2] * (unsigned)A.cell_sz + (unsigned)C[1] * (unsigned)A.cell_sy + (unsigned)C[0])) * 6;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const typename Real3<T>::V4 v = Real3<T>::load(p + q);
            a[4 * q] = v.x; a[4 * q + 1] = v.y; a[4 * q + 2] = v.z; a[4 * q + 3] = v.w;
        }
        if (SPH) {
            rc = (T)fma((double)C[2], A.T0.fv.h[2], A.T0.fv.lo[2]);
            const float2 v = __ldg(A.row_sc + C[1]);
            sc = (T)v.x; cc = (T)v.y;
        }
    }

    // SPH: r cos(theta) and r of the point at offsets p of the frame
    __device__ __forceinline__ void polar(const T p[3], T &rcos, T &r) const
    {
        const T d = p[1], d2 = d * d;
        const T cd = fma(d2, fma(d2, fma(d2, T(-1.0 / 720.0), T(1.0 / 24.0)), T(-0.5)), T(1.));
        const T sd = d * fma(d2, fma(d2, T(1.0 / 120.0), T(-1.0 / 6.0)), T(1.));
        r = rc + p[2];
        rcos = r * fma(cc, cd, -(sc * sd));
    }

    // |b| of the field vector and, with SPH, b -> coordinate rates and k -> coordinate deviation rates at offsets p:
    // orthonormal components x (1 / (r cos theta), 1 / r, 1)  (PAPER.md:83-85 eq. 2, :125-135 eq. 6-7)
    __device__ __forceinline__ T to_rates(const T p[3], T b[3], T *k) const
    {
        const T bn = norm3r_fast<T>(b);
        if (SPH) {
            T rcos, r;
            polar(p, rcos, r);
            const T m0 = Real3<T>::rcp(rcos), m1 = Real3<T>::rcp(r);
            b[0] *= m0; b[1] *= m1;
            if (DEV) { k[3 % NV] *= m0; k[4 % NV] *= m1; k[6 % NV] *= m0; k[7 % NV] *= m1; }
        }
        return bn;
    }

    // Makes the cached cell the one containing the point at offsets p (reading A8: the index is clamped to the grid,
    // the offset is not) by a neighbour step per axis, and moves the frame of p and of the line's own point with it.
    // Consecutive evaluation points are at most half a cell apart (|b| <= 1, h = step_frac cell), so one step suffices.
    // The "still inside" test is one unsigned compare per axis on the bit pattern: 0 <= p < h.
    __device__ __forceinline__ void enter_cell(const Args &A, T p[3])
    {
        if (!(Real3<T>::bits(p[0]) < A.hbits[0] && Real3<T>::bits(p[1]) < A.hbits[1] && Real3<T>::bits(p[2]) < A.hbits[2])) {
            // one level of divergence: a lane that is only extrapolating beyond the edge of the grid (no neighbour to
            // step to) reloads the cell it already has
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const bool dn = p[d] < T(0.) && C[d] > 0, up = p[d] >= A.hf[d] && C[d] < A.cmax[d];
                C[d] += up ? 1 : (dn ? -1 : 0);
                const T sh = up ? A.hf[d] : (dn ? -A.hf[d] : T(0.));
                p[d] -= sh; y[d] -= sh;
            }
            load_cell(A);
        }
    }

    // Field evaluation at offsets d inside the cached cell fused with the deviation products (as LineState2::stage).
    __device__ __forceinline__ void stage(const T d[3], const T *ys, T b[3], T *k)
    {
        const T dx = d[0], dy = d[1], dz = d[2];
        T v[3], g[9];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const T *q = a + 8 * c;
            const T P = fma(q[7], dz, q[3]), Q = fma(q[5], dz, q[1]), R = fma(q[6], dz, q[2]), S = fma(q[4], dz, q[0]);
            const T E = fma(P, dy, Q), F = fma(R, dy, S);
            v[c] = fma(E, dx, F);
            if (DEV || INTERP) {
                g[3 * c] = E;
                g[3 * c + 1] = fma(P, dx, R);
                g[3 * c + 2] = fma(fma(q[7], dy, q[5]), dx, fma(q[6], dy, q[4]));
            }
        }
        if (!INTERP) {
#pragma unroll
            for (int c = 0; c < 3; ++c) b[c] = v[c];
        } else
        {
            // reading A2: b = B/|B|, J = (G - u (u^T G))/|B|
            const T nn = sqrt(fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0])));
            if (nn < (sizeof(T) == 4 ? T(1e-37) : T(1e-300))) {
#pragma unroll
                for (int c = 0; c < 3; ++c) b[c] = T(0.);
#pragma unroll
                for (int q = 0; q < 9; ++q) g[q] = T(0.);
            } else {
                const T inv = T(1.0) / nn;
                const T u[3] = { v[0] * inv, v[1] * inv, v[2] * inv };
#pragma unroll
                for (int c = 0; c < 3; ++c) b[c] = u[c];
                if (DEV) {
#pragma unroll
                    for (int e = 0; e < 3; ++e) {
                        const T uG = fma(u[2], g[6 + e], fma(u[1], g[3 + e], u[0] * g[e]));
#pragma unroll
                        for (int c = 0; c < 3; ++c) g[3 * c + e] = (g[3 * c + e] - u[c] * uG) * inv;
                    }
                }
            }
        }
        if (DEV) {
#pragma unroll
            for (int w = 0; w < 2; ++w)
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    k[(3 + 3 * w + c) % NV] = fma(g[3 * c + 2], ys[(5 + 3 * w) % NV], fma(g[3 * c + 1], ys[(4 + 3 * w) % NV], g[3 * c] * ys[(3 + 3 * w) % NV]));
        }
    }

    // Starts a line at the seed x with the orthonormal pair bs (a^, b^ of O2, from seed_basis3_kernel; unused without
    // DEV) for record slot sl (false if it ended at once: seed outside the trace box).  The seed's cell is found once,
    // in fp64, exactly as O1 does (floor of (x - lo)/h, clamped).
    __device__ __forceinline__ bool start(const Args &A, const double x[3], const double *bs, uint32_t sl)
    {
        const TraceArgs &G = A.T0;
        slot = sl;
        back = (long long)sl >= G.n;
        L = 0.0; lam = 0.0; nsteps = 0; phase = 0;
        if (!inside_box(G, x)) {
            double out[REC_DOUBLES];
#pragma unroll
            for (int c = 0; c < REC_DOUBLES; ++c) out[c] = c < 3 ? x[c] : 0.0;
            out[10] = __hiloint2double((int)(255u | REC_SEED_OUTSIDE), 0);
            double2 *r2 = reinterpret_cast<double2 *>(G.rec + (size_t)slot * REC_DOUBLES);
#pragma unroll
            for (int c = 0; c < REC_DOUBLES / 2; ++c) r2[c] = make_double2(out[2 * c], out[2 * c + 1]);
            return false;
        }
        frame_of(A, x);
#pragma unroll
        for (int c = 3; c < NV; ++c) y[c] = (T)bs[(c - 3) % 6];
        load_cell(A);
        if (SPH && DEV) {     // orthonormal pair -> coordinate deviations (eq. 8 inverted)
            T rcos, r;
            polar(y, rcos, r);
            const T m0 = Real3<T>::rcp(rcos), m1 = Real3<T>::rcp(r);
            y[3 % NV] *= m0; y[4 % NV] *= m1; y[6 % NV] *= m0; y[7 % NV] *= m1;
        }
        return true;
    }

    // Frame (cell index C, offsets y[0..2]) of the absolute point x
    __device__ __forceinline__ void frame_of(const Args &A, const double x[3])
    {
        const TraceArgs &G = A.T0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double u = (x[d] - G.fv.lo[d]) * G.inv_h[d];
            int i = (int)floor(u);
            i = max(0, min(i, A.cmax[d]));
            C[d] = i;
            y[d] = (T)(x[d] - fma((double)i, G.fv.h[d], G.fv.lo[d]));
        }
    }

    // Starts work item q of the queue
    __device__ bool init(const Args &A, long long q)
    {
        const TraceArgs &G = A.T0;
        long long pos; int dir;
        if (G.interleave) { pos = q >> 1; dir = (int)(q & 1); } else { dir = q >= G.n ? 1 : 0; pos = q - (long long)dir * G.n; }
        const uint32_t si = G.perm[pos];
        const double x[3] = { G.seeds[3 * (size_t)si], G.seeds[3 * (size_t)si + 1], G.seeds[3 * (size_t)si + 2] };
        double bs[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
        if (DEV) {
            const double2 *__restrict__ bp = reinterpret_cast<const double2 *>(G.basis + 6 * (size_t)pos);
            const double2 b0 = bp[0], b1 = bp[1], b2 = bp[2];
            bs[0] = b0.x; bs[1] = b0.y; bs[2] = b1.x; bs[3] = b1.y; bs[4] = b2.x; bs[5] = b2.y;
        }
        return start(A, x, bs, (uint32_t)((long long)dir * G.n + pos));
    }

    // Writes the per-direction record in fp64: position = origin of the frame cell + offset; `snap` >= 0 puts the
    // coordinate of that axis exactly on the face it landed on.
    __device__ void finish(const Args &A, int face, uint32_t flags, int snap)
    {
        const TraceArgs &G = A.T0;
        double out[REC_DOUBLES];
#pragma unroll
        for (int d = 0; d < 3; ++d) out[d] = fma((double)C[d], G.fv.h[d], G.fv.lo[d]) + (double)y[d];
        if (snap >= 0) {
            const double bd = (face & 1) ? (snap == 0 ? G.box_hi[0] : (snap == 1 ? G.box_hi[1] : G.box_hi[2]))
                                         : (snap == 0 ? G.box_lo[0] : (snap == 1 ? G.box_lo[1] : G.box_lo[2]));
            if (snap == 0) out[0] = bd; else if (snap == 1) out[1] = bd; else out[2] = bd;
        }
#pragma unroll
        for (int c = 3; c < 9; ++c) out[c] = c < NV ? (double)y[c % NV] : 0.0;
        out[9] = L;
        out[10] = __hiloint2double((int)((uint32_t)face | flags), (int)nsteps);
        out[11] = lam;
        double2 *r2 = reinterpret_cast<double2 *>(G.rec + (size_t)slot * REC_DOUBLES);
#pragma unroll
        for (int c = 0; c < REC_DOUBLES / 2; ++c) r2[c] = make_double2(out[2 * c], out[2 * c + 1]);
    }

    // Offset, in the current frame, of the face (axis, upper?) of the trace box.
    __device__ __forceinline__ T face_offset(const Args &A, int axis, bool upper) const
    {
        const int cd = axis == 0 ? C[0] : (axis == 1 ? C[1] : C[2]);
        const int cb = upper ? (axis == 0 ? A.ch[0] : (axis == 1 ? A.ch[1] : A.ch[2])) : (axis == 0 ? A.cl[0] : (axis == 1 ? A.cl[1] : A.cl[2]));
        const T ob = upper ? (axis == 0 ? A.off_hi[0] : (axis == 1 ? A.off_hi[1] : A.off_hi[2]))
                               : (axis == 0 ? A.off_lo[0] : (axis == 1 ? A.off_lo[1] : A.off_lo[2]));
        const T hd = axis == 0 ? A.hf[0] : (axis == 1 ? A.hf[1] : A.hf[2]);
        return fma((T)(cb - cd), hd, ob);
    }

    // Is the point at offsets e of the frame cell inside the closed trace box?  Cells strictly between the cells that
    // hold the faces of the box need one unsigned compare per axis; the others compare the offset with the face's.
    __device__ __forceinline__ bool inside3(const Args &A, const T e[3]) const
    {
        if ((unsigned)(C[0] - A.cl[0] - 1) < A.cw[0] && (unsigned)(C[1] - A.cl[1] - 1) < A.cw[1] && (unsigned)(C[2] - A.cl[2] - 1) < A.cw[2])
            return true;
        bool in = true;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const bool lo_ok = C[d] > A.cl[d] || (C[d] == A.cl[d] && e[d] >= A.off_lo[d]);
            const bool hi_ok = C[d] < A.ch[d] || (C[d] == A.ch[d] && e[d] <= A.off_hi[d]);
            in = in && lo_ok && hi_ok;
        }
        return in;
    }

    // Scheduling fence (LineState2::tie): the offsets of the next evaluation are made to depend on `after` through an
    // integer OR with (bits & tie_zero), tie_zero a kernel argument that is always 0, so that ptxas keeps the independent
    // work placed after enter_cell() between the table loads of a cell change and their first use.
    __device__ __forceinline__ static void tie(const Args &A, T d[3], T after)
    {
        if (sizeof(T) == 4) {
            const int t = __float_as_int((float)after) & (int)A.T0.tie_zero;
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] = (T)__int_as_float(__float_as_int((float)d[c]) | t);
        } else {
            const int t = __double2loint((double)after) & (int)A.T0.tie_zero;
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] = (T)__hiloint2double(__double2hiint((double)d[c]), __double2loint((double)d[c]) | t);
        }
    }

    // Step size of a trial step from the line's point (reading A5; spherical: physical cell edges, reading A19)
    __device__ __forceinline__ T step_size(const Args &A) const
    {
        T h = A.h_step;
        if (SPH) {
            T rcos, r;
            polar(y, rcos, r);
            h = A.step_frac * fmin(rcos * A.hf[0], fmin(r * A.hf[1], A.hf[2]));
        }
        if (lam + (double)h > A.T0.max_length) h = (T)(A.T0.max_length - lam);
        return h;
    }

    // One step of size hs from y given k1 = (b, k[3..]) and bn = |b| at y (all three consumed): trial end ys (position
    // offsets in the frame of the trial end's cell, to which y has been moved as well; deviation components) and the
    // length accL of the step.  Four evaluations per RK4 step in all; the cached cell on return is that of ys.
    __device__ __forceinline__ void trial(const Args &A, T hs, T b[3], T *k, T bn, T *ys, T &accL)
    {
        const TraceArgs &G = A.T0;
        T acc[NV];
        const T shs = back ? -hs : hs;
        if (G.method == QSL_EULER) {
#pragma unroll
            for (int c = 0; c < NV; ++c) ys[c] = fma(shs, c < 3 ? b[c] : k[c], y[c]);
            enter_cell(A, ys);
            accL = hs * bn;
            return;
        }
        const T half = T(0.5) * shs;
#pragma unroll
        for (int c = 0; c < 3; ++c) ys[c] = fma(half, b[c], y[c]);
        enter_cell(A, ys);
#pragma unroll
        for (int c = 0; c < NV; ++c) { acc[c] = c < 3 ? b[c] : k[c]; if (c >= 3) ys[c] = fma(half, k[c], y[c]); }
        accL = bn;
        tie(A, ys, ys[NV - 1]);
        // ---- stage 2
        stage(ys, ys, b, k);
        T bnS = T(0.);             // SPH: |b| is taken before the scaling to coordinate rates
        if (SPH) bnS = to_rates(ys, b, k);
        {
            T xn[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) xn[c] = fma(half, b[c], y[c]);
            enter_cell(A, xn);
            bn = SPH ? bnS : norm3r_fast<T>(b);
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                const T kc = c < 3 ? b[c] : k[c];
                acc[c] = fma(T(2.), kc, acc[c]); ys[c] = c < 3 ? xn[c] : fma(half, kc, y[c]);
            }
            accL = fma(T(2.), bn, accL);
        }
        // ---- stage 3
        stage(ys, ys, b, k);
        if (SPH) bnS = to_rates(ys, b, k);
        {
            T xn[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) xn[c] = fma(shs, b[c], y[c]);
            enter_cell(A, xn);
            bn = SPH ? bnS : norm3r_fast<T>(b);
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                const T kc = c < 3 ? b[c] : k[c];
                acc[c] = fma(T(2.), kc, acc[c]); ys[c] = c < 3 ? xn[c] : fma(shs, kc, y[c]);
            }
            accL = fma(T(2.), bn, accL);
            tie(A, ys, accL);
        }
        // ---- stage 4
        stage(ys, ys, b, k);
        if (SPH) bnS = to_rates(ys, b, k);
        {
            const T fL = hs * (T(1.0) / T(6.0)), f = back ? -fL : fL;
            T xn[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) xn[c] = fma(f, b[c] + acc[c], y[c]);
            enter_cell(A, xn);             // the trial end is where the next attempt starts if it is accepted
            bn = SPH ? bnS : norm3r_fast<T>(b);
#pragma unroll
            for (int c = 0; c < NV; ++c) ys[c] = c < 3 ? xn[c] : fma(f, k[c] + acc[c], y[c]);
            accL = fL * (bn + accL);
        }
    }

    // One attempt of the trace kernel proper (as LineState2::advance): a trial step from y, committed if its end is
    // inside the closed trace box; a line whose trial step leaves the box is recorded as it stands with REC_LANDING and
    // landed by landing3_kernel.  Returns true when the line has left this kernel.
    __device__ __forceinline__ bool advance(const Args &A)
    {
        const TraceArgs &G = A.T0;
        T b[3], k[NV], ys[NV], accL;
        {
            T p0[3] = { y[0], y[1], y[2] };
            enter_cell(A, p0);
            stage(p0, y, b, k);
            const T bn = to_rates(p0, b, k);
            // O4: stall / caps are tested on k1 before the step
            if (!(bn >= A.null_eps) || (long long)nsteps >= G.max_steps || lam >= G.max_length) {
                finish(A, 255, !(bn >= A.null_eps) ? (nsteps == 0 ? REC_NULL_AT_SEED : REC_STALL) : REC_CAP, -1);
                return true;
            }
            const T h = step_size(A);
            trial(A, h, b, k, bn, ys, accL);
            if (inside3(A, ys)) {
#pragma unroll
                for (int c = 0; c < NV; ++c) y[c] = ys[c];
                L += (double)accL; lam += (double)h; ++nsteps;
                return false;
            }
        }
        finish(A, 255, REC_LANDING, -1);
        return true;
    }

    // The landing of one line (reading A4; as LineState2::land) from the state the trace kernel recorded: the trial step
    // again, the chord, then step(hp), Newton, step(hp), Newton, step(hp), Newton, step(hp) -> snap onto the face, with
    // k1 at y evaluated once.  Returns the number of steps added to the line.
    __device__ unsigned land(const Args &A)
    {
        T b1[3], k1[NV], b[3], k[NV], ys[NV], accL;
        {
            T p0[3] = { y[0], y[1], y[2] };
            enter_cell(A, p0);
            stage(p0, y, b1, k1);
        }
        const T bn1 = to_rates(y, b1, k1);
        const T h = step_size(A);
#pragma unroll
        for (int c = 0; c < NV; ++c) { if (c < 3) b[c] = b1[c]; else k[c] = k1[c]; }
        trial(A, h, b, k, bn1, ys, accL);
        // first face crossed by the chord: smallest fraction, tie -> lowest axis, then low face (reading A4)
        T phi = INFINITY; int ax = -1, fc = 255; T bd = T(0.);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const bool lo_v = C[d] < A.cl[d] || (C[d] == A.cl[d] && ys[d] < A.off_lo[d]);
            const bool hi_v = C[d] > A.ch[d] || (C[d] == A.ch[d] && ys[d] > A.off_hi[d]);
            if (lo_v || hi_v) {
                const T fo = face_offset(A, d, !lo_v);
                const T f = (fo - y[d]) / (ys[d] - y[d]);
                if (f < phi) { phi = f; ax = d; fc = 2 * d + (lo_v ? 0 : 1); bd = fo; }
            }
        }
        if (ax < 0) { finish(A, 255, REC_STALL, -1); return 0; }   // non-finite trial point
        const T yd = ax == 0 ? y[0] : (ax == 1 ? y[1] : y[2]);
        if (yd == bd) {
            // the line starts on the face it leaves through: the landing of O4 is one zero-length step
            ++nsteps;
            finish(A, fc, 0, ax);
            return 1;
        }
        T hp = phi * h;
        for (int it = 0; it < 4; ++it) {
#pragma unroll
            for (int c = 0; c < NV; ++c) { if (c < 3) b[c] = b1[c]; else k[c] = k1[c]; }
            trial(A, hp, b, k, bn1, ys, accL);
            if (it == 3) break;
            // Newton update of hp from the field at the trial end (its cell is the cached one), clamped to [0, h]
            stage(ys, y, b, k);
            to_rates(ys, b, k);
            const T bdn = ax == 0 ? b[0] : (ax == 1 ? b[1] : b[2]);
            const T xd = ax == 0 ? ys[0] : (ax == 1 ? ys[1] : ys[2]);
            const T gg = back ? -bdn : bdn, r = xd - face_offset(A, ax, (fc & 1) != 0);
            if (gg != T(0.)) {
                const T hn = hp - r / gg;
                if (hn == hn) hp = fmin(fmax(hn, T(0.)), h);
            }
        }
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = ys[c];
        L += (double)accL; lam += (double)hp; ++nsteps;
        finish(A, fc, 0, ax);
        return 1;
    }
};

// O2 (PAPER.md:160 eq. 9, :163; reading A7) in fp64 from the packed node samples (S = their storage type), one thread per
// seed in sorted order: (a^, b^) = 6 doubles per seed for LineState3::init.  Once per line: not worth an fp32 variant.
template <typename S, bool INTERP>
__global__ void __launch_bounds__(128) seed_basis3_kernel(const TraceArgs A, double *__restrict__ basis)
{
    const long long pos = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= A.n) return;
    const uint32_t si = A.perm[pos];
    const double x[3] = { A.seeds[3 * (size_t)si], A.seeds[3 * (size_t)si + 1], A.seeds[3 * (size_t)si + 2] };
    double o[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    if (inside_box(A, x)) {
        double b[3], J[9], m, hmin;
        evaluate<S, false, INTERP, false, false>(A, x, b, J, m, hmin);
        const double inv = 1.0 / norm3(b);
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

#ifndef QSL_T3_THREADS
#define QSL_T3_THREADS 128
#endif
#ifndef QSL_T3_MIN_BLOCKS_LQ
#define QSL_T3_MIN_BLOCKS_LQ 5
#endif
#ifndef QSL_T3_MIN_BLOCKS_L
#define QSL_T3_MIN_BLOCKS_L 8
#endif
#ifndef QSL_T3_MIN_BLOCKS_LQ64
#define QSL_T3_MIN_BLOCKS_LQ64 3
#endif
#ifndef QSL_T3_MIN_BLOCKS_L64
#define QSL_T3_MIN_BLOCKS_L64 4
#endif
// Persistent grid; work items (one direction of one line) are staged per warp in shared memory, up to QSL_T3_CHUNK
// consecutive items of the Morton order per pop of the global counter (staged_queue, trace_kernels.cuh); a lane whose
// line ended takes the next staged item.
#ifndef QSL_T3_CHUNK
#define QSL_T3_CHUNK 8
#endif
template <typename T, bool DEV, bool INTERP, bool REFILL, bool SPH = false>
__global__ void __launch_bounds__(QSL_T3_THREADS, sizeof(T) == 4 ? (DEV ? QSL_T3_MIN_BLOCKS_LQ : QSL_T3_MIN_BLOCKS_L)
                                                                  : (DEV ? QSL_T3_MIN_BLOCKS_LQ64 : QSL_T3_MIN_BLOCKS_L64))
    trace3_kernel(const Trace3Args<T> A)
{
    LineState3<T, DEV, INTERP, SPH> ls;
    const TraceArgs &G = A.T0;
    const long long n_items = 2 * G.n;
    unsigned long long my_steps = 0;
    if (!REFILL) {
        const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (q < n_items) {
            ls.nsteps = 0;
            if (ls.init(A, q)) { while (!ls.advance(A)) {} }
            my_steps = ls.nsteps;
        }
    } else {
        staged_queue<DEV, QSL_T3_THREADS, QSL_T3_CHUNK>(
            G, [&](const double *x, const double *bs, uint32_t sl) { return ls.start(A, x, bs, sl); },
            [&]() { if (!ls.advance(A)) return false; my_steps += ls.nsteps; return true; });
    }
    if (G.total_steps) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_steps += __shfl_xor_sync(0xffffffffu, my_steps, o);
        if ((threadIdx.x & 31) == 0 && my_steps) atomicAdd(G.total_steps, my_steps);
    }
}

// The landings of all lines of a launch (reading A4): one thread per per-direction record (see landing_kernel).  The
// frame of the recorded point is found again as for a seed (fp64 cell search, offset rounded to T).
template <typename T, bool DEV, bool INTERP, bool SPH = false>
__global__ void __launch_bounds__(128) landing3_kernel(const Trace3Args<T> A)
{
    const TraceArgs &G = A.T0;
    const long long sl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned added = 0;
    if (sl < 2 * G.n) {
        const double2 *__restrict__ r2 = reinterpret_cast<const double2 *>(G.rec + (size_t)sl * REC_DOUBLES);
        const double2 w5 = r2[5];
        if ((uint32_t)__double2hiint(w5.x) & REC_LANDING) {
            LineState3<T, DEV, INTERP, SPH> ls;
            constexpr int NV = LineState3<T, DEV, INTERP, SPH>::NV;
            double v[10];
#pragma unroll
            for (int c = 0; c < 5; ++c) { const double2 t = r2[c]; v[2 * c] = t.x; v[2 * c + 1] = t.y; }
            ls.frame_of(A, v);
#pragma unroll
            for (int c = 3; c < NV; ++c) ls.y[c] = (T)v[c];
            ls.L = v[9]; ls.lam = w5.y; ls.nsteps = (uint32_t)__double2loint(w5.x);
            ls.slot = (uint32_t)sl; ls.back = sl >= G.n; ls.phase = 0;
            ls.load_cell(A);
            added = ls.land(A);
        }
    }
    if (G.total_steps) {
        const unsigned m = __ballot_sync(0xffffffffu, added != 0);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(G.total_steps, (unsigned long long)__popc(m));
    }
}

}  // namespace qsl
