// Device code of the field-line tracer: field evaluation, fused RK step of the 10-component
// state (x, delta1, delta2, L), termination + landing, per-direction records, and the Q/L epilogue.
//
//  PAPER.md:79  (eq. 1)   d x/d lambda = B^(x)
//  PAPER.md:95  (eq. 3)   B^(x) = sum_v B^{v+c} f_v(x - x_c; h_c), trilinear kernels eq. (4)
//  PAPER.md:119 (eq. 5)   d delta/d lambda = (delta . grad) B^, gradient taken analytically on the kernels (:123, :137)
//  PAPER.md:141           fixed-step integrators (Euler in the paper; RK4 by BASELINE.json, reading A5)
//  PAPER.md:163, 165      integrate forwards and backwards to any boundary of the box / to a maximum length
//  PAPER.md:156, 174, 176 (eq. 11) perpendicular projection and Q at the end points
#pragma once
#include <math.h>

#include "qsl_internal.cuh"

namespace qsl {

// ---------------------------------------------------------------------------------------------------------------
// Kernel arguments
struct TraceArgs {
    FieldView fv;
    double inv_h[3];             // 1 / uniform spacing
    double box_lo[3], box_hi[3];
    double h_uniform;            // step_frac * min_d h_d on a uniform grid
    unsigned h_hi[3];            // high words of the uniform spacings (in-cell test of the cell-table kernel)
    double step_frac, max_length, null_eps;
    long long max_steps;
    int method;
    int interleave;              // work item q -> (pos, dir): interleave ? (q >> 1, q & 1) : (q % n, q / n)
    long long n;                 // number of seeds
    const double *seeds;         // n*3, caller order
    const uint32_t *perm;        // sorted position -> seed index
    double *rec;                 // 2n per-direction records of REC_DOUBLES doubles, index = dir*n + pos
    unsigned long long *total_steps;
    unsigned long long *queue;   // work counter of the persistent kernel
    const double *basis;         // cell-table kernel, QSL_TRACE_LQ: n*6 (a^, b^) per seed in sorted order (seed_basis_kernel)
    unsigned tie_zero;           // cell-table kernel: always 0 (operand of the scheduling fence LineState2::tie)
};

// Per-direction record written once when a line ends: x[3], d1[3], d2[3], L, (nsteps, face|flags) as two uint32, lambda.
constexpr int REC_DOUBLES = 12;
constexpr uint32_t REC_STALL = 1u << 8, REC_CAP = 1u << 9, REC_SEED_OUTSIDE = 1u << 10, REC_NULL_AT_SEED = 1u << 11;
// Record flag of the cell-table and cell-frame kernels: the trial step from the recorded state leaves the trace box, the landing of
// reading A4 is still to be done (landing_kernel / landing3_kernel clear it).  Bits 8..11 are the status flags above.
constexpr uint32_t REC_LANDING = 1u << 12;

// ---------------------------------------------------------------------------------------------------------------
// The work queue of the persistent table kernels (trace2_kernel, trace_ck_kernel, trace3_kernel).  Work items (one
// direction of one line) are taken from the global counter by the WARP, up to CHUNK consecutive items of the Morton
// order at a time, and their seeds (and orthonormal pairs, DEV) are staged in shared memory by all lanes at once; a lane
// whose line has ended takes the next staged item with a few LDS instead of going through three dependent global round
// trips (counter -> permutation -> seed) while the other 31 lanes of its warp wait (profiles/r2d: 5 % of the issue
// cycles of cfg2).  The chunk shrinks with the work left (remaining / (4 x warps of the grid), at least the number of
// lanes waiting), so that at the end of a launch no warp sits on staged items other warps could be running; a small
// CHUNK keeps the lines in flight close together in the Morton order (cfg4: 47 GB of DRAM traffic with 8, 86 GB with 32).
//   start(x, bs, slot) -> bool   begins the line of a staged item in this lane (false: it ended at once)
//   advance() -> bool            one attempt of this lane's line (true: the line has left the kernel)
template <bool DEV, int THREADS, int CHUNK, class Start, class Advance>
__device__ __forceinline__ void staged_queue(const TraceArgs &A, Start start, Advance advance)
{
    constexpr int NP = DEV ? 9 : 3;
    __shared__ double pool_v[THREADS / 32][NP][32];
    __shared__ uint32_t pool_slot[THREADS / 32][32];
    const long long n_items = 2 * A.n;
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const long long n_warps = (long long)gridDim.x * (THREADS / 32);
    int pool_n = 0, pool_head = 0;              // warp-uniform
    long long left = n_items;                   // work left in the queue when this warp last looked
    bool have = false, drained = false;         // drained: warp-uniform
    while (true) {
        unsigned need = __ballot_sync(0xffffffffu, !have);
        while (need) {
            if (pool_n == 0) {
                if (drained) break;
                long long want = left / (4 * n_warps);
                want = max((long long)__popc(need), min(want, (long long)CHUNK));
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(A.queue, (unsigned long long)want);
                base = __shfl_sync(0xffffffffu, base, 0);
                left = n_items - (long long)base;
                const int got = left <= 0 ? 0 : (int)min(left, want);
                left -= got;
                if (got < (int)want) drained = true;
                if ((int)lane < got) {
                    const long long q = (long long)base + lane;
                    long long pos; int dir;
                    if (A.interleave) { pos = q >> 1; dir = (int)(q & 1); } else { dir = q >= A.n ? 1 : 0; pos = q - (long long)dir * A.n; }
                    const uint32_t si = A.perm[pos];
                    pool_slot[w][lane] = (uint32_t)((long long)dir * A.n + pos);
#pragma unroll
                    for (int c = 0; c < 3; ++c) pool_v[w][c][lane] = A.seeds[3 * (size_t)si + c];
                    if (DEV) {
                        const double2 *__restrict__ bp = reinterpret_cast<const double2 *>(A.basis + 6 * (size_t)pos);
                        const double2 b0 = bp[0], b1 = bp[1], b2 = bp[2];
                        pool_v[w][3 % NP][lane] = b0.x; pool_v[w][4 % NP][lane] = b0.y; pool_v[w][5 % NP][lane] = b1.x;
                        pool_v[w][6 % NP][lane] = b1.y; pool_v[w][7 % NP][lane] = b2.x; pool_v[w][8 % NP][lane] = b2.y;
                    }
                }
                __syncwarp();
                pool_n = got; pool_head = 0;
                if (got == 0) break;
            }
            const int rank = __popc(need & ((1u << lane) - 1u));
            if (!have && rank < pool_n) {
                const int e = pool_head + rank;
                const double x[3] = { pool_v[w][0][e], pool_v[w][1][e], pool_v[w][2][e] };
                double bs[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
                if (DEV) {
#pragma unroll
                    for (int c = 0; c < 6; ++c) bs[c] = pool_v[w][(3 + c) % NP][e];
                }
                have = start(x, bs, pool_slot[w][e]);
            }
            const int served = min(pool_n, __popc(need));
            pool_head += served; pool_n -= served;
            __syncwarp();
            need = __ballot_sync(0xffffffffu, !have);
        }
        if (!__any_sync(0xffffffffu, have)) break;
        if (have) {
            if (advance()) have = false;
        }
    }
}

template <typename S> struct Sample4;
template <> struct Sample4<float> { using type = float4; };
template <> struct Sample4<double> { using type = double4; };

// One gather per cell corner: LDG.128 for a float4 sample, one 256-bit LDG (sm_100) for a double4 sample.
__device__ __forceinline__ float4 load_sample(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ double4 load_sample(const double4 *p)
{
    double4 r;
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// ---------------------------------------------------------------------------------------------------------------
// Cell location (PAPER.md:93: "identify the cell within the input array within which x lies"; :97 h_c).
// Reading A8: index clamped to [0, n-2], fraction not clamped.
template <bool STRETCHED>
__device__ __forceinline__ void locate(const TraceArgs &A, int d, int n, double x, int &i, double &t, double &inv_h, double &hc)
{
    if (!STRETCHED) {
        const double u = (x - A.fv.lo[d]) * A.inv_h[d];
        int ii = (int)floor(u);                       // NaN converts to 0
        ii = max(0, min(ii, n - 2));
        i = ii;
        t = u - (double)ii;
        inv_h = A.inv_h[d];
        hc = A.fv.h[d];
    } else {
        const double *__restrict__ xs = A.fv.axis[d];
        int lo = 0, hi = n - 1;                       // largest i with xs[i] <= x, clamped to [0, n-2]
        if (x >= xs[n - 1]) lo = n - 2;
        else if (x >= xs[0]) {
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(xs + mid) <= x) lo = mid; else hi = mid; }
        }
        lo = min(lo, n - 2);
        const double x0 = __ldg(xs + lo), x1 = __ldg(xs + lo + 1);
        hc = x1 - x0;
        inv_h = 1.0 / hc;
        t = (x - x0) * inv_h;
        i = lo;
    }
}

// Trilinear value and analytic gradient of one component from its 8 corner samples:
// lerp along x, then y, then z; the differences formed on the way are the gradient numerators.
template <bool WITH_J>
__device__ __forceinline__ void trilinear(double c000, double c100, double c010, double c110, double c001, double c101,
                                          double c011, double c111, double tx, double ty, double tz, double &val,
                                          double &gx, double &gy, double &gz)
{
    const double dx00 = c100 - c000, dx10 = c110 - c010, dx01 = c101 - c001, dx11 = c111 - c011;
    const double v00 = fma(tx, dx00, c000), v10 = fma(tx, dx10, c010), v01 = fma(tx, dx01, c001), v11 = fma(tx, dx11, c011);
    const double dy0 = v10 - v00, dy1 = v11 - v01;
    const double v0 = fma(ty, dy0, v00), v1 = fma(ty, dy1, v01);
    const double dz = v1 - v0;
    val = fma(tz, dz, v0);
    if (WITH_J) {
        gz = dz;
        gy = fma(tz, dy1 - dy0, dy0);
        const double gx0 = fma(ty, dx10 - dx00, dx00), gx1 = fma(ty, dx11 - dx01, dx01);
        gx = fma(tz, gx1 - gx0, gx0);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Higher-order interpolation ("trilinear, triquadratic (Dodgson 1997) and tricubic
// (Keys 1981) ... 8, 27, or 64 vertices"; eq. (3): kernels f_v(x - x_c; h_c) in the units of the cell containing x;
// :123, :137: the gradient is taken analytically on the kernels).  Reading A18 of DESIGN.md:
//   ORDER 3  Keys' cubic convolution (a = -1/2) on the nodes i-1 .. i+2 of each axis, t = (x - x_i)/h_i; a node outside
//            the grid takes Keys' boundary value f_-1 = 3 f_0 - 3 f_1 + f_2 (mirrored at the upper end);
//   ORDER 2  Dodgson's interpolating quadratic (r = 1) on the node nearest to x (t >= 1/2 -> i + 1) and its two
//            neighbours, s = t - (j - i); outside the grid the linear extrapolation f_-1 = 2 f_0 - f_1.
// Per axis: node indices (clamped; a folded node has weight 0), weights and d weight / dx.
template <int ORDER>
__device__ __forceinline__ void axis_stencil(int n, int i, double t, double inv_h, int idx[ORDER + 1], double w[ORDER + 1],
                                             double dw[ORDER + 1])
{
    if (ORDER == 3) {
        const double t2 = t * t, t3 = t2 * t;
        w[0] = 0.5 * ((-t3 + 2.0 * t2) - t);        dw[0] = 0.5 * ((-3.0 * t2 + 4.0 * t) - 1.0);
        w[1] = 0.5 * ((3.0 * t3 - 5.0 * t2) + 2.0); dw[1] = 0.5 * (9.0 * t2 - 10.0 * t);
        w[2] = 0.5 * ((-3.0 * t3 + 4.0 * t2) + t);  dw[2] = 0.5 * ((-9.0 * t2 + 8.0 * t) + 1.0);
        w[ORDER] = 0.5 * (t3 - t2);                 dw[ORDER] = 0.5 * (3.0 * t2 - 2.0 * t);
#pragma unroll
        for (int k = 0; k <= ORDER; ++k) { idx[k] = i - 1 + k; dw[k] *= inv_h; }
        if (idx[0] < 0) {
            w[1] += 3.0 * w[0]; w[2] -= 3.0 * w[0]; w[ORDER] += w[0]; w[0] = 0.0;
            dw[1] += 3.0 * dw[0]; dw[2] -= 3.0 * dw[0]; dw[ORDER] += dw[0]; dw[0] = 0.0;
            idx[0] = 0;
        }
        if (idx[ORDER] > n - 1) {
            w[2] += 3.0 * w[ORDER]; w[1] -= 3.0 * w[ORDER]; w[0] += w[ORDER]; w[ORDER] = 0.0;
            dw[2] += 3.0 * dw[ORDER]; dw[1] -= 3.0 * dw[ORDER]; dw[0] += dw[ORDER]; dw[ORDER] = 0.0;
            idx[ORDER] = n - 1;
        }
    } else {
        const int up = t >= 0.5 ? 1 : 0;
        const int j = i + up;
        const double s = t - (double)up;
        w[0] = s * s - 0.5 * s;   dw[0] = (2.0 * s - 0.5) * inv_h;
        w[1] = 1.0 - 2.0 * s * s; dw[1] = (-4.0 * s) * inv_h;
        w[2] = s * s + 0.5 * s;   dw[2] = (2.0 * s + 0.5) * inv_h;
#pragma unroll
        for (int k = 0; k < 3; ++k) idx[k] = j - 1 + k;
        if (idx[0] < 0) {
            w[1] += 2.0 * w[0]; w[2] -= w[0]; w[0] = 0.0;
            dw[1] += 2.0 * dw[0]; dw[2] -= dw[0]; dw[0] = 0.0;
            idx[0] = 0;
        }
        if (idx[2] > n - 1) {
            w[1] += 2.0 * w[2]; w[0] -= w[2]; w[2] = 0.0;
            dw[1] += 2.0 * dw[2]; dw[0] -= dw[2]; dw[2] = 0.0;
            idx[2] = n - 1;
        }
    }
}

// Separable tensor-product sum over the (ORDER + 1)^3 stencil: x innermost (value and d/dx of every component), then y,
// then z.  val[4] = (v0, v1, v2, |B| sample), g[c*3 + d] = d v_c / d x_d.
template <typename S, bool STRETCHED, bool WITH_J, bool WITH_M, int ORDER>
__device__ __forceinline__ void interpolate_ho(const TraceArgs &A, const double x[3], double val[4], double g[9], double &hmin)
{
    using S4 = typename Sample4<S>::type;
    constexpr int NS = ORDER + 1;
    int i, j, k; double tx, ty, tz, ihx, ihy, ihz, hx, hy, hz;
    locate<STRETCHED>(A, 0, A.fv.nx, x[0], i, tx, ihx, hx);
    locate<STRETCHED>(A, 1, A.fv.ny, x[1], j, ty, ihy, hy);
    locate<STRETCHED>(A, 2, A.fv.nz, x[2], k, tz, ihz, hz);
    hmin = fmin(hx, fmin(hy, hz));
    int ix[NS], iy[NS], iz[NS];
    double wx[NS], dwx[NS], wy[NS], dwy[NS], wz[NS], dwz[NS];
    axis_stencil<ORDER>(A.fv.nx, i, tx, ihx, ix, wx, dwx);
    axis_stencil<ORDER>(A.fv.ny, j, ty, ihy, iy, wy, dwy);
    axis_stencil<ORDER>(A.fv.nz, k, tz, ihz, iz, wz, dwz);
    constexpr int NC = WITH_M ? 4 : 3;
#pragma unroll
    for (int q = 0; q < 4; ++q) val[q] = 0.0;
#pragma unroll
    for (int q = 0; q < 9; ++q) g[q] = 0.0;
    const S4 *__restrict__ base = (const S4 *)A.fv.samples;
#pragma unroll
    for (int c = 0; c < NS; ++c) {
        double vy[NC], gxy[3], gyy[3];          // sums over the (x, y) plane c: value, d/dx, d/dy
#pragma unroll
        for (int q = 0; q < NC; ++q) vy[q] = 0.0;
#pragma unroll
        for (int q = 0; q < 3; ++q) { gxy[q] = 0.0; gyy[q] = 0.0; }
#pragma unroll
        for (int b = 0; b < NS; ++b) {
            const S4 *__restrict__ row = base + ((size_t)iz[c] * A.fv.ny + iy[b]) * A.fv.nx;
            double vx[NC], gx[3];
#pragma unroll
            for (int q = 0; q < NC; ++q) vx[q] = 0.0;
#pragma unroll
            for (int q = 0; q < 3; ++q) gx[q] = 0.0;
#pragma unroll
            for (int a = 0; a < NS; ++a) {
                const S4 sm = load_sample(row + ix[a]);
                const double sv[4] = { (double)sm.x, (double)sm.y, (double)sm.z, (double)sm.w };
#pragma unroll
                for (int q = 0; q < NC; ++q) vx[q] = fma(wx[a], sv[q], vx[q]);
                if (WITH_J) {
#pragma unroll
                    for (int q = 0; q < 3; ++q) gx[q] = fma(dwx[a], sv[q], gx[q]);
                }
            }
#pragma unroll
            for (int q = 0; q < NC; ++q) vy[q] = fma(wy[b], vx[q], vy[q]);
            if (WITH_J) {
#pragma unroll
                for (int q = 0; q < 3; ++q) { gxy[q] = fma(wy[b], gx[q], gxy[q]); gyy[q] = fma(dwy[b], vx[q], gyy[q]); }
            }
        }
#pragma unroll
        for (int q = 0; q < NC; ++q) val[q] = fma(wz[c], vy[q], val[q]);
        if (WITH_J) {
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                g[q * 3 + 0] = fma(wz[c], gxy[q], g[q * 3 + 0]);
                g[q * 3 + 1] = fma(wz[c], gyy[q], g[q * 3 + 1]);
                g[q * 3 + 2] = fma(dwz[c], vy[q], g[q * 3 + 2]);
            }
        }
    }
}

// Evaluate(x) -> b[3], J[9] (J[c*3+d] = d b_c / d x_d), optionally m = |B| and the cell size (O1 of DESIGN.md).
template <typename S, bool STRETCHED, bool INTERP, bool WITH_J, bool WITH_M, int ORDER = 1>
__device__ __forceinline__ void evaluate(const TraceArgs &A, const double x[3], double b[3], double J[9], double &m, double &hmin)
{
    using S4 = typename Sample4<S>::type;
    if (ORDER != 1) {
        // paper mode only (NORMALIZE_FIRST): the interpolant of the pre-normalised samples is used as it is
        double val[4], gg[9];
        interpolate_ho<S, STRETCHED, WITH_J, WITH_M, ORDER == 1 ? 2 : ORDER>(A, x, val, gg, hmin);
#pragma unroll
        for (int c = 0; c < 3; ++c) b[c] = val[c];
        if (WITH_J) {
#pragma unroll
            for (int q = 0; q < 9; ++q) J[q] = gg[q];
        }
        m = val[3];
        return;
    }
    int i, j, k; double tx, ty, tz, ihx, ihy, ihz, hx, hy, hz;
    locate<STRETCHED>(A, 0, A.fv.nx, x[0], i, tx, ihx, hx);
    locate<STRETCHED>(A, 1, A.fv.ny, x[1], j, ty, ihy, hy);
    locate<STRETCHED>(A, 2, A.fv.nz, x[2], k, tz, ihz, hz);
    hmin = fmin(hx, fmin(hy, hz));
    const int nx = A.fv.nx, sxy = A.fv.nx * A.fv.ny;
    const S4 *__restrict__ p = (const S4 *)A.fv.samples + ((size_t)k * A.fv.ny + j) * nx + i;
    const S4 s000 = load_sample(p), s100 = load_sample(p + 1), s010 = load_sample(p + nx), s110 = load_sample(p + nx + 1);
    const S4 s001 = load_sample(p + sxy), s101 = load_sample(p + sxy + 1), s011 = load_sample(p + sxy + nx),
             s111 = load_sample(p + sxy + nx + 1);
    double v[3], g[9];
    trilinear<WITH_J>(s000.x, s100.x, s010.x, s110.x, s001.x, s101.x, s011.x, s111.x, tx, ty, tz, v[0], g[0], g[1], g[2]);
    trilinear<WITH_J>(s000.y, s100.y, s010.y, s110.y, s001.y, s101.y, s011.y, s111.y, tx, ty, tz, v[1], g[3], g[4], g[5]);
    trilinear<WITH_J>(s000.z, s100.z, s010.z, s110.z, s001.z, s101.z, s011.z, s111.z, tx, ty, tz, v[2], g[6], g[7], g[8]);
    if (WITH_J) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { g[c * 3 + 0] *= ihx; g[c * 3 + 1] *= ihy; g[c * 3 + 2] *= ihz; }
    }
    if (!INTERP) {
        // paper mode: the interpolant of the pre-normalised samples is used as is
#pragma unroll
        for (int c = 0; c < 3; ++c) b[c] = v[c];
        if (WITH_J) {
#pragma unroll
            for (int q = 0; q < 9; ++q) J[q] = g[q];
        }
        if (WITH_M) {
            double dummy0, dummy1, dummy2;
            trilinear<false>(s000.w, s100.w, s010.w, s110.w, s001.w, s101.w, s011.w, s111.w, tx, ty, tz, m, dummy0, dummy1, dummy2);
        }
    } else {
        // reading A2: interpolate B, then normalise: b = B/|B|, J = (G - u (u^T G))/|B|, m = |B|
        const double n2 = fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0]));
        const double nn = sqrt(n2);
        if (nn < 1e-300) {
#pragma unroll
            for (int c = 0; c < 3; ++c) b[c] = 0.0;
            if (WITH_J) {
#pragma unroll
                for (int q = 0; q < 9; ++q) J[q] = 0.0;
            }
            m = 0.0;
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
            m = nn;
        }
    }
}

__device__ __forceinline__ double norm3(const double v[3]) { return sqrt(fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0]))); }
__device__ __forceinline__ double dot3(const double a[3], const double b[3]) { return fma(a[2], b[2], fma(a[1], b[1], a[0] * b[0])); }

__device__ __forceinline__ bool inside_box(const TraceArgs &A, const double x[3])
{
    return x[0] >= A.box_lo[0] && x[0] <= A.box_hi[0] && x[1] >= A.box_lo[1] && x[1] <= A.box_hi[1] &&
           x[2] >= A.box_lo[2] && x[2] <= A.box_hi[2];
}

// ---------------------------------------------------------------------------------------------------------------
// One work item = one direction of one field line, advanced by a small state machine so that every lane of a warp
// runs the same code whatever its phase:
//   phase 0      trial RK step of size h; accepted if the trial point is inside the closed trace box
//   phase 1..3   landing (reading A4): step of size hp from the same state, then one Newton update of hp from the
//                field at the trial end (evaluated as a "5th stage" through the same evaluate call site)
//   phase 4      final step of size hp, snap onto the face, done
// NV = 9 with deviation vectors (QSL_TRACE_LQ), 3 without (QSL_TRACE_L): x and L are bit-identical in both modes.
// Spherical geometry (reading A19): axes (phi, theta, r) = (longitude, latitude, radius), components in
// the orthonormal basis.  PAPER.md:83-85 (eq. 2): r cos(theta) phi' = B^_phi, r theta' = B^_theta, r' = B^_r, and
// PAPER.md:125-135 (eq. 6, 7) for the coordinate deviations with the gradient acting on the kernels only: every
// coordinate rate is the orthonormal component times mf = (1/(r cos theta), 1/r, 1).
template <bool SPH>
__device__ __forceinline__ void metric(const double *u, double mf[3])
{
    if (SPH) { mf[0] = 1.0 / (u[2] * cos(u[1])); mf[1] = 1.0 / u[2]; mf[2] = 1.0; }
    else { mf[0] = 1.0; mf[1] = 1.0; mf[2] = 1.0; }
}

// The same metric factors without a call to cos() per evaluation point.  The cell-table kernel carries (sin, cos) of the
// latitude of the line's current point; a stage point's latitude differs from it by dt = O(step / r), so
// cos(theta + dt) = cos(theta) cos(dt) - sin(theta) sin(dt) with cos(dt), sin(dt) from their Taylor polynomials through
// dt^8 / dt^9 (truncation below 2^-64 for |dt| <= 1/16; anything larger falls back to sincos()).  1 / (r cos theta) is one
// hardware reciprocal seed + two Newton steps (within an ulp), and 1 / r = cos(theta) / (r cos(theta)).  The plain
// definition (reading A19: cos() and two divisions) differs by a few ulp of the metric factors, far below the parity gates.
__device__ __forceinline__ void sincos_small(double dt, double &s, double &c)
{
    const double t2 = dt * dt;
    c = fma(t2, fma(t2, fma(t2, fma(t2, 1.0 / 40320.0, -1.0 / 720.0), 1.0 / 24.0), -0.5), 1.0);
    s = dt * fma(t2, fma(t2, fma(t2, fma(t2, 1.0 / 362880.0, -1.0 / 5040.0), 1.0 / 120.0), -1.0 / 6.0), 1.0);
}
__device__ __forceinline__ double rcp_fast(double d)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    r = fma(r, fma(-d, r, 1.0), r);
    return fma(r, fma(-d, r, 1.0), r);
}
// (sin, cos) of theta0 + dt from (st0, ct0) = (sin, cos)(theta0)
__device__ __forceinline__ void sincos_shift(double st0, double ct0, double dt, double &s, double &c)
{
    if (fabs(dt) <= 0.0625) {
        double sd, cd;
        sincos_small(dt, sd, cd);
        s = fma(st0, cd, ct0 * sd);
        c = fma(ct0, cd, -(st0 * sd));
    } else {
        // far from the anchor (never on the path of a fixed-step line): exact functions of the sum of the two angles
        const double th = atan2(st0, ct0) + dt;
        sincos(th, &s, &c);
    }
}
__device__ __forceinline__ void metric_shift(double r, double st0, double ct0, double dt, double mf[3])
{
    double s, c;
    sincos_shift(st0, ct0, dt, s, c);
    const double q = rcp_fast(r * c);
    mf[0] = q; mf[1] = q * c; mf[2] = 1.0;
}

template <typename S, bool DEV, bool STRETCHED, bool INTERP, int ORDER = 1, bool SPH = false>
struct LineState {
    static constexpr int NV = DEV ? 9 : 3;
    double y[NV];        // x, delta1, delta2
    double L, lam, hp, bound;
    uint32_t nsteps;
    int phase, axis, face;
    double sgn;
    long long slot;      // record index dir*n + pos

    // Initialises from work item q.  Returns false if the item ended at once (seed outside / null at seed).
    __device__ bool init(const TraceArgs &A, long long q)
    {
        long long pos; int dir;
        if (A.interleave) { pos = q >> 1; dir = (int)(q & 1); } else { dir = q >= A.n ? 1 : 0; pos = q - (long long)dir * A.n; }
        slot = (long long)dir * A.n + pos;
        sgn = dir ? -1.0 : 1.0;
        const uint32_t si = A.perm[pos];
        double x[3] = { A.seeds[3 * (size_t)si], A.seeds[3 * (size_t)si + 1], A.seeds[3 * (size_t)si + 2] };
        L = 0.0; lam = 0.0; nsteps = 0; phase = 0; axis = 0; face = 255; hp = 0.0; bound = 0.0;
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = c < 3 ? x[c] : 0.0;
        if (!inside_box(A, x)) { finish(A, REC_SEED_OUTSIDE); return false; }
        double b[3], J[9], m, hmin;
        evaluate<S, STRETCHED, INTERP, false, false, ORDER>(A, x, b, J, m, hmin);
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
            double a[3] = { -u[0] * ue, -u[1] * ue, -u[2] * ue };
            if (e == 0) a[0] += 1.0; else if (e == 1) a[1] += 1.0; else a[2] += 1.0;
            const double ia = 1.0 / norm3(a);
            a[0] *= ia; a[1] *= ia; a[2] *= ia;
            y[3 % NV] = a[0]; y[4 % NV] = a[1]; y[5 % NV] = a[2];
            y[6 % NV] = u[1] * a[2] - u[2] * a[1];
            y[7 % NV] = u[2] * a[0] - u[0] * a[2];
            y[8 % NV] = u[0] * a[1] - u[1] * a[0];
            if (SPH) {
                // the pair is orthonormal in the orthonormal basis; the state carries coordinate deviations (eq. 8 inverted)
                double mf[3];
                metric<SPH>(x, mf);
#pragma unroll
                for (int c = 0; c < 3; ++c) { y[(3 + c) % NV] *= mf[c]; y[(6 + c) % NV] *= mf[c]; }
            }
        }
        return true;
    }

    __device__ void finish(const TraceArgs &A, uint32_t flags)
    {
        double *r = A.rec + (size_t)slot * REC_DOUBLES;
        double out[REC_DOUBLES] = {};
#pragma unroll
        for (int c = 0; c < 9; ++c) out[c] = c < NV ? y[c % NV] : 0.0;
        out[9] = L;
        const uint32_t w1 = (uint32_t)face | flags;
        out[10] = __hiloint2double((int)w1, (int)nsteps);
        out[11] = lam;
        double2 *r2 = reinterpret_cast<double2 *>(r);
#pragma unroll
        for (int c = 0; c < REC_DOUBLES / 2; ++c) r2[c] = make_double2(out[2 * c], out[2 * c + 1]);
    }

    // Advances the line by one attempt (one trial step, one landing iteration, or the final landing step).
    // Returns true when the line has ended (its record is written).
    __device__ bool advance(const TraceArgs &A)
    {
        double acc[NV], accL = 0.0, ys[NV], yn[NV], Ln = L;
        double hs = phase == 0 ? 0.0 : hp, h = 0.0;
        const int last = A.method == QSL_EULER ? 0 : 3;
#pragma unroll
        for (int c = 0; c < NV; ++c) { acc[c] = 0.0; ys[c] = y[c]; yn[c] = y[c]; }
#pragma unroll 1
        for (int st = 0;; ++st) {
            double b[3], J[9], m, hmin;
            evaluate<S, STRETCHED, INTERP, DEV, false, ORDER>(A, ys, b, J, m, hmin);
            const double bn = norm3(b);
            if (st == 0 && phase == 0) {
                // O4: stall / caps are tested on k1 before the step; h from the cell containing x
                if (!(bn >= A.null_eps)) { finish(A, REC_STALL); return true; }
                if ((long long)nsteps >= A.max_steps || lam >= A.max_length) { finish(A, REC_CAP); return true; }
                h = STRETCHED ? A.step_frac * hmin : A.h_uniform;
                if (SPH)   // physical cell edges (r cos(theta) h_phi, r h_theta, h_r) of the cell containing x (uniform axes)
                    h = A.step_frac * fmin(ys[2] * cos(ys[1]) * A.fv.h[0], fmin(ys[2] * A.fv.h[1], A.fv.h[2]));
                if (lam + h > A.max_length) h = A.max_length - lam;
                hs = h;
            }
            double mf[3];
            metric<SPH>(ys, mf);
            if (st > last) {
                // landing, "5th stage": b at the trial end -> one Newton update of hp (clamped to [0, h_full])
                const double bd = axis == 0 ? b[0] : (axis == 1 ? b[1] : b[2]);
                const double xd = axis == 0 ? yn[0] : (axis == 1 ? yn[1] : yn[2]);
                const double g = sgn * bd * (axis == 0 ? mf[0] : (axis == 1 ? mf[1] : mf[2])), r = xd - bound;
                if (g != 0.0) {
                    double hn = hp - r / g;
                    if (hn == hn) hp = fmin(fmax(hn, 0.0), hfull());
                }
                ++phase;
                return false;
            }
            // stage derivative k = (s b, s J d1, s J d2, |b|)  (PAPER.md:79 eq. 1, :119 eq. 5; reading A3 for L)
            double k[NV];
#pragma unroll
            for (int c = 0; c < 3; ++c) k[c] = SPH ? sgn * b[c] * mf[c] : sgn * b[c];
            if (DEV) {
#pragma unroll
                for (int v = 0; v < 2; ++v)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const double jd = fma(J[c * 3 + 2], ys[(3 + 3 * v + 2) % NV],
                                              fma(J[c * 3 + 1], ys[(3 + 3 * v + 1) % NV], J[c * 3] * ys[(3 + 3 * v) % NV]));
                        k[(3 + 3 * v + c) % NV] = SPH ? sgn * jd * mf[c] : sgn * jd;
                    }
            }
            const double w = (st == 0 || st == last) ? 1.0 : 2.0;
#pragma unroll
            for (int c = 0; c < NV; ++c) acc[c] = fma(w, k[c], acc[c]);
            accL = fma(w, bn, accL);
            if (st == last) {
                const double f = A.method == QSL_EULER ? hs : hs * (1.0 / 6.0);
#pragma unroll
                for (int c = 0; c < NV; ++c) yn[c] = fma(f, acc[c], y[c]);
                Ln = fma(f, accL, L);
                if (phase >= 1 && phase <= 3) {
#pragma unroll
                    for (int c = 0; c < NV; ++c) ys[c] = yn[c];
                    continue;
                }
                break;
            }
            const double ch = st == 2 ? hs : 0.5 * hs;
#pragma unroll
            for (int c = 0; c < NV; ++c) ys[c] = fma(ch, k[c], y[c]);
        }
        if (phase == 0) {
            if (inside_box(A, yn)) {
#pragma unroll
                for (int c = 0; c < NV; ++c) y[c] = yn[c];
                L = Ln; lam += h; ++nsteps;
                return false;
            }
            // first face crossed by the chord: smallest fraction, tie -> lowest axis (reading A4)
            double phi = INFINITY; int ax = -1, fc = 255; double bd = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (yn[d] < A.box_lo[d]) {
                    const double f = (A.box_lo[d] - y[d]) / (yn[d] - y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d; bd = A.box_lo[d]; }
                } else if (yn[d] > A.box_hi[d]) {
                    const double f = (A.box_hi[d] - y[d]) / (yn[d] - y[d]);
                    if (f < phi) { phi = f; ax = d; fc = 2 * d + 1; bd = A.box_hi[d]; }
                }
            }
            if (ax < 0) { finish(A, REC_STALL); return true; }   // non-finite trial point
            axis = ax; face_pending = fc; bound = bd; hp = phi * h; hfull_ = h; phase = 1;
            return false;
        }
        // phase 4: final landing step
#pragma unroll
        for (int c = 0; c < NV; ++c) y[c] = yn[c];
        if (axis == 0) y[0] = bound; else if (axis == 1) y[1] = bound; else y[2] = bound;
        L = Ln; lam += hp; ++nsteps; face = face_pending;
        finish(A, 0);
        return true;
    }

    int face_pending;
    double hfull_;
    __device__ __forceinline__ double hfull() const { return hfull_; }
};

// ---------------------------------------------------------------------------------------------------------------
// Kernels.  REFILL = false: one work item per thread (grid covers 2n items).  REFILL = true: persistent warps, a lane
// whose line ended pops the next item from a global counter (warp-aggregated atomic), so ragged line lengths do not
// idle lanes (north_star, "persistent trace kernel with a global work queue that refills lanes as lines terminate").
template <typename S, bool DEV, bool STRETCHED, bool INTERP, bool REFILL, int ORDER = 1, bool SPH = false>
__global__ void __launch_bounds__(128) trace_kernel(const TraceArgs A)
{
    LineState<S, DEV, STRETCHED, INTERP, ORDER, SPH> ls;
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
                else { have = ls.init(A, q); if (!have) my_steps += 0; }
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

// ---------------------------------------------------------------------------------------------------------------
// Epilogue: one thread per seed combines its forward and backward records.
struct EpilogueArgs {
    TraceArgs T;
    int with_dev;
    qsl_trace_out out;
};

struct EndProj { double a[3], b[3], m; };

template <typename S, bool STRETCHED, bool INTERP, int ORDER = 1, bool SPH = false>
__device__ void project_end(const TraceArgs &A, const double *r, int face, bool bnd, EndProj &E)
{
    // delta_perp = delta - B^(B^ . delta) with B^ re-normalised at the end point.
    // Reading A1 (bnd): slide along the field onto the end face instead, and weight by the normal field component.
    double b[3], J[9], m, hmin;
    evaluate<S, STRETCHED, INTERP, false, true, ORDER>(A, r, b, J, m, hmin);
    const double inv = 1.0 / norm3(b);
    const double u[3] = { b[0] * inv, b[1] * inv, b[2] * inv };
    double d1[3], d2[3];
    {   // PAPER.md:156 (eq. 8): delta x_phi = r cos(theta) delta phi, delta x_theta = r delta theta, delta x_r = delta r
        double mf[3];
        metric<SPH>(r, mf);
#pragma unroll
        for (int c = 0; c < 3; ++c) { d1[c] = SPH ? r[3 + c] / mf[c] : r[3 + c]; d2[c] = SPH ? r[6 + c] / mf[c] : r[6 + c]; }
    }
    double c1, c2;
    if (bnd && face != 255) {
        const int ax = face >> 1;
        const double un = ax == 0 ? u[0] : (ax == 1 ? u[1] : u[2]);
        c1 = (ax == 0 ? d1[0] : (ax == 1 ? d1[1] : d1[2])) / un;
        c2 = (ax == 0 ? d2[0] : (ax == 1 ? d2[1] : d2[2])) / un;
        E.m = m * fabs(un);
    } else {
        c1 = dot3(u, d1); c2 = dot3(u, d2);
        E.m = m;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) { E.a[c] = d1[c] - u[c] * c1; E.b[c] = d2[c] - u[c] * c2; }
}

__device__ __forceinline__ double q_eq11(const EndProj &F, const EndProj &B, double m0)
{
    // PAPER.md:174 (eq. 11): Q = B_F B_B / B_0^2 [ a_F^2 b_B^2 + a_B^2 b_F^2 - 2 (a_B . b_B)(a_F . b_F) ]
    const double aF2 = dot3(F.a, F.a), bF2 = dot3(F.b, F.b), aB2 = dot3(B.a, B.a), bB2 = dot3(B.b, B.b);
    const double abF = dot3(F.a, F.b), abB = dot3(B.a, B.b);
    return (F.m * B.m) / (m0 * m0) * ((aF2 * bB2 + aB2 * bF2) - 2.0 * (abB * abF));
}

template <typename S, bool STRETCHED, bool INTERP, int ORDER = 1, bool SPH = false>
__global__ void __launch_bounds__(128) epilogue_kernel(const EpilogueArgs E)
{
    const TraceArgs &A = E.T;
    const long long pos = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= A.n) return;
    const size_t si = A.perm[pos];
    double rf[REC_DOUBLES], rb[REC_DOUBLES];
    {
        const double2 *pf = reinterpret_cast<const double2 *>(A.rec + (size_t)pos * REC_DOUBLES);
        const double2 *pb = reinterpret_cast<const double2 *>(A.rec + (size_t)(A.n + pos) * REC_DOUBLES);
#pragma unroll
        for (int c = 0; c < REC_DOUBLES / 2; ++c) {
            const double2 a = pf[c], b = pb[c];
            rf[2 * c] = a.x; rf[2 * c + 1] = a.y; rb[2 * c] = b.x; rb[2 * c + 1] = b.y;
        }
    }
    const uint32_t wf = (uint32_t)__double2hiint(rf[10]), wb = (uint32_t)__double2hiint(rb[10]);
    const uint32_t nsf = (uint32_t)__double2loint(rf[10]), nsb = (uint32_t)__double2loint(rb[10]);
    int ff = (int)(wf & 255u), fb = (int)(wb & 255u);
    uint32_t st = 0;
    if (wf & REC_SEED_OUTSIDE) st |= QSL_ST_SEED_OUTSIDE;
    if (wf & REC_NULL_AT_SEED) st |= QSL_ST_NULL_AT_SEED;
    const qsl_trace_out &O = E.out;
    const double qnan = __longlong_as_double(0x7ff8000000000000ll);
    if (st) {
        for (int c = 0; c < 3; ++c) { if (O.end_f) O.end_f[3 * si + c] = qnan; if (O.end_b) O.end_b[3 * si + c] = qnan; }
        if (O.L) O.L[si] = qnan;
        if (O.q_perp) O.q_perp[si] = qnan;
        if (O.q_bnd) O.q_bnd[si] = qnan;
        if (O.face_f) O.face_f[si] = 255;
        if (O.face_b) O.face_b[si] = 255;
        if (O.nsteps_f) O.nsteps_f[si] = 0;
        if (O.nsteps_b) O.nsteps_b[si] = 0;
        if (O.dev_f) for (int c = 0; c < 6; ++c) O.dev_f[6 * si + c] = qnan;
        if (O.dev_b) for (int c = 0; c < 6; ++c) O.dev_b[6 * si + c] = qnan;
        if (O.status) O.status[si] = st;
        return;
    }
    if (wf & REC_STALL) st |= QSL_ST_STALL_F;
    if (wb & REC_STALL) st |= QSL_ST_STALL_B;
    if (wf & REC_CAP) st |= QSL_ST_CAP_F;
    if (wb & REC_CAP) st |= QSL_ST_CAP_B;
    if ((ff != 255 && ff != 4) || (fb != 255 && fb != 4)) st |= QSL_ST_OPEN;
    for (int c = 0; c < 3; ++c) { if (O.end_f) O.end_f[3 * si + c] = rf[c]; if (O.end_b) O.end_b[3 * si + c] = rb[c]; }
    if (O.L) O.L[si] = rf[9] + rb[9];
    if (O.face_f) O.face_f[si] = (unsigned char)ff;
    if (O.face_b) O.face_b[si] = (unsigned char)fb;
    if (O.nsteps_f) O.nsteps_f[si] = nsf;
    if (O.nsteps_b) O.nsteps_b[si] = nsb;
    if (O.status) O.status[si] = st;
    if (!E.with_dev) {
        if (O.q_perp) O.q_perp[si] = qnan;
        if (O.q_bnd) O.q_bnd[si] = qnan;
        if (O.dev_f) for (int c = 0; c < 6; ++c) O.dev_f[6 * si + c] = qnan;
        if (O.dev_b) for (int c = 0; c < 6; ++c) O.dev_b[6 * si + c] = qnan;
        return;
    }
    if (O.dev_f) for (int c = 0; c < 6; ++c) O.dev_f[6 * si + c] = rf[3 + c];
    if (O.dev_b) for (int c = 0; c < 6; ++c) O.dev_b[6 * si + c] = rb[3 + c];
    if (O.q_perp || O.q_bnd) {
        // B_0 = |B| at the seed
        const double x0[3] = { A.seeds[3 * si], A.seeds[3 * si + 1], A.seeds[3 * si + 2] };
        double b0[3], J[9], m0, hmin;
        evaluate<S, STRETCHED, INTERP, false, true, ORDER>(A, x0, b0, J, m0, hmin);
        EndProj PF, PB;
        if (O.q_perp) {
            project_end<S, STRETCHED, INTERP, ORDER, SPH>(A, rf, ff, false, PF);
            project_end<S, STRETCHED, INTERP, ORDER, SPH>(A, rb, fb, false, PB);
            O.q_perp[si] = q_eq11(PF, PB, m0);
        }
        if (O.q_bnd) {
            project_end<S, STRETCHED, INTERP, ORDER, SPH>(A, rf, ff, true, PF);
            project_end<S, STRETCHED, INTERP, ORDER, SPH>(A, rb, fb, true, PB);
            O.q_bnd[si] = q_eq11(PF, PB, m0);
        }
    }
}

}  // namespace qsl
