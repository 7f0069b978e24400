// FLEDGE maps.  PAPER.md:190: "the gradient magnitude from the Sobel operator (i.e. a 2D or 3D
// gradient of FLL convolved with a simple smoothing function) applied to a 2D or 3D map of the length of field lines".
// Reading A10: un-normalised weights, difference [-1,0,+1] along the axis, smoothing [1,2,1] along the others, edges
// replicated.  The stencil is separable: every lane folds the other axes of its own column in registers, then the
// axis-0 taps are exchanged between neighbouring lanes with warp shuffles (no shared memory).
#include <math.h>

#include "qsl_internal.cuh"

namespace qsl {

constexpr int FL_THREADS = 128;
constexpr int FL_VALID = 30;   // outputs per warp: lanes 1..30; lanes 0 and 31 carry the halo columns

constexpr int FL_ROWS = 32;    // rows (axis 1) one warp marches over, keeping a rolling window of three rows in registers

// Folds the axis-1 / axis-2 taps of one column.  a[o2][o1] are the clamped neighbours of the column.
// A: smooth x smooth, B: diff along axis 1 (smooth along 2), C: diff along axis 2 (smooth along 1).
// (used by the sparse levels, where every neighbour is a look-up)
template <int NDIM>
__device__ __forceinline__ void fold_column(const double a[3][3], double &A, double &B, double &C)
{
    if (NDIM == 2) {
        A = (a[0][0] + a[0][2]) + 2.0 * a[0][1];
        B = a[0][2] - a[0][0];
        C = 0.0;
    } else {
        double s1[3], d1[3];
#pragma unroll
        for (int o2 = 0; o2 < 3; ++o2) {
            s1[o2] = (a[o2][0] + a[o2][2]) + 2.0 * a[o2][1];
            d1[o2] = a[o2][2] - a[o2][0];
        }
        A = (s1[0] + s1[2]) + 2.0 * s1[1];
        B = (d1[0] + d1[2]) + 2.0 * d1[1];
        C = s1[2] - s1[0];
    }
}

// Axis-0 taps across lanes: G0 = A(i+1) - A(i-1), G1 = B(i-1) + 2 B(i) + B(i+1), G2 likewise from C.
template <int NDIM>
__device__ __forceinline__ double combine_lanes(double A, double B, double C)
{
    const unsigned full = 0xffffffffu;
    const double Am = __shfl_up_sync(full, A, 1), Ap = __shfl_down_sync(full, A, 1);
    const double Bm = __shfl_up_sync(full, B, 1), Bp = __shfl_down_sync(full, B, 1);
    const double G0 = Ap - Am, G1 = (Bm + Bp) + 2.0 * B;
    double ss = fma(G1, G1, G0 * G0);
    if (NDIM == 3) {
        const double Cm = __shfl_up_sync(full, C, 1), Cp = __shfl_down_sync(full, C, 1);
        const double G2 = (Cm + Cp) + 2.0 * C;
        ss = fma(G2, G2, ss);
    }
    return sqrt(ss);
}

// One row of one column: the axis-2 taps folded (3-D), or the value itself (2-D).  P: [1,2,1] along axis 2, D: [-1,0,1]
// along axis 2, cen: the value at the row itself.
template <int NDIM>
__device__ __forceinline__ void load_row(const double *__restrict__ L, long long d0, long long d1, long long d2, long long cc,
                                         long long y, long long c2, double &P, double &D, double &cen)
{
    if (NDIM == 2) {
        cen = __ldg(L + y * d0 + cc);
        P = cen; D = 0.0;
    } else {
        const long long zm = max(c2 - 1, 0ll), zp = min(c2 + 1, d2 - 1);
        const double lm = __ldg(L + (zm * d1 + y) * d0 + cc), lp = __ldg(L + (zp * d1 + y) * d0 + cc);
        cen = __ldg(L + (c2 * d1 + y) * d0 + cc);
        P = (lm + lp) + 2.0 * cen;
        D = lp - lm;
    }
}

// Dense map.  A warp owns a strip of FL_VALID columns (axis 0; lanes 0 and 31 carry the halo columns) of one axis-2 plane
// and marches over FL_ROWS rows of axis 1 with the folded rows y-1, y, y+1 in registers: every value is loaded once per
// strip and plane it contributes to (3 loads per output in 3-D, 1 in 2-D, + the halo) instead of 9 / 3.
template <int NDIM>
__global__ void __launch_bounds__(FL_THREADS) fledge_dense_kernel(long long d0, long long d1, long long d2,
                                                                  const double *__restrict__ L, double *__restrict__ S)
{
    const unsigned lane = threadIdx.x & 31u;
    const long long strips = (d0 + FL_VALID - 1) / FL_VALID;
    const long long bands = (d1 + FL_ROWS - 1) / FL_ROWS;
    const long long tasks = strips * bands * d2;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long t = (((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5); t < tasks; t += warps) {
        const long long strip = t % strips, rest = t / strips;
        const long long band = rest % bands, c2 = rest / bands;
        const long long col = strip * FL_VALID - 1 + lane;               // lane 0 / 31 = halo
        const long long cc = min(max(col, 0ll), d0 - 1);                 // edge replication
        const long long y0 = band * FL_ROWS, y1 = min(y0 + FL_ROWS, d1);
        double P0, D0, c0, P1, D1, c1, P2, D2, cn;
        load_row<NDIM>(L, d0, d1, d2, cc, max(y0 - 1, 0ll), c2, P0, D0, c0);
        load_row<NDIM>(L, d0, d1, d2, cc, y0, c2, P1, D1, c1);
        for (long long y = y0; y < y1; ++y) {
            load_row<NDIM>(L, d0, d1, d2, cc, min(y + 1, d1 - 1), c2, P2, D2, cn);
            const double A = (P0 + P2) + 2.0 * P1, B = P2 - P0, C = (D0 + D2) + 2.0 * D1;
            double s = combine_lanes<NDIM>(A, B, C);
            // the centre tap has weight 0 in every G_d; O6 still lets a non-finite L anywhere in the stencil poison S
            if (!isfinite(c1)) s = __longlong_as_double(0x7ff8000000000000ll);
            if (lane >= 1 && lane <= FL_VALID && col < d0) S[(c2 * d1 + y) * d0 + col] = s;
            P0 = P1; D0 = D1; P1 = P2; D1 = D2; c1 = cn;
        }
    }
}

// Dense 2-D map, the kernel qsl_fledge_dense launches for ndim = 2.  Same strips of FL_VALID columns and the same
// arithmetic (and bits) as fledge_dense_kernel<2>; what differs is the shape of the march (profiles/r2g: the kernel above
// has one load in flight per warp and row, 13.7 of its 19 stall cycles per issue are long_scoreboard): one warp per CTA, so
// that task index and bounds are provably warp-uniform (no WARPSYNC pair around the shuffles, loop control on the uniform
// datapath), 32-bit index arithmetic with one moving pointer, and the rows taken FL2_GROUP at a time - their loads are all
// requested before the first of them is used.
#ifndef QSL_FL2_ROWS
#define QSL_FL2_ROWS 64
#endif
#ifndef QSL_FL2_GROUP
#define QSL_FL2_GROUP 8
#endif
constexpr int FL2_ROWS = QSL_FL2_ROWS, FL2_GROUP = QSL_FL2_GROUP;
__global__ void __launch_bounds__(32, 32) fledge_dense2_kernel(int d0, int d1, int rows, const double *__restrict__ L,
                                                              double *__restrict__ S)
{
    constexpr int G = FL2_GROUP;
    const int lane = threadIdx.x;
    const int strips = (d0 + FL_VALID - 1) / FL_VALID;
    const int bands = (d1 + rows - 1) / rows;                            // rows: rows per band, a multiple of G
    const long long tasks = (long long)strips * bands;
    for (long long t = blockIdx.x; t < tasks; t += gridDim.x) {
        const int strip = (int)(t % strips), band = (int)(t / strips);
        const int col = strip * FL_VALID - 1 + lane;                     // lane 0 / 31 = halo
        const int cc = min(max(col, 0), d0 - 1);                         // edge replication
        const int y0 = band * rows, y1 = min(y0 + rows, d1);
        const bool mine = lane >= 1 && lane <= FL_VALID && col < d0;
        const double *__restrict__ q = L + (long long)y0 * d0 + cc;      // row y of the lane's column
        double *__restrict__ so = S + (long long)y0 * d0 + col;
        double w[G + 2];                                                 // rows y - 1, y, y + 1 .. y + G
        w[0] = __ldg(y0 > 0 ? q - d0 : q);
        w[1] = __ldg(q);
        for (int y = y0; y < y1; y += G) {
#pragma unroll
            for (int k = 0; k < G; ++k) {                                // row y + k + 1, clamped to the last row
                q += y + k + 1 < d1 ? d0 : 0;
                w[k + 2] = __ldg(q);
            }
#pragma unroll
            for (int k = 0; k < G; ++k) {
                const double A = (w[k] + w[k + 2]) + 2.0 * w[k + 1], B = w[k + 2] - w[k];
                double s = combine_lanes<2>(A, B, 0.0);
                if (!isfinite(w[k + 1])) s = __longlong_as_double(0x7ff8000000000000ll);
                if (mine && y + k < y1) so[(long long)k * d0] = s;
            }
            so += (long long)G * d0;
            w[0] = w[G]; w[1] = w[G + 1];
        }
    }
}

// Dense 3-D map, each value loaded once (+ halo): a warp owns a strip of FL_VALID columns x a band of FL3_ROWS rows and
// marches along axis 2 over a chunk of FL3_PLANES planes, holding the raw values of its column for the rows of the band
// (+ one halo row on either side) of the planes z-1, z, z+1 in registers.  Per plane step: FL3_ROWS + 2 loads per lane
// for FL3_ROWS outputs instead of 3 per output.  Measured on a 512 x 512 x 256 map, 128-thread CTAs with 64-bit index
// arithmetic: 8 rows (168 registers) 0.48 ms, 4 rows at 5 CTAs / SM 0.46 ms, 2 rows at 8 CTAs / SM (64 registers) 0.40 ms,
// the row-marching kernel 0.45 ms: the kernel wants resident warps more than it wants fewer loads (the repeated loads hit
// L2).  The form below (2 rows, single-warp CTAs, 32-bit indices, moving pointers, rotating windows): 0.294 ms = 0.56 of
// the copy rate (profiles/r2g).  The folds are taken in the order of the kernel above (axis 2, then axis 1, then axis 0
// across lanes), so both give the same bits.
#ifndef QSL_FL3_ROWS
#define QSL_FL3_ROWS 2
#endif
#ifndef QSL_FL3_MINB
#define QSL_FL3_MINB 32
#endif
constexpr int FL3_ROWS = QSL_FL3_ROWS;
constexpr int FL3_PLANES = 64;
__global__ void __launch_bounds__(32, QSL_FL3_MINB) fledge_dense3_kernel(int d0, int d1, int d2,
                                                                   const double *__restrict__ L, double *__restrict__ S)
{
    // One warp per CTA: the task index then depends on blockIdx alone and the compiler sees that the march is
    // warp-uniform (task loop and bounds on the uniform datapath, no WARPSYNC / ENDCOLLECTIVE pair around every shuffle).
    // All per-task index arithmetic in 32 bits (the launcher checks that a plane has fewer than 2^31 values); inside the
    // march only pointers move, by one plane per step, and the three plane windows rotate by name (three steps per
    // trip) instead of being copied: the first version spent 55 % of its instructions on 64-bit index arithmetic, the
    // bounds tests of the rows, register moves and spills (profiles/r2g).
    constexpr int R = FL3_ROWS;
    const int lane = threadIdx.x;
    const int strips = (d0 + FL_VALID - 1) / FL_VALID;
    const int bands = (d1 + R - 1) / R;
    const int chunks = (d2 + FL3_PLANES - 1) / FL3_PLANES;
    const long long tasks = (long long)strips * bands * chunks;
    const long long plane = (long long)d1 * d0;
    for (long long t = blockIdx.x; t < tasks; t += gridDim.x) {
        const int strip = (int)(t % strips);
        const int rest = (int)(t / strips);
        const int band = rest % bands, chunk = rest / bands;
        const int col = strip * FL_VALID - 1 + lane;                     // lane 0 / 31 = halo
        const int cc = min(max(col, 0), d0 - 1);                         // edge replication
        const int y0 = band * R, z0 = chunk * FL3_PLANES, z1 = min(z0 + FL3_PLANES, d2);
        const double *__restrict__ row[R + 2];                           // the (clamped) rows of the plane loaded last
        double vm[R + 2], vc[R + 2], vp[R + 2];
        {
            const double *__restrict__ pm = L + (long long)max(z0 - 1, 0) * plane + cc;
            const long long up = z0 > 0 ? plane : 0;                     // plane z0 - 1 -> plane z0
#pragma unroll
            for (int r = 0; r < R + 2; ++r) {
                const double *__restrict__ q = pm + (long long)min(max(y0 - 1 + r, 0), d1 - 1) * d0;
                vm[r] = __ldg(q); vc[r] = __ldg(q + up);
                row[r] = q + up;
            }
        }
        const bool mine = lane >= 1 && lane <= FL_VALID && col < d0;
        double *__restrict__ so = S + (long long)z0 * plane + (long long)y0 * d0 + col;
        // one plane step: a = plane z - 1, b = plane z, c <- plane z + 1
        auto plane_step = [&](int z, const double *a, const double *b, double *c) {
            const long long step = z + 1 < d2 ? plane : 0;               // the plane above the last one is the last one
#pragma unroll
            for (int r = 0; r < R + 2; ++r) { row[r] += step; c[r] = __ldg(row[r]); }
            double P[R + 2], D[R + 2];
#pragma unroll
            for (int r = 0; r < R + 2; ++r) { P[r] = (a[r] + c[r]) + 2.0 * b[r]; D[r] = c[r] - a[r]; }
#pragma unroll
            for (int r = 1; r <= R; ++r) {
                const double A = (P[r - 1] + P[r + 1]) + 2.0 * P[r], B = P[r + 1] - P[r - 1], C = (D[r - 1] + D[r + 1]) + 2.0 * D[r];
                double s = combine_lanes<3>(A, B, C);
                if (!isfinite(b[r])) s = __longlong_as_double(0x7ff8000000000000ll);
                if (mine && y0 + r - 1 < d1) so[(long long)(r - 1) * d0] = s;
            }
            so += plane;
        };
        int z = z0;
        for (; z + 3 <= z1; z += 3) {
            plane_step(z, vm, vc, vp);
            plane_step(z + 1, vc, vp, vm);
            plane_step(z + 2, vp, vm, vc);
        }
        if (z < z1) {
            plane_step(z, vm, vc, vp);
            if (z + 1 < z1) plane_step(z + 1, vc, vp, vm);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Sparse levels: the same stencil on the virtual lattice n_d 2^level; a neighbour that was not refined takes the L
// of its nearest existing ancestor.  Cells are found by walking down from the dense level 0 through the child_base
// links written by qsl_refine (child_base[l][i] = index at level l+1 of the first child of cell i, or -1).
constexpr int MAX_LEVELS = 16;
struct SparseArgs {
    int ndim, level;
    long long n0[3];
    long long count;
    const uint32_t *coords;                 // cells of `level`
    const double *L[MAX_LEVELS];            // L[0] = dense level 0
    const long long *child_base[MAX_LEVELS];
    double *S;
};

// One thread per cell of `level`.  The 27 (9) neighbours of a cell have at most two distinct ancestors per axis at every
// coarser level (c - 1 and c + 1 shifted down; c's own ancestor is one of them), so only 2^NDIM walks go down the
// child_base links to level - 1 instead of 27 (9); the neighbours then read their L through the child_base of their
// parent's slot, or take the L of the ancestor at which that slot's walk ended (not refined further).
template <int NDIM>
__global__ void __launch_bounds__(FL_THREADS) fledge_sparse_kernel(const SparseArgs A)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.count) return;
    const int lev = A.level;
    constexpr int NS = 1 << NDIM;
    long long nb[3][3];                              // clamped neighbour coordinates per axis
    long long par[3][2];                             // their two candidate parents (level lev - 1)
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const long long dim = d < NDIM ? A.n0[d] << lev : 1;
        const long long c = d < NDIM ? (long long)A.coords[i * NDIM + d] : 0;
#pragma unroll
        for (int o = 0; o < 3; ++o) nb[d][o] = min(max(c + o - 1, 0ll), dim - 1);
        par[d][0] = nb[d][0] >> 1; par[d][1] = nb[d][2] >> 1;
    }
    long long slot_base[NS];                         // index at level lev of the first child of the slot's cell, or -1
    double slot_val[NS];                             // L of the ancestor the slot's walk ended at (slot_base < 0)
#pragma unroll
    for (int sl = 0; sl < NS; ++sl) {
        const long long q0 = par[0][sl & 1], q1 = par[1][(sl >> 1) & 1], q2 = NDIM == 3 ? par[2][(sl >> 2) & 1] : 0;
        const int top = lev - 1;                      // level of (q0, q1, q2)
        long long idx = ((NDIM == 3 ? (q2 >> top) : 0) * A.n0[1] + (q1 >> top)) * A.n0[0] + (q0 >> top);
        long long base = 0; double val = 0.0; bool ended = false;
        for (int l = 1; l <= top; ++l) {
            base = __ldg(A.child_base[l - 1] + idx);
            if (base < 0) { val = __ldg(A.L[l - 1] + idx); ended = true; break; }
            const int sh = top - l;
            int bits = (int)((q0 >> sh) & 1) | ((int)((q1 >> sh) & 1) << 1);
            if (NDIM == 3) bits |= (int)((q2 >> sh) & 1) << 2;
            idx = base + bits;
        }
        if (!ended) {
            base = __ldg(A.child_base[top] + idx);
            if (base < 0) { val = __ldg(A.L[top] + idx); ended = true; }
        }
        slot_base[sl] = ended ? -1 : base;
        slot_val[sl] = val;
    }
    double As[3], Bs[3], Cs[3], centre = 0.0;
#pragma unroll
    for (int o0 = 0; o0 < 3; ++o0) {
        double a[3][3];
#pragma unroll
        for (int o2 = 0; o2 < (NDIM == 3 ? 3 : 1); ++o2) {
#pragma unroll
            for (int o1 = 0; o1 < 3; ++o1) {
                const long long x = nb[0][o0], y = nb[1][o1], z = NDIM == 3 ? nb[2][o2] : 0;
                int sl = ((x >> 1) != par[0][0] ? 1 : 0) | ((y >> 1) != par[1][0] ? 2 : 0);
                int bits = (int)(x & 1) | ((int)(y & 1) << 1);
                if (NDIM == 3) { sl |= (z >> 1) != par[2][0] ? 4 : 0; bits |= (int)(z & 1) << 2; }
                const long long base = slot_base[sl];
                a[o2][o1] = base < 0 ? slot_val[sl] : __ldg(A.L[lev] + base + bits);
            }
        }
        fold_column<NDIM>(a, As[o0], Bs[o0], Cs[o0]);
        if (o0 == 1) centre = a[NDIM == 3 ? 1 : 0][1];
    }
    const double G0 = As[2] - As[0], G1 = (Bs[0] + Bs[2]) + 2.0 * Bs[1];
    double ss = fma(G1, G1, G0 * G0);
    if (NDIM == 3) {
        const double G2 = (Cs[0] + Cs[2]) + 2.0 * Cs[1];
        ss = fma(G2, G2, ss);
    }
    A.S[i] = isfinite(centre) ? sqrt(ss) : __longlong_as_double(0x7ff8000000000000ll);
}

}  // namespace qsl

using namespace qsl;

extern "C" int qsl_fledge_dense(int ndim, const long long dims[3], const double *L, double *S, void *stream)
{
    if ((ndim != 2 && ndim != 3) || !dims || !L || !S) return QSL_EINVAL;
    const long long d0 = dims[0], d1 = dims[1], d2 = ndim == 3 ? dims[2] : 1;
    if (d0 < 1 || d1 < 1 || d2 < 1) return QSL_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const long long strips = (d0 + FL_VALID - 1) / FL_VALID;
    const long long tasks = strips * ((d1 + FL_ROWS - 1) / FL_ROWS) * d2;
    const int wpb = FL_THREADS / 32;
    long long blocks = (tasks + wpb - 1) / wpb;
    const long long cap = (long long)sm_count() * 32;      // a multiple of the SM count; warps stride over the tasks
    if (blocks > cap) blocks = cap;
    count_launch();
    if (ndim == 2 && d0 < (1ll << 31) - 64 && d1 < (1ll << 31) - 64) {
        // rows per band: FL2_ROWS on a large map; fewer (a multiple of the group, at least two groups) on a map too small
        // to give every SM its 32 single-warp CTAs otherwise
        long long rows = FL2_ROWS;
        const long long want = (long long)sm_count() * 32;
        while (rows > 2 * FL2_GROUP && strips * ((d1 + rows - 1) / rows) < want) rows >>= 1;
        const long long tasks2 = strips * ((d1 + rows - 1) / rows), cap2 = want * 8;
        fledge_dense2_kernel<<<(unsigned)(tasks2 < cap2 ? tasks2 : cap2), 32, 0, s>>>((int)d0, (int)d1, (int)rows, L, S);
    } else if (ndim == 2) fledge_dense_kernel<2><<<(unsigned)blocks, FL_THREADS, 0, s>>>(d0, d1, d2, L, S);
    else if (d2 >= 8 && d0 * d1 < (1ll << 31) && d2 < (1ll << 31)) {
        // deep enough along axis 2 for the plane-marching kernel to amortise its two halo planes
        const long long tasks3 = strips * ((d1 + FL3_ROWS - 1) / FL3_ROWS) * ((d2 + FL3_PLANES - 1) / FL3_PLANES);
        const long long cap3 = (long long)sm_count() * QSL_FL3_MINB * 8;   // single-warp CTAs, a few waves of them
        fledge_dense3_kernel<<<(unsigned)(tasks3 < cap3 ? tasks3 : cap3), 32, 0, s>>>((int)d0, (int)d1, (int)d2, L, S);
    } else fledge_dense_kernel<3><<<(unsigned)blocks, FL_THREADS, 0, s>>>(d0, d1, d2, L, S);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

extern "C" int qsl_fledge_sparse(const qsl_levels *lv, int level, double *S, void *stream)
{
    if (!lv || !lv->lat || !S || level < 1 || level >= MAX_LEVELS || lv->nlevels < level + 1) return QSL_EINVAL;
    if (!lv->L0 || !lv->count || !lv->coords || !lv->L || !lv->child_base) return QSL_EINVAL;
    const int ndim = lv->lat->ndim;
    if (ndim != 2 && ndim != 3) return QSL_EINVAL;
    SparseArgs A;
    A.ndim = ndim; A.level = level;
    for (int d = 0; d < 3; ++d) A.n0[d] = d < ndim ? lv->lat->n[d] : 1;
    for (int d = 0; d < ndim; ++d)
        if (A.n0[d] < 1 || (A.n0[d] << level) > 0xffffffffll) return QSL_ERANGE;
    A.count = lv->count[level];
    if (A.count < 0) return QSL_EINVAL;
    if (A.count == 0) return QSL_OK;
    A.coords = lv->coords[level];
    A.L[0] = lv->L0;
    for (int l = 1; l <= level; ++l) { A.L[l] = lv->L[l]; if (!A.L[l]) return QSL_EINVAL; }
    for (int l = 0; l < level; ++l) { A.child_base[l] = lv->child_base[l]; if (!A.child_base[l]) return QSL_EINVAL; }
    if (!A.coords) return QSL_EINVAL;
    A.S = S;
    cudaStream_t s = (cudaStream_t)stream;
    const long long blocks = (A.count + FL_THREADS - 1) / FL_THREADS;
    count_launch();
    if (ndim == 2) fledge_sparse_kernel<2><<<(unsigned)blocks, FL_THREADS, 0, s>>>(A);
    else fledge_sparse_kernel<3><<<(unsigned)blocks, FL_THREADS, 0, s>>>(A);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}
