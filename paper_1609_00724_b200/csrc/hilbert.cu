// The paper's own adaptive refinement (section 3.6) as device kernels: samples
// ordered along a Hilbert curve, a new sample "halfway along the Hilbert curve" between two successive samples whose
// field-line lengths differ by more than a threshold, the pass on a shifted curve and
// the converter back to a rectilinear array (max Q per cell, log Q interpolated along the curve into empty cells,
// PAPER.md:202).  The paper does this on the host (~50 lines of C++); here only the per-pass count of new
// samples reaches the host.  Readings H0-H4: DESIGN.md A17.
//
// H0: the curve is Skilling's ("Programming the Hilbert curve", 2004): coordinates -> "transposed" index by the
// inverse-undo / Gray-encode loops, then the bits of the ndim words interleaved, axis 0 most significant.
#include <math.h>

#include "qsl_internal.cuh"
#include "scan.cuh"

namespace qsl {

template <int ND>
__device__ __forceinline__ unsigned long long hilbert_key(const uint32_t c[ND], int bits)
{
    uint32_t X[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) X[d] = c[d];
    const uint32_t M = 1u << (bits - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {                 // inverse undo
        const uint32_t P = Q - 1;
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            if (X[i] & Q) X[0] ^= P;                           // invert
            else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }   // exchange
        }
    }
#pragma unroll
    for (int i = 1; i < ND; ++i) X[i] ^= X[i - 1];             // Gray encode
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[ND - 1] & Q) t ^= Q - 1;
#pragma unroll
    for (int i = 0; i < ND; ++i) X[i] ^= t;
    unsigned long long key = 0;
    for (int b = bits - 1; b >= 0; --b)
#pragma unroll
        for (int d = 0; d < ND; ++d) key = (key << 1) | ((X[d] >> b) & 1u);
    return key;
}

template <int ND>
__device__ __forceinline__ void hilbert_cell(unsigned long long key, int bits, uint32_t c[ND])
{
    uint32_t X[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) X[d] = 0;
    for (int b = bits - 1; b >= 0; --b)
#pragma unroll
        for (int d = 0; d < ND; ++d) X[d] |= (uint32_t)((key >> (b * ND + (ND - 1 - d))) & 1ull) << b;
    const uint32_t N = 2u << (bits - 1);
    uint32_t t = X[ND - 1] >> 1;                               // Gray decode
#pragma unroll
    for (int i = ND - 1; i > 0; --i) X[i] ^= X[i - 1];
    X[0] ^= t;
    for (uint32_t Q = 2; Q != N; Q <<= 1) {                    // undo excess work
        const uint32_t P = Q - 1;
#pragma unroll
        for (int i = ND - 1; i >= 0; --i) {
            if (X[i] & Q) X[0] ^= P;
            else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
#pragma unroll
    for (int d = 0; d < ND; ++d) c[d] = X[d];
}

struct HilbertLat {
    int ndim, R;
    long long n[3];             // level-0 lattice
    double origin[3], e[3][3];
};

// H1: centre of a fine cell, origin + sum_d (c_d + 0.5)/(n_d 2^R) e_d: one IEEE division and an fma chain (as O7)
template <int ND>
__device__ __forceinline__ void fine_position(const HilbertLat &A, const uint32_t c[ND], double pos[3])
{
    double w[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) w[d] = __ddiv_rn((double)c[d] + 0.5, (double)(A.n[d] << A.R));
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double p = __fma_rn(w[0], A.e[0][k], A.origin[k]);
        p = __fma_rn(w[1], A.e[1][k], p);
        if (ND == 3) p = __fma_rn(w[ND - 1], A.e[2][k], p);
        pos[k] = p;
    }
}

template <int ND>
__device__ __forceinline__ bool fine_inside(const HilbertLat &A, const int c[ND])
{
    bool in = true;
#pragma unroll
    for (int d = 0; d < ND; ++d) in = in && c[d] >= 0 && (long long)c[d] < (A.n[d] << A.R);
    return in;
}

template <int ND>
__global__ void __launch_bounds__(256) hilbert_keys_kernel(int bits, int shift, long long n, const uint32_t *__restrict__ coords,
                                                           unsigned long long *__restrict__ keys)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t c[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) c[d] = coords[ND * i + d] + (uint32_t)shift;
    keys[i] = hilbert_key<ND>(c, bits);
}

template <int ND>
__global__ void __launch_bounds__(256) hilbert_cells_kernel(int bits, int shift, long long n, const unsigned long long *__restrict__ keys,
                                                            uint32_t *__restrict__ coords)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t c[ND];
    hilbert_cell<ND>(keys[i], bits, c);
#pragma unroll
    for (int d = 0; d < ND; ++d) coords[ND * i + d] = c[d] - (uint32_t)shift;
}

// Level-0 samples in dense order (c2 n1 + c1) n0 + c0: fine cell c0 2^R + 2^(R-1), and its centre
template <int ND>
__global__ void __launch_bounds__(256) hilbert_level0_kernel(const HilbertLat A, long long n, uint32_t *__restrict__ coords,
                                                             double *__restrict__ seeds)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long r = i;
    uint32_t c[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        const long long c0 = r % A.n[d];
        r /= A.n[d];
        c[d] = (uint32_t)((c0 << A.R) + ((1ll << A.R) >> 1));
        coords[ND * i + d] = c[d];
    }
    double pos[3];
    fine_position<ND>(A, c, pos);
    seeds[3 * i] = pos[0]; seeds[3 * i + 1] = pos[1]; seeds[3 * i + 2] = pos[2];
}

// H2 / H3: flag[i] = 1 if a sample is to be inserted between samples i and i+1 of the (possibly shifted) curve order
template <int ND>
__global__ void __launch_bounds__(256) hilbert_flag_kernel(const HilbertLat A, int bits, int shift, long long n,
                                                           const unsigned long long *__restrict__ keys, const double *__restrict__ L,
                                                           double thr, uint32_t *__restrict__ flag)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t f = 0;
    if (i + 1 < n) {
        const double a = L[i], b = L[i + 1];
        const unsigned long long k0 = keys[i], k1 = keys[i + 1];
        if (isfinite(a) && isfinite(b) && fabs(b - a) > thr && k1 - k0 >= 2ull) {
            uint32_t c[ND]; int ci[ND];
            hilbert_cell<ND>((k0 + k1) >> 1, bits, c);
#pragma unroll
            for (int d = 0; d < ND; ++d) ci[d] = (int)c[d] - shift;
            f = fine_inside<ND>(A, ci) ? 1u : 0u;
        }
    }
    flag[i] = f;
}

template <int ND>
__global__ void __launch_bounds__(256) hilbert_emit_kernel(const HilbertLat A, int bits, int shift, long long n,
                                                           const unsigned long long *__restrict__ keys, const uint32_t *__restrict__ flag,
                                                           const unsigned long long *__restrict__ offset, long long capacity,
                                                           long long *__restrict__ left, uint32_t *__restrict__ new_coords,
                                                           double *__restrict__ new_seeds)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || !flag[i]) return;
    const long long j = (long long)offset[i];
    if (j >= capacity) return;
    uint32_t c[ND];
    hilbert_cell<ND>((keys[i] + keys[i + 1]) >> 1, bits, c);
#pragma unroll
    for (int d = 0; d < ND; ++d) { c[d] -= (uint32_t)shift; new_coords[ND * j + d] = c[d]; }
    left[j] = i;
    double pos[3];
    fine_position<ND>(A, c, pos);
    new_seeds[3 * j] = pos[0]; new_seeds[3 * j + 1] = pos[1]; new_seeds[3 * j + 2] = pos[2];
}

// Merge of the payload of the old samples and of the new ones (new sample j goes right after old sample left[j]; left
// is ascending): old i -> i + #{j : left[j] < i}, new j -> left[j] + 1 + j.  Payload elements are `words` 32-bit words.
__global__ void __launch_bounds__(256) hilbert_merge_kernel(long long n_old, long long n_new, const long long *__restrict__ left,
                                                            int words, const uint32_t *__restrict__ a, const uint32_t *__restrict__ b,
                                                            uint32_t *__restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_old + n_new) return;
    const uint32_t *src; long long dst;
    if (i < n_old) {
        long long lo = 0, hi = n_new;                      // first j with left[j] >= i
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if (left[mid] < i) lo = mid + 1; else hi = mid; }
        dst = i + lo; src = a + (size_t)i * words;
    } else {
        const long long j = i - n_old;
        dst = left[j] + 1 + j; src = b + (size_t)j * words;
    }
    for (int w = 0; w < words; ++w) out[(size_t)dst * words + w] = src[w];
}

__global__ void __launch_bounds__(256) gather_words_kernel(long long n, const uint32_t *__restrict__ perm, int words,
                                                           const uint32_t *__restrict__ src, uint32_t *__restrict__ dst)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const size_t s = (size_t)perm[i] * words;
    for (int w = 0; w < words; ++w) dst[(size_t)i * words + w] = src[s + w];
}

__global__ void __launch_bounds__(256) iota_u32_kernel(long long n, uint32_t *p)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = (uint32_t)i;
}

// ---- H4 converter --------------------------------------------------------------------------------------------------
// order-preserving image of a finite double in an unsigned 64-bit integer (0 is below every image: "no sample yet")
__device__ __forceinline__ unsigned long long ordered_bits(double v)
{
    const unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double from_ordered_bits(unsigned long long o)
{
    const unsigned long long u = (o >> 63) ? (o & 0x7fffffffffffffffull) : ~o;
    return __longlong_as_double((long long)u);
}

template <int ND>
__global__ void __launch_bounds__(256) convert_max_kernel(const HilbertLat A, int bits, int r, long long n,
                                                          const unsigned long long *__restrict__ keys, const double *__restrict__ Q,
                                                          unsigned long long *__restrict__ acc, uint32_t *__restrict__ usable)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double q = Q[i];
    usable[i] = (isfinite(q) && q > 0.0) ? 1u : 0u;
    if (!isfinite(q)) return;
    uint32_t c[ND];
    hilbert_cell<ND>(keys[i], bits, c);
    long long f = 0;
#pragma unroll
    for (int d = ND - 1; d >= 0; --d) f = f * (A.n[d] << r) + (long long)(c[d] >> (A.R - r));
    atomicMax(acc + f, ordered_bits(q));
}

__global__ void __launch_bounds__(256) compact_usable_kernel(long long n, const uint32_t *__restrict__ usable,
                                                             const unsigned long long *__restrict__ offset,
                                                             const unsigned long long *__restrict__ keys, const double *__restrict__ Q,
                                                             unsigned long long *__restrict__ uk, double *__restrict__ uq)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || !usable[i]) return;
    uk[offset[i]] = keys[i]; uq[offset[i]] = Q[i];
}

template <int ND>
__global__ void __launch_bounds__(256) convert_fill_kernel(const HilbertLat A, int bits, int r, long long n_cells,
                                                           const unsigned long long *__restrict__ acc,
                                                           const unsigned long long *__restrict__ n_usable_p,
                                                           const unsigned long long *__restrict__ uk, const double *__restrict__ uq,
                                                           double *__restrict__ out)
{
    const long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_cells) return;
    const unsigned long long a = acc[f];
    if (a) { out[f] = from_ordered_bits(a); return; }
    const long long m = (long long)*n_usable_p;
    double v = __longlong_as_double(0x7ff8000000000000ll);
    if (m > 0) {
        long long rem = f;
        uint32_t c[ND];
#pragma unroll
        for (int d = 0; d < ND; ++d) { const long long dim = A.n[d] << r; c[d] = (uint32_t)(rem % dim) << (A.R - r); rem /= dim; }
        const unsigned long long span = 1ull << (ND * (A.R - r));
        const unsigned long long k0 = hilbert_key<ND>(c, bits) & ~(span - 1ull), k1 = k0 + span, kc = k0 + span / 2;
        long long lo = 0, hi = m;                             // first usable key >= k0
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if (uk[mid] < k0) lo = mid + 1; else hi = mid; }
        const long long p = lo - 1;
        hi = m;                                               // first usable key >= k1 (the range holds no usable key...
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if (uk[mid] < k1) lo = mid + 1; else hi = mid; }
        const long long q = lo;                               // ... unless it holds only non-positive Q: skipped here)
        if (p >= 0 && q < m) {
            const double t = (double)(kc - uk[p]) / (double)(uk[q] - uk[p]);
            const double la = log10(uq[p]), lb = log10(uq[q]);
            v = pow(10.0, la + t * (lb - la));
        } else if (p >= 0) v = uq[p];
        else if (q < m) v = uq[q];
    }
    out[f] = v;
}

}  // namespace qsl

using namespace qsl;

static int make_lat(const qsl_lattice *lat, int R, HilbertLat &A)
{
    if (!lat || (lat->ndim != 2 && lat->ndim != 3) || R < 0 || R > 20) return QSL_EINVAL;
    A.ndim = lat->ndim; A.R = R;
    for (int d = 0; d < 3; ++d) {
        A.n[d] = d < lat->ndim ? lat->n[d] : 1;
        if (A.n[d] < 1 || (A.n[d] << R) > (1ll << 30)) return QSL_ERANGE;
        A.origin[d] = lat->origin[d];
        A.e[0][d] = lat->e0[d]; A.e[1][d] = lat->e1[d]; A.e[2][d] = lat->ndim == 3 ? lat->e2[d] : 0.0;
    }
    return QSL_OK;
}

static int curve_bits(const HilbertLat &A)
{
    long long m = 1;
    for (int d = 0; d < A.ndim; ++d) m = (A.n[d] << A.R) > m ? (A.n[d] << A.R) : m;
    int bits = 0;
    while (((m - 1) >> bits) > 0) ++bits;
    return bits < 1 ? 1 : bits;
}

static inline unsigned grid_for(long long n) { return (unsigned)((n + 255) / 256); }

extern "C" {

int qsl_hilbert_bits(const qsl_lattice *lat, int R)
{
    HilbertLat A;
    const int rc = make_lat(lat, R, A);
    if (rc != QSL_OK) return rc;
    const int bits = curve_bits(A);
    return (bits + 1) * A.ndim > 63 ? QSL_ERANGE : bits;       // the shifted curve has one bit more per axis
}

int qsl_hilbert_level0(const qsl_lattice *lat, int R, unsigned int *coords, double *seeds, void *stream)
{
    HilbertLat A;
    int rc = make_lat(lat, R, A);
    if (rc != QSL_OK) return rc;
    if (!coords || !seeds) return QSL_EINVAL;
    const long long n = A.n[0] * A.n[1] * A.n[2];
    cudaStream_t s = (cudaStream_t)stream;
    count_launch();
    if (A.ndim == 2) hilbert_level0_kernel<2><<<grid_for(n), 256, 0, s>>>(A, n, coords, seeds);
    else hilbert_level0_kernel<3><<<grid_for(n), 256, 0, s>>>(A, n, coords, seeds);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

int qsl_hilbert_keys(int ndim, int bits, int shift, long long n, const unsigned int *coords, unsigned long long *keys, void *stream)
{
    if ((ndim != 2 && ndim != 3) || bits < 1 || bits * ndim > 63 || bits > 31 || shift < 0 || n < 0) return QSL_EINVAL;
    if ((long long)shift >= (1ll << bits)) return QSL_EINVAL;      // coords + shift would leave the curve's cube
    if (n == 0) return QSL_OK;
    if (!coords || !keys) return QSL_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    count_launch();
    if (ndim == 2) hilbert_keys_kernel<2><<<grid_for(n), 256, 0, s>>>(bits, shift, n, coords, keys);
    else hilbert_keys_kernel<3><<<grid_for(n), 256, 0, s>>>(bits, shift, n, coords, keys);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

int qsl_hilbert_cells(int ndim, int bits, int shift, long long n, const unsigned long long *keys, unsigned int *coords, void *stream)
{
    if ((ndim != 2 && ndim != 3) || bits < 1 || bits * ndim > 63 || bits > 31 || shift < 0 || n < 0) return QSL_EINVAL;
    if ((long long)shift >= (1ll << bits)) return QSL_EINVAL;      // coords + shift would leave the curve's cube
    if (n == 0) return QSL_OK;
    if (!coords || !keys) return QSL_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    count_launch();
    if (ndim == 2) hilbert_cells_kernel<2><<<grid_for(n), 256, 0, s>>>(bits, shift, n, keys, coords);
    else hilbert_cells_kernel<3><<<grid_for(n), 256, 0, s>>>(bits, shift, n, keys, coords);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

int qsl_sort_keys64(long long n, unsigned long long *keys, unsigned int *perm, int key_bits, void *stream)
{
    if (n < 0 || n >= (1ll << 32) || key_bits < 1 || key_bits > 64) return QSL_EINVAL;
    if (n == 0) return QSL_OK;
    if (!keys || !perm) return QSL_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    count_launch();
    iota_u32_kernel<<<grid_for(n), 256, 0, s>>>(n, perm);
    QSL_CUDA(cudaGetLastError());
    void *kt = nullptr, *vt = nullptr;
    int rc = scratch_alloc(&kt, sizeof(unsigned long long) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&vt, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = radix_sort_pairs64(keys, perm, (unsigned long long *)kt, (uint32_t *)vt, n, key_bits, s);
    scratch_free(kt, s); scratch_free(vt, s);
    return rc;
}

int qsl_gather(long long n, const unsigned int *perm, int elem_bytes, const void *src, void *dst, void *stream)
{
    if (n < 0 || elem_bytes < 4 || (elem_bytes & 3)) return QSL_EINVAL;
    if (n == 0) return QSL_OK;
    if (!perm || !src || !dst) return QSL_EINVAL;
    count_launch();
    gather_words_kernel<<<grid_for(n), 256, 0, (cudaStream_t)stream>>>(n, perm, elem_bytes / 4, (const uint32_t *)src, (uint32_t *)dst);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

int qsl_hilbert_refine(const qsl_lattice *lat, int R, int shift, long long n, const unsigned long long *keys, const double *L,
                       double thr, long long capacity, long long *left, unsigned int *new_coords, double *new_seeds,
                       long long *n_new, void *stream)
{
    HilbertLat A;
    int rc = make_lat(lat, R, A);
    if (rc != QSL_OK) return rc;
    if (!n_new || n < 0 || shift < 0 || capacity < 0 || !(thr >= 0.0)) return QSL_EINVAL;
    *n_new = 0;
    if (n < 2) return QSL_OK;
    if (!keys || !L || (capacity > 0 && (!left || !new_coords || !new_seeds))) return QSL_EINVAL;
    // the shifted curve has one bit more per axis than the lattice's cube: shifts up to the size of that cube fit
    if ((long long)shift > (1ll << curve_bits(A))) return QSL_EINVAL;
    const int bits = curve_bits(A) + (shift ? 1 : 0);
    if (bits * A.ndim > 63) return QSL_ERANGE;
    cudaStream_t s = (cudaStream_t)stream;
    void *flag = nullptr, *offset = nullptr, *tiles = nullptr, *total = nullptr;
    rc = scratch_alloc(&flag, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&offset, sizeof(unsigned long long) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&tiles, sizeof(unsigned long long) * (size_t)((n + SCAN_TILE - 1) / SCAN_TILE), s);
    if (rc == QSL_OK) rc = scratch_alloc(&total, sizeof(unsigned long long), s);
    unsigned long long m = 0;
    if (rc == QSL_OK) {
        count_launch();
        if (A.ndim == 2) hilbert_flag_kernel<2><<<grid_for(n), 256, 0, s>>>(A, bits, shift, n, keys, L, thr, (uint32_t *)flag);
        else hilbert_flag_kernel<3><<<grid_for(n), 256, 0, s>>>(A, bits, shift, n, keys, L, thr, (uint32_t *)flag);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess)
            e = exclusive_scan_u32(n, (const uint32_t *)flag, (unsigned long long *)offset, (unsigned long long *)tiles,
                                   (unsigned long long *)total, s);
        if (e == cudaSuccess && capacity > 0) {
            count_launch();
            if (A.ndim == 2)
                hilbert_emit_kernel<2><<<grid_for(n), 256, 0, s>>>(A, bits, shift, n, keys, (const uint32_t *)flag,
                                                                   (const unsigned long long *)offset, capacity, left, new_coords, new_seeds);
            else
                hilbert_emit_kernel<3><<<grid_for(n), 256, 0, s>>>(A, bits, shift, n, keys, (const uint32_t *)flag,
                                                                   (const unsigned long long *)offset, capacity, left, new_coords, new_seeds);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(&m, total, sizeof m, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);          // the count is the one number that reaches the host
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(flag, s); scratch_free(offset, s); scratch_free(tiles, s); scratch_free(total, s);
    if (rc == QSL_OK) {
        *n_new = (long long)m;
        if ((long long)m > capacity) rc = QSL_ERANGE;               // *n_new tells the capacity needed
    }
    return rc;
}

int qsl_hilbert_merge(long long n_old, long long n_new, const long long *left, int elem_bytes, const void *old_vals,
                      const void *new_vals, void *out, void *stream)
{
    if (n_old < 0 || n_new < 0 || elem_bytes < 4 || (elem_bytes & 3)) return QSL_EINVAL;
    if (n_old + n_new == 0) return QSL_OK;
    if (!out || (n_old && !old_vals) || (n_new && (!new_vals || !left))) return QSL_EINVAL;
    count_launch();
    hilbert_merge_kernel<<<grid_for(n_old + n_new), 256, 0, (cudaStream_t)stream>>>(n_old, n_new, left, elem_bytes / 4,
                                                                                     (const uint32_t *)old_vals, (const uint32_t *)new_vals,
                                                                                     (uint32_t *)out);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}

int qsl_hilbert_convert(const qsl_lattice *lat, int R, int r, long long n, const unsigned long long *keys, const double *Q,
                        double *out, void *stream)
{
    HilbertLat A;
    int rc = make_lat(lat, R, A);
    if (rc != QSL_OK) return rc;
    if (r < 0 || r > R || n < 0 || !out || (n > 0 && (!keys || !Q))) return QSL_EINVAL;
    const int bits = curve_bits(A);
    if (bits * A.ndim > 63) return QSL_ERANGE;
    long long n_cells = 1;
    for (int d = 0; d < A.ndim; ++d) n_cells *= A.n[d] << r;
    cudaStream_t s = (cudaStream_t)stream;
    void *acc = nullptr, *usable = nullptr, *offset = nullptr, *tiles = nullptr, *total = nullptr, *uk = nullptr, *uq = nullptr;
    const long long nn = n > 0 ? n : 1;
    rc = scratch_alloc(&acc, sizeof(unsigned long long) * (size_t)n_cells, s);
    if (rc == QSL_OK) rc = scratch_alloc(&usable, sizeof(uint32_t) * (size_t)nn, s);
    if (rc == QSL_OK) rc = scratch_alloc(&offset, sizeof(unsigned long long) * (size_t)nn, s);
    if (rc == QSL_OK) rc = scratch_alloc(&tiles, sizeof(unsigned long long) * (size_t)((nn + SCAN_TILE - 1) / SCAN_TILE), s);
    if (rc == QSL_OK) rc = scratch_alloc(&total, sizeof(unsigned long long), s);
    if (rc == QSL_OK) rc = scratch_alloc(&uk, sizeof(unsigned long long) * (size_t)nn, s);
    if (rc == QSL_OK) rc = scratch_alloc(&uq, sizeof(double) * (size_t)nn, s);
    if (rc == QSL_OK) {
        cudaError_t e = cudaMemsetAsync(acc, 0, sizeof(unsigned long long) * (size_t)n_cells, s);
        if (e == cudaSuccess) e = cudaMemsetAsync(total, 0, sizeof(unsigned long long), s);
        if (e == cudaSuccess && n > 0) {
            count_launch();
            if (A.ndim == 2) convert_max_kernel<2><<<grid_for(n), 256, 0, s>>>(A, bits, r, n, keys, Q, (unsigned long long *)acc, (uint32_t *)usable);
            else convert_max_kernel<3><<<grid_for(n), 256, 0, s>>>(A, bits, r, n, keys, Q, (unsigned long long *)acc, (uint32_t *)usable);
            e = cudaGetLastError();
            if (e == cudaSuccess)
                e = exclusive_scan_u32(n, (const uint32_t *)usable, (unsigned long long *)offset, (unsigned long long *)tiles,
                                       (unsigned long long *)total, s);
            if (e == cudaSuccess) {
                count_launch();
                compact_usable_kernel<<<grid_for(n), 256, 0, s>>>(n, (const uint32_t *)usable, (const unsigned long long *)offset, keys, Q,
                                                                  (unsigned long long *)uk, (double *)uq);
                e = cudaGetLastError();
            }
        }
        if (e == cudaSuccess) {
            count_launch();
            if (A.ndim == 2)
                convert_fill_kernel<2><<<grid_for(n_cells), 256, 0, s>>>(A, bits, r, n_cells, (const unsigned long long *)acc,
                                                                         (const unsigned long long *)total, (const unsigned long long *)uk,
                                                                         (const double *)uq, out);
            else
                convert_fill_kernel<3><<<grid_for(n_cells), 256, 0, s>>>(A, bits, r, n_cells, (const unsigned long long *)acc,
                                                                         (const unsigned long long *)total, (const unsigned long long *)uk,
                                                                         (const double *)uq, out);
            e = cudaGetLastError();
        }
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(acc, s); scratch_free(usable, s); scratch_free(offset, s); scratch_free(tiles, s); scratch_free(total, s);
    scratch_free(uk, s); scratch_free(uq, s);
    return rc;
}

}  // extern "C"
