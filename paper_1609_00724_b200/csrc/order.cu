// Seed ordering.  PAPER.md:196-198 orders the samples along a space-filling curve so that
// neighbours on the curve are close in space (Hilbert in the paper); here the seeds are ordered by the Morton code of
// the field cell they start in, so that the lanes of a warp gather from neighbouring cells.  The order never changes a
// result: outputs are scattered back to the caller's order.
//
// The sort is a hand-written stable LSD radix sort on 32-bit keys (8-bit digits): per pass a per-warp-chunk digit
// histogram, one exclusive scan of the (digit-major) count table, and a scatter in which every warp ranks its 32 keys
// with __match_any_sync and keeps its running digit offsets in shared memory.
#include "qsl_internal.cuh"
#include "scan.cuh"

namespace qsl {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_CHUNK = 2048;                      // keys per warp per pass

__device__ __forceinline__ uint32_t spread3(uint32_t v)   // 10 bits -> every third bit
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__device__ __forceinline__ int cell_of(const FieldView &fv, int d, int n, double x)
{
    int i;
    if (!fv.stretched) {
        i = (int)floor((x - fv.lo[d]) / fv.h[d]);
    } else {
        const double *xs = fv.axis[d];
        int lo = 0, hi = n - 1;
        if (x >= xs[n - 1]) lo = n - 2;
        else if (x >= xs[0]) { while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (xs[mid] <= x) lo = mid; else hi = mid; } }
        i = lo;
    }
    return max(0, min(i, n - 2));
}

__global__ void __launch_bounds__(256) morton_key_kernel(const FieldView fv, long long n, const double *__restrict__ seeds,
                                                         int shift, uint32_t *__restrict__ keys, uint32_t *__restrict__ vals)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int cx = cell_of(fv, 0, fv.nx, seeds[3 * i]) >> shift;
    const int cy = cell_of(fv, 1, fv.ny, seeds[3 * i + 1]) >> shift;
    const int cz = cell_of(fv, 2, fv.nz, seeds[3 * i + 2]) >> shift;
    keys[i] = spread3((uint32_t)cx) | (spread3((uint32_t)cy) << 1) | (spread3((uint32_t)cz) << 2);
    vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(256) iota_kernel(long long n, uint32_t *perm)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) perm[i] = (uint32_t)i;
}

// counts[digit * n_chunks + chunk] = number of keys of `chunk` whose current digit is `digit`
template <typename K>
__global__ void __launch_bounds__(SORT_THREADS) sort_hist_kernel(long long n, const K *__restrict__ keys, int shift,
                                                                 long long n_chunks, uint32_t *__restrict__ counts)
{
    __shared__ uint32_t h[SORT_WARPS][256];
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (int b = lane; b < 256; b += 32) h[w][b] = 0;
    __syncwarp();
    const long long chunk = (long long)blockIdx.x * SORT_WARPS + w;
    if (chunk < n_chunks) {
        const long long lo = chunk * SORT_CHUNK, hi = min(lo + SORT_CHUNK, n);
        for (long long i = lo + lane; i < hi; i += 32) atomicAdd(&h[w][(uint32_t)(keys[i] >> shift) & 255u], 1u);
        __syncwarp();
        for (int b = lane; b < 256; b += 32) counts[(long long)b * n_chunks + chunk] = h[w][b];
    }
}

template <typename K>
__global__ void __launch_bounds__(SORT_THREADS) sort_scatter_kernel(long long n, const K *__restrict__ keys,
                                                                    const uint32_t *__restrict__ vals, int shift, long long n_chunks,
                                                                    const unsigned long long *__restrict__ offsets,
                                                                    K *__restrict__ keys_out, uint32_t *__restrict__ vals_out)
{
    __shared__ unsigned long long base[SORT_WARPS][256];
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const long long chunk = (long long)blockIdx.x * SORT_WARPS + w;
    if (chunk >= n_chunks) return;
    for (int b = lane; b < 256; b += 32) base[w][b] = offsets[(long long)b * n_chunks + chunk];
    __syncwarp();
    const long long lo = chunk * SORT_CHUNK, hi = min(lo + SORT_CHUNK, n);
    for (long long i0 = lo; i0 < hi; i0 += 32) {
        const long long i = i0 + lane;
        const bool live = i < hi;
        const K k = live ? keys[i] : (K)0;
        const uint32_t v = live ? vals[i] : 0u;
        const uint32_t digit = live ? ((uint32_t)(k >> shift) & 255u) : 256u + lane;   // dead lanes match nobody
        const unsigned peers = __match_any_sync(0xffffffffu, digit);
        const unsigned rank = __popc(peers & ((1u << lane) - 1u));
        unsigned long long dst = 0;
        if (live) dst = base[w][digit] + rank;                                    // stable: lanes in key order
        __syncwarp();
        if (live && rank == 0) base[w][digit] += __popc(peers);                   // one writer per digit
        __syncwarp();
        if (live) { keys_out[dst] = k; vals_out[dst] = v; }
    }
}

template <typename K>
static int radix_sort_pairs_t(K *keys, uint32_t *vals, K *keys_tmp, uint32_t *vals_tmp, long long n, int key_bits,
                              cudaStream_t s)
{
    // sorts in place: an even number of passes ping-pongs back into keys / vals, an odd number ends with two copies
    // (cheaper than a whole extra pass over zero digits)
    const int passes = (key_bits + 7) / 8;
    const long long n_chunks = (n + SORT_CHUNK - 1) / SORT_CHUNK;
    const long long table = 256 * n_chunks;
    void *counts = nullptr, *offsets = nullptr, *tiles = nullptr, *total = nullptr;
    int rc = scratch_alloc(&counts, sizeof(uint32_t) * (size_t)table, s);
    if (rc == QSL_OK) rc = scratch_alloc(&offsets, sizeof(unsigned long long) * (size_t)table, s);
    if (rc == QSL_OK) rc = scratch_alloc(&tiles, sizeof(unsigned long long) * (size_t)((table + SCAN_TILE - 1) / SCAN_TILE), s);
    if (rc == QSL_OK) rc = scratch_alloc(&total, sizeof(unsigned long long), s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        const unsigned blocks = (unsigned)((n_chunks + SORT_WARPS - 1) / SORT_WARPS);
        K *ki = keys, *ko = keys_tmp;
        uint32_t *vi = vals, *vo = vals_tmp;
        for (int p = 0; p < passes && e == cudaSuccess; ++p) {
            count_launch();
            sort_hist_kernel<K><<<blocks, SORT_THREADS, 0, s>>>(n, ki, 8 * p, n_chunks, (uint32_t *)counts);
            e = exclusive_scan_u32(table, (const uint32_t *)counts, (unsigned long long *)offsets, (unsigned long long *)tiles,
                                   (unsigned long long *)total, s);
            if (e != cudaSuccess) break;
            count_launch();
            sort_scatter_kernel<K><<<blocks, SORT_THREADS, 0, s>>>(n, ki, vi, 8 * p, n_chunks, (const unsigned long long *)offsets, ko, vo);
            e = cudaGetLastError();
            K *t = ki; ki = ko; ko = t;
            uint32_t *u = vi; vi = vo; vo = u;
        }
        if (e == cudaSuccess && ki != keys) {
            e = cudaMemcpyAsync(keys, ki, sizeof(K) * (size_t)n, cudaMemcpyDeviceToDevice, s);
            if (e == cudaSuccess) e = cudaMemcpyAsync(vals, vi, sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToDevice, s);
        }
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(counts, s); scratch_free(offsets, s); scratch_free(tiles, s); scratch_free(total, s);
    return rc;
}

int radix_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, long long n, int key_bits,
                     cudaStream_t s)
{
    return radix_sort_pairs_t<uint32_t>(keys, vals, keys_tmp, vals_tmp, n, key_bits, s);
}

int radix_sort_pairs64(unsigned long long *keys, uint32_t *vals, unsigned long long *keys_tmp, uint32_t *vals_tmp, long long n,
                       int key_bits, cudaStream_t s)
{
    return radix_sort_pairs_t<unsigned long long>(keys, vals, keys_tmp, vals_tmp, n, key_bits, s);
}

int morton_order(const FieldView &fv, long long n, const double *seeds, uint32_t *perm, bool sort, cudaStream_t s)
{
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (!sort || n < 2) {
        count_launch();
        iota_kernel<<<blocks, 256, 0, s>>>(n, perm);
        QSL_CUDA(cudaGetLastError());
        return QSL_OK;
    }
    int maxn = fv.nx > fv.ny ? fv.nx : fv.ny;
    if (fv.nz > maxn) maxn = fv.nz;
    int shift = 0;
    while (((maxn - 1) >> shift) > 1023) ++shift;       // 10 bits per axis
    int bits = 0;
    while (bits < 10 && ((maxn - 1) >> shift) >> bits) ++bits;
    void *keys = nullptr, *kt = nullptr, *vt = nullptr;
    int rc = scratch_alloc(&keys, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&kt, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = scratch_alloc(&vt, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) {
        count_launch();
        morton_key_kernel<<<blocks, 256, 0, s>>>(fv, n, seeds, shift, (uint32_t *)keys, perm);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) rc = record_cuda(e);
        else rc = radix_sort_pairs((uint32_t *)keys, perm, (uint32_t *)kt, (uint32_t *)vt, n, 3 * bits, s);
    }
    scratch_free(keys, s); scratch_free(kt, s); scratch_free(vt, s);
    return rc;
}

}  // namespace qsl

// Test hook (not in qsl.h's compute path): sorts key/value pairs on the device; used by the GPU tests of the sort.
extern "C" int qsl_debug_sort_pairs(unsigned int *keys, unsigned int *vals, long long n, int key_bits, void *stream)
{
    if (n < 0 || (n > 0 && (!keys || !vals)) || key_bits < 1 || key_bits > 32) return QSL_EINVAL;
    if (n == 0) return QSL_OK;
    cudaStream_t s = (cudaStream_t)stream;
    void *kt = nullptr, *vt = nullptr;
    int rc = qsl::scratch_alloc(&kt, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = qsl::scratch_alloc(&vt, sizeof(uint32_t) * (size_t)n, s);
    if (rc == QSL_OK) rc = qsl::radix_sort_pairs(keys, vals, (uint32_t *)kt, (uint32_t *)vt, n, key_bits, s);
    qsl::scratch_free(kt, s); qsl::scratch_free(vt, s);
    return rc;
}
