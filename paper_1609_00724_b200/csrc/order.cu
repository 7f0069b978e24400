// Seed ordering.  PAPER.md:196-198 orders the samples along a space-filling curve so that
// neighbours on the curve are close in space (Hilbert in the paper); here the seeds are ordered by the Morton code of
// the field cell they start in, so that the lanes of a warp gather from neighbouring cells.  The order never changes a
// result: outputs are scattered back to the caller's order.
//
// The sort is a hand-written stable LSD radix sort on 32- or 64-bit keys (8-bit digits): per pass a per-tile digit
// histogram, one exclusive scan of the (digit-major) count table, and a scatter that sorts a tile of 2048 keys by the
// digit in shared memory (warps rank their keys with warp votes) and writes it out run by run.
#include "qsl_internal.cuh"
#include "scan.cuh"

namespace qsl {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
template <typename K> struct SortTile { static constexpr int value = sizeof(K) == 8 ? 2048 : 2048; };   // keys per block per pass (static shared memory <= 48 KB)

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

// counts[digit * n_tiles + tile] = number of keys of `tile` whose current digit is `digit`.  One block per tile of
// SORT_TILE keys; per-warp histograms in shared memory (no cross-warp atomics), summed at the end.
template <typename K>
__global__ void __launch_bounds__(SORT_THREADS) sort_hist_kernel(long long n, const K *__restrict__ keys, int shift,
                                                                 long long n_tiles, uint32_t *__restrict__ counts)
{
    constexpr int SORT_TILE = SortTile<K>::value;
    __shared__ uint32_t h[SORT_WARPS][256];
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (int b = lane; b < 256; b += 32) h[w][b] = 0;
    __syncwarp();
    const long long tile = blockIdx.x;
    const long long lo = tile * SORT_TILE + (long long)w * (SORT_TILE / SORT_WARPS), hi = min(lo + SORT_TILE / SORT_WARPS, n);
    for (long long i = lo + lane; i < hi; i += 32) atomicAdd(&h[w][(uint32_t)(keys[i] >> shift) & 255u], 1u);
    __syncthreads();
    uint32_t c = 0;
#pragma unroll
    for (int q = 0; q < SORT_WARPS; ++q) c += h[q][threadIdx.x];
    counts[(long long)threadIdx.x * n_tiles + tile] = c;
}

// Scatter of one pass.  A block owns a tile of SORT_TILE consecutive keys (warp w the w-th eighth of it, 32 keys per
// round, so that index order = (warp, round, lane) order and the ranking below is stable):
//   1. every warp ranks its keys among the keys of the same digit it has seen so far (warp votes per round + a
//      running per-warp digit counter in shared memory);
//   2. thread d adds up the eight warp counters of digit d (-> the warps' bases inside the digit) and a block-wide
//      exclusive scan of the digit totals gives the place of digit d inside the tile;
//   3. keys and values are written to shared memory at their place in the tile sorted by digit;
//   4. the tile is written out in that order: entry e of digit d goes to offsets[d][tile] + (e - start of d in the
//      tile), so neighbouring threads store to neighbouring addresses within a digit's run (16 keys on average for
//      uniformly distributed digits, whole rows for the nearly sorted keys of a seed lattice) instead of 32 unrelated
//      sectors per store instruction.
// The live lanes of the warp that hold the same 8-bit digit as this lane: nine warp votes and their masks on the integer
// pipe.  __match_any_sync gives the same set in one instruction, but MATCH runs on the address-divergence unit, which
// takes one step per distinct value of the warp: with it the scatter kernel sat at 82 % of that unit's issue rate
// (profiles/r2h), 565 us per pass of 6.7e7 random keys.
__device__ __forceinline__ unsigned same_digit_lanes(uint32_t digit, bool live)
{
    unsigned peers = __ballot_sync(0xffffffffu, live);
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const bool bit = (digit >> b) & 1u;
        const unsigned v = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? v : ~v;
    }
    return peers;
}

// 5 CTAs of 256 threads per SM: 48 registers, no spill (un-capped ptxas takes 82 and the sort is 25 % slower; 6 / 8 CTAs
// spill: profiles/r2g)
#ifndef QSL_SORT_MINB
#define QSL_SORT_MINB 5
#endif
template <typename K>
__global__ void __launch_bounds__(SORT_THREADS, QSL_SORT_MINB) sort_scatter_kernel(long long n, const K *__restrict__ keys,
                                                                    const uint32_t *__restrict__ vals, int shift, long long n_tiles,
                                                                    const unsigned long long *__restrict__ offsets,
                                                                    K *__restrict__ keys_out, uint32_t *__restrict__ vals_out)
{
    constexpr int SORT_TILE = SortTile<K>::value;
    constexpr int ROUNDS = SORT_TILE / SORT_THREADS;        // 32-key rounds per warp
    __shared__ K s_key[SORT_TILE];
    __shared__ uint32_t s_val[SORT_TILE];
    __shared__ uint32_t cnt[SORT_WARPS][256];               // running digit counters, then the warps' bases inside a digit
    __shared__ uint32_t d_start[256];                       // place of a digit inside the tile
    __shared__ unsigned long long g_base[256];              // where the tile's keys of a digit go in the output
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const long long tile = blockIdx.x;
    for (int b = lane; b < 256; b += 32) cnt[w][b] = 0;
    g_base[threadIdx.x] = offsets[(long long)threadIdx.x * n_tiles + tile];
    __syncwarp();
    const long long lo = tile * SORT_TILE + (long long)w * (SORT_TILE / SORT_WARPS);
    const long long tile_n = min((long long)SORT_TILE, n - tile * SORT_TILE);
    K k[ROUNDS]; uint32_t v[ROUNDS]; uint32_t dr[ROUNDS];   // dr = digit | rank inside (warp, digit) << 8
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
        const long long i = lo + r * 32 + lane;
        const bool live = i < n;
        k[r] = live ? keys[i] : (K)0;
        v[r] = live ? vals[i] : 0u;
        const uint32_t digit = live ? ((uint32_t)(k[r] >> shift) & 255u) : 0u;
        const unsigned peers = same_digit_lanes(digit, live);                             // dead lanes match nobody
        const unsigned rank = __popc(peers & ((1u << lane) - 1u));
        uint32_t before = 0;
        if (live) before = cnt[w][digit];
        __syncwarp();
        if (live && rank == 0) cnt[w][digit] = before + __popc(peers);                    // one writer per digit
        __syncwarp();
        dr[r] = live ? (digit | ((before + rank) << 8)) : 0xffffffffu;
    }
    __syncthreads();
    {
        // digit d = threadIdx.x: exclusive prefix over the warps, total -> exclusive scan over the digits
        uint32_t run = 0;
#pragma unroll
        for (int q = 0; q < SORT_WARPS; ++q) { const uint32_t c = cnt[q][threadIdx.x]; cnt[q][threadIdx.x] = run; run += c; }
        unsigned long long total;
        d_start[threadIdx.x] = (uint32_t)block_exclusive_scan((unsigned long long)run, total);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
        if (dr[r] != 0xffffffffu) {
            const uint32_t digit = dr[r] & 255u, e = d_start[digit] + cnt[w][digit] + (dr[r] >> 8);
            s_key[e] = k[r]; s_val[e] = v[r];
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < tile_n; e += SORT_THREADS) {
        const K kk = s_key[e];
        const uint32_t digit = (uint32_t)(kk >> shift) & 255u;
        const unsigned long long dst = g_base[digit] + (unsigned)(e - d_start[digit]);
        keys_out[dst] = kk; vals_out[dst] = s_val[e];
    }
}

template <typename K>
static int radix_sort_pairs_t(K *keys, uint32_t *vals, K *keys_tmp, uint32_t *vals_tmp, long long n, int key_bits,
                              cudaStream_t s)
{
    // sorts in place: an even number of passes ping-pongs back into keys / vals, an odd number ends with two copies
    // (cheaper than a whole extra pass over zero digits)
    const int passes = (key_bits + 7) / 8;
    const long long n_chunks = (n + SortTile<K>::value - 1) / SortTile<K>::value;   // one block per tile
    const long long table = 256 * n_chunks;
    void *counts = nullptr, *offsets = nullptr, *tiles = nullptr, *total = nullptr;
    int rc = scratch_alloc(&counts, sizeof(uint32_t) * (size_t)table, s);
    if (rc == QSL_OK) rc = scratch_alloc(&offsets, sizeof(unsigned long long) * (size_t)table, s);
    if (rc == QSL_OK) rc = scratch_alloc(&tiles, sizeof(unsigned long long) * (size_t)((table + SCAN_TILE - 1) / SCAN_TILE), s);
    if (rc == QSL_OK) rc = scratch_alloc(&total, sizeof(unsigned long long), s);
    cudaError_t e = cudaSuccess;
    if (rc == QSL_OK) {
        const unsigned blocks = (unsigned)n_chunks;
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
