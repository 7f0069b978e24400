// Device-wide exclusive prefix sum of 32-bit counts into 64-bit offsets (hand-written, three kernels):
// per-tile sums -> single-block scan of the tile sums -> per-tile scan with the tile offset added.
#pragma once
#include "qsl_internal.cuh"

namespace qsl {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;                       // per thread
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ unsigned long long warp_inclusive_scan(unsigned long long v, unsigned lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= (unsigned)o) v += t;
    }
    return v;
}

// Exclusive scan over the threads of a block (blockDim.x <= 1024); returns the block total in `total`.
__device__ __forceinline__ unsigned long long block_exclusive_scan(unsigned long long v, unsigned long long &total)
{
    __shared__ unsigned long long warp_sums[32];
    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const unsigned long long inc = warp_inclusive_scan(v, lane);
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const unsigned nw = (blockDim.x + 31) >> 5;
        unsigned long long w = lane < nw ? warp_sums[lane] : 0ull;
        w = warp_inclusive_scan(w, lane);
        warp_sums[lane] = w;
    }
    __syncthreads();
    const unsigned long long before = wid == 0 ? 0ull : warp_sums[wid - 1];
    total = warp_sums[((blockDim.x + 31) >> 5) - 1];
    __syncthreads();
    return before + inc - v;
}

static __global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums(long long n, const uint32_t *__restrict__ in,
                                                               unsigned long long *__restrict__ tile_sums)
{
    const long long base = (long long)blockIdx.x * SCAN_TILE;
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const long long i = base + (long long)k * SCAN_THREADS + threadIdx.x;
        if (i < n) s += in[i];
    }
    unsigned long long total;
    block_exclusive_scan(s, total);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// Single block: exclusive scan of m values in place; writes the grand total to *total_out (if not NULL).
static __global__ void __launch_bounds__(1024) scan_single_block(long long m, unsigned long long *__restrict__ v,
                                                          unsigned long long *__restrict__ total_out)
{
    unsigned long long carry = 0;
    for (long long base = 0; base < m; base += blockDim.x) {
        const long long i = base + threadIdx.x;
        const unsigned long long x = i < m ? v[i] : 0ull;
        unsigned long long total;
        const unsigned long long ex = block_exclusive_scan(x, total);
        if (i < m) v[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

static __global__ void __launch_bounds__(SCAN_THREADS) scan_tiles(long long n, const uint32_t *__restrict__ in,
                                                           const unsigned long long *__restrict__ tile_offsets,
                                                           unsigned long long *__restrict__ out)
{
    // thread t owns SCAN_ITEMS consecutive elements so that the scan order is the element order
    const long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
    uint32_t x[SCAN_ITEMS];
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { x[k] = base + k < n ? in[base + k] : 0u; s += x[k]; }
    unsigned long long total;
    unsigned long long ex = block_exclusive_scan(s, total) + tile_offsets[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += x[k];
    }
}

// Small inputs: one block does the whole scan (one launch instead of three).
static __global__ void __launch_bounds__(1024) scan_small_u32(long long n, const uint32_t *__restrict__ in,
                                                       unsigned long long *__restrict__ out,
                                                       unsigned long long *__restrict__ total_out)
{
    unsigned long long carry = 0;
    for (long long base = 0; base < n; base += blockDim.x) {
        const long long i = base + threadIdx.x;
        const unsigned long long x = i < n ? in[i] : 0ull;
        unsigned long long total;
        const unsigned long long ex = block_exclusive_scan(x, total);
        if (i < n) out[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}
constexpr long long SCAN_SMALL = 32768;

// out[i] = sum_{j<i} in[i]; *total (device, optional) = sum of all.  `tile_sums` scratch: ceil(n / SCAN_TILE) entries.
static inline cudaError_t exclusive_scan_u32(long long n, const uint32_t *in, unsigned long long *out,
                                             unsigned long long *tile_sums, unsigned long long *total, cudaStream_t s)
{
    const long long tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (tiles == 0) return cudaMemsetAsync(total, 0, sizeof(unsigned long long), s);
    if (n <= SCAN_SMALL) {
        count_launch();
        scan_small_u32<<<1, 1024, 0, s>>>(n, in, out, total);
        return cudaGetLastError();
    }
    count_launch();
    scan_tile_sums<<<(unsigned)tiles, SCAN_THREADS, 0, s>>>(n, in, tile_sums);
    count_launch();
    scan_single_block<<<1, 1024, 0, s>>>(tiles, tile_sums, total);
    count_launch();
    scan_tiles<<<(unsigned)tiles, SCAN_THREADS, 0, s>>>(n, in, tile_sums, out);
    return cudaGetLastError();
}

}  // namespace qsl
