// Threshold and refinement.
// refine where the field-line-length jump "surpasses a certain threshold"; new samples are
// inserted where it does.  BASELINE.json configs[2]: "where the FLEDGE value exceeds the 95th percentile".
// Reading A11: tau = nearest-rank order statistic of the finite level-0 values; strict >; 2x refinement per axis.
//   qsl_select: exact radix select on the order-preserving 64-bit image of the doubles (8 passes of 8 bits), all on device.
//   qsl_refine: flag -> exclusive scan -> stable stream compaction; every flagged cell emits its 2^D children.
#include <math.h>

#include "qsl_internal.cuh"
#include "scan.cuh"

namespace qsl {

// ---------------------------------------------------------------------------------------------------------------
// radix select
struct SelectState {
    unsigned long long prefix;      // high digits of the answer found so far
    unsigned long long rank;        // 0-based rank still to be located inside the current bucket
    unsigned long long n_finite;
    unsigned long long n_cand16;    // values that share the answer's top 16 bits (known after pass 1)
    unsigned int overflow;          // pass 2: some block found more candidates than its segment holds
    unsigned int pad;
    unsigned int hist[256];
};

__device__ __forceinline__ unsigned long long ordered_key(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double key_to_double(unsigned long long k)
{
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

// One pass of the radix select: histogram of digit `pass` over the values that share the digits found so far.
// Passes 0 and 1 read S.  Pass 2 reads S once more and, if no more than `cap` / 2 values share the answer's top 16 bits
// (sign, exponent, 4 bits of mantissa), also keeps the ordered keys of those values: block b appends the ones it meets to
// its own segment cand[b seg .. (b + 1) seg) (slots from a counter in shared memory, the count to blk_cnt[b]; no global
// atomics), and passes 3 - 7 - same grid - read their block's segment instead of S.  For a FLEDGE map the candidates are
// a few per cent of the values: three reads of S instead of eight.  With more candidates than that (a near-constant
// map), or if a block's segment overflows, every pass reads S, as before.
__global__ void __launch_bounds__(256) select_hist_kernel(long long n, const double *__restrict__ S, int pass,
                                                          SelectState *__restrict__ st, unsigned long long *__restrict__ cand,
                                                          unsigned int *__restrict__ blk_cnt, unsigned long long cap)
{
    __shared__ unsigned int h[256];
    __shared__ unsigned int s_n;
    h[threadIdx.x] = 0;
    if (threadIdx.x == 0) s_n = 0;
    __syncthreads();
    const int shift = 56 - 8 * pass;
    const unsigned long long prefix = st->prefix;
    const bool use_cand = cand != nullptr && 2 * st->n_cand16 <= cap && !st->overflow;   // the same in every thread of the grid
    const unsigned long long seg = cap / gridDim.x;
    unsigned long long *__restrict__ mine = cand + (size_t)blockIdx.x * seg;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const unsigned lane = threadIdx.x & 31u;
    if (pass >= 3 && use_cand) {
        const unsigned m = blk_cnt[blockIdx.x];
        for (unsigned i = threadIdx.x; i < m; i += blockDim.x) {
            const unsigned long long k = mine[i];
            if ((k >> (shift + 8)) == (prefix >> (shift + 8))) atomicAdd(&h[(k >> shift) & 255u], 1u);
        }
    } else if (!(pass == 2 && use_cand)) {
        // plain pass over S (the compiler unrolls it: several loads in flight per thread)
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
            const double v = S[i];
            if (!isfinite(v)) continue;
            const unsigned long long k = ordered_key(v);
            if (pass == 0 || (k >> (shift + 8)) == (prefix >> (shift + 8))) atomicAdd(&h[(k >> shift) & 255u], 1u);
        }
    } else {
        // pass 2 with compaction
        // warp-uniform loop bounds (every lane of a warp takes part in the vote of the compaction); four loads in
        // flight per thread (the vote keeps the compiler from unrolling the loop itself)
        constexpr int U = 4;
        const double qnan = __longlong_as_double(0x7ff8000000000000ll);
        for (long long b = (long long)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); b < n; b += U * stride) {
            double v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { const long long i = b + u * stride + lane; v[u] = i < n ? S[i] : qnan; }
            unsigned long long k[U]; unsigned m[U]; unsigned tot = 0;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                k[u] = ordered_key(v[u]);
                const bool match = isfinite(v[u]) && (k[u] >> (shift + 8)) == (prefix >> (shift + 8));
                if (match) atomicAdd(&h[(k[u] >> shift) & 255u], 1u);
                m[u] = __ballot_sync(0xffffffffu, match);
                tot += __popc(m[u]);
            }
            if (tot) {                                   // one slot request per warp and trip
                unsigned slot = 0;
                if (lane == 0) slot = atomicAdd(&s_n, tot);
                slot = __shfl_sync(0xffffffffu, slot, 0);
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const unsigned at = slot + __popc(m[u] & ((1u << lane) - 1u));
                    if (((m[u] >> lane) & 1u) && at < seg) mine[at] = k[u];
                    slot += __popc(m[u]);
                }
            }
        }
    }
    __syncthreads();
    if (h[threadIdx.x]) atomicAdd(&st->hist[threadIdx.x], h[threadIdx.x]);
    if (pass == 2 && use_cand && threadIdx.x == 0) {
        blk_cnt[blockIdx.x] = s_n;
        if (s_n > seg) atomicExch(&st->overflow, 1u);
    }
}

__global__ void __launch_bounds__(256) select_pick_kernel(int pass, double p, SelectState *__restrict__ st, double *__restrict__ tau)
{
    const unsigned int mine = st->hist[threadIdx.x];
    unsigned long long total;
    const unsigned long long before = block_exclusive_scan((unsigned long long)mine, total);
    if (pass == 0 && threadIdx.x == 0) {
        st->n_finite = total;
        long long r = (long long)ceil(p * (double)total);         // nearest rank: the ceil(p N)-th smallest
        if (r < 1) r = 1;
        if (r > (long long)total) r = (long long)total;
        st->rank = total ? (unsigned long long)(r - 1) : 0ull;
    }
    __syncthreads();
    const unsigned long long rank = st->rank;
    const bool hit = mine != 0 && rank >= before && rank < before + mine;
    __syncthreads();
    if (hit) {
        const int shift = 56 - 8 * pass;
        st->prefix |= (unsigned long long)threadIdx.x << shift;
        st->rank = rank - before;
        if (pass == 1) st->n_cand16 = mine;
    }
    st->hist[threadIdx.x] = 0;
    __syncthreads();
    if (pass == 7 && threadIdx.x == 0)
        *tau = st->n_finite ? key_to_double(st->prefix) : __longlong_as_double(0x7ff8000000000000ll);
}

// ---------------------------------------------------------------------------------------------------------------
// refine
struct RefineArgs {
    int ndim, level;
    long long n;
    const uint32_t *coords;          // NULL: dense level-0 lattice in index order
    const double *S;
    const double *tau;
    long long n0[3];
    double origin[3], e[3][3];
    long long capacity;
    uint32_t *child_coords;
    double *child_seeds;
    long long *child_base;
};

// Refinement in three launches without a flag or an offset array: (1) flagged cells per tile of RF_TILE cells, straight
// from S and tau; (2) exclusive scan of the tile counts (one block); (3) per tile: the flags again, a block-wide
// exclusive scan, and the children of every flagged cell written at (tile offset + rank) << NDIM - the stable
// compaction of O7.  Per cell 8 B of S twice and 8 B of child_base, per child 4 NDIM + 24 B.
constexpr int RF_THREADS = 256;
constexpr int RF_ITEMS = 8;                          // consecutive cells per thread (the scan order is the cell order)
constexpr int RF_TILE = RF_THREADS * RF_ITEMS;

__global__ void __launch_bounds__(RF_THREADS) refine_count_kernel(long long n, const double *__restrict__ S,
                                                                  const double *__restrict__ tau,
                                                                  unsigned long long *__restrict__ tile_counts)
{
    const double t = *tau;
    const long long base = (long long)blockIdx.x * RF_TILE;
    unsigned long long c = 0;
#pragma unroll
    for (int k = 0; k < RF_ITEMS; ++k) {
        const long long i = base + (long long)k * RF_THREADS + threadIdx.x;      // coalesced: the count needs no order
        if (i < n) c += S[i] > t ? 1u : 0u;                                      // NaN never flags
    }
    unsigned long long total;
    block_exclusive_scan(c, total);
    if (threadIdx.x == 0) tile_counts[blockIdx.x] = total;
}

// The children of a tile form one contiguous run of the output (tile offset << NDIM onwards), so the block writes them
// cooperatively - one thread per coordinate word, then one thread per child for its position - instead of every flagged
// cell's thread writing its own 2^NDIM children (36 B each) at a stride: neighbouring threads store to neighbouring
// addresses.  The arithmetic per child (one IEEE division per axis, the fma chain) is unchanged.
template <int NDIM>
__global__ void __launch_bounds__(RF_THREADS) refine_emit_kernel(const RefineArgs A, const unsigned long long *__restrict__ tile_offs)
{
    __shared__ unsigned char s_flag[RF_TILE];
    __shared__ unsigned short s_rank[RF_TILE];      // rank of a flagged cell among the flagged cells of the tile
    __shared__ unsigned short s_cell[RF_TILE];      // the r-th flagged cell of the tile
    __shared__ uint32_t s_c[RF_TILE][NDIM];         // and its lattice coordinates
    const double t = *A.tau;
    const long long base = (long long)blockIdx.x * RF_TILE;
    // flags of the tile, loaded with coalesced accesses
#pragma unroll
    for (int k = 0; k < RF_ITEMS; ++k) {
        const int e = k * RF_THREADS + threadIdx.x;
        s_flag[e] = base + e < A.n && A.S[base + e] > t ? 1 : 0;                // NaN never flags
    }
    __syncthreads();
    // thread t ranks RF_ITEMS consecutive cells, so that the scan order is the cell order (stable compaction)
    unsigned long long mine = 0;
#pragma unroll
    for (int k = 0; k < RF_ITEMS; ++k) mine += s_flag[threadIdx.x * RF_ITEMS + k];
    unsigned long long total;
    unsigned rank = (unsigned)block_exclusive_scan(mine, total);
    const long long first0 = (long long)tile_offs[blockIdx.x] << NDIM;          // first child of the tile
#pragma unroll
    for (int k = 0; k < RF_ITEMS; ++k) {
        const int e = threadIdx.x * RF_ITEMS + k;
        if (s_flag[e]) { s_rank[e] = (unsigned short)rank; s_cell[rank] = (unsigned short)e; ++rank; }
    }
    __syncthreads();
    const int flagged = (int)total;
    if (A.child_base) {
        for (int e = threadIdx.x; e < RF_TILE && base + e < A.n; e += RF_THREADS)
            A.child_base[base + e] = s_flag[e] ? first0 + ((long long)s_rank[e] << NDIM) : -1ll;
    }
    // coordinates of the flagged cells
    for (int r = threadIdx.x; r < flagged; r += RF_THREADS) {
        const long long i = base + s_cell[r];
        if (A.coords) {
#pragma unroll
            for (int d = 0; d < NDIM; ++d) s_c[r][d] = A.coords[i * NDIM + d];
        } else {
            s_c[r][0] = (uint32_t)(i % A.n0[0]);
            s_c[r][1] = (uint32_t)((i / A.n0[0]) % A.n0[1]);
            if (NDIM == 3) s_c[r][NDIM - 1] = (uint32_t)(i / (A.n0[0] * A.n0[1]));
        }
    }
    __syncthreads();
    // children that fit the caller's buffers (the host reports QSL_ERANGE if some did not)
    long long room = A.capacity - first0;
    if (room <= 0) return;
    const int children = (int)min((long long)flagged << NDIM, room);
    // child coordinates: one thread per 32-bit word of the run
    for (int w = threadIdx.x; w < children * NDIM; w += RF_THREADS) {
        const int j = w / NDIM, d = w - j * NDIM;
        A.child_coords[first0 * NDIM + w] = 2u * s_c[j >> NDIM][d] + (uint32_t)(((j & ((1 << NDIM) - 1)) >> d) & 1);
    }
    double inv_den[3];
#pragma unroll
    for (int d = 0; d < NDIM; ++d) inv_den[d] = (double)(A.n0[d] << (A.level + 1));
    // child positions: one thread per child
    for (int j = threadIdx.x; j < children; j += RF_THREADS) {
        const int r = j >> NDIM, ch = j & ((1 << NDIM) - 1);
        double w[3] = { 0.0, 0.0, 0.0 };
#pragma unroll
        for (int d = 0; d < NDIM; ++d) {
            const uint32_t cc = 2u * s_c[r][d] + (uint32_t)((ch >> d) & 1);
            w[d] = __ddiv_rn((double)cc + 0.5, inv_den[d]);      // one IEEE division, as in the definition
        }
        double *__restrict__ o = A.child_seeds + 3 * (first0 + j);
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            double pos = __fma_rn(w[0], A.e[0][q], A.origin[q]);
            pos = __fma_rn(w[1], A.e[1][q], pos);
            if (NDIM == 3) pos = __fma_rn(w[2], A.e[2][q], pos);
            o[q] = pos;
        }
    }
}

}  // namespace qsl

using namespace qsl;

extern "C" int qsl_select(long long n, const double *S, double p, double *tau, void *stream)
{
    if (n < 0 || (n > 0 && !S) || !tau || !(p >= 0.0 && p <= 1.0)) return QSL_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    void *stp = nullptr, *cand = nullptr;
    int rc = scratch_alloc(&stp, sizeof(SelectState), s);
    if (rc != QSL_OK) return rc;
    long long blocks = (n + 255) / 256;
    const long long cap_blocks = (long long)sm_count() * 8;
    if (blocks > cap_blocks) blocks = cap_blocks;
    if (blocks < 1) blocks = 1;
    // candidate buffer of pass 2: room for a quarter of the values in one segment per block (+ the blocks' counts); a map
    // with more candidates than half of that keeps reading S
    const unsigned long long cap = n >= 65536 ? (unsigned long long)(n / 4) : 0ull;
    if (cap) {
        rc = scratch_alloc(&cand, sizeof(unsigned long long) * (size_t)cap + sizeof(unsigned int) * (size_t)blocks, s);
        if (rc != QSL_OK) { scratch_free(stp, s); return rc; }
    }
    unsigned int *blk_cnt = cand ? (unsigned int *)((unsigned long long *)cand + cap) : nullptr;
    SelectState *st = (SelectState *)stp;
    cudaError_t e = cudaMemsetAsync(st, 0, sizeof(SelectState), s);
    for (int pass = 0; pass < 8 && e == cudaSuccess; ++pass) {
        count_launch();
        select_hist_kernel<<<(unsigned)blocks, 256, 0, s>>>(n, S, pass, st, (unsigned long long *)cand, blk_cnt, cap);
        count_launch();
        select_pick_kernel<<<1, 256, 0, s>>>(pass, p, st, tau);
        e = cudaGetLastError();
    }
    scratch_free(cand, s);
    scratch_free(stp, s);
    if (e != cudaSuccess) return record_cuda(e);
    return QSL_OK;
}

extern "C" int qsl_refine(int ndim, int level, long long n, const unsigned int *coords, const double *S, const double *tau,
                          const qsl_lattice *lat, long long capacity, unsigned int *child_coords, double *child_seeds,
                          long long *child_base, long long *n_children, void *stream)
{
    if ((ndim != 2 && ndim != 3) || level < 0 || level > 14 || n < 0 || !lat || !tau || !n_children || capacity < 0) return QSL_EINVAL;
    if (n > 0 && (!S || (capacity > 0 && (!child_coords || !child_seeds)))) return QSL_EINVAL;
    if (lat->ndim != ndim) return QSL_EINVAL;
    if (!coords) {
        const long long dense = lat->n[0] * lat->n[1] * (ndim == 3 ? lat->n[2] : 1);
        if (level != 0 || n != dense) return QSL_EINVAL;
    }
    for (int d = 0; d < ndim; ++d)
        if (lat->n[d] < 1 || (lat->n[d] << (level + 1)) > 0xffffffffll) return QSL_ERANGE;
    *n_children = 0;
    if (n == 0) return QSL_OK;
    cudaStream_t s = (cudaStream_t)stream;
    RefineArgs A;
    A.ndim = ndim; A.level = level; A.n = n; A.coords = coords; A.S = S; A.tau = tau;
    for (int d = 0; d < 3; ++d) {
        A.n0[d] = d < ndim ? lat->n[d] : 1;
        A.origin[d] = lat->origin[d];
        A.e[0][d] = lat->e0[d]; A.e[1][d] = lat->e1[d]; A.e[2][d] = lat->e2[d];
    }
    A.capacity = capacity; A.child_coords = child_coords; A.child_seeds = child_seeds; A.child_base = child_base;

    void *tiles = nullptr, *total = nullptr;
    const long long ntiles = (n + RF_TILE - 1) / RF_TILE;
    int rc = scratch_alloc(&tiles, sizeof(unsigned long long) * (size_t)ntiles, s);
    if (rc == QSL_OK) rc = scratch_alloc(&total, sizeof(unsigned long long), s);
    unsigned long long h_total = 0;
    if (rc == QSL_OK) {
        count_launch();
        refine_count_kernel<<<(unsigned)ntiles, RF_THREADS, 0, s>>>(n, S, tau, (unsigned long long *)tiles);
        count_launch();
        scan_single_block<<<1, 1024, 0, s>>>(ntiles, (unsigned long long *)tiles, (unsigned long long *)total);
        count_launch();
        if (ndim == 2) refine_emit_kernel<2><<<(unsigned)ntiles, RF_THREADS, 0, s>>>(A, (const unsigned long long *)tiles);
        else refine_emit_kernel<3><<<(unsigned)ntiles, RF_THREADS, 0, s>>>(A, (const unsigned long long *)tiles);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpyAsync(&h_total, total, sizeof(h_total), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) rc = record_cuda(e);
    }
    scratch_free(tiles, s); scratch_free(total, s);
    if (rc != QSL_OK) return rc;
    *n_children = (long long)(h_total << ndim);
    if (*n_children > capacity) return QSL_ERANGE;
    return QSL_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// qsl_refine for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
// the per-tile counts of the compaction live in a file-scope device array instead of the stream-ordered pool, and the
// child count stays on the device (no host synchronisation).  Same kernels, same arithmetic, same outputs as qsl_refine.
//
// The array is part of the library image: every GPU that loads libqsl holds its 256 KiB (+ 256 B) until the process
// exits.  All calls on a device share it and it keeps the last call's contents; nothing in it has to start at zero
// (refine_count_kernel writes every tile count of the call, scan_single_block the total, before either is read).  Two
// calls that overlap on the GPU (different streams) race on it: serialise them.
namespace qsl {

constexpr long long RF_NOALLOC_MAX_TILES = QSL_REFINE_NOALLOC_MAX_CELLS / RF_TILE;
static_assert(QSL_REFINE_NOALLOC_MAX_CELLS % RF_TILE == 0, "the limit is a whole number of tiles");
// [0, MAX_TILES): tile counts, then their exclusive scan; [MAX_TILES]: the number of flagged cells
static __device__ __align__(256) unsigned long long g_refine_noalloc_scratch[RF_NOALLOC_MAX_TILES + 32];

__global__ void refine_noalloc_total_kernel(const unsigned long long *__restrict__ flagged, int ndim,
                                            long long *__restrict__ n_children)
{
    *n_children = (long long)(*flagged << ndim);
}

// Device address of the array on the current device.  In host code the array's name is a host-side stand-in, not a
// device address: the address comes from cudaGetSymbolAddress, asked once per device with that device current.
static int refine_noalloc_scratch(unsigned long long **out)
{
    static unsigned long long *cache[64];
    int dev = 0;
    QSL_CUDA(cudaGetDevice(&dev));
    unsigned long long *ptr = dev >= 0 && dev < 64 ? cache[dev] : nullptr;
    if (!ptr) {
        QSL_CUDA(cudaGetSymbolAddress((void **)&ptr, g_refine_noalloc_scratch));
        if (!ptr) return QSL_ECUDA;
        if (dev >= 0 && dev < 64) cache[dev] = ptr;
    }
    *out = ptr;
    return QSL_OK;
}

}  // namespace qsl

extern "C" int qsl_refine_noalloc(int ndim, int level, long long n, const unsigned int *coords, const double *S,
                                  const double *tau, const qsl_lattice *lat, long long capacity, unsigned int *child_coords,
                                  double *child_seeds, long long *child_base, long long *n_children, void *stream)
{
    if ((ndim != 2 && ndim != 3) || level < 0 || level > 14 || n < 0 || !lat || !tau || !n_children || capacity < 0) return QSL_EINVAL;
    if (n > 0 && (!S || (capacity > 0 && (!child_coords || !child_seeds)))) return QSL_EINVAL;
    if (lat->ndim != ndim) return QSL_EINVAL;
    if (!coords) {
        const long long dense = lat->n[0] * lat->n[1] * (ndim == 3 ? lat->n[2] : 1);
        if (level != 0 || n != dense) return QSL_EINVAL;
    }
    for (int d = 0; d < ndim; ++d)
        if (lat->n[d] < 1 || (lat->n[d] << (level + 1)) > 0xffffffffll) return QSL_ERANGE;
    if (n > QSL_REFINE_NOALLOC_MAX_CELLS) return QSL_ETOOBIG;       // the fixed scratch array holds no more tile counts
    cudaStream_t s = (cudaStream_t)stream;
    if (n == 0) {
        QSL_CUDA(cudaMemsetAsync(n_children, 0, sizeof(long long), s));
        return QSL_OK;
    }
    unsigned long long *tiles = nullptr;
    int rc = refine_noalloc_scratch(&tiles);
    if (rc != QSL_OK) return rc;
    unsigned long long *total = tiles + RF_NOALLOC_MAX_TILES;
    RefineArgs A;
    A.ndim = ndim; A.level = level; A.n = n; A.coords = coords; A.S = S; A.tau = tau;
    for (int d = 0; d < 3; ++d) {
        A.n0[d] = d < ndim ? lat->n[d] : 1;
        A.origin[d] = lat->origin[d];
        A.e[0][d] = lat->e0[d]; A.e[1][d] = lat->e1[d]; A.e[2][d] = lat->e2[d];
    }
    A.capacity = capacity; A.child_coords = child_coords; A.child_seeds = child_seeds; A.child_base = child_base;
    const long long ntiles = (n + RF_TILE - 1) / RF_TILE;
    count_launch();
    refine_count_kernel<<<(unsigned)ntiles, RF_THREADS, 0, s>>>(n, S, tau, tiles);
    count_launch();
    scan_single_block<<<1, 1024, 0, s>>>(ntiles, tiles, total);
    count_launch();
    if (ndim == 2) refine_emit_kernel<2><<<(unsigned)ntiles, RF_THREADS, 0, s>>>(A, tiles);
    else refine_emit_kernel<3><<<(unsigned)ntiles, RF_THREADS, 0, s>>>(A, tiles);
    count_launch();
    refine_noalloc_total_kernel<<<1, 1, 0, s>>>(total, ndim, n_children);
    QSL_CUDA(cudaGetLastError());
    return QSL_OK;
}
