// Field packing and library plumbing.
// PAPER.md:178 (fn. 9): "To speed up the code, we first normalize the magnetic field data cubes, and only then
// interpolate them"; B_F, B_B, B_0 are unnormalised magnitudes, so |B| rides along as the 4th sample.
#include <math.h>
#include <new>

#include "qsl_internal.cuh"

namespace qsl {

int g_last_cuda_error = 0;
long long g_launches = 0;
int record_cuda(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    cudaGetLastError();  // clear the sticky-free error state
    return e == cudaErrorMemoryAllocation ? QSL_ENOMEM : QSL_ECUDA;
}

// Scratch comes from a PRIVATE stream-ordered memory pool per device (release threshold = never: repeated calls do not go
// back to the OS), so that the library does not change the behaviour of the device's default pool under other users of
// cudaMallocAsync in the process.  The per-device table is filled on first use; the hooks that read it (and
// g_last_cuda_error, the launch counter and the profiling event pool of trace.cu) are not thread-safe: one host thread
// drives the library at a time.
constexpr int MAX_DEVICES = 64;
static cudaMemPool_t g_pool[MAX_DEVICES];
static bool g_pool_made[MAX_DEVICES];
static int g_sm_count[MAX_DEVICES];

static int current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return -1;
    return dev;
}

int scratch_alloc(void **p, size_t bytes, cudaStream_t s)
{
    if (bytes == 0) bytes = 16;
    const int dev = current_device();
    if (dev >= 0 && !g_pool_made[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        if (cudaMemPoolCreate(&g_pool[dev], &props) == cudaSuccess) {
            uint64_t keep = UINT64_MAX;
            cudaMemPoolSetAttribute(g_pool[dev], cudaMemPoolAttrReleaseThreshold, &keep);
            g_pool_made[dev] = true;
        } else {
            cudaGetLastError();
        }
    }
    if (dev >= 0 && g_pool_made[dev]) QSL_CUDA(cudaMallocFromPoolAsync(p, bytes, g_pool[dev], s));
    else QSL_CUDA(cudaMallocAsync(p, bytes, s));      // no private pool: the device's default pool, untouched
    return QSL_OK;
}
void scratch_free(void *p, cudaStream_t s)
{
    if (p) cudaFreeAsync(p, s);
}

int sm_count()
{
    const int dev = current_device();
    if (dev < 0) return 148;
    if (g_sm_count[dev] == 0 &&
        cudaDeviceGetAttribute(&g_sm_count[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        g_sm_count[dev] = 148;
    return g_sm_count[dev];
}

// One thread per node.  All arithmetic is explicit-rounding fp64 (no FMA contraction) so that the packed samples are
// bit-identical to the definition in qsl.h: round inputs to the storage type, m = sqrt((bx*bx + by*by) + bz*bz),
// v = B/m (IEEE), round.
template <typename S4, typename S>
__global__ void __launch_bounds__(256) pack_kernel(long long n, const double *__restrict__ bx, const double *__restrict__ by,
                                                   const double *__restrict__ bz, int interp_mode, S4 *__restrict__ out)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (; p < n; p += stride) {
        const double x = (double)(S)bx[p], y = (double)(S)by[p], z = (double)(S)bz[p];
        double m = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)));
        double vx = x, vy = y, vz = z;
        if (interp_mode == QSL_NORMALIZE_FIRST) {
            if (m < 1e-300) { vx = vy = vz = 0.0; m = 0.0; }
            else { vx = __ddiv_rn(x, m); vy = __ddiv_rn(y, m); vz = __ddiv_rn(z, m); }
        }
        S4 o;
        o.x = (S)vx; o.y = (S)vy; o.z = (S)vz; o.w = (S)m;
        out[p] = o;
    }
}

// Per-cell polynomial table of the V2 trace kernel: the trilinear interpolant of each component c (eq. 3,
// :101-107 eq. 4) inside cell (i, j, k), written in monomials of the physical offset d = x - x_cell,
//     v_c(d) = sum_{m in {0,1}^3} a[c][m] dx^{m0} dy^{m1} dz^{m2},      m = m0 + 2 m1 + 4 m2,
// so that value and analytic gradient cost 11 FMAs per component instead of 25 from the corners.
// The coefficients are finite differences of the 8 corner samples (converted exactly to fp64) divided by the cell
// edges; 24 doubles = 192 B per cell, component-major, cell index (k (ny-1) + j)(nx-1) + i.
// O4 = double4 (192 B per cell, the fp64 kernels) or float4 (coefficients rounded to fp32, 96 B per cell, QSL_ARITH_F32).
// Each block builds the entries of CT_THREADS consecutive cells (one thread per cell: 8 corner gathers that neighbouring
// threads share through L1) into a shared-memory tile and then writes the tile - one contiguous run of global memory -
// with fully coalesced stores; a thread storing its own 192 bytes directly makes every warp store touch 32 lines.
constexpr int CT_THREADS = 128;
constexpr int CT_PAD = 25;                       // tile row stride in coefficients: conflict-free column writes
template <typename S4, typename O4>
__global__ void __launch_bounds__(CT_THREADS) cell_table_kernel(FieldView fv, O4 *__restrict__ cells)
{
    using E = decltype(O4().x);
    __shared__ E tile[CT_THREADS * CT_PAD];
    const int cx = fv.nx - 1, cy = fv.ny - 1, cz = fv.nz - 1;
    const long long n_cells = (long long)cx * cy * cz;
    const long long n_tiles = (n_cells + CT_THREADS - 1) / CT_THREADS;
    const S4 *__restrict__ smp = (const S4 *)fv.samples;
    E *__restrict__ out = reinterpret_cast<E *>(cells);
    for (long long tl = blockIdx.x; tl < n_tiles; tl += gridDim.x) {
        const long long p = tl * CT_THREADS + threadIdx.x;
        if (p < n_cells) {
            const int i = (int)(p % cx), j = (int)((p / cx) % cy), k = (int)(p / ((long long)cx * cy));
            const double ihx = 1.0 / (fv.axis[0][i + 1] - fv.axis[0][i]), ihy = 1.0 / (fv.axis[1][j + 1] - fv.axis[1][j]),
                         ihz = 1.0 / (fv.axis[2][k + 1] - fv.axis[2][k]);
            const size_t base = ((size_t)k * fv.ny + j) * fv.nx + i, sy = (size_t)fv.nx, sz = (size_t)fv.nx * fv.ny;
            const S4 s[8] = { smp[base], smp[base + 1], smp[base + sy], smp[base + sy + 1],
                              smp[base + sz], smp[base + sz + 1], smp[base + sz + sy], smp[base + sz + sy + 1] };
            E *row = tile + threadIdx.x * CT_PAD;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double v[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) v[q] = c == 0 ? (double)s[q].x : (c == 1 ? (double)s[q].y : (double)s[q].z);
                // finite differences along x, then y, then z (in place): v[m] becomes the coefficient of monomial m in t
#pragma unroll
                for (int q = 0; q < 8; q += 2) v[q + 1] -= v[q];
#pragma unroll
                for (int q = 0; q < 8; q += 4) { v[q + 2] -= v[q]; v[q + 3] -= v[q + 1]; }
#pragma unroll
                for (int q = 0; q < 4; ++q) v[q + 4] -= v[q];
                row[8 * c + 0] = (E)v[0];
                row[8 * c + 1] = (E)(v[1] * ihx);
                row[8 * c + 2] = (E)(v[2] * ihy);
                row[8 * c + 3] = (E)(v[3] * (ihx * ihy));
                row[8 * c + 4] = (E)(v[4] * ihz);
                row[8 * c + 5] = (E)(v[5] * (ihx * ihz));
                row[8 * c + 6] = (E)(v[6] * (ihy * ihz));
                row[8 * c + 7] = (E)(v[7] * ((ihx * ihy) * ihz));
            }
        }
        __syncthreads();
        const long long first = tl * CT_THREADS;
        const int live = (int)min((long long)CT_THREADS, n_cells - first) * 24;   // coefficients in this tile
        E *__restrict__ dst = out + first * 24;
        for (int g = threadIdx.x; g < live; g += CT_THREADS) dst[g] = tile[(g / 24) * CT_PAD + g % 24];
        __syncthreads();
    }
}

__global__ void row_sincos_kernel(int n, const double *__restrict__ theta, float2 *__restrict__ out)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double sn, cs;
    sincos(theta[j], &sn, &cs);
    out[j] = make_float2((float)sn, (float)cs);
}

}  // namespace qsl

using namespace qsl;

extern "C" {

const char *qsl_strerror(int code)
{
    switch (code) {
        case QSL_OK: return "ok";
        case QSL_EINVAL: return "invalid argument";
        case QSL_ENOMEM: return "out of memory";
        case QSL_ECUDA: return "CUDA runtime error (see qsl_last_cuda_error)";
        case QSL_ERANGE: return "size out of range";
        case QSL_ETOOBIG: return "input larger than the fixed scratch of this no-allocation entry point";
        default: return "unknown error";
    }
}
int qsl_last_cuda_error(void) { return g_last_cuda_error; }
long long qsl_launch_count(void) { return g_launches; }
int qsl_version(void) { return 100; }
int qsl_compiled_arch(void)
{
#ifdef QSL_TARGET_ARCH
    return QSL_TARGET_ARCH;
#else
    return 0;
#endif
}

int qsl_field_create(qsl_field **out, const qsl_grid_desc *d, const double *bx, const double *by, const double *bz,
                     void *stream)
{
    if (!out || !d || !bx || !by || !bz) return QSL_EINVAL;
    *out = nullptr;
    if (d->nx < 2 || d->ny < 2 || d->nz < 2) return QSL_EINVAL;
    if (d->sample_type != QSL_F32 && d->sample_type != QSL_F64) return QSL_EINVAL;
    if (d->interp_mode != QSL_NORMALIZE_FIRST && d->interp_mode != QSL_INTERP_FIRST) return QSL_EINVAL;
    if (d->layout < QSL_LAYOUT_CELL_TABLE || d->layout > QSL_LAYOUT_CELL_TABLES_BOTH) return QSL_EINVAL;
    if (d->interp_order != QSL_TRILINEAR && d->interp_order != QSL_TRIQUADRATIC && d->interp_order != QSL_TRICUBIC) return QSL_EINVAL;
    if (d->geometry != QSL_CARTESIAN && d->geometry != QSL_SPHERICAL) return QSL_EINVAL;
    const bool sph = d->geometry == QSL_SPHERICAL;
    if (sph && (d->stretched || d->interp_mode != QSL_NORMALIZE_FIRST || d->interp_order != QSL_TRILINEAR)) return QSL_EINVAL;
    const bool ho = d->interp_order != QSL_TRILINEAR;           // gather-kernel fields: node samples only, paper mode only
    if (d->interp_order != QSL_TRILINEAR) {
        const int need = d->interp_order == QSL_TRICUBIC ? 4 : 3;
        if (d->nx < need || d->ny < need || d->nz < need || d->interp_mode != QSL_NORMALIZE_FIRST) return QSL_EINVAL;
    }
    const bool want64 = !ho && (d->layout == QSL_LAYOUT_CELL_TABLE || d->layout == QSL_LAYOUT_CELL_TABLES_BOTH);
    const bool want32 = !ho && (d->layout == QSL_LAYOUT_CELL_TABLE_F32 || d->layout == QSL_LAYOUT_CELL_TABLES_BOTH);
    if (want32 && (d->sample_type != QSL_F32 || d->stretched)) return QSL_EINVAL;   // fp32 arithmetic: fp32 samples, uniform grid
    const long long n = (long long)d->nx * d->ny * d->nz;
    if (n >= (1ll << 31)) return QSL_ERANGE;   // node index is 32-bit inside the gather
    const int dims[3] = { d->nx, d->ny, d->nz };
    const double *host_axes[3] = { d->xs, d->ys, d->zs };
    if (d->stretched) {
        for (int a = 0; a < 3; ++a) {
            if (!host_axes[a]) return QSL_EINVAL;
            for (int i = 1; i < dims[a]; ++i)
                if (!(host_axes[a][i] > host_axes[a][i - 1])) return QSL_EINVAL;
        }
    } else {
        for (int a = 0; a < 3; ++a)
            if (!(d->hi[a] > d->lo[a])) return QSL_EINVAL;
    }
    cudaStream_t s = (cudaStream_t)stream;
    qsl_field *f = new (std::nothrow) qsl_field();
    if (!f) return QSL_ENOMEM;
    f->d_samples = nullptr;
    f->d_cells = nullptr;
    f->d_cells32 = nullptr;
    f->d_row_sc = nullptr;
    f->view.cells = nullptr;
    f->view.row_sc = nullptr;
    for (int a = 0; a < 3; ++a) f->d_axis[a] = nullptr;
    f->sample_type = d->sample_type;
    f->n_nodes = n;
    const size_t sbytes = (size_t)n * 4 * (d->sample_type == QSL_F32 ? 4 : 8);
    f->bytes = sbytes;
    cudaError_t e = cudaMalloc(&f->d_samples, sbytes);
    if (e != cudaSuccess) { delete f; return record_cuda(e); }
    FieldView &v = f->view;
    v.samples = f->d_samples;
    v.nx = d->nx; v.ny = d->ny; v.nz = d->nz;
    v.stretched = d->stretched ? 1 : 0;
    v.interp_mode = d->interp_mode;
    v.order = d->interp_order != QSL_TRILINEAR ? d->interp_order : 1;
    v.spherical = sph ? 1 : 0;
    for (int a = 0; a < 3; ++a) {
        // node coordinates: given (stretched) or lo + i*h (uniform), always resident for the locate of the stretched path
        double *tmp = new (std::nothrow) double[dims[a]];
        if (!tmp) { qsl_field_destroy(f); return QSL_ENOMEM; }
        if (d->stretched) {
            for (int i = 0; i < dims[a]; ++i) tmp[i] = host_axes[a][i];
            v.lo[a] = tmp[0]; v.hi[a] = tmp[dims[a] - 1];
        } else {
            v.lo[a] = d->lo[a]; v.hi[a] = d->hi[a];
            const double h = (d->hi[a] - d->lo[a]) / (double)(dims[a] - 1);
            for (int i = 0; i < dims[a]; ++i) tmp[i] = d->lo[a] + (double)i * h;
        }
        v.h[a] = (v.hi[a] - v.lo[a]) / (double)(dims[a] - 1);
        e = cudaMalloc(&f->d_axis[a], sizeof(double) * dims[a]);
        if (e == cudaSuccess) e = cudaMemcpyAsync(f->d_axis[a], tmp, sizeof(double) * dims[a], cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);   // tmp is pageable host memory
        delete[] tmp;
        if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
        v.axis[a] = f->d_axis[a];
        f->bytes += sizeof(double) * dims[a];
    }
    const int threads = 256;
    const int blocks = (int)((n + threads - 1) / threads < (long long)sm_count() * 16 ? (n + threads - 1) / threads : (long long)sm_count() * 16);
    count_launch();
    if (d->sample_type == QSL_F32)
        pack_kernel<float4, float><<<blocks, threads, 0, s>>>(n, bx, by, bz, d->interp_mode, (float4 *)f->d_samples);
    else
        pack_kernel<double4, double><<<blocks, threads, 0, s>>>(n, bx, by, bz, d->interp_mode, (double4 *)f->d_samples);
    e = cudaGetLastError();
    if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
    if (want64) {
        const long long n_cells = (long long)(d->nx - 1) * (d->ny - 1) * (d->nz - 1);
        const size_t cbytes = (size_t)n_cells * 24 * sizeof(double);
        e = cudaMalloc(&f->d_cells, cbytes);
        if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
        f->bytes += cbytes;
        const long long want = (n_cells + CT_THREADS - 1) / CT_THREADS, cap = (long long)sm_count() * 16;
        const int cblocks = (int)(want < cap ? want : cap);
        count_launch();
        if (d->sample_type == QSL_F32) cell_table_kernel<float4, double4><<<cblocks, CT_THREADS, 0, s>>>(f->view, (double4 *)f->d_cells);
        else cell_table_kernel<double4, double4><<<cblocks, CT_THREADS, 0, s>>>(f->view, (double4 *)f->d_cells);
        e = cudaGetLastError();
        if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
        f->view.cells = f->d_cells;
    }
    if (want32) {
        const long long n_cells = (long long)(d->nx - 1) * (d->ny - 1) * (d->nz - 1);
        if (n_cells >= (1ll << 31)) { qsl_field_destroy(f); return QSL_ERANGE; }   // 32-bit cell index in the fp32 kernel
        const size_t cbytes = (size_t)n_cells * 24 * sizeof(float);
        e = cudaMalloc(&f->d_cells32, cbytes);
        if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
        f->bytes += cbytes;
        const long long want = (n_cells + CT_THREADS - 1) / CT_THREADS, cap = (long long)sm_count() * 16;
        const int cblocks = (int)(want < cap ? want : cap);
        count_launch();
        cell_table_kernel<float4, float4><<<cblocks, CT_THREADS, 0, s>>>(f->view, (float4 *)f->d_cells32);
        e = cudaGetLastError();
        if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
        if (sph) {
            // (sin, cos) of the latitude of every node row, in fp64 and rounded once: the fp32 kernel's frame (reading A19)
            e = cudaMalloc(&f->d_row_sc, sizeof(float2) * (size_t)d->ny);
            if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
            f->bytes += sizeof(float2) * (size_t)d->ny;
            count_launch();
            row_sincos_kernel<<<(d->ny + 127) / 128, 128, 0, s>>>(d->ny, f->d_axis[1], (float2 *)f->d_row_sc);
            e = cudaGetLastError();
            if (e != cudaSuccess) { qsl_field_destroy(f); return record_cuda(e); }
            f->view.row_sc = (const float2 *)f->d_row_sc;
        }
    }
    *out = f;
    return QSL_OK;
}

int qsl_field_destroy(qsl_field *f)
{
    if (!f) return QSL_OK;
    if (f->d_samples) cudaFree(f->d_samples);
    if (f->d_cells) cudaFree(f->d_cells);
    if (f->d_cells32) cudaFree(f->d_cells32);
    if (f->d_row_sc) cudaFree(f->d_row_sc);
    for (int a = 0; a < 3; ++a)
        if (f->d_axis[a]) cudaFree(f->d_axis[a]);
    delete f;
    return QSL_OK;
}

int qsl_field_export(const qsl_field *f, void *packed_out, void *stream)
{
    if (!f || !packed_out) return QSL_EINVAL;
    const size_t sbytes = (size_t)f->n_nodes * 4 * (f->sample_type == QSL_F32 ? 4 : 8);
    QSL_CUDA(cudaMemcpyAsync(packed_out, f->d_samples, sbytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return QSL_OK;
}

long long qsl_field_bytes(const qsl_field *f) { return f ? (long long)f->bytes : 0; }

}  // extern "C"
