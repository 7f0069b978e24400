// Internal declarations shared by the translation units of libqsl (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qsl.h"

namespace qsl {

// Last CUDA error seen by any entry point (qsl_last_cuda_error).
extern int g_last_cuda_error;
int record_cuda(cudaError_t e);

#define QSL_CUDA(call)                                                            \
    do {                                                                          \
        cudaError_t e__ = (call);                                                 \
        if (e__ != cudaSuccess) return ::qsl::record_cuda(e__);                   \
    } while (0)

// Stream-ordered scratch allocation (released to the pool, not to the OS, between calls).
int scratch_alloc(void **p, size_t bytes, cudaStream_t s);
void scratch_free(void *p, cudaStream_t s);

int sm_count();

// Number of kernels launched by the library so far (qsl_launch_count; bench.py's gpu_launches).
extern long long g_launches;
inline void count_launch() { ++g_launches; }

// Device view of a packed field: AoS samples (v0, v1, v2, |B|), x fastest.
struct FieldView {
    const void *samples;      // float4* or double4*
    const void *cells;        // double4[6] per cell: monomial coefficients of the trilinear interpolant, or NULL
    int nx, ny, nz;
    int stretched;
    int interp_mode;
    int spherical;            // axes are (longitude, latitude, radius), components in the orthonormal basis (reading A19)
    int order;                // interpolation order: 1 trilinear, 2 triquadratic (Dodgson), 3 tricubic (Keys)
    double lo[3], hi[3];
    double h[3];              // uniform spacing (hi - lo)/(n - 1)
    const double *axis[3];    // device node coordinates (always present)
    const float2 *row_sc;     // spherical fields with the fp32 table: (sin, cos) of the latitude of node row j, else NULL
};

// Sort (key, value) pairs by 32-bit key, ascending, stable.  Hand-written LSD radix sort (order.cu).
int radix_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, long long n,
                     int key_bits, cudaStream_t s);
int radix_sort_pairs64(unsigned long long *keys, uint32_t *vals, unsigned long long *keys_tmp, uint32_t *vals_tmp, long long n,
                       int key_bits, cudaStream_t s);
// perm (n) = seed indices ordered by the Morton code of the seed's field cell; identity if !sort.
int morton_order(const FieldView &fv, long long n, const double *seeds, uint32_t *perm, bool sort, cudaStream_t s);

}  // namespace qsl

struct qsl_field {
    qsl::FieldView view;
    void *d_samples;
    void *d_cells;
    void *d_cells32;          // fp32 coefficient table of the QSL_ARITH_F32 kernel, or NULL
    void *d_row_sc;           // float2[ny] behind view.row_sc, or NULL
    double *d_axis[3];
    int sample_type;
    long long n_nodes;
    size_t bytes;
};
