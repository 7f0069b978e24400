/* qsl.h -- C ABI of libqsl: B200-native (sm_100a) field-line tracing, squashing factor Q, field-line length L,
 * FLEDGE edge maps and adaptive seed refinement, after Tassev & Savcheva, "QSL Squasher" (arXiv:1609.00724).
 * Citations are "PAPER.md:<line>" of the paper text plus the section / equation they fall in; readings of silent
 * or ambiguous passages (A1..A19) are listed in DESIGN.md.
 *
 * Conventions
 *  - Every function returns int: 0 = QSL_OK, < 0 = error (see qsl_strerror).  Nothing throws or aborts across the ABI.
 *  - Unless marked "host", every array argument is a DEVICE pointer owned by the caller (e.g. torch.Tensor.data_ptr());
 *    the library neither frees nor retains it.  The one exception is qsl_field_create, which copies its input into a
 *    library-owned packed buffer released by qsl_field_destroy.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls are asynchronous on that
 *    stream except where a count is returned to the host (qsl_refine's n_children, qsl_hilbert_refine's n_new), which
 *    synchronises the stream.
 *    Scratch memory is taken from the stream-ordered CUDA memory pool of the current device.
 *  - Per-line problems are not errors: they are bits of the per-seed `status` output.
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns QSL_ECUDA.
 */
#ifndef QSL_H
#define QSL_H

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes ------------------------------------------------------------------------------------------ */
#define QSL_OK       0
#define QSL_EINVAL  (-1)   /* bad argument (NULL pointer, size < minimum, unknown enum, inconsistent sizes)       */
#define QSL_ENOMEM  (-2)   /* device or host allocation failed                                                    */
#define QSL_ECUDA   (-3)   /* a CUDA runtime call failed (qsl_last_cuda_error() gives the cudaError_t)             */
#define QSL_ERANGE  (-4)   /* a size exceeds what the implementation indexes (e.g. > 2^31 - 1 nodes per axis)      */
#define QSL_ETOOBIG (-5)   /* the input exceeds the fixed scratch of a *_noalloc entry point (use the pooled one)   */
const char *qsl_strerror(int code);
int qsl_last_cuda_error(void);
/* Library version and the SM architecture the kernels were compiled for (e.g. 100 for sm_100a). */
int qsl_version(void);
int qsl_compiled_arch(void);

/* ---- enums ------------------------------------------------------------------------------------------------ */
enum { QSL_F32 = 0, QSL_F64 = 1 };                       /* storage type of the packed field samples             */
enum { QSL_NORMALIZE_FIRST = 0, QSL_INTERP_FIRST = 1 };  /* PAPER.md:178 (fn. 9) = NORMALIZE_FIRST, the default   */
enum { QSL_RK4 = 0, QSL_EULER = 1, QSL_CK45 = 2 };       /* PAPER.md:141; RK4: BASELINE.json configs (reading A5);
                                                            CK45: adaptive Cash-Karp 5(4), PAPER.md:141, :143 (reading A16) */
enum { QSL_TRACE_L = 0, QSL_TRACE_LQ = 1 };              /* L only (FLEDGE pass) | L and Q                        */
enum { QSL_LAYOUT_CELL_TABLE = 0, QSL_LAYOUT_NODES_ONLY = 1,    /* what qsl_field_create keeps in HBM (see qsl_grid_desc) */
       QSL_LAYOUT_CELL_TABLE_F32 = 2, QSL_LAYOUT_CELL_TABLES_BOTH = 3 };
enum { QSL_TRILINEAR = 0, QSL_TRIQUADRATIC = 2, QSL_TRICUBIC = 3 };   /* interpolation scheme (reading A18) */
enum { QSL_CARTESIAN = 0, QSL_SPHERICAL = 1 };                        /* geometry of the grid axes    */
enum { QSL_ARITH_F64 = 0, QSL_ARITH_F32 = 1 };           /* arithmetic of the integrator (F32 only with F32 samples) */

/* status bits of qsl_trace_out.status */
#define QSL_ST_SEED_OUTSIDE 1u    /* seed not inside the closed trace box: all outputs NaN / 255 / 0             */
#define QSL_ST_NULL_AT_SEED 2u    /* |b(seed)| < null_eps: all outputs NaN / 255 / 0                             */
#define QSL_ST_STALL_F      4u    /* |b| < null_eps met while integrating forwards (line stops there, face 255)   */
#define QSL_ST_STALL_B      8u
#define QSL_ST_CAP_F        16u   /* max_steps or max_length reached forwards                      */
#define QSL_ST_CAP_B        32u
#define QSL_ST_OPEN         64u   /* an end lies on a face other than -z of the trace box     */

/* tuning flags of qsl_trace_params.flags (results never depend on them) */
#define QSL_FLAG_NO_SORT    1u    /* do not Morton-order the seeds before tracing                                  */
#define QSL_FLAG_NO_REFILL  2u    /* one work item per thread instead of the persistent work queue                 */
#define QSL_FLAG_KERNEL_V1  4u    /* corner kernel: 8 AoS sample gathers per RK stage instead of the per-cell table  */
#define QSL_FLAG_KERNEL_FRAME 8u  /* fp64 on a uniform grid: the cell-frame kernel (integer cell index + offset, the
                                     design of the fp32 kernel) instead of the absolute-coordinate cell-table kernel  */

/* ---- field (PAPER.md:54 input cubes; :93-107 eq. 3-4 interpolation; :178 normalise-then-interpolate) --------- */
typedef struct qsl_field qsl_field;          /* opaque, library-owned */

typedef struct {
    int nx, ny, nz;              /* nodes per axis, each >= 2; sample index = (k*ny + j)*nx + i (x fastest)      */
    int stretched;               /* 0: uniform nodes lo + i (hi - lo)/(n - 1); 1: node coordinates xs, ys, zs     */
    double lo[3], hi[3];         /* grid box (ignored when stretched: taken from the coordinate arrays)           */
    const double *xs, *ys, *zs;  /* HOST arrays of nx, ny, nz strictly increasing coordinates; only if stretched  */
    int sample_type;             /* QSL_F32 | QSL_F64: storage type of the packed samples                         */
    int interp_mode;             /* QSL_NORMALIZE_FIRST (paper) | QSL_INTERP_FIRST (reading A2)                   */
    int layout;                  /* QSL_LAYOUT_CELL_TABLE (default): besides the packed node samples, keep per cell the
                                    24 fp64 monomial coefficients of its trilinear interpolant (192 B per cell; 6x the
                                    fp64 samples, 12x the fp32 samples) - what the fast trace kernel reads.
                                    QSL_LAYOUT_NODES_ONLY: packed samples only; qsl_trace then gathers 8 corners per
                                    RK stage (the slower QSL_FLAG_KERNEL_V1 path), for fields too large for the table.
                                    QSL_LAYOUT_CELL_TABLE_F32: the same coefficients rounded to fp32 (96 B per cell),
                                    the table of QSL_ARITH_F32; fp32 samples on a uniform grid only (else QSL_EINVAL;
                                    Cartesian or spherical);
                                    QSL_ARITH_F64 traces of such a field run the corner kernel.
                                    QSL_LAYOUT_CELL_TABLES_BOTH: the fp64 and the fp32 table                          */
    int interp_order;            /* QSL_TRILINEAR (0, default; eq. 3-4) | QSL_TRIQUADRATIC (Dodgson 1997, 27
                                    vertices) | QSL_TRICUBIC (Keys 1981, 64 vertices): PAPER.md:91-93, gradients taken
                                    analytically on the kernels (:123, :137).  The higher orders need >= 3 / >= 4 nodes per
                                    axis and QSL_NORMALIZE_FIRST (else QSL_EINVAL), keep the node samples only (layout is
                                    ignored) and are traced by the gather kernel in fp64 with QSL_RK4 / QSL_EULER         */
    int geometry;                /* QSL_CARTESIAN (0, default) | QSL_SPHERICAL: the axes are (longitude phi, latitude theta,
                                    radius r), angles in radians, and bx, by, bz are the components in the orthonormal basis
                                    (phi^, theta^, r^) (PAPER.md:83-87 eq. 2, :111).  Seeds, trace box and end points are
                                    then (phi, theta, r); lines follow eq. (2), deviations eq. (6)-(7) as printed (without
                                    the metric-derivative terms), Q uses eq. (8); dev_f / dev_b are coordinate
                                    deviations.  Uniform axes, QSL_NORMALIZE_FIRST, QSL_TRILINEAR only (else QSL_EINVAL).
                                    fp64 arithmetic: RK4 / Euler / CK45 in the cell-table kernels (fp64 table layouts) and in the
                                    gather kernels (QSL_LAYOUT_NODES_ONLY / QSL_FLAG_KERNEL_V1); fp32 arithmetic
                                    (QSL_ARITH_F32, RK4 / Euler) on the fp32 table layouts of an fp32-sampled field         */
} qsl_grid_desc;

/* Packs the three component cubes (DEVICE, fp64, nx*ny*nz each) into one AoS array of (b^x, b^y, b^z, |B|) samples
 * [NORMALIZE_FIRST] or (Bx, By, Bz, |B|) [INTERP_FIRST], rounded to sample_type: inputs are first rounded to
 * sample_type, |B| and B/|B| are formed in fp64 with IEEE sqrt / division, then rounded; |B| < 1e-300 gives zeros.
 * Errors: QSL_EINVAL (NULL, n < 2, non-increasing coordinates, unknown enum), QSL_ERANGE, QSL_ENOMEM, QSL_ECUDA.  */
int qsl_field_create(qsl_field **out, const qsl_grid_desc *desc, const double *bx, const double *by,
                     const double *bz, void *stream);
int qsl_field_destroy(qsl_field *f);
/* Test hook: copies the packed samples (nx*ny*nz*4 values of sample_type) to `packed_out` (DEVICE). */
int qsl_field_export(const qsl_field *f, void *packed_out, void *stream);
/* Bytes of device memory held by the field. */
long long qsl_field_bytes(const qsl_field *f);

/* ---- trace (PAPER.md:79 eq. 1; :119 eq. 5; :141 integrators; :156-176 eq. 9-11 Q; :163 boundaries; :165 cap) --- */
typedef struct {
    double box_lo[3], box_hi[3]; /* trace box, inside the grid box; may be smaller (raised lower boundary) */
    int method;                  /* QSL_RK4 | QSL_EULER | QSL_CK45 (fp64 arithmetic; every layout, order and geometry) */
    double step_frac;            /* h = step_frac * min_d h_c,d of the cell containing x; > 0   */
    int mode;                    /* QSL_TRACE_L | QSL_TRACE_LQ                                                      */
    int arith;                   /* QSL_ARITH_F64 | QSL_ARITH_F32                                                   */
    double max_length;           /* cap on the affine parameter lambda per direction; +inf = off     */
    long long max_steps;         /* cap on accepted steps per direction; >= 1                                       */
    double null_eps;             /* stall threshold on |b|                                                          */
    unsigned int flags;          /* QSL_FLAG_*                                                                      */
    double tol;                  /* QSL_CK45 only (> 0): error allowed per step on the position, in units of the
                                    smallest edge of the current cell (PAPER.md:143 uses 1e-2).  The step is
                                    step_frac * min_d h_c,d * 2^j, j in [-20, +2]: a step whose error estimate
                                    |x5 - x4|_max exceeds tol is halved and retried, one below tol/64 doubles the next */
} qsl_trace_params;

typedef struct {                 /* every member may be NULL (output not wanted); n = number of seeds               */
    double *end_f, *end_b;       /* n*3: end points forwards (along +B) / backwards                                 */
    double *L;                   /* n: field-line length L_F + L_B                              */
    double *q_perp;              /* n: eq. (11) verbatim, field-perpendicular projections            */
    double *q_bnd;               /* n: the same bracket with projections along the field onto the end faces and the
                                    normal field components (Titov's Q for face-to-face mapping; reading A1)        */
    unsigned char *face_f, *face_b;       /* n: 0..5 = -x,+x,-y,+y,-z,+z of the trace box; 255 = none (stall / cap) */
    unsigned int *status;        /* n: QSL_ST_* bits                                                                */
    unsigned int *nsteps_f, *nsteps_b;    /* n: accepted steps per direction (the landing step counts once)         */
    double *dev_f, *dev_b;       /* n*6: raw deviation vectors (delta1, delta2) at each end (QSL_TRACE_LQ only)      */
} qsl_trace_out;

/* Traces n seeds (DEVICE, n*3 fp64) forwards and backwards and writes the requested outputs in seed order.
 * total_steps (DEVICE, optional) receives the number of accepted RK steps summed over all lines and directions.
 * n = 0 is valid.  Errors: QSL_EINVAL, QSL_ENOMEM, QSL_ECUDA.                                                       */
int qsl_trace(const qsl_field *f, const qsl_trace_params *p, long long n, const double *seeds,
              const qsl_trace_out *out, unsigned long long *total_steps, void *stream);

/* ---- FLEDGE (Sobel gradient magnitude of the field-line-length map; reading A10) ----------------- */
typedef struct {
    int ndim;                    /* 2 or 3                                                                          */
    long long n[3];              /* level-0 seed lattice dims (n[2] = 1 for 2-D)                                    */
    double origin[3], e0[3], e1[3], e2[3];  /* seed(c) at level l = origin + sum_d (c_d + 0.5)/(n_d 2^l) e_d         */
} qsl_lattice;

typedef struct {
    const qsl_lattice *lat;      /* host                                                                            */
    int nlevels;                 /* number of levels described, >= level + 1                                        */
    const double *L0;            /* DEVICE, dense level-0 map, index (c2*n1 + c1)*n0 + c0                           */
    const long long *count;      /* host [nlevels]; count[0] ignored (level 0 is dense)                             */
    const unsigned int *const *coords;  /* host array [nlevels] of DEVICE pointers: count[l]*ndim integer coords at
                                           level l, in the order qsl_refine emitted them; [0] ignored                */
    const double *const *L;      /* host array [nlevels] of DEVICE pointers: count[l] lengths; [0] ignored          */
    const long long *const *child_base; /* host array [nlevels] of DEVICE pointers: child_base[l][i] = index at level
                                           l+1 of the first of the 2^ndim children of cell i of level l, or -1 if the
                                           cell was not refined (as written by qsl_refine); entries for l >= level
                                           are not read                                                              */
} qsl_levels;

/* Dense map: dims d0 x d1 (x d2), index (c2*d1 + c1)*d0 + c0.  S = sqrt(sum_d G_d^2), G_d = difference [-1,0,1] along
 * d, smoothing [1,2,1] along the other axes, un-normalised, edges replicated.  Non-finite L propagates to S.       */
int qsl_fledge_dense(int ndim, const long long dims[3], const double *L, double *S, void *stream);
/* Sparse level >= 1: the same stencil on the virtual lattice n_d 2^level, a missing neighbour takes the L of its
 * nearest existing ancestor (level 0 is dense).  S (DEVICE) has count[level] entries.                              */
int qsl_fledge_sparse(const qsl_levels *lv, int level, double *S, void *stream);

/* ---- threshold and refinement (BASELINE.json configs[2],[4]; reading A11) --------------------- */
/* tau (DEVICE, 1 double) = the ceil(p N)-th smallest of the N finite values of S (nearest rank); NaN if N = 0.       */
int qsl_select(long long n, const double *S, double p, double *tau, void *stream);
/* For each cell i with S[i] > *tau (NaN never flags), in input order, emits 2^ndim children: coord' = 2 coord + bit
 * (child-index bit d -> axis d) and position = origin + sum_d w_d e_d, w_d = (coord'_d + 0.5)/(n_d 2^(level+1)),
 * accumulated with fma, axis 0 first (bit-reproducible).  coords = NULL means "the dense level-0 lattice in index
 * order" (then level must be 0 and n = n0*n1*n2).  tau is a DEVICE pointer (as written by qsl_select).
 * child_coords (n_out*ndim), child_seeds (n_out*3) hold up to capacity children; child_base (n, optional) receives the
 * index of each cell's first child or -1.  n_children (host) is written after synchronising the stream; if it exceeds
 * `capacity` nothing beyond capacity was written and QSL_ERANGE is returned (call again with larger buffers).       */
int qsl_refine(int ndim, int level, long long n, const unsigned int *coords, const double *S, const double *tau,
               const qsl_lattice *lat, long long capacity, unsigned int *child_coords, double *child_seeds,
               long long *child_base, long long *n_children, void *stream);

/* qsl_refine for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc).  Same operation, same kernels and the same bits in child_coords / child_seeds / child_base as
 * qsl_refine (reading A11), with two differences:
 *  - it calls no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library routine: the per-tile counts of the
 *    stream compaction live in a file-scope device array of the library (256 KiB, held by every GPU that loads libqsl
 *    until the process exits), which limits the call to n <= QSL_REFINE_NOALLOC_MAX_CELLS cells (cfg5's dense level
 *    0 just fits); a larger n returns QSL_ETOOBIG and launches nothing - use qsl_refine;
 *  - n_children is a DEVICE pointer (1 long long) written on the stream; the call never synchronises.  If the count
 *    exceeds `capacity`, nothing beyond capacity was written (no error can be reported: compare on the device or
 *    after the caller's own synchronisation).
 * All calls on a device share the scratch array and it keeps the last call's contents; nothing in it needs clearing
 * (every word a call reads it has written first).  Calls that overlap on the GPU (two streams) race on it: serialise
 * them.  Errors: QSL_EINVAL, QSL_ERANGE (as qsl_refine), QSL_ETOOBIG, QSL_ECUDA.                                      */
#define QSL_REFINE_NOALLOC_MAX_CELLS 67108864LL
int qsl_refine_noalloc(int ndim, int level, long long n, const unsigned int *coords, const double *S, const double *tau,
                       const qsl_lattice *lat, long long capacity, unsigned int *child_coords, double *child_seeds,
                       long long *child_base, long long *n_children, void *stream);

/* ---- test hook ------------------------------------------------------------------------------------------------- */
/* Stable ascending sort of n (key, value) pairs (DEVICE, in place) on the low key_bits (1..32) of the keys: the
 * hand-written LSD radix sort that qsl_trace uses to Morton-order its seeds (PAPER.md:196-198 orders samples along a
 * space-filling curve), exposed so that tests can check it on its own.                                              */
int qsl_debug_sort_pairs(unsigned int *keys, unsigned int *vals, long long n, int key_bits, void *stream);

/* ---- the paper's own refinement along a Hilbert curve (section 3.6; reading A17) -------- *
 * A sample sits at the centre of a cell of the finest lattice n_d 2^R ("fine cell", integer coordinates c); its position
 * is origin + sum_d (c_d + 0.5)/(n_d 2^R) e_d.  Its place along the curve is the 64-bit key of c on the Hilbert curve
 * (Skilling 2004) of `bits` = qsl_hilbert_bits(lat, R) bits per axis; the shifted curve of PAPER.md:204 is the curve of
 * bits + 1 bits through the cells c + shift.  All arrays are DEVICE pointers; coordinates are n*ndim uint32.            */
/* Bits per axis of the cube bounding the finest lattice (>= 1), or QSL_EINVAL / QSL_ERANGE ((bits + 1) ndim > 63).       */
int qsl_hilbert_bits(const qsl_lattice *lat, int R);
/* Level-0 samples in dense order (c2 n1 + c1) n0 + c0: fine cell c0 2^R + 2^(R-1) and its centre (seeds: n*3 fp64).      */
int qsl_hilbert_level0(const qsl_lattice *lat, int R, unsigned int *coords, double *seeds, void *stream);
/* keys[i] = position along the curve of `bits` bits per axis of the cell coords[i] + shift; and the inverse.  coords[i] +
 * shift must stay below 2^bits (the caller's duty; shift >= 2^bits is rejected with QSL_EINVAL, and qsl_hilbert_refine
 * rejects a shift larger than the cube of the un-shifted curve, which is what its one extra bit per axis can hold).      */
int qsl_hilbert_keys(int ndim, int bits, int shift, long long n, const unsigned int *coords, unsigned long long *keys,
                     void *stream);
int qsl_hilbert_cells(int ndim, int bits, int shift, long long n, const unsigned long long *keys, unsigned int *coords,
                      void *stream);
/* Sorts keys ascending in place (stable LSD radix sort on key_bits bits) and writes the permutation: the sorted keys[i] is
 * the input keys[perm[i]].  qsl_gather: dst[i] = src[perm[i]] for elements of elem_bytes (a multiple of 4) bytes.          */
int qsl_sort_keys64(long long n, unsigned long long *keys, unsigned int *perm, int key_bits, void *stream);
int qsl_gather(long long n, const unsigned int *perm, int elem_bytes, const void *src, void *dst, void *stream);
/* One refinement pass over n samples sorted by `keys` (the keys of the shifted curve if shift != 0):
 * between successive samples i, i+1 with both L finite, |L[i+1] - L[i]| > thr and keys[i+1] - keys[i] >= 2 a new sample
 * at key (keys[i] + keys[i+1]) >> 1 - "halfway along the Hilbert curve" - unless that cell (displaced back by shift) lies
 * outside the lattice.  Writes, in curve order, left[j] = i, the fine cell and the position of every new sample, and the
 * count to *n_new (HOST; synchronises the stream).  QSL_ERANGE if the count exceeds `capacity` (*n_new = needed).         */
int qsl_hilbert_refine(const qsl_lattice *lat, int R, int shift, long long n, const unsigned long long *keys, const double *L,
                       double thr, long long capacity, long long *left, unsigned int *new_coords, double *new_seeds,
                       long long *n_new, void *stream);
/* Merges a payload array of the old samples with that of the new ones, keeping the curve order: new sample j goes right
 * after old sample left[j] (left ascending, as written by qsl_hilbert_refine).  out: n_old + n_new elements.               */
int qsl_hilbert_merge(long long n_old, long long n_new, const long long *left, int elem_bytes, const void *old_vals,
                      const void *new_vals, void *out, void *stream);
/* Converter: samples sorted by their un-shifted keys -> dense map on the lattice n_d 2^r (r <= R), index
 * (c2 d1 + c1) d0 + c0: the maximum of the finite Q inside a cell; a cell without sample takes 10^(log10 Q interpolated
 * linearly in the key between the last sample with Q > 0 before the cell's key range and the first after it, at the middle
 * of the range); one-sided at the ends of the curve; NaN if there is no such sample at all.                                 */
int qsl_hilbert_convert(const qsl_lattice *lat, int R, int r, long long n, const unsigned long long *keys, const double *Q,
                        double *out, void *stream);

/* ---- measurement hooks (bench.py) ------------------------------------------------------------------ *
 * Threading: the library keeps per-process state without locks (last CUDA error, launch counter, the profiling event
 * pool below, one private stream-ordered scratch pool per device): drive it from one host thread at a time.             */
/* qsl_profile_enable(1): every later qsl_trace records a CUDA event pair around its trace kernel (the dominant
 * kernel) on the caller's stream (up to 256 launches between two reads).  qsl_profile_trace_kernel_ms waits for the pairs
 * recorded since the previous read (or enable), returns their summed device time in milliseconds and their number per
 * trace mode (host arrays indexed by QSL_TRACE_L, QSL_TRACE_LQ) and forgets them; QSL_EINVAL if there were none.      */
/* Number of kernels the library has launched in this process so far (bench.py's gpu_launches). */
long long qsl_launch_count(void);
int qsl_profile_enable(int on);
int qsl_profile_trace_kernel_ms(double ms[2], long long launches[2]);
/* (The roofline denominators bench.py measures on the device are not part of this library: include/qsl_peaks.h.) */

#ifdef __cplusplus
}
#endif
#endif /* QSL_H */
