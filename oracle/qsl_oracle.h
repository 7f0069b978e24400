/* oracle/qsl_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU restatement of the QSL Squasher hot path (Tassev & Savcheva, arXiv:1609.00724),
 * written from the paper with the readings listed in DESIGN.md ("Readings of the paper").
 * It shares no code with the CUDA path under paper_1609_00724_b200/ and may be used only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Parity pins (tests/test_oracle_pins.py): P1 uniform field Q = 2; P2 hyperbolic closed forms; P3 invariances;
 * P4 finite-difference Jacobian (Pariat & Demoulin style); P5 bounds; P6 RK4 order;
 * P8 scipy.ndimage.sobel; P9 numpy order statistic; P10 brute-force refinement; P12 mode consistency.
 * Rows f1-f4: tests/test_oracle_ck45.py (Cash-Karp: single-step orders 5 / 4 against the exact flow, deviation =
 * derivative of the step map, closed forms, controller invariants), tests/test_oracle_interp.py (Dodgson / Keys kernels:
 * interpolation, linear / quadratic reproduction, C1 / C0, gradient = derivative, convergence orders),
 * tests/test_oracle_spherical.py (monopole Q = 2, dipole line geometry, Cartesian limit), and for oracle/hilbert.py
 * tests/test_oracle_hilbert.py (curve properties, purpose of each pass, merge and converter by brute force).
 * On configs 2-5 no closed form exists: there the oracle itself is the reference ("parity pinned on the
 * analytic cases P1-P6, unpinned in absolute terms on configs 2-5").
 */
#ifndef QSL_ORACLE_H
#define QSL_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_F32 = 0, ORC_F64 = 1 };
enum { ORC_NORMALIZE_FIRST = 0, ORC_INTERP_FIRST = 1 };
enum { ORC_CARTESIAN = 0, ORC_SPHERICAL = 1 };
enum { ORC_TRILINEAR = 1, ORC_TRIQUADRATIC = 2, ORC_TRICUBIC = 3 };
enum { ORC_RK4 = 0, ORC_EULER = 1, ORC_CK45 = 2 };   /* CK45: adaptive Cash-Karp 5(4) */
enum { ORC_TRACE_L = 0, ORC_TRACE_LQ = 1 };

enum {
    ORC_ST_SEED_OUTSIDE = 1u, ORC_ST_NULL_AT_SEED = 2u, ORC_ST_STALL_F = 4u, ORC_ST_STALL_B = 8u,
    ORC_ST_CAP_F = 16u, ORC_ST_CAP_B = 32u, ORC_ST_OPEN = 64u
};

typedef struct {
    int nx, ny, nz;            /* nodes per axis; flat index (k*ny + j)*nx + i                         */
    int stretched;             /* 0: uniform on [lo,hi]; 1: node coordinates xs, ys, zs                 */
    double lo[3], hi[3];
    const double *xs, *ys, *zs;
    int interp_mode;           /* ORC_NORMALIZE_FIRST (paper) | ORC_INTERP_FIRST          */
    const double *packed;      /* n*4 doubles (v0,v1,v2,m): output of orc_field_pack                    */
    int order;                 /* 0 / ORC_TRILINEAR | ORC_TRIQUADRATIC | ORC_TRICUBIC (reading A18) */
    int geometry;              /* ORC_CARTESIAN (0) | ORC_SPHERICAL: axes = (longitude phi, latitude theta, radius r),
                                  components in the orthonormal basis (phi^, theta^, r^)  */
} orc_field;

typedef struct {
    double box_lo[3], box_hi[3];
    int method;                /* ORC_RK4 | ORC_EULER | ORC_CK45                                         */
    double step_frac;          /* h = step_frac * min_d h_c,d                                            */
    int mode;                  /* ORC_TRACE_L | ORC_TRACE_LQ                                             */
    double max_length;         /* cap on the affine parameter per direction; inf = off    */
    long long max_steps;
    double null_eps;
    double basis_angle;        /* rotation of (a, b) about B at the seed -- pin P3 only                  */
    double tol;                /* ORC_CK45: error per step allowed on x, in units of min_d h_c,d         */
} orc_trace_params;

typedef struct {
    double *end_f, *end_b;     /* n*3                                                                    */
    double *L, *q_perp, *q_bnd;
    uint8_t *face_f, *face_b;  /* 0..5 = -x,+x,-y,+y,-z,+z ; 255 = none                                  */
    uint32_t *status, *nsteps_f, *nsteps_b;
    double *dev_f, *dev_b;     /* n*6: raw (delta1, delta2) at each end; may be NULL                     */
} orc_trace_out;

/* O0 (PAPER.md:178 fn. 9, :176): samples -> packed (v,m) rounded to the storage type, widened to double. */
void orc_field_pack(long long n_nodes, const double *bx, const double *by, const double *bz,
                    int sample_type, int interp_mode, double *packed);

/* O1 (PAPER.md:93-107 eq. 3-4, :123, :137): b[3], J[9] (J[c*3+d] = d b_c / d x_d), m, h_cell[3]. */
void orc_evaluate(const orc_field *F, const double x[3], double b[3], double J[9], double *m, double hc[3]);
/* One Cash-Karp 5(4) step of size h of the state y = (x, delta1, delta2, L): yn = 5th-order result, err3 = y5 - y4 of x. */
void orc_ck_step(const orc_field *F, int with_dev, double s, const double y[10], double h, double yn[10], double err3[3]);

/* O2-O5 (PAPER.md:79 eq.1, :119 eq.5, :141, :156-176 eq.9-11, :163, :165). */
void orc_trace(const orc_field *F, const orc_trace_params *P, long long n, const double *seeds,
               const orc_trace_out *out, unsigned long long *total_steps, int nthreads);

/* O6: Sobel gradient magnitude of the field-line-length map. */
void orc_fledge_dense(int ndim, const long long dims[3], const double *L, double *S);
void orc_fledge_sparse(int ndim, const long long n0[3], int level, const double *L0,
                       const long long *count /* [level+1], count[0] unused */,
                       const uint32_t *const *coords /* [level+1] */, const double *const *L /* [level+1] */,
                       double *S /* count[level] */);

/* O7 (BASELINE.json configs[2],[4]). */
double orc_select(long long n, const double *S, double p);
long long orc_refine(int ndim, int level, long long n, const uint32_t *coords, const double *S, double tau,
                     const long long n0[3], const double origin[3], const double e0[3], const double e1[3],
                     const double e2[3], uint32_t *child_coords, double *child_seeds);

#ifdef __cplusplus
}
#endif
#endif
