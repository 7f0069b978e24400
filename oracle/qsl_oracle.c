/* oracle/qsl_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see qsl_oracle.h).
 *
 * Plain fp64, one field line at a time, OpenMP threads over seeds.  Every function follows the passage it
 * cites, in the paper's order and notation; readings of silent / ambiguous passages are those of DESIGN.md
 * (A1..A14).  Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no FMA contraction: arithmetic is
 * exactly as written; the only fused operation is the explicit fma() of the refinement positions, O7).
 */
#include "qsl_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------------ O0 */
/* PAPER.md:178 (fn. 9): "we first normalize the magnetic field data cubes, and only then interpolate them";
 * B_F, B_B, B_0 are the unnormalised magnitudes, so |B| is kept as a 4th sample.           */
static double round_to(double v, int sample_type) { return sample_type == ORC_F32 ? (double)(float)v : v; }

void orc_field_pack(long long n_nodes, const double *bx, const double *by, const double *bz,
                    int sample_type, int interp_mode, double *packed)
{
    for (long long p = 0; p < n_nodes; ++p) {
        double B[3] = { round_to(bx[p], sample_type), round_to(by[p], sample_type), round_to(bz[p], sample_type) };
        double m = sqrt((B[0] * B[0] + B[1] * B[1]) + B[2] * B[2]);
        double v[3];
        if (interp_mode == ORC_NORMALIZE_FIRST) {
            if (m < 1e-300) { v[0] = v[1] = v[2] = 0.0; m = 0.0; }
            else { v[0] = B[0] / m; v[1] = B[1] / m; v[2] = B[2] / m; }
        } else {
            v[0] = B[0]; v[1] = B[1]; v[2] = B[2];
        }
        packed[4 * p + 0] = round_to(v[0], sample_type);
        packed[4 * p + 1] = round_to(v[1], sample_type);
        packed[4 * p + 2] = round_to(v[2], sample_type);
        packed[4 * p + 3] = round_to(m, sample_type);
    }
}

/* ------------------------------------------------------------------------------------------------ O1 */
/* "identify the cell within the input array within which x lies ... denote by c that vertex,
 * which lies closest to the origin"; h_c = physical dimensions of that cell.
 * Reading A8: node-sampled grid, index clamped to [0, n-2], fraction NOT clamped (linear extrapolation).  */
static void locate_axis(const orc_field *F, int d, double x, int *i_out, double *t_out, double *h_out)
{
    const int n = d == 0 ? F->nx : (d == 1 ? F->ny : F->nz);
    int i;
    if (!F->stretched) {
        const double h = (F->hi[d] - F->lo[d]) / (double)(n - 1);
        const double u = (x - F->lo[d]) / h;
        double fi = floor(u);
        if (!(fi >= 0.0)) fi = 0.0;                 /* also catches NaN */
        if (fi > (double)(n - 2)) fi = (double)(n - 2);
        i = (int)fi;
        *t_out = u - (double)i;
        *h_out = h;
    } else {
        const double *xs = d == 0 ? F->xs : (d == 1 ? F->ys : F->zs);
        /* largest i with xs[i] <= x, clamped to [0, n-2] */
        int lo = 0, hi = n - 1;                      /* invariant: xs[lo] <= x < xs[hi] (after clamping) */
        if (!(x >= xs[0])) i = 0;
        else if (x >= xs[n - 1]) i = n - 2;
        else {
            while (hi - lo > 1) { int mid = (lo + hi) / 2; if (xs[mid] <= x) lo = mid; else hi = mid; }
            i = lo;
        }
        if (i > n - 2) i = n - 2;
        const double h = xs[i + 1] - xs[i];
        *t_out = (x - xs[i]) / h;
        *h_out = h;
    }
    *i_out = i;
}

/* PAPER.md:95 (eq. 3): B^(x) = sum_v B^{v+c} f_v(x - x_c; h_c); PAPER.md:101-107 (eq. 4): trilinear kernels
 * f_{abc} = w_a(x0/h0) w_b(x1/h1) w_c(x2/h2), w_0(t) = 1-t, w_1(t) = t.  PAPER.md:123, 137: the gradient acts
 * only on the kernels and is taken analytically: d w_0/dx = -1/h, d w_1/dx = +1/h.                         */
static void finish_evaluate(const orc_field *F, const double val[4], double grad[4][3], double b[3], double J[9], double *m)
{
    if (F->interp_mode == ORC_NORMALIZE_FIRST) {
        /* the interpolant of the pre-normalised samples, "not guaranteed to be a unit vector" */
        for (int c = 0; c < 3; ++c) { b[c] = val[c]; for (int d = 0; d < 3; ++d) J[c * 3 + d] = grad[c][d]; }
        *m = val[3];
    } else {
        /* reading A2: interpolate B, then normalise: b = B/|B|, J = (G - u (u^T G))/|B| */
        const double n = sqrt((val[0] * val[0] + val[1] * val[1]) + val[2] * val[2]);
        if (n < 1e-300) { for (int c = 0; c < 3; ++c) b[c] = 0.0; for (int q = 0; q < 9; ++q) J[q] = 0.0; *m = 0.0; }
        else {
            double u[3] = { val[0] / n, val[1] / n, val[2] / n };
            for (int d = 0; d < 3; ++d) {
                const double uG = (u[0] * grad[0][d] + u[1] * grad[1][d]) + u[2] * grad[2][d];
                for (int c = 0; c < 3; ++c) J[c * 3 + d] = (grad[c][d] - u[c] * uG) / n;
            }
            for (int c = 0; c < 3; ++c) b[c] = u[c];
            *m = n;
        }
    }
}

/* "The available interpolation schemes are trilinear, triquadratic (Dodgson 1997) and tricubic (Keys
 * 1981) ... The interpolation kernels cover 8, 27, or 64 vertices neighboring that cell"; eq. (3): the kernels are
 * functions of (x - x_c)/h_c of the cell containing x, whatever the spacing of the neighbouring cells.  Reading A18,
 * written out as its plain definition: per axis the interpolant is  sum_nodes f(node) K(u_node),  u_node = distance
 * from the node to x in units of the cell containing x, K the published one-dimensional kernel:
 *  tricubic     Keys' cubic convolution kernel with a = -1/2:
 *               K(u) = 3/2 u^3 - 5/2 u^2 + 1 (0 <= u <= 1),  -1/2 u^3 + 5/2 u^2 - 4 u + 2 (1 <= u <= 2),  0 beyond,
 *               on the nodes i-1 .. i+2, whose distances to x are u = t+1, t, 1-t, 2-t with t = (x - x_i)/h_i;
 *  triquadratic Dodgson's interpolating quadratic kernel (r = 1):
 *               K(u) = 1 - 2 u^2 (u <= 1/2),  u^2 - 5/2 u + 3/2 (1/2 <= u <= 3/2),  0 beyond,
 *               on the node j nearest to x (t >= 1/2 -> j = i + 1) and its two neighbours, distances 1+s, |s|, 1-s with
 *               s = t - (j - i).
 * Which piece of K a stencil node takes follows from its place in the stencil (inner / outer node), and u is the
 * distance written as the expression above, positive for x inside the cell.  Reading A8 (cell index clamped, fraction
 * not): for a stage point outside the grid, t < 0 or t > 1, the same expressions are used, i.e. the polynomial of the
 * boundary cell is continued, as the trilinear kernels 1-t, t are.
 * The gradient acts on the kernels only: d/dx K(u) = K'(u) (du/dt) / h with du/dt = +-1. */
static double keys_piece(int outer, double u, double *dk)
{
    if (!outer) { *dk = 4.5 * u * u - 5.0 * u; return (1.5 * u * u * u - 2.5 * u * u) + 1.0; }
    *dk = (-1.5 * u * u + 5.0 * u) - 4.0;
    return ((-0.5 * u * u * u + 2.5 * u * u) - 4.0 * u) + 2.0;
}

static double dodgson_piece(int outer, double u, double *dk)
{
    if (!outer) { *dk = -4.0 * u; return 1.0 - 2.0 * u * u; }
    *dk = 2.0 * u - 2.5;
    return (u * u - 2.5 * u) + 1.5;
}

/* Reading A18, boundary rule: a stencil node outside the grid takes the extrapolated VALUE
 *   tricubic (Keys 1981, his boundary condition):  f_-1 = 3 f_0 - 3 f_1 + f_2,  f_n = 3 f_{n-1} - 3 f_{n-2} + f_{n-3};
 *   triquadratic (linear extrapolation):           f_-1 = 2 f_0 - f_1,          f_n = 2 f_{n-1} - f_{n-2},
 * applied axis by axis (x, then y, then z) to the packed samples (b^_x, b^_y, b^_z, |B|). */
static void sample_ext(const orc_field *F, int ix, int iy, int iz, double out[4])
{
    const int nn[3] = { F->nx, F->ny, F->nz };
    int id[3] = { ix, iy, iz };
    for (int d = 0; d < 3; ++d) {
        if (id[d] >= 0 && id[d] <= nn[d] - 1) continue;
        const int e = id[d] < 0 ? 0 : nn[d] - 1, st = id[d] < 0 ? 1 : -1;      /* edge node and the inward direction */
        double f0[4], f1[4], f2[4];
        int q[3] = { id[0], id[1], id[2] };
        q[d] = e;          sample_ext(F, q[0], q[1], q[2], f0);
        q[d] = e + st;     sample_ext(F, q[0], q[1], q[2], f1);
        if (F->order == ORC_TRICUBIC) {
            q[d] = e + 2 * st; sample_ext(F, q[0], q[1], q[2], f2);
            for (int c = 0; c < 4; ++c) out[c] = (3.0 * f0[c] - 3.0 * f1[c]) + f2[c];
        } else {
            for (int c = 0; c < 4; ++c) out[c] = 2.0 * f0[c] - f1[c];
        }
        return;
    }
    const double *sp = F->packed + 4 * (((long long)iz * F->ny + iy) * F->nx + ix);
    for (int c = 0; c < 4; ++c) out[c] = sp[c];
}

/* Stencil of one axis: first node index (may be -1, last may be n: sample_ext supplies the value), kernel weights and
 * their x-derivatives.  Returns the number of stencil nodes. */
static int axis_stencil(int order, int i, double t, double h, int *first, double w[4], double dw[4])
{
    if (order == ORC_TRICUBIC) {
        *first = i - 1;
        const double u[4] = { t + 1.0, t, 1.0 - t, 2.0 - t }, sg[4] = { 1.0, 1.0, -1.0, -1.0 };
        for (int k = 0; k < 4; ++k) { w[k] = keys_piece(k == 0 || k == 3, u[k], &dw[k]); dw[k] = sg[k] * dw[k] / h; }
        return 4;
    }
    const int j = t >= 0.5 ? i + 1 : i;              /* nearest node */
    const double s = t - (double)(j - i);
    *first = j - 1;
    const double u[3] = { 1.0 + s, s, 1.0 - s }, sg[3] = { 1.0, 1.0, -1.0 };
    for (int k = 0; k < 3; ++k) { w[k] = dodgson_piece(k != 1, u[k], &dw[k]); dw[k] = sg[k] * dw[k] / h; }
    return 3;
}

void orc_evaluate(const orc_field *F, const double x[3], double b[3], double J[9], double *m, double hc[3])
{
    int i[3]; double t[3], h[3];
    for (int d = 0; d < 3; ++d) locate_axis(F, d, x[d], &i[d], &t[d], &h[d]);
    if (F->order == ORC_TRIQUADRATIC || F->order == ORC_TRICUBIC) {
        int first[3], cnt[3]; double ww[3][4], dww[3][4];
        for (int d = 0; d < 3; ++d) cnt[d] = axis_stencil(F->order, i[d], t[d], h[d], &first[d], ww[d], dww[d]);
        double val[4] = { 0, 0, 0, 0 }, grad[4][3] = { { 0 } };
        for (int c = 0; c < cnt[2]; ++c)
            for (int bb = 0; bb < cnt[1]; ++bb)
                for (int a = 0; a < cnt[0]; ++a) {
                    double sv[4];
                    sample_ext(F, first[0] + a, first[1] + bb, first[2] + c, sv);
                    const double f = ww[0][a] * ww[1][bb] * ww[2][c];
                    const double f0 = dww[0][a] * ww[1][bb] * ww[2][c];
                    const double f1 = ww[0][a] * dww[1][bb] * ww[2][c];
                    const double f2 = ww[0][a] * ww[1][bb] * dww[2][c];
                    for (int q = 0; q < 4; ++q) {
                        val[q] += sv[q] * f;
                        grad[q][0] += sv[q] * f0; grad[q][1] += sv[q] * f1; grad[q][2] += sv[q] * f2;
                    }
                }
        finish_evaluate(F, val, grad, b, J, m);
        if (hc) { hc[0] = h[0]; hc[1] = h[1]; hc[2] = h[2]; }
        return;
    }
    double w[3][2], dw[3][2];
    for (int d = 0; d < 3; ++d) {
        w[d][0] = 1.0 - t[d]; w[d][1] = t[d];
        dw[d][0] = -1.0 / h[d]; dw[d][1] = 1.0 / h[d];
    }
    double val[4] = { 0, 0, 0, 0 }, grad[4][3] = { { 0 } };
    for (int c = 0; c < 2; ++c)
        for (int bb = 0; bb < 2; ++bb)
            for (int a = 0; a < 2; ++a) {
                const long long p = ((long long)(i[2] + c) * F->ny + (i[1] + bb)) * F->nx + (i[0] + a);
                const double *s = F->packed + 4 * p;
                const double f = w[0][a] * w[1][bb] * w[2][c];
                const double f0 = dw[0][a] * w[1][bb] * w[2][c];
                const double f1 = w[0][a] * dw[1][bb] * w[2][c];
                const double f2 = w[0][a] * w[1][bb] * dw[2][c];
                for (int q = 0; q < 4; ++q) {
                    val[q] += s[q] * f;
                    grad[q][0] += s[q] * f0; grad[q][1] += s[q] * f1; grad[q][2] += s[q] * f2;
                }
            }
    finish_evaluate(F, val, grad, b, J, m);
    if (hc) { hc[0] = h[0]; hc[1] = h[1]; hc[2] = h[2]; }
}

static double norm3(const double v[3]) { return sqrt((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]); }
static double dot3(const double a[3], const double b[3]) { return (a[0] * b[0] + a[1] * b[1]) + a[2] * b[2]; }

/* ------------------------------------------------------------------------------------------------ O3 */
/* State y = (x[3], delta1[3], delta2[3], L).  f(y) = (s b, s J delta1, s J delta2, |b|):
 * PAPER.md:79 (eq. 1) d x/d lambda = B^(x); PAPER.md:119 (eq. 5) d delta/d lambda = (delta . grad) B^;
 * reading A3: L = integral of |b_interp| d lambda (arc length of the numerical curve) as a 10th component. */
/* Spherical geometry (reading A19): y = (phi, theta, r, delta phi, delta theta, delta r, ..., L), angles in radians,
 * theta = latitude.  PAPER.md:83-85 (eq. 2): r cos(theta) phi' = B^_phi, r theta' = B^_theta, r' = B^_r.
 * PAPER.md:125-135 (eq. 6, 7): r cos(theta) (delta phi)' = (delta u . grad_u) B^_phi, r (delta theta)' = (delta u . grad_u)
 * B^_theta, (delta r)' = (delta u . grad_u) B^_r with grad_u = (d/dphi, d/dtheta, d/dr) acting on the interpolation kernels
 * only - as printed, i.e. without the derivatives of the metric factors (fn. 8).                     */
static void metric(const orc_field *F, const double y[10], double mf[3])
{
    if (F->geometry == ORC_SPHERICAL) { mf[0] = 1.0 / (y[2] * cos(y[1])); mf[1] = 1.0 / y[2]; mf[2] = 1.0; }
    else { mf[0] = mf[1] = mf[2] = 1.0; }
}

static void rhs(const orc_field *F, int with_dev, double s, const double y[10], double dy[10], double *bnorm,
                double hc[3])
{
    double b[3], J[9], m, mf[3];
    orc_evaluate(F, y, b, J, &m, hc);
    metric(F, y, mf);
    for (int c = 0; c < 3; ++c) dy[c] = s * b[c] * mf[c];
    for (int v = 0; v < 2; ++v) {
        const double *dl = y + 3 + 3 * v;
        for (int c = 0; c < 3; ++c)
            dy[3 + 3 * v + c] = with_dev ? s * ((J[c * 3 + 0] * dl[0] + J[c * 3 + 1] * dl[1]) + J[c * 3 + 2] * dl[2]) * mf[c] : 0.0;
    }
    dy[9] = norm3(b);
    if (bnorm) *bnorm = dy[9];
    if (hc && F->geometry == ORC_SPHERICAL) { hc[0] *= y[2] * cos(y[1]); hc[1] *= y[2]; }   /* physical cell edges */
}

/* Cash & Karp (1990) embedded pair, the scheme behind the paper's adaptive stepper: six stages,
 * nodes c, coupling a, 5th-order weights b5 (the propagated solution) and 4th-order weights b4 of the embedded
 * solution; y5 - y4 estimates the local error.  Written out as printed in the literature.                    */
static const double CK_A[6][5] = {
    { 0.0, 0.0, 0.0, 0.0, 0.0 },
    { 1.0 / 5.0, 0.0, 0.0, 0.0, 0.0 },
    { 3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0 },
    { 3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0.0, 0.0 },
    { -11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0.0 },
    { 1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0 } };
static const double CK_B5[6] = { 37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0 };
static const double CK_B4[6] = { 2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0, 277.0 / 14336.0, 1.0 / 4.0 };

/* One Cash-Karp step of size h from y given k1 = f(y): yn = 5th-order solution, err3 = (y5 - y4) of the position. */
static void ck_step(const orc_field *F, int with_dev, double s, const double y[10], const double k1[10], double h,
                    double yn[10], double err3[3])
{
    double k[6][10], yt[10];
    memcpy(k[0], k1, sizeof k[0]);
    for (int i = 1; i < 6; ++i) {
        for (int q = 0; q < 10; ++q) {
            double acc = 0.0;
            for (int j = 0; j < i; ++j) acc += CK_A[i][j] * k[j][q];
            yt[q] = y[q] + h * acc;
        }
        rhs(F, with_dev, s, yt, k[i], NULL, NULL);
    }
    for (int q = 0; q < 10; ++q) {
        double a5 = 0.0;
        for (int i = 0; i < 6; ++i) a5 += CK_B5[i] * k[i][q];
        yn[q] = y[q] + h * a5;
    }
    for (int d = 0; d < 3; ++d) {
        double e = 0.0;
        for (int i = 0; i < 6; ++i) e += (CK_B5[i] - CK_B4[i]) * k[i][d];
        err3[d] = h * e;
    }
}

/* Pin hook: one Cash-Karp step from y (k1 computed here). */
void orc_ck_step(const orc_field *F, int with_dev, double s, const double y[10], double h, double yn[10], double err3[3])
{
    double k1[10];
    rhs(F, with_dev, s, y, k1, NULL, NULL);
    ck_step(F, with_dev, s, y, k1, h, yn, err3);
}

static void take_step(const orc_field *F, const orc_trace_params *P, int with_dev, double s,
                      const double y[10], const double k1[10], double h, double yn[10])
{
    if (P->method == ORC_EULER) {
        for (int q = 0; q < 10; ++q) yn[q] = y[q] + h * k1[q];
        return;
    }
    if (P->method == ORC_CK45) {
        double err3[3];
        ck_step(F, with_dev, s, y, k1, h, yn, err3);
        return;
    }
    double k2[10], k3[10], k4[10], yt[10];
    for (int q = 0; q < 10; ++q) yt[q] = y[q] + (0.5 * h) * k1[q];
    rhs(F, with_dev, s, yt, k2, NULL, NULL);
    for (int q = 0; q < 10; ++q) yt[q] = y[q] + (0.5 * h) * k2[q];
    rhs(F, with_dev, s, yt, k3, NULL, NULL);
    for (int q = 0; q < 10; ++q) yt[q] = y[q] + h * k3[q];
    rhs(F, with_dev, s, yt, k4, NULL, NULL);
    for (int q = 0; q < 10; ++q) yn[q] = y[q] + (h / 6.0) * ((k1[q] + 2.0 * k2[q]) + (2.0 * k3[q] + k4[q]));
}

static int inside_box(const orc_trace_params *P, const double x[3])
{
    for (int d = 0; d < 3; ++d) if (!(x[d] >= P->box_lo[d] && x[d] <= P->box_hi[d])) return 0;
    return 1;
}

typedef struct { double y[10]; double lam; uint32_t nsteps; int face; int stall, cap; } dir_result;

/* ------------------------------------------------------------------------------------------------ O4 */
/* integrate "forwards to lambda_F, and then backwards to lambda_B ... for which x(lambda)
 * reaches the boundary of the region ... (irrespective of which boundary: bottom, top or side)";
 * optional fixed maximum field-line length.  Reading A4 (landing: chord fraction, exactly
 * three Newton updates, snap), A9 (stall / cap).                                                          */
static void trace_direction(const orc_field *F, const orc_trace_params *P, int with_dev, double s,
                            const double y0[10], dir_result *R)
{
    double y[10]; memcpy(y, y0, sizeof y);
    double lam = 0.0; uint32_t nsteps = 0;
    R->face = 255; R->stall = 0; R->cap = 0;
    /* ORC_CK45 (reading A16): the step is h = step_frac * min_d h_c,d * 2^j with the integer j in [-20, +2] as
     * the controller state.  After a trial step the error e = max_d |y5_d - y4_d| / (tol * min_d h_c,d) of the
     * POSITION decides: e > 1 (and j > -20) rejects and halves (j - 1); an accepted step with e < 1/64 doubles
     * the next one (j + 1, at most +2).  Halving / doubling is exact in binary floating point, so two
     * implementations take identical decisions; controlling x only keeps x and L independent of the mode.  */
    int j = 0;
    for (;;) {
        double k1[10], bnorm, hc[3];                   /* hc = h_c of the cell containing x */
        rhs(F, with_dev, s, y, k1, &bnorm, hc);
        if (!(bnorm >= P->null_eps)) { R->stall = 1; break; }
        if ((long long)nsteps >= P->max_steps) { R->cap = 1; break; }
        if (lam >= P->max_length) { R->cap = 1; break; }
        const double hmin = fmin(hc[0], fmin(hc[1], hc[2]));
        double h = P->step_frac * hmin;
        if (P->method == ORC_CK45) h = ldexp(h, j);
        if (lam + h > P->max_length) h = P->max_length - lam;
        double yn[10];
        if (P->method == ORC_CK45) {
            double err3[3];
            ck_step(F, with_dev, s, y, k1, h, yn, err3);
            const double e = fmax(fabs(err3[0]), fmax(fabs(err3[1]), fabs(err3[2]))) / (P->tol * hmin);
            if (e > 1.0 && j > -20) { --j; continue; }                     /* reject: halve and retry from y */
            if (inside_box(P, yn)) {
                memcpy(y, yn, sizeof y); lam += h; ++nsteps;
                if (e < 1.0 / 64.0 && j < 2) ++j;
                continue;
            }
        } else {
            take_step(F, P, with_dev, s, y, k1, h, yn);
            if (inside_box(P, yn)) { memcpy(y, yn, sizeof y); lam += h; ++nsteps; continue; }
        }
        /* the trial point left the box: first face crossed by the chord (smallest fraction; tie -> lowest
         * axis; one axis cannot violate both of its faces) */
        double phi = INFINITY, bound = 0.0; int axis = -1, face = 255;
        for (int d = 0; d < 3; ++d) {
            if (yn[d] < P->box_lo[d]) {
                double f = (P->box_lo[d] - y[d]) / (yn[d] - y[d]);
                if (f < phi) { phi = f; axis = d; face = 2 * d; bound = P->box_lo[d]; }
            } else if (yn[d] > P->box_hi[d]) {
                double f = (P->box_hi[d] - y[d]) / (yn[d] - y[d]);
                if (f < phi) { phi = f; axis = d; face = 2 * d + 1; bound = P->box_hi[d]; }
            }
        }
        if (axis < 0) { R->stall = 1; break; }         /* non-finite trial point */
        double hp = phi * h;
        for (int it = 0; it < 3; ++it) {               /* exactly three Newton updates of the step length */
            double yt[10], bt[3], Jt[9], mt;
            take_step(F, P, with_dev, s, y, k1, hp, yt);
            orc_evaluate(F, yt, bt, Jt, &mt, NULL);
            double mft[3]; metric(F, yt, mft);
            const double g = s * bt[axis] * mft[axis];
            const double r = yt[axis] - bound;
            if (g != 0.0) {
                double hn = hp - r / g;
                if (hn == hn) { if (hn < 0.0) hn = 0.0; if (hn > h) hn = h; hp = hn; }
            }
        }
        take_step(F, P, with_dev, s, y, k1, hp, yn);
        yn[axis] = bound;                              /* snap exactly onto the face */
        memcpy(y, yn, sizeof y); lam += hp; ++nsteps; R->face = face;
        break;
    }
    memcpy(R->y, y, sizeof y); R->lam = lam; R->nsteps = nsteps;
}

/* ------------------------------------------------------------------------------------------------ O5 */
/* delta x_perp = delta x - B^ (B^ . delta x), B^ evaluated at x(lambda) and explicitly
 * re-normalised.  PAPER.md:169 (eq. 10): a_F, a_B, b_F, b_B.  PAPER.md:174 (eq. 11):
 *   Q = B_F B_B / B_0^2 [ a_F^2 b_B^2 + a_B^2 b_F^2 - 2 (a_B . b_B)(a_F . b_F) ].
 * Reading A1: q_perp is eq. (11) verbatim; q_bnd uses the projection along the field onto the boundary
 * face (normal n_E) and the normal field component, which is Titov's Q for boundary-to-boundary mapping. */
typedef struct { double a[3], b[3], m; } end_proj;

static void project_end(const orc_field *F, const dir_result *R, int bnd, end_proj *E)
{
    double bE[3], J[9], mE;
    orc_evaluate(F, R->y, bE, J, &mE, NULL);
    const double nb = norm3(bE);
    const double u[3] = { bE[0] / nb, bE[1] / nb, bE[2] / nb };
    double d1[3], d2[3];
    {   /* PAPER.md:156 (eq. 8): delta x_phi = r cos(theta) delta phi, delta x_theta = r delta theta, delta x_r = delta r */
        double mf[3]; metric(F, R->y, mf);
        for (int c = 0; c < 3; ++c) { d1[c] = R->y[3 + c] / mf[c]; d2[c] = R->y[6 + c] / mf[c]; }
    }
    if (bnd && R->face != 255) {
        const int ax = R->face / 2;                    /* n_E = unit vector of that axis */
        const double un = u[ax];
        const double c1 = d1[ax] / un, c2 = d2[ax] / un;
        for (int c = 0; c < 3; ++c) { E->a[c] = d1[c] - u[c] * c1; E->b[c] = d2[c] - u[c] * c2; }
        E->m = mE * fabs(un);
    } else {
        const double c1 = dot3(u, d1), c2 = dot3(u, d2);
        for (int c = 0; c < 3; ++c) { E->a[c] = d1[c] - u[c] * c1; E->b[c] = d2[c] - u[c] * c2; }
        E->m = mE;
    }
}

static double q_eq11(const end_proj *Fw, const end_proj *Bw, double m0)
{
    const double aF2 = dot3(Fw->a, Fw->a), bF2 = dot3(Fw->b, Fw->b);
    const double aB2 = dot3(Bw->a, Bw->a), bB2 = dot3(Bw->b, Bw->b);
    const double abF = dot3(Fw->a, Fw->b), abB = dot3(Bw->a, Bw->b);
    return (Fw->m * Bw->m) / (m0 * m0) * ((aF2 * bB2 + aB2 * bF2) - 2.0 * (abB * abF));
}

static void trace_one(const orc_field *F, const orc_trace_params *P, const double seed[3], long long idx,
                      const orc_trace_out *O, unsigned long long *steps)
{
    const double nan = NAN;
    uint32_t st = 0;
    double b0[3], J0[9], m0;
    int ok = inside_box(P, seed);
    if (!ok) st |= ORC_ST_SEED_OUTSIDE;
    if (ok) {
        orc_evaluate(F, seed, b0, J0, &m0, NULL);
        if (!(norm3(b0) >= P->null_eps)) { st |= ORC_ST_NULL_AT_SEED; ok = 0; }
    }
    if (!ok) {
        for (int c = 0; c < 3; ++c) { if (O->end_f) O->end_f[3 * idx + c] = nan; if (O->end_b) O->end_b[3 * idx + c] = nan; }
        if (O->L) O->L[idx] = nan;
        if (O->q_perp) O->q_perp[idx] = nan;
        if (O->q_bnd) O->q_bnd[idx] = nan;
        if (O->face_f) O->face_f[idx] = 255;
        if (O->face_b) O->face_b[idx] = 255;
        if (O->nsteps_f) O->nsteps_f[idx] = 0;
        if (O->nsteps_b) O->nsteps_b[idx] = 0;
        if (O->dev_f) for (int c = 0; c < 6; ++c) O->dev_f[6 * idx + c] = nan;
        if (O->dev_b) for (int c = 0; c < 6; ++c) O->dev_b[6 * idx + c] = nan;
        if (O->status) O->status[idx] = st;
        return;
    }
    /* O2. PAPER.md:160 (eq. 9), :163: a^, b^ and B^(x0) form an orthonormal basis.  Reading A7: e = axis of
     * the smallest |u_d| (tie -> lowest d), a^ = (e - u (u.e))/|..|, b^ = u x a^.                         */
    const double nb0 = norm3(b0);
    const double u[3] = { b0[0] / nb0, b0[1] / nb0, b0[2] / nb0 };
    int e = 0;
    if (fabs(u[1]) < fabs(u[e])) e = 1;
    if (fabs(u[2]) < fabs(u[e])) e = 2;
    double a[3] = { -u[0] * u[e], -u[1] * u[e], -u[2] * u[e] };
    a[e] += 1.0;
    const double na = norm3(a);
    for (int c = 0; c < 3; ++c) a[c] /= na;
    double bp[3] = { u[1] * a[2] - u[2] * a[1], u[2] * a[0] - u[0] * a[2], u[0] * a[1] - u[1] * a[0] };
    if (P->basis_angle != 0.0) {                       /* pin P3: any orthonormal pair must give the same Q */
        const double cs = cos(P->basis_angle), sn = sin(P->basis_angle);
        for (int c = 0; c < 3; ++c) { const double a0 = a[c], b1 = bp[c]; a[c] = cs * a0 + sn * b1; bp[c] = cs * b1 - sn * a0; }
    }
    const int with_dev = P->mode == ORC_TRACE_LQ;
    {   /* the pair is orthonormal in the orthonormal basis; the state carries coordinate deviations (eq. 8 inverted) */
        double y00[10] = { seed[0], seed[1], seed[2] }, mf[3];
        metric(F, y00, mf);
        for (int c = 0; c < 3; ++c) { a[c] *= mf[c]; bp[c] *= mf[c]; }
    }
    double y0[10] = { seed[0], seed[1], seed[2], a[0], a[1], a[2], bp[0], bp[1], bp[2], 0.0 };
    if (!with_dev) for (int c = 3; c < 9; ++c) y0[c] = 0.0;
    dir_result RF, RB;
    trace_direction(F, P, with_dev, +1.0, y0, &RF);
    trace_direction(F, P, with_dev, -1.0, y0, &RB);
    if (RF.stall) st |= ORC_ST_STALL_F;
    if (RB.stall) st |= ORC_ST_STALL_B;
    if (RF.cap) st |= ORC_ST_CAP_F;
    if (RB.cap) st |= ORC_ST_CAP_B;
    /* open lines reach the top or a side boundary; here: an end on a face other than -z */
    if ((RF.face != 255 && RF.face != 4) || (RB.face != 255 && RB.face != 4)) st |= ORC_ST_OPEN;
    for (int c = 0; c < 3; ++c) { if (O->end_f) O->end_f[3 * idx + c] = RF.y[c]; if (O->end_b) O->end_b[3 * idx + c] = RB.y[c]; }
    if (O->L) O->L[idx] = RF.y[9] + RB.y[9];           /* field-line length */
    if (O->face_f) O->face_f[idx] = (uint8_t)RF.face;
    if (O->face_b) O->face_b[idx] = (uint8_t)RB.face;
    if (O->nsteps_f) O->nsteps_f[idx] = RF.nsteps;
    if (O->nsteps_b) O->nsteps_b[idx] = RB.nsteps;
    if (O->status) O->status[idx] = st;
    if (O->dev_f) for (int c = 0; c < 6; ++c) O->dev_f[6 * idx + c] = with_dev ? RF.y[3 + c] : nan;
    if (O->dev_b) for (int c = 0; c < 6; ++c) O->dev_b[6 * idx + c] = with_dev ? RB.y[3 + c] : nan;
    if (with_dev) {
        end_proj EF, EB;
        project_end(F, &RF, 0, &EF); project_end(F, &RB, 0, &EB);
        if (O->q_perp) O->q_perp[idx] = q_eq11(&EF, &EB, m0);
        project_end(F, &RF, 1, &EF); project_end(F, &RB, 1, &EB);
        if (O->q_bnd) O->q_bnd[idx] = q_eq11(&EF, &EB, m0);
    } else {
        if (O->q_perp) O->q_perp[idx] = nan;
        if (O->q_bnd) O->q_bnd[idx] = nan;
    }
    *steps += RF.nsteps + RB.nsteps;
}

void orc_trace(const orc_field *F, const orc_trace_params *P, long long n, const double *seeds,
               const orc_trace_out *out, unsigned long long *total_steps, int nthreads)
{
    unsigned long long tot = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    (void)nthreads;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : tot)
    for (long long i = 0; i < n; ++i) {
        unsigned long long s = 0;
        trace_one(F, P, seeds + 3 * i, i, out, &s);
        tot += s;
    }
    if (total_steps) *total_steps = tot;
}

/* ------------------------------------------------------------------------------------------------ O6 */
/* "the gradient magnitude from the Sobel operator (i.e. a 2D or 3D gradient of FLL convolved
 * with a simple smoothing function) applied to a 2D or 3D map of the length of field lines".
 * Reading A10: un-normalised weights diff = [-1,0,+1], smooth = [1,2,1]; out-of-range neighbours replicate
 * the edge sample.  G_d = sum over the 3^D neighbourhood, offsets visited axis 2 outermost, axis 0
 * innermost; S = sqrt(G_0^2 + G_1^2 (+ G_2^2)).                                                           */
typedef double (*cell_value_fn)(const void *ctx, const long long c[3]);

static double sobel_at(int ndim, const long long dims[3], const long long c[3], cell_value_fn get, const void *ctx)
{
    static const double diffw[3] = { -1.0, 0.0, 1.0 }, smoothw[3] = { 1.0, 2.0, 1.0 };
    double G[3] = { 0.0, 0.0, 0.0 };
    const int o2lo = ndim == 3 ? -1 : 0, o2hi = ndim == 3 ? 1 : 0;
    for (int o2 = o2lo; o2 <= o2hi; ++o2)
        for (int o1 = -1; o1 <= 1; ++o1)
            for (int o0 = -1; o0 <= 1; ++o0) {
                long long nb[3] = { c[0] + o0, c[1] + o1, c[2] + o2 };
                for (int d = 0; d < ndim; ++d) { if (nb[d] < 0) nb[d] = 0; if (nb[d] > dims[d] - 1) nb[d] = dims[d] - 1; }
                const double v = get(ctx, nb);
                const int o[3] = { o0, o1, o2 };
                for (int d = 0; d < ndim; ++d) {
                    double w = diffw[o[d] + 1];
                    for (int e = 0; e < ndim; ++e) if (e != d) w *= smoothw[o[e] + 1];
                    G[d] += w * v;
                }
            }
    double ss = 0.0;
    for (int d = 0; d < ndim; ++d) ss += G[d] * G[d];
    return sqrt(ss);
}

typedef struct { const long long *dims; const double *L; } dense_ctx;
static double dense_get(const void *ctx, const long long c[3])
{
    const dense_ctx *D = (const dense_ctx *)ctx;
    return D->L[(c[2] * D->dims[1] + c[1]) * D->dims[0] + c[0]];
}

void orc_fledge_dense(int ndim, const long long dims_in[3], const double *L, double *S)
{
    long long dims[3] = { dims_in[0], dims_in[1], ndim == 3 ? dims_in[2] : 1 };
    dense_ctx ctx = { dims, L };
#pragma omp parallel for collapse(2) schedule(static)
    for (long long c2 = 0; c2 < dims[2]; ++c2)
        for (long long c1 = 0; c1 < dims[1]; ++c1)
            for (long long c0 = 0; c0 < dims[0]; ++c0) {
                const long long c[3] = { c0, c1, c2 };
                S[(c2 * dims[1] + c1) * dims[0] + c0] = sobel_at(ndim, dims, c, dense_get, &ctx);
            }
}

/* Sparse level l >= 1: the same stencil on the virtual lattice of dims n_d 2^l; a neighbour that was not
 * refined takes the L of its nearest existing ancestor (coords >> 1 per level up; level 0 is dense).      */
typedef struct { unsigned long long key; long long idx; } key_idx;
static int key_cmp(const void *a, const void *b)
{
    const key_idx *x = (const key_idx *)a, *y = (const key_idx *)b;
    return x->key < y->key ? -1 : (x->key > y->key ? 1 : 0);
}
typedef struct {
    int ndim, level; const long long *n0; const double *L0;
    const long long *count; key_idx *const *table; const double *const *L;
} sparse_ctx;
static unsigned long long lin_key(int ndim, const long long n0[3], int level, const long long c[3])
{
    const unsigned long long d0 = (unsigned long long)n0[0] << level, d1 = (unsigned long long)n0[1] << level;
    return ((unsigned long long)(ndim == 3 ? c[2] : 0) * d1 + (unsigned long long)c[1]) * d0 + (unsigned long long)c[0];
}
static double sparse_get(const void *ctx, const long long c_in[3])
{
    const sparse_ctx *C = (const sparse_ctx *)ctx;
    long long c[3] = { c_in[0], c_in[1], c_in[2] };
    for (int l = C->level; l >= 1; --l) {
        key_idx probe = { lin_key(C->ndim, C->n0, l, c), 0 };
        const key_idx *hit = (const key_idx *)bsearch(&probe, C->table[l], (size_t)C->count[l], sizeof(key_idx), key_cmp);
        if (hit) return C->L[l][hit->idx];
        for (int d = 0; d < 3; ++d) c[d] >>= 1;
    }
    return C->L0[lin_key(C->ndim, C->n0, 0, c)];
}

void orc_fledge_sparse(int ndim, const long long n0[3], int level, const double *L0, const long long *count,
                       const uint32_t *const *coords, const double *const *L, double *S)
{
    key_idx **table = (key_idx **)calloc((size_t)level + 1, sizeof(key_idx *));
    for (int l = 1; l <= level; ++l) {
        table[l] = (key_idx *)malloc(sizeof(key_idx) * (size_t)(count[l] > 0 ? count[l] : 1));
        for (long long i = 0; i < count[l]; ++i) {
            long long c[3] = { coords[l][i * ndim + 0], coords[l][i * ndim + 1], ndim == 3 ? coords[l][i * ndim + 2] : 0 };
            table[l][i].key = lin_key(ndim, n0, l, c); table[l][i].idx = i;
        }
        qsort(table[l], (size_t)count[l], sizeof(key_idx), key_cmp);
    }
    const long long dims[3] = { n0[0] << level, n0[1] << level, ndim == 3 ? n0[2] << level : 1 };
    sparse_ctx ctx = { ndim, level, n0, L0, count, table, L };
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < count[level]; ++i) {
        const long long c[3] = { coords[level][i * ndim + 0], coords[level][i * ndim + 1],
                                 ndim == 3 ? coords[level][i * ndim + 2] : 0 };
        S[i] = sobel_at(ndim, dims, c, sparse_get, &ctx);
    }
    for (int l = 1; l <= level; ++l) free(table[l]);
    free(table);
}

/* ------------------------------------------------------------------------------------------------ O7 */
/* refine where the FLL jump "surpasses a certain threshold"; BASELINE.json configs[2]: "where the
 * FLEDGE value exceeds the 95th percentile".  Reading A11: tau = the ceil(p N)-th smallest of the N finite
 * values (nearest rank); strict >; NaN never flags.                                                       */
static int dbl_cmp(const void *a, const void *b)
{
    const double x = *(const double *)a, y = *(const double *)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}
double orc_select(long long n, const double *S, double p)
{
    double *f = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    long long N = 0;
    for (long long i = 0; i < n; ++i) if (isfinite(S[i])) f[N++] = S[i];
    if (N == 0) { free(f); return NAN; }
    qsort(f, (size_t)N, sizeof(double), dbl_cmp);
    long long rank = (long long)ceil(p * (double)N);
    if (rank < 1) rank = 1;
    if (rank > N) rank = N;
    const double tau = f[rank - 1];
    free(f);
    return tau;
}

/* when the threshold is surpassed new samples are inserted between the old ones; here (north_star,
 * reading A11) each flagged cell is split 2x per axis.  Children are emitted for each flagged cell in input
 * order, child index bit d -> axis d: coord' = 2 coord + bit, position = origin + sum_d w_d e_d with
 * w_d = (coord'_d + 0.5)/(n_d 2^(level+1)) (one IEEE division) accumulated with fma, axis 0 first.          */
long long orc_refine(int ndim, int level, long long n, const uint32_t *coords, const double *S, double tau,
                     const long long n0[3], const double origin[3], const double e0[3], const double e1[3],
                     const double e2[3], uint32_t *child_coords, double *child_seeds)
{
    long long m = 0;
    const int nchild = 1 << ndim;
    for (long long i = 0; i < n; ++i) {
        if (!(S[i] > tau)) continue;
        for (int ch = 0; ch < nchild; ++ch) {
            double w[3] = { 0.0, 0.0, 0.0 };
            for (int d = 0; d < ndim; ++d) {
                const uint32_t cc = 2u * coords[i * ndim + d] + (uint32_t)((ch >> d) & 1);
                child_coords[m * ndim + d] = cc;
                w[d] = ((double)cc + 0.5) / (double)(n0[d] << (level + 1));
            }
            for (int k = 0; k < 3; ++k) {
                double pos = fma(w[0], e0[k], origin[k]);
                pos = fma(w[1], e1[k], pos);
                if (ndim == 3) pos = fma(w[2], e2[k], pos);
                child_seeds[3 * m + k] = pos;
            }
            ++m;
        }
    }
    return m;
}
