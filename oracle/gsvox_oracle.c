/*
 * gsvox_oracle.c — fp64 CPU brute-force oracle for the 3D Gaussian voxelizer.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2503_22139_b200/)
 * may import, link or call this file.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs use it.  It shares no code,
 * header, table or helper with the CUDA path.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md):
 *   Eq. 4  G_i(x) = rho_i * exp(-1/2 (x-p_i)^T Sigma_i^-1 (x-p_i))
 *   Eq. 5  sigma(x) = sum_i G_i(x)            ("voxelization")
 *   PAPER.md:104         the voxelizer is differentiable wrt all Gaussian params
 *   PAPER.md:108         signed values are allowed ("negative-permitting")
 * The paper is silent on the parameterisation of Sigma, the cutoff, the voxel
 * convention and the layout; those follow BASELINE.json north_star and the
 * readings A1..A16 of SURVEY.md section 8(c), restated in DESIGN.md:
 *   Sigma = R S S^T R^T, S = diag(s), R from the normalised quaternion (w,x,y,z);
 *   support of Gaussian i = the axis-aligned box |x_k - p_k| <= kappa*sqrt(Sigma_kk)
 *   (kappa = 3 in the product), voxel CENTRES tested, bounds inclusive, clipped to
 *   the grid; no other test inside the box; backward treats the box as frozen.
 *
 * Method: the truncated sum IS the definition, so this file is that definition
 * written out: for every Gaussian, for every voxel of its box, one exp().  The
 * only liberty taken is the loop nest used for threading (forward: each thread
 * owns whole z-slices and visits Gaussians in index order; backward: each thread
 * owns whole Gaussians), which changes no arithmetic.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off matters: the box bounds (reading A5) must be evaluated with
 * one IEEE-754 rounding per operation so that any other correctly rounded fp64
 * implementation of the same operation sequence gets the identical integers.
 *
 * Pins (tests/test_oracle_pins.py): closed-form Gaussian integral, box-truncated
 * closed form, survey-script worked values (tests/golden/), separability,
 * linearity, superposition, rotation identities, scipy rotation matrices,
 * numpy.linalg.inv covariances, ellipsoid-tangent boxes, central finite
 * differences, closed-form gradients.  Parity of the paper's whole-system
 * accuracy tables (II/III) is unpinned and out of scope.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL -1
#define ORACLE_ENOMEM -2

typedef struct {
    double p[3];      /* centre, world units (exact promotion of the fp32 input)   */
    double s[3];      /* standard deviations                                       */
    double qn;        /* |q|                                                        */
    double qh[4];     /* normalised quaternion (r, x, y, z)                         */
    double R[9];      /* row-major rotation matrix                                  */
    double M[9];      /* Sigma^-1 = R diag(1/s^2) R^T, row-major, world units       */
    int32_t lo[3];    /* inclusive voxel box, already clipped to the grid           */
    int32_t hi[3];
    int skipped;      /* degenerate input: contributes nothing, all gradients zero  */
    int empty;        /* box does not meet the grid                                 */
} gauss_t;

int gsvox_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* SURVEY 8(b) "Degenerate Gaussians": any non-finite parameter, any scale <= 0
 * or |q| = 0 -> skipped. */
static int degenerate(const double p[3], const double s[3], const double q[4])
{
    for (int k = 0; k < 3; ++k) {
        if (!isfinite(p[k]) || !isfinite(s[k]) || !(s[k] > 0.0)) return 1;
    }
    for (int k = 0; k < 4; ++k)
        if (!isfinite(q[k])) return 1;
    if (q[0] == 0.0 && q[1] == 0.0 && q[2] == 0.0 && q[3] == 0.0) return 1;
    return 0;
}

/* Steps 1-5 of the forward definition, operation order of reading
 * A5.  Every line below is one rounded fp64 operation per operator. */
static void geometry(const float *pos, const float *scale, const float *quat,
                     const double o[3], const double h[3], const int32_t dims[3],
                     double kappa, gauss_t *g)
{
    double q[4];
    for (int k = 0; k < 3; ++k) { g->p[k] = (double)pos[k]; g->s[k] = (double)scale[k]; }
    for (int k = 0; k < 4; ++k) q[k] = (double)quat[k];
    memset(g->R, 0, sizeof g->R); memset(g->M, 0, sizeof g->M);
    g->qn = 0.0; g->empty = 1;
    for (int k = 0; k < 3; ++k) { g->lo[k] = 0; g->hi[k] = -1; }
    g->skipped = degenerate(g->p, g->s, q);
    if (g->skipped) return;

    /* step 1: q^ = q/|q|, q = (r,x,y,z) scalar first (reading A2) */
    double n2 = ((q[0] * q[0] + q[1] * q[1]) + q[2] * q[2]) + q[3] * q[3];
    double n = sqrt(n2);
    g->qn = n;
    double r = q[0] / n, x = q[1] / n, y = q[2] / n, z = q[3] / n;
    g->qh[0] = r; g->qh[1] = x; g->qh[2] = y; g->qh[3] = z;

    /* step 2: rotation matrix, entries exactly as written in SURVEY 8(c) step 2 */
    double *R = g->R;
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - r * z);       R[2] = 2.0 * (x * z + r * y);
    R[3] = 2.0 * (x * y + r * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - r * x);
    R[6] = 2.0 * (x * z - r * y);       R[7] = 2.0 * (y * z + r * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);

    /* step 3: M = R diag(1/s^2) R^T (closed form of Sigma^-1, Sigma = R S S^T R^T) */
    double is2[3];
    for (int k = 0; k < 3; ++k) is2[k] = 1.0 / (g->s[k] * g->s[k]);
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            double acc = 0.0;
            for (int j = 0; j < 3; ++j) acc += R[3 * a + j] * is2[j] * R[3 * b + j];
            g->M[3 * a + b] = acc;
        }

    /* steps 4-5: half-extents r_k = kappa*sqrt(Sigma_kk), integer box (A3, A4, A5) */
    g->empty = 0;
    for (int k = 0; k < 3; ++k) {
        double s0 = g->s[0] * g->s[0], s1 = g->s[1] * g->s[1], s2 = g->s[2] * g->s[2];
        double Skk = ((R[3 * k] * R[3 * k]) * s0 + (R[3 * k + 1] * R[3 * k + 1]) * s1)
                     + (R[3 * k + 2] * R[3 * k + 2]) * s2;
        double rk = kappa * sqrt(Skk);
        double lo = ceil(((g->p[k] - rk) - o[k]) / h[k]);
        double hi = floor(((g->p[k] + rk) - o[k]) / h[k]);
        double top = (double)(dims[k] - 1);
        if (lo < 0.0) lo = 0.0;
        if (hi > top) hi = top;
        if (!(hi >= lo)) { g->empty = 1; }
        else { g->lo[k] = (int32_t)lo; g->hi[k] = (int32_t)hi; }
    }
    if (g->empty)
        for (int k = 0; k < 3; ++k) { g->lo[k] = 0; g->hi[k] = -1; }
}

static int check_grid(const float *origin, const float *spacing, const int32_t *dims)
{
    if (!origin || !spacing || !dims) return 0;
    for (int k = 0; k < 3; ++k) {
        if (!(spacing[k] > 0.0f) || !isfinite(spacing[k]) || !isfinite(origin[k])) return 0;
        if (dims[k] < 1) return 0;
    }
    return 1;
}

static gauss_t *all_geometry(const float *pos, const float *scale, const float *quat, int64_t n,
                             const float *origin, const float *spacing, const int32_t *dims,
                             double kappa)
{
    gauss_t *G = (gauss_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(gauss_t));
    if (!G) return NULL;
    double o[3], h[3];
    for (int k = 0; k < 3; ++k) { o[k] = (double)origin[k]; h[k] = (double)spacing[k]; }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i)
        geometry(pos + 3 * i, scale + 3 * i, quat + 4 * i, o, h, dims, kappa, &G[i]);
    return G;
}

/* ---------------------------------------------------------------------------
 * Per-Gaussian geometry, exported so tests can pin it and compare the CUDA
 * preprocess against it (integer boxes bit-identical, reading A5).
 *   M_out  [n,6]  xx,xy,xz,yy,yz,zz of Sigma^-1 (world units)   (may be NULL)
 *   R_out  [n,9]  row-major rotation                            (may be NULL)
 *   box    [n,6]  lo_x,lo_y,lo_z,hi_x,hi_y,hi_z inclusive; empty/skipped -> 0,0,0,-1,-1,-1
 *   flags  [n]    bit0 = skipped (degenerate), bit1 = empty box  (may be NULL)
 * ------------------------------------------------------------------------- */
int gsvox_oracle_geometry(const float *pos, const float *scale, const float *quat, int64_t n,
                          const float *origin, const float *spacing, const int32_t *dims,
                          double kappa, double *M_out, double *R_out, int32_t *box, uint8_t *flags)
{
    if (n < 0 || !check_grid(origin, spacing, dims) || (n > 0 && (!pos || !scale || !quat)))
        return ORACLE_EINVAL;
    gauss_t *G = all_geometry(pos, scale, quat, n, origin, spacing, dims, kappa);
    if (!G) return ORACLE_ENOMEM;
    for (int64_t i = 0; i < n; ++i) {
        const gauss_t *g = &G[i];
        if (M_out) {
            M_out[6 * i + 0] = g->M[0]; M_out[6 * i + 1] = g->M[1]; M_out[6 * i + 2] = g->M[2];
            M_out[6 * i + 3] = g->M[4]; M_out[6 * i + 4] = g->M[5]; M_out[6 * i + 5] = g->M[8];
        }
        if (R_out) memcpy(R_out + 9 * i, g->R, sizeof g->R);
        if (box) {
            for (int k = 0; k < 3; ++k) { box[6 * i + k] = g->lo[k]; box[6 * i + 3 + k] = g->hi[k]; }
        }
        if (flags) flags[i] = (uint8_t)((g->skipped ? 1 : 0) | ((g->empty && !g->skipped) ? 2 : 0));
    }
    free(G);
    return ORACLE_OK;
}

/* Eq. 4 exponent for one voxel: x = o + idx*h (reading A6), d = x - p. */
static inline double gauss_value(const gauss_t *g, const double o[3], const double h[3],
                                 int i, int j, int k, double d[3])
{
    d[0] = (o[0] + (double)i * h[0]) - g->p[0];
    d[1] = (o[1] + (double)j * h[1]) - g->p[1];
    d[2] = (o[2] + (double)k * h[2]) - g->p[2];
    const double *M = g->M;
    double qf = d[0] * (M[0] * d[0] + M[1] * d[1] + M[2] * d[2])
              + d[1] * (M[3] * d[0] + M[4] * d[1] + M[5] * d[2])
              + d[2] * (M[6] * d[0] + M[7] * d[1] + M[8] * d[2]);
    return exp(-0.5 * qf);
}

/* ---------------------------------------------------------------------------
 * Forward, Eq. 5 with the box cutoff (step 6 of the definition).
 *   weight [n,C] fp32;  out [C,nz,ny,nx] fp64, overwritten (reading A7)
 *   pairs_out: number of (Gaussian, voxel) pairs inside the cutoff = P_def
 * ------------------------------------------------------------------------- */
int gsvox_oracle_forward(const float *pos, const float *scale, const float *quat,
                         const float *weight, int64_t n, int32_t C,
                         const float *origin, const float *spacing, const int32_t *dims,
                         double kappa, double *out, int64_t *pairs_out)
{
    if (n < 0 || C < 1 || !check_grid(origin, spacing, dims) || !out ||
        (n > 0 && (!pos || !scale || !quat || !weight)))
        return ORACLE_EINVAL;
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t V = (int64_t)nx * ny * nz;
    gauss_t *G = all_geometry(pos, scale, quat, n, origin, spacing, dims, kappa);
    if (!G) return ORACLE_ENOMEM;
    double o[3], h[3];
    for (int k = 0; k < 3; ++k) { o[k] = (double)origin[k]; h[k] = (double)spacing[k]; }
    memset(out, 0, (size_t)V * (size_t)C * sizeof(double));
    int64_t pairs = 0;

    /* each thread owns whole z-slices; Gaussians visited in index order */
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : pairs)
    for (int k = 0; k < nz; ++k) {
        for (int64_t gi = 0; gi < n; ++gi) {
            const gauss_t *g = &G[gi];
            if (g->skipped || g->empty || k < g->lo[2] || k > g->hi[2]) continue;
            const float *w = weight + (int64_t)C * gi;
            for (int j = g->lo[1]; j <= g->hi[1]; ++j)
                for (int i = g->lo[0]; i <= g->hi[0]; ++i) {
                    double d[3];
                    double e = gauss_value(g, o, h, i, j, k, d);
                    int64_t v = ((int64_t)k * ny + j) * nx + i;
                    for (int c = 0; c < C; ++c) out[(int64_t)c * V + v] += (double)w[c] * e;
                    ++pairs;
                }
        }
    }
    if (pairs_out) *pairs_out = pairs;
    free(G);
    return ORACLE_OK;
}

/* Forward at a list of voxels only (linear voxel index v = (k*ny + j)*nx + i):
 * the same definition, one voxel at a time, for spot checks at full size.
 *   out [C, m] fp64 */
int gsvox_oracle_forward_at(const float *pos, const float *scale, const float *quat,
                            const float *weight, int64_t n, int32_t C,
                            const float *origin, const float *spacing, const int32_t *dims,
                            double kappa, const int64_t *voxels, int64_t m, double *out)
{
    if (n < 0 || C < 1 || m < 0 || !check_grid(origin, spacing, dims) ||
        (m > 0 && (!voxels || !out)) || (n > 0 && (!pos || !scale || !quat || !weight)))
        return ORACLE_EINVAL;
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    gauss_t *G = all_geometry(pos, scale, quat, n, origin, spacing, dims, kappa);
    if (!G) return ORACLE_ENOMEM;
    double o[3], h[3];
    for (int k = 0; k < 3; ++k) { o[k] = (double)origin[k]; h[k] = (double)spacing[k]; }
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t t = 0; t < m; ++t) {
        int64_t v = voxels[t];
        if (v < 0 || v >= (int64_t)nx * ny * nz) { bad = 1; continue; }
        int i = (int)(v % nx), j = (int)((v / nx) % ny), k = (int)(v / ((int64_t)nx * ny));
        for (int c = 0; c < C; ++c) out[(int64_t)c * m + t] = 0.0;
        for (int64_t gi = 0; gi < n; ++gi) {
            const gauss_t *g = &G[gi];
            if (g->skipped || g->empty) continue;
            if (i < g->lo[0] || i > g->hi[0] || j < g->lo[1] || j > g->hi[1] ||
                k < g->lo[2] || k > g->hi[2]) continue;
            double d[3];
            double e = gauss_value(g, o, h, i, j, k, d);
            for (int c = 0; c < C; ++c)
                out[(int64_t)c * m + t] += (double)weight[(int64_t)C * gi + c] * e;
        }
    }
    free(G);
    return bad ? ORACLE_EINVAL : ORACLE_OK;
}

/* Backward for one Gaussian (the "Definition (backward)" block of SURVEY 8(c)). */
static void backward_one(const gauss_t *g, const float *w, int32_t C, const float *grad_out,
                         const double o[3], const double h[3], int nx, int ny, int64_t V,
                         double *gw, double *gp, double *gs, double *gq)
{
    for (int c = 0; c < C; ++c) gw[c] = 0.0;
    for (int k = 0; k < 3; ++k) { gp[k] = 0.0; gs[k] = 0.0; }
    for (int k = 0; k < 4; ++k) gq[k] = 0.0;
    if (g->skipped || g->empty) return;

    double DM[9];                      /* dL/dM = -1/2 sum a d d^T */
    memset(DM, 0, sizeof DM);
    const double *M = g->M, *R = g->R;
    for (int k = g->lo[2]; k <= g->hi[2]; ++k)
        for (int j = g->lo[1]; j <= g->hi[1]; ++j)
            for (int i = g->lo[0]; i <= g->hi[0]; ++i) {
                double d[3];
                double e = gauss_value(g, o, h, i, j, k, d);
                int64_t v = ((int64_t)k * ny + j) * nx + i;
                double a = 0.0;
                for (int c = 0; c < C; ++c) {
                    double gc = (double)grad_out[(int64_t)c * V + v];
                    gw[c] += gc * e;                    /* dL/dw_c = sum g_c G     */
                    a += gc * (double)w[c];
                }
                a *= e;                                 /* a = (sum_c g_c w_c) G   */
                for (int r = 0; r < 3; ++r)             /* dL/dp = sum a M d       */
                    gp[r] += a * (M[3 * r] * d[0] + M[3 * r + 1] * d[1] + M[3 * r + 2] * d[2]);
                for (int r = 0; r < 3; ++r)
                    for (int c2 = 0; c2 < 3; ++c2) DM[3 * r + c2] += -0.5 * a * d[r] * d[c2];
            }

    /* dL/ds_k = -2 (R^T D_M R)_kk / s_k^3 */
    for (int k = 0; k < 3; ++k) {
        double acc = 0.0;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) acc += R[3 * a + k] * DM[3 * a + b] * R[3 * b + k];
        gs[k] = -2.0 * acc / (g->s[k] * g->s[k] * g->s[k]);
    }
    /* D_R = 2 D_M R diag(1/s^2) */
    double DR[9];
    for (int a = 0; a < 3; ++a)
        for (int k = 0; k < 3; ++k) {
            double acc = 0.0;
            for (int b = 0; b < 3; ++b) acc += DM[3 * a + b] * R[3 * b + k];
            DR[3 * a + k] = 2.0 * acc / (g->s[k] * g->s[k]);
        }
    /* dL/dq^_j = <dR/dq^_j, D_R> */
    double r = g->qh[0], x = g->qh[1], y = g->qh[2], z = g->qh[3];
    double dRr[9] = { 0, -2 * z, 2 * y,    2 * z, 0, -2 * x,    -2 * y, 2 * x, 0 };
    double dRx[9] = { 0, 2 * y, 2 * z,     2 * y, -4 * x, -2 * r,   2 * z, 2 * r, -4 * x };
    double dRy[9] = { -4 * y, 2 * x, 2 * r,   2 * x, 0, 2 * z,    -2 * r, 2 * z, -4 * y };
    double dRz[9] = { -4 * z, -2 * r, 2 * x,  2 * r, -4 * z, 2 * y,   2 * x, 2 * y, 0 };
    double gh[4] = { 0, 0, 0, 0 };
    for (int t = 0; t < 9; ++t) {
        gh[0] += dRr[t] * DR[t]; gh[1] += dRx[t] * DR[t];
        gh[2] += dRy[t] * DR[t]; gh[3] += dRz[t] * DR[t];
    }
    /* through the normalisation: dL/dq = (dL/dq^ - q^ (q^ . dL/dq^)) / |q|  (reading A2) */
    double dot = g->qh[0] * gh[0] + g->qh[1] * gh[1] + g->qh[2] * gh[2] + g->qh[3] * gh[3];
    for (int t = 0; t < 4; ++t) gq[t] = (gh[t] - g->qh[t] * dot) / g->qn;
}

/* ---------------------------------------------------------------------------
 * Backward over all Gaussians.
 *   grad_out [C,nz,ny,nx] fp32;  gw [n,C], gp [n,3], gs [n,3], gq [n,4] fp64, overwritten
 * ------------------------------------------------------------------------- */
int gsvox_oracle_backward(const float *pos, const float *scale, const float *quat,
                          const float *weight, int64_t n, int32_t C,
                          const float *origin, const float *spacing, const int32_t *dims,
                          double kappa, const float *grad_out,
                          double *gw, double *gp, double *gs, double *gq)
{
    if (n < 0 || C < 1 || !check_grid(origin, spacing, dims) ||
        (n > 0 && (!pos || !scale || !quat || !weight || !grad_out || !gw || !gp || !gs || !gq)))
        return ORACLE_EINVAL;
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t V = (int64_t)nx * ny * nz;
    gauss_t *G = all_geometry(pos, scale, quat, n, origin, spacing, dims, kappa);
    if (!G) return ORACLE_ENOMEM;
    double o[3], h[3];
    for (int k = 0; k < 3; ++k) { o[k] = (double)origin[k]; h[k] = (double)spacing[k]; }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t gi = 0; gi < n; ++gi)
        backward_one(&G[gi], weight + (int64_t)C * gi, C, grad_out, o, h, nx, ny, V,
                     gw + (int64_t)C * gi, gp + 3 * gi, gs + 3 * gi, gq + 4 * gi);
    free(G);
    return ORACLE_OK;
}

/* Backward for a list of Gaussian ids only (spot checks at full size).
 *   ids [m];  gw [m,C], gp [m,3], gs [m,3], gq [m,4] */
int gsvox_oracle_backward_for(const float *pos, const float *scale, const float *quat,
                              const float *weight, int64_t n, int32_t C,
                              const float *origin, const float *spacing, const int32_t *dims,
                              double kappa, const float *grad_out, const int64_t *ids, int64_t m,
                              double *gw, double *gp, double *gs, double *gq)
{
    if (n < 0 || C < 1 || m < 0 || !check_grid(origin, spacing, dims) ||
        (m > 0 && (!ids || !pos || !scale || !quat || !weight || !grad_out || !gw || !gp || !gs || !gq)))
        return ORACLE_EINVAL;
    for (int64_t t = 0; t < m; ++t)
        if (ids[t] < 0 || ids[t] >= n) return ORACLE_EINVAL;
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t V = (int64_t)nx * ny * nz;
    double o[3], h[3];
    for (int k = 0; k < 3; ++k) { o[k] = (double)origin[k]; h[k] = (double)spacing[k]; }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t t = 0; t < m; ++t) {
        int64_t gi = ids[t];
        gauss_t g;
        geometry(pos + 3 * gi, scale + 3 * gi, quat + 4 * gi, o, h, dims, kappa, &g);
        backward_one(&g, weight + (int64_t)C * gi, C, grad_out, o, h, nx, ny, V,
                     gw + (int64_t)C * t, gp + 3 * t, gs + 3 * t, gq + 4 * t);
    }
    return ORACLE_OK;
}
