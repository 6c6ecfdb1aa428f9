/*
 * OSOG forward-render ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, float64 CPU restatement of what the hot path computes, written from the paper
 * and the readings listed in DESIGN.md section 3.  It shares no code,
 * header, table or helper with the CUDA path under paper_2606_21381_b200/csrc and is imported only
 * by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * What is computed (per frame, pixel (i,j) = row i, column j, centre x=(j+1/2)p, y=(i+1/2)p):
 *
 *   OPD[i,j] = sum over particles n, ascending n, of (n_p[n] - n_medium) * thickness_n(x-cx, y-cy)
 *
 * - the integrand of Eq. 2 ("integral of [n_p(z) - n_m] dz") for piecewise-constant
 *   n_p, summed over particles as Eq. 7's accumulate=True does.  Off-canvas
 *   pixels are simply not part of the frame ("strict boolean masking").
 *
 * thickness_n(dx,dy) = length of the intersection of the vertical line (dx,dy,.) with the body:
 *   kind 0  ellipsoid  { q : q^T M q <= 1 },  M = R diag(1/a^2,1/b^2,1/c^2) R^T   (not in the paper:
 *           BASELINE.json north_star, "ellipsoid quadratic"); solved as a quadratic in z.
 *   kind 1  capped tetragonal prism = intersection of 12 half-spaces  A x <= b  (Eq. 1),
 *           evaluated by the generic loop over planes: enter = max over planes with n_z<0 of g/n_z,
 *           exit = min over planes with n_z>0 of g/n_z, g = b - n_x dx - n_y dy; a plane with n_z==0
 *           empties the line when g<0.
 *
 * Precision: float64 throughout; the float32 inputs are promoted exactly.  No tiling, no bounding
 * boxes; `mode` 1 ("bcircle") skips pixels farther from the centre than the body's circumradius,
 * which is trivially conservative and is shown bit-identical to mode 0 ("full") by the tests.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): sphere closed form, axis-aligned ellipsoid,
 * Schur-complement projection, prism closed forms, volume invariance, vertex/plane consistency,
 * permutation invariance, integer translation, supersampled ray marching by inside-test only.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define OSOG_ORACLE_MAX_PLANES 16

/* Hamilton unit quaternion (w,x,y,z) -> active rotation matrix body->world, row-major R[3*r+c].
 * No renormalisation (reading A4). */
void osog_oracle_rot_from_quat(const double q[4], double R[9])
{
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
    R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
    R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

/* Ellipsoid: points q with q^T M q <= 1, M = R D R^T, D = diag(1/a^2, 1/b^2, 1/c^2).
 * On the line q = (dx, dy, z):  A z^2 + 2 Bq z + C <= 0  with
 *   A = M_zz,  Bq = M_xz dx + M_yz dy,  C = M_xx dx^2 + 2 M_xy dx dy + M_yy dy^2 - 1,
 * so the chord length is 2 sqrt(Bq^2 - A C) / A when the discriminant is positive, else 0. */
double osog_oracle_thickness_ellipsoid(const double R[9], double a, double b, double c,
                                       double dx, double dy)
{
    const double D[3] = { 1.0 / (a * a), 1.0 / (b * b), 1.0 / (c * c) };
    double M[9];
    for (int r = 0; r < 3; ++r)
        for (int s = 0; s < 3; ++s) {
            double acc = 0.0;
            for (int k = 0; k < 3; ++k) acc += R[3 * r + k] * D[k] * R[3 * s + k];
            M[3 * r + s] = acc;
        }
    const double A  = M[8];
    const double Bq = M[2] * dx + M[5] * dy;
    const double C  = M[0] * dx * dx + 2.0 * M[1] * dx * dy + M[4] * dy * dy - 1.0;
    const double disc = Bq * Bq - A * C;
    return disc > 0.0 ? 2.0 * sqrt(disc) / A : 0.0;
}

/* Body-frame half-spaces of the capped tetragonal prism (reading A5/A6): square
 * cross-section of side s in body x,y; prismatic part |z| <= L/2; a four-sided pyramid of height hc
 * on each end with apex (0,0,+-(L/2+hc)).  12 planes, un-normalised normals:
 *   +-(1,0,0), +-(0,1,0)                      with b = s/2
 *   (+-hc, 0, +-s/2), (0, +-hc, +-s/2)        with b = hc*s/2 + s*L/4     (all sign choices)
 * Returns the number of planes (12). */
int osog_oracle_prism_planes(double s, double L, double hc, double A[][3], double b[])
{
    int m = 0;
    const double sgn[2] = { 1.0, -1.0 };
    for (int k = 0; k < 2; ++k) { A[m][0] = sgn[k]; A[m][1] = 0.0; A[m][2] = 0.0; b[m] = 0.5 * s; ++m; }
    for (int k = 0; k < 2; ++k) { A[m][0] = 0.0; A[m][1] = sgn[k]; A[m][2] = 0.0; b[m] = 0.5 * s; ++m; }
    const double bc = hc * s * 0.5 + s * L * 0.25;
    for (int kz = 0; kz < 2; ++kz)
        for (int kx = 0; kx < 2; ++kx) { A[m][0] = sgn[kx] * hc; A[m][1] = 0.0; A[m][2] = sgn[kz] * 0.5 * s; b[m] = bc; ++m; }
    for (int kz = 0; kz < 2; ++kz)
        for (int ky = 0; ky < 2; ++ky) { A[m][0] = 0.0; A[m][1] = sgn[ky] * hc; A[m][2] = sgn[kz] * 0.5 * s; b[m] = bc; ++m; }
    return m;
}

/* Eq. 1: P = { x | A x <= b }, planes given in WORLD axes relative to the centre.
 * Length of { z : A (dx,dy,z) <= b }. */
double osog_oracle_thickness_polyhedron(int M, const double A[][3], const double b[],
                                        double dx, double dy)
{
    double enter = -INFINITY, exit_ = INFINITY;
    for (int k = 0; k < M; ++k) {
        const double g = b[k] - A[k][0] * dx - A[k][1] * dy;
        const double nz = A[k][2];
        if (nz > 0.0)      { const double z = g / nz; if (z < exit_) exit_ = z; }
        else if (nz < 0.0) { const double z = g / nz; if (z > enter) enter = z; }
        else if (g < 0.0)  return 0.0;
    }
    const double t = exit_ - enter;
    return t > 0.0 ? t : 0.0;
}

/* World-frame planes of prism n: normal R n_hat, same offset b. */
static int prism_world_planes(const double R[9], double s, double L, double hc,
                              double Aw[][3], double b[])
{
    double Ab[OSOG_ORACLE_MAX_PLANES][3];
    const int M = osog_oracle_prism_planes(s, L, hc, Ab, b);
    for (int k = 0; k < M; ++k)
        for (int r = 0; r < 3; ++r)
            Aw[k][r] = R[3 * r + 0] * Ab[k][0] + R[3 * r + 1] * Ab[k][1] + R[3 * r + 2] * Ab[k][2];
    return M;
}

/* A particle takes part iff every parameter is finite and all three dimensions are positive
 * (error behaviour: others are skipped). */
int osog_oracle_particle_valid(float cx, float cy, float qw, float qx, float qy, float qz,
                               float d0, float d1, float d2, float n_p, uint8_t kind)
{
    const double v[10] = { cx, cy, qw, qx, qy, qz, d0, d1, d2, n_p };
    for (int k = 0; k < 10; ++k) if (!isfinite(v[k])) return 0;
    if (!(d0 > 0.0f) || !(d1 > 0.0f) || !(d2 > 0.0f)) return 0;
    return kind <= 1;
}

/* Thickness of one particle at offset (dx,dy) from its centre; q = (w,x,y,z), dims = (d0,d1,d2). */
double osog_oracle_thickness(uint8_t kind, const double q[4], const double dims[3], double dx, double dy)
{
    double R[9];
    osog_oracle_rot_from_quat(q, R);
    if (kind == 0) return osog_oracle_thickness_ellipsoid(R, dims[0], dims[1], dims[2], dx, dy);
    double Aw[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
    const int M = prism_world_planes(R, dims[0], dims[1], dims[2], Aw, b);
    return osog_oracle_thickness_polyhedron(M, Aw, b, dx, dy);
}

/* Circumradius of the body (largest distance of any of its points from the centre):
 * ellipsoid: largest semi-axis; prism: largest vertex norm over (+-s/2,+-s/2,+-L/2), (0,0,+-(L/2+hc)). */
double osog_oracle_circumradius(uint8_t kind, float d0, float d1, float d2)
{
    if (kind == 0) return fmax((double)d0, fmax((double)d1, (double)d2));
    const double s = d0, L = d1, hc = d2;
    return fmax(sqrt(0.5 * s * s + 0.25 * L * L), 0.5 * L + hc);
}

/* One frame of OPD.  Particle arrays hold this frame's N particles.  mode 0 = full, 1 = bcircle.
 * opd is row-major [H*W], overwritten.  Rows are split over OpenMP threads; for each pixel the
 * particle loop runs in ascending index, so the summation order is fixed. */
void osog_oracle_render_opd(int64_t N,
                            const float *cx, const float *cy,
                            const float *qw, const float *qx, const float *qy, const float *qz,
                            const float *d0, const float *d1, const float *d2,
                            const float *n_p, const uint8_t *kind,
                            int H, int W, double pitch, double n_medium, int mode, double *opd)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < H; ++i) {
        const double y = (i + 0.5) * pitch;
        for (int j = 0; j < W; ++j) opd[(size_t)i * W + j] = 0.0;
        for (int64_t n = 0; n < N; ++n) {
            if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                            d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
            const double dy = y - (double)cy[n];
            const double dn = (double)n_p[n] - n_medium;
            const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
            double R[9];
            osog_oracle_rot_from_quat(q, R);
            double Aw[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
            int M = 0;
            if (kind[n] == 1) M = prism_world_planes(R, d0[n], d1[n], d2[n], Aw, b);
            double r2 = INFINITY;
            if (mode == 1) {
                const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
                r2 = r * r;
                if (dy * dy > r2) continue;
            }
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                const double t = kind[n] == 0
                    ? osog_oracle_thickness_ellipsoid(R, d0[n], d1[n], d2[n], dx, dy)
                    : osog_oracle_thickness_polyhedron(M, Aw, b, dx, dy);
                opd[(size_t)i * W + j] += dn * t;
            }
        }
    }
}

/* Workload statistic (not part of the rendered result): number of (particle, pixel) pairs of one frame
 * whose thickness is positive, counted separately for ellipsoids (pairs[0]) and prisms (pairs[1]).
 * These are the "true covered pairs" of SURVEY.md section 8(d): the units of arithmetic the method
 * cannot avoid.  Same loops and the same thickness functions as osog_oracle_render_opd. */
void osog_oracle_count_covered(int64_t N,
                               const float *cx, const float *cy,
                               const float *qw, const float *qx, const float *qy, const float *qz,
                               const float *d0, const float *d1, const float *d2,
                               const float *n_p, const uint8_t *kind,
                               int H, int W, double pitch, int mode, int64_t pairs[2])
{
    int64_t ne = 0, np = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : ne, np)
    for (int i = 0; i < H; ++i) {
        const double y = (i + 0.5) * pitch;
        for (int64_t n = 0; n < N; ++n) {
            if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                            d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
            const double dy = y - (double)cy[n];
            const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
            double R[9];
            osog_oracle_rot_from_quat(q, R);
            double Aw[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
            int M = 0;
            if (kind[n] == 1) M = prism_world_planes(R, d0[n], d1[n], d2[n], Aw, b);
            double r2 = INFINITY;
            if (mode == 1) {
                const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
                r2 = r * r;
                if (dy * dy > r2) continue;
            }
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                const double t = kind[n] == 0
                    ? osog_oracle_thickness_ellipsoid(R, d0[n], d1[n], d2[n], dx, dy)
                    : osog_oracle_thickness_polyhedron(M, Aw, b, dx, dy);
                if (t > 0.0) { if (kind[n] == 0) ++ne; else ++np; }
            }
        }
    }
    pairs[0] = ne;
    pairs[1] = np;
}

/* ---- G-buffer extras ("depth maps ... strict instance masks"; reading A24) ----------
 * Chord of the vertical line (dx, dy, .) through the body: [*z_enter, *z_exit] relative to the centre; returns 1 when the
 * chord has positive length (the same condition as thickness > 0), else 0.  Ellipsoid: roots of A z^2 + 2 Bq z + C = 0,
 * z = (-Bq -+ sqrt(disc)) / A; polyhedron: enter / exit of the Eq. 1 plane loop. */
int osog_oracle_chord(uint8_t kind, const double R[9], const double dims[3], double dx, double dy,
                      double *z_enter, double *z_exit)
{
    if (kind == 0) {
        const double a = dims[0], b = dims[1], c = dims[2];
        const double D[3] = { 1.0 / (a * a), 1.0 / (b * b), 1.0 / (c * c) };
        double M[9];
        for (int r = 0; r < 3; ++r)
            for (int s = 0; s < 3; ++s) {
                double acc = 0.0;
                for (int k = 0; k < 3; ++k) acc += R[3 * r + k] * D[k] * R[3 * s + k];
                M[3 * r + s] = acc;
            }
        const double A  = M[8];
        const double Bq = M[2] * dx + M[5] * dy;
        const double C  = M[0] * dx * dx + 2.0 * M[1] * dx * dy + M[4] * dy * dy - 1.0;
        const double disc = Bq * Bq - A * C;
        if (!(disc > 0.0)) return 0;
        const double sq = sqrt(disc);
        *z_enter = (-Bq - sq) / A;
        *z_exit  = (-Bq + sq) / A;
        return 1;
    }
    double Aw[OSOG_ORACLE_MAX_PLANES][3], bb[OSOG_ORACLE_MAX_PLANES];
    const int M = prism_world_planes(R, dims[0], dims[1], dims[2], Aw, bb);
    double enter = -INFINITY, exit_ = INFINITY;
    for (int k = 0; k < M; ++k) {
        const double g = bb[k] - Aw[k][0] * dx - Aw[k][1] * dy;
        const double nz = Aw[k][2];
        if (nz > 0.0)      { const double z = g / nz; if (z < exit_) exit_ = z; }
        else if (nz < 0.0) { const double z = g / nz; if (z > enter) enter = z; }
        else if (g < 0.0)  return 0;
    }
    if (!(exit_ - enter > 0.0)) return 0;
    *z_enter = enter;
    *z_exit = exit_;
    return 1;
}

/* Slope (dz/dx, dz/dy) of the body's TOP surface at (dx, dy): the analytic height gradient of the visible surface that "falls
 * out of the same ray test" (N = <-dh/dx, -dh/dy, 1>).  Ellipsoid: the surface is the level
 * set F(p) = p^T M p = 1; at the exit point p = (dx, dy, z_exit) its normal is grad F = 2 M p, so dz/dx = -(M p)_x / (M p)_z.
 * Prism: the active exit plane n . p = b gives dz/dx = -n_x / n_z.  Returns 0 (and leaves slope untouched) where the chord
 * is empty. */
int osog_oracle_top_slope(uint8_t kind, const double R[9], const double dims[3], double dx, double dy, double slope[2])
{
    double ze, zx;
    if (!osog_oracle_chord(kind, R, dims, dx, dy, &ze, &zx)) return 0;
    if (kind == 0) {
        const double D[3] = { 1.0 / (dims[0] * dims[0]), 1.0 / (dims[1] * dims[1]), 1.0 / (dims[2] * dims[2]) };
        double M[9];
        for (int r = 0; r < 3; ++r)
            for (int s = 0; s < 3; ++s) {
                double acc = 0.0;
                for (int k = 0; k < 3; ++k) acc += R[3 * r + k] * D[k] * R[3 * s + k];
                M[3 * r + s] = acc;
            }
        const double p[3] = { dx, dy, zx };
        double g[3];
        for (int r = 0; r < 3; ++r) g[r] = M[3 * r] * p[0] + M[3 * r + 1] * p[1] + M[3 * r + 2] * p[2];
        slope[0] = -g[0] / g[2];
        slope[1] = -g[1] / g[2];
        return 1;
    }
    double Aw[OSOG_ORACLE_MAX_PLANES][3], bb[OSOG_ORACLE_MAX_PLANES];
    const int M = prism_world_planes(R, dims[0], dims[1], dims[2], Aw, bb);
    double exit_ = INFINITY;
    int ke = -1;
    for (int k = 0; k < M; ++k) {
        const double nz = Aw[k][2];
        if (nz > 0.0) { const double z = (bb[k] - Aw[k][0] * dx - Aw[k][1] * dy) / nz; if (z < exit_) { exit_ = z; ke = k; } }
    }
    slope[0] = -Aw[ke][0] / Aw[ke][2];
    slope[1] = -Aw[ke][1] / Aw[ke][2];
    return 1;
}

/* Depth and instance-id maps of one frame (reading A24): for every pixel, among the particles whose chord there has
 * positive length, the one whose top surface  cz[n] + z_exit  is highest (+z points at the objective); ties go to the
 * smallest index.  top_id[i*W+j] = that particle's index (-1: no particle), depth[i*W+j] = the height of its top
 * surface in um (0 where top_id is -1).  cz may be NULL (all zero).  mode as in osog_oracle_render_opd. */
void osog_oracle_render_gbuffer(int64_t N,
                                const float *cx, const float *cy, const float *cz,
                                const float *qw, const float *qx, const float *qy, const float *qz,
                                const float *d0, const float *d1, const float *d2,
                                const float *n_p, const uint8_t *kind,
                                int H, int W, double pitch, int mode, int32_t *top_id, double *depth, double *normal)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < H; ++i) {
        const double y = (i + 0.5) * pitch;
        for (int j = 0; j < W; ++j) {
            top_id[(size_t)i * W + j] = -1; depth[(size_t)i * W + j] = 0.0;
            if (normal != NULL) normal[2 * ((size_t)i * W + j)] = normal[2 * ((size_t)i * W + j) + 1] = 0.0;
        }
        for (int64_t n = 0; n < N; ++n) {
            if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                            d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
            if (cz != NULL && !isfinite((double)cz[n])) continue;
            const double dy = y - (double)cy[n];
            const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
            const double dims[3] = { d0[n], d1[n], d2[n] };
            double R[9];
            osog_oracle_rot_from_quat(q, R);
            double r2 = INFINITY;
            if (mode == 1) {
                const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
                r2 = r * r;
                if (dy * dy > r2) continue;
            }
            const double zc = cz != NULL ? (double)cz[n] : 0.0;
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                double ze, zx;
                if (!osog_oracle_chord(kind[n], R, dims, dx, dy, &ze, &zx)) continue;
                const double top = zc + zx;
                const size_t px = (size_t)i * W + j;
                if (top_id[px] < 0 || top > depth[px]) {
                    top_id[px] = (int32_t)n; depth[px] = top;
                    if (normal != NULL) osog_oracle_top_slope(kind[n], R, dims, dx, dy, normal + 2 * px);   /* slope of the owner's top */
                }
            }
        }
    }
}

/* ---- first step of the backward pass ("the gradient of the final image with respect to
 * the initial state tensor"): adjoint of the OPD sum with respect to the refractive indices.  OPD[px] = sum_n (n_p[n] -
 * n_medium) t_n[px] is linear in n_p, so for an upstream gradient G = dL/dOPD (one frame, row-major [H*W]) the gradient
 * is  dL/dn_p[n] = sum over pixels of G[px] * t_n[px]  (pixels in row-major order, fp64 sum).  Invalid particles get 0. */
void osog_oracle_backward_np(int64_t N,
                             const float *cx, const float *cy,
                             const float *qw, const float *qx, const float *qy, const float *qz,
                             const float *d0, const float *d1, const float *d2,
                             const float *n_p, const uint8_t *kind,
                             int H, int W, double pitch, int mode, const float *G, double *g_np)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t n = 0; n < N; ++n) {
        g_np[n] = 0.0;
        if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                        d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
        const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
        double R[9];
        osog_oracle_rot_from_quat(q, R);
        double Aw[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
        int M = 0;
        if (kind[n] == 1) M = prism_world_planes(R, d0[n], d1[n], d2[n], Aw, b);
        double r2 = INFINITY;
        if (mode == 1) {
            const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
            r2 = r * r;
        }
        double acc = 0.0;
        for (int i = 0; i < H; ++i) {
            const double dy = (i + 0.5) * pitch - (double)cy[n];
            if (dy * dy > r2) continue;
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                const double t = kind[n] == 0
                    ? osog_oracle_thickness_ellipsoid(R, d0[n], d1[n], d2[n], dx, dy)
                    : osog_oracle_thickness_polyhedron(M, Aw, b, dx, dy);
                acc += (double)G[(size_t)i * W + j] * t;
            }
        }
        g_np[n] = acc;
    }
}

/* Gradient of the thickness with respect to the ray's lateral position (dx, dy) (equivalently minus the gradient with
 * respect to the particle's centre).  Ellipsoid: t = 2 sqrt(disc) / A with disc = Bq^2 - A C, so
 *   dt/dx = (d disc / dx) / (A sqrt(disc)),  d disc / dx = 2 Bq M_xz - 2 A (M_xx dx + M_xy dy)   (likewise y);
 * polyhedron: t = exit - enter with exit = g_e / n_ez on the active exit plane e (the arg min) and enter on the active
 * entry plane f (the arg max), g = b - n_x dx - n_y dy, so dt/dx = -n_ex / n_ez + n_fx / n_fz  (likewise y).
 * Where the chord is empty the gradient is 0.  (At the measure-zero set where two planes tie the first one is taken.) */
void osog_oracle_thickness_grad(uint8_t kind, const double R[9], const double dims[3], double dx, double dy, double grad[2])
{
    grad[0] = grad[1] = 0.0;
    if (kind == 0) {
        const double D[3] = { 1.0 / (dims[0] * dims[0]), 1.0 / (dims[1] * dims[1]), 1.0 / (dims[2] * dims[2]) };
        double M[9];
        for (int r = 0; r < 3; ++r)
            for (int s = 0; s < 3; ++s) {
                double acc = 0.0;
                for (int k = 0; k < 3; ++k) acc += R[3 * r + k] * D[k] * R[3 * s + k];
                M[3 * r + s] = acc;
            }
        const double A  = M[8];
        const double Bq = M[2] * dx + M[5] * dy;
        const double C  = M[0] * dx * dx + 2.0 * M[1] * dx * dy + M[4] * dy * dy - 1.0;
        const double disc = Bq * Bq - A * C;
        if (!(disc > 0.0)) return;
        const double sq = sqrt(disc);
        grad[0] = (2.0 * Bq * M[2] - 2.0 * A * (M[0] * dx + M[1] * dy)) / (A * sq);
        grad[1] = (2.0 * Bq * M[5] - 2.0 * A * (M[1] * dx + M[4] * dy)) / (A * sq);
        return;
    }
    double Aw[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
    const int M = prism_world_planes(R, dims[0], dims[1], dims[2], Aw, b);
    double enter = -INFINITY, exit_ = INFINITY;
    int ke = -1, kf = -1;
    for (int k = 0; k < M; ++k) {
        const double g = b[k] - Aw[k][0] * dx - Aw[k][1] * dy;
        const double nz = Aw[k][2];
        if (nz > 0.0)      { const double z = g / nz; if (z < exit_) { exit_ = z; ke = k; } }
        else if (nz < 0.0) { const double z = g / nz; if (z > enter) { enter = z; kf = k; } }
        else if (g < 0.0)  return;
    }
    if (!(exit_ - enter > 0.0)) return;
    grad[0] = -Aw[ke][0] / Aw[ke][2] + Aw[kf][0] / Aw[kf][2];
    grad[1] = -Aw[ke][1] / Aw[ke][2] + Aw[kf][1] / Aw[kf][2];
}

/* Second step of the backward pass: dL/d(cx, cy)[n] = -(n_p[n] - n_medium) * sum over pixels of G[px] * grad t_n[px]
 * (the thickness depends on the pixel position minus the centre).  g_c is [N][2]. */
void osog_oracle_backward_centre(int64_t N,
                                 const float *cx, const float *cy,
                                 const float *qw, const float *qx, const float *qy, const float *qz,
                                 const float *d0, const float *d1, const float *d2,
                                 const float *n_p, const uint8_t *kind,
                                 int H, int W, double pitch, double n_medium, int mode, const float *G, double *g_c)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t n = 0; n < N; ++n) {
        g_c[2 * n] = g_c[2 * n + 1] = 0.0;
        if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                        d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
        const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
        const double dims[3] = { d0[n], d1[n], d2[n] };
        double R[9];
        osog_oracle_rot_from_quat(q, R);
        double r2 = INFINITY;
        if (mode == 1) {
            const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
            r2 = r * r;
        }
        double ax = 0.0, ay = 0.0;
        for (int i = 0; i < H; ++i) {
            const double dy = (i + 0.5) * pitch - (double)cy[n];
            if (dy * dy > r2) continue;
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                double gr[2];
                osog_oracle_thickness_grad(kind[n], R, dims, dx, dy, gr);
                ax += (double)G[(size_t)i * W + j] * gr[0];
                ay += (double)G[(size_t)i * W + j] * gr[1];
            }
        }
        const double dn = (double)n_p[n] - n_medium;
        g_c[2 * n] = -dn * ax;
        g_c[2 * n + 1] = -dn * ay;
    }
}


/* ---- third step of the backward pass: gradient of the thickness with respect to the
 * particle's SHAPE parameters: grad[0..2] = dt/d(d0, d1, d2) (semi-axes a, b, c or side s, length L, cap height hc),
 * grad[3..6] = dt/d(qw, qx, qy, qz) (the four quaternion components as independent variables of the rotation formula of
 * osog_oracle_rot_from_quat, which does not renormalise: reading A4).  Chain rule written out:
 *   ellipsoid: M = R D R^T, D = diag(1/a^2, 1/b^2, 1/c^2);  dM = dR D R^T + R dD R^T + R D dR^T;
 *              A = M_zz, Bq = M_xz dx + M_yz dy, C = M_xx dx^2 + 2 M_xy dx dy + M_yy dy^2 - 1, disc = Bq^2 - A C,
 *              t = 2 sqrt(disc) / A  =>  dt = d(disc) / (A sqrt(disc)) - 2 sqrt(disc) dA / A^2,
 *              d(disc) = 2 Bq dBq - C dA - A dC;
 *   prism:     plane k: world normal n = R n_hat, offset b; z_k = (b - n_x dx - n_y dy) / n_z;
 *              dz_k = (db - dn_x dx - dn_y dy - z_k dn_z) / n_z, dn = dR n_hat + R dn_hat;
 *              t = z_e - z_f on the active exit plane e (arg min) and entry plane f (arg max)  =>  dt = dz_e - dz_f.
 * Where the chord is empty the gradient is 0. */
static void rot_derivatives(const double q[4], double dR[4][9])
{
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    const double dw[9] = { 0.0, -2.0 * z, 2.0 * y,   2.0 * z, 0.0, -2.0 * x,   -2.0 * y, 2.0 * x, 0.0 };
    const double dx[9] = { 0.0, 2.0 * y, 2.0 * z,    2.0 * y, -4.0 * x, -2.0 * w,   2.0 * z, 2.0 * w, -4.0 * x };
    const double dy[9] = { -4.0 * y, 2.0 * x, 2.0 * w,   2.0 * x, 0.0, 2.0 * z,   -2.0 * w, 2.0 * z, -4.0 * y };
    const double dz[9] = { -4.0 * z, -2.0 * w, 2.0 * x,   2.0 * w, -4.0 * z, 2.0 * y,   2.0 * x, 2.0 * y, 0.0 };
    for (int k = 0; k < 9; ++k) { dR[0][k] = dw[k]; dR[1][k] = dx[k]; dR[2][k] = dy[k]; dR[3][k] = dz[k]; }
}

void osog_oracle_thickness_param_grad(uint8_t kind, const double q[4], const double dims[3], double dx, double dy,
                                      double grad[7])
{
    for (int p = 0; p < 7; ++p) grad[p] = 0.0;
    double R[9], dR[4][9];
    osog_oracle_rot_from_quat(q, R);
    rot_derivatives(q, dR);
    if (kind == 0) {
        const double D[3] = { 1.0 / (dims[0] * dims[0]), 1.0 / (dims[1] * dims[1]), 1.0 / (dims[2] * dims[2]) };
        double M[9];
        for (int r = 0; r < 3; ++r)
            for (int s = 0; s < 3; ++s) {
                double acc = 0.0;
                for (int k = 0; k < 3; ++k) acc += R[3 * r + k] * D[k] * R[3 * s + k];
                M[3 * r + s] = acc;
            }
        const double A  = M[8];
        const double Bq = M[2] * dx + M[5] * dy;
        const double C  = M[0] * dx * dx + 2.0 * M[1] * dx * dy + M[4] * dy * dy - 1.0;
        const double disc = Bq * Bq - A * C;
        if (!(disc > 0.0)) return;
        const double sq = sqrt(disc);
        for (int p = 0; p < 7; ++p) {
            double dM[9];
            for (int r = 0; r < 3; ++r)
                for (int s = 0; s < 3; ++s) {
                    double acc = 0.0;
                    if (p < 3) {                       /* dD: only entry p of the diagonal, d(1/a^2)/da = -2/a^3 */
                        const double dDp = -2.0 / (dims[p] * dims[p] * dims[p]);
                        acc = R[3 * r + p] * dDp * R[3 * s + p];
                    } else {
                        const double *dRq = dR[p - 3];
                        for (int k = 0; k < 3; ++k) acc += dRq[3 * r + k] * D[k] * R[3 * s + k] + R[3 * r + k] * D[k] * dRq[3 * s + k];
                    }
                    dM[3 * r + s] = acc;
                }
            const double dA  = dM[8];
            const double dBq = dM[2] * dx + dM[5] * dy;
            const double dC  = dM[0] * dx * dx + 2.0 * dM[1] * dx * dy + dM[4] * dy * dy;
            const double ddisc = 2.0 * Bq * dBq - C * dA - A * dC;
            grad[p] = ddisc / (A * sq) - 2.0 * sq * dA / (A * A);
        }
        return;
    }
    /* prism: body planes and their derivatives in (s, L, hc), in the construction order of osog_oracle_prism_planes */
    const double s_ = dims[0], L_ = dims[1], hc = dims[2];
    double Ab[OSOG_ORACLE_MAX_PLANES][3], b[OSOG_ORACLE_MAX_PLANES];
    const int M = osog_oracle_prism_planes(s_, L_, hc, Ab, b);
    double dAb[OSOG_ORACLE_MAX_PLANES][3][3], db[OSOG_ORACLE_MAX_PLANES][3];   /* [plane][parameter][component] */
    for (int k = 0; k < M; ++k)
        for (int p = 0; p < 3; ++p) { db[k][p] = 0.0; for (int c = 0; c < 3; ++c) dAb[k][p][c] = 0.0; }
    for (int k = 0; k < 4; ++k) db[k][0] = 0.5;                                  /* side planes: b = s/2 */
    for (int k = 4; k < 12; ++k) {
        /* cap planes: normal (+-hc, 0, +-s/2) or (0, +-hc, +-s/2), b = hc s/2 + s L/4 */
        db[k][0] = 0.5 * hc + 0.25 * L_;  db[k][1] = 0.25 * s_;  db[k][2] = 0.5 * s_;
        const int lateral = k < 8 ? 0 : 1;                                       /* which lateral component carries +-hc */
        dAb[k][2][lateral] = Ab[k][lateral] > 0.0 ? 1.0 : -1.0;                  /* d(+-hc)/dhc */
        dAb[k][0][2] = Ab[k][2] > 0.0 ? 0.5 : -0.5;                              /* d(+-s/2)/ds */
    }
    double Aw[OSOG_ORACLE_MAX_PLANES][3];
    for (int k = 0; k < M; ++k)
        for (int r = 0; r < 3; ++r)
            Aw[k][r] = R[3 * r + 0] * Ab[k][0] + R[3 * r + 1] * Ab[k][1] + R[3 * r + 2] * Ab[k][2];
    double enter = -INFINITY, exit_ = INFINITY;
    int ke = -1, kf = -1;
    for (int k = 0; k < M; ++k) {
        const double g = b[k] - Aw[k][0] * dx - Aw[k][1] * dy;
        const double nz = Aw[k][2];
        if (nz > 0.0)      { const double z = g / nz; if (z < exit_) { exit_ = z; ke = k; } }
        else if (nz < 0.0) { const double z = g / nz; if (z > enter) { enter = z; kf = k; } }
        else if (g < 0.0)  return;
    }
    if (!(exit_ - enter > 0.0)) return;
    const int act[2] = { ke, kf };
    const double zact[2] = { exit_, enter };
    for (int p = 0; p < 7; ++p) {
        double dz[2];
        for (int a = 0; a < 2; ++a) {
            const int k = act[a];
            double dn[3], dbk;
            if (p < 3) {
                dbk = db[k][p];
                for (int r = 0; r < 3; ++r)
                    dn[r] = R[3 * r + 0] * dAb[k][p][0] + R[3 * r + 1] * dAb[k][p][1] + R[3 * r + 2] * dAb[k][p][2];
            } else {
                dbk = 0.0;
                const double *dRq = dR[p - 3];
                for (int r = 0; r < 3; ++r)
                    dn[r] = dRq[3 * r + 0] * Ab[k][0] + dRq[3 * r + 1] * Ab[k][1] + dRq[3 * r + 2] * Ab[k][2];
            }
            dz[a] = (dbk - dn[0] * dx - dn[1] * dy - zact[a] * dn[2]) / Aw[k][2];
        }
        grad[p] = dz[0] - dz[1];
    }
}

/* dL/d(d0, d1, d2, qw, qx, qy, qz)[n] = (n_p[n] - n_medium) * sum over pixels of G[px] * dt_n/dtheta[px];  g_p is [N][7]. */
void osog_oracle_backward_params(int64_t N,
                                 const float *cx, const float *cy,
                                 const float *qw, const float *qx, const float *qy, const float *qz,
                                 const float *d0, const float *d1, const float *d2,
                                 const float *n_p, const uint8_t *kind,
                                 int H, int W, double pitch, double n_medium, int mode, const float *G, double *g_p)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t n = 0; n < N; ++n) {
        for (int p = 0; p < 7; ++p) g_p[7 * n + p] = 0.0;
        if (!osog_oracle_particle_valid(cx[n], cy[n], qw[n], qx[n], qy[n], qz[n],
                                        d0[n], d1[n], d2[n], n_p[n], kind[n])) continue;
        const double q[4] = { qw[n], qx[n], qy[n], qz[n] };
        const double dims[3] = { d0[n], d1[n], d2[n] };
        double r2 = INFINITY;
        if (mode == 1) {
            const double r = osog_oracle_circumradius(kind[n], d0[n], d1[n], d2[n]) * (1.0 + 1e-9);
            r2 = r * r;
        }
        double acc[7] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
        for (int i = 0; i < H; ++i) {
            const double dy = (i + 0.5) * pitch - (double)cy[n];
            if (dy * dy > r2) continue;
            for (int j = 0; j < W; ++j) {
                const double dx = (j + 0.5) * pitch - (double)cx[n];
                if (dx * dx + dy * dy > r2) continue;
                double gr[7];
                osog_oracle_thickness_param_grad(kind[n], q, dims, dx, dy, gr);
                for (int p = 0; p < 7; ++p) acc[p] += (double)G[(size_t)i * W + j] * gr[p];
            }
        }
        const double dn = (double)n_p[n] - n_medium;
        for (int p = 0; p < 7; ++p) g_p[7 * n + p] = dn * acc[p];
    }
}
