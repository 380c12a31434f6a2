/* cbct_oracle.c -- fp64 CPU ORACLE for the cone-beam projector pair.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or constant with the CUDA path
 * (paper_1008_2042_b200/csrc) and neither includes the other.
 *
 * What it computes (citations: /root/reference/PAPER.md line + section; SURVEY.md §8(c) reading):
 *   orc_forward*      g = P f   PAPER.md:73 Eq. 1, discretised as the midpoint rule on a global,
 *                               source-anchored t-grid with zero-padded trilinear interpolation
 *                               (north_star "fixed step ... trilinear").
 *   orc_back_scatter  f = P^T g the matrix transpose of the above, written as the literal scatter
 *                               ("updating voxel values along all ray lines").
 *   orc_back_gather*  f = P^T g the same transpose, voxel-driven ("one thread per
 *                               voxel"), loop structure of SURVEY.md §8(c) c.3 gather form.
 *   orc_back_eq3      the paper's own approximate adjoint, Eq. 3 with bilinear
 *                               detector interpolation.  Used only as a pin.
 *   orc_sample_count  algorithmic sample count: sum over rays of chord(padded box)/step.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): analytic ellipsoid chords, uniform-slab closed form,
 * symmetry, adjoint identity to 1e-12, explicit 8x8x4 system matrix, scatter==gather, Eq. 3 within
 * the paper's "<1 %".  No function here is "parity unpinned".
 *
 * Everything is plain loops in double precision.  No clipping, blocking or reordering beyond what
 * the definition states; OpenMP only distributes independent outputs (rays / voxels / views).
 *
 * Geometry (Fig. 1 is missing from PAPER.md:89; convention of SURVEY.md §8(c) c.1):
 *   world mm, origin = isocentre, z = rotation axis
 *   voxel centre   x = ox + (ix - (nx-1)/2) dx   (same for y, z);   f[z][y][x], x fastest
 *   source         x_S = (SAD cos th, SAD sin th, 0)
 *   detector       d = c_D + u e_u + v e_v,  c_D = -(SDD-SAD)(cos th, sin th, 0),
 *                  e_u = (-sin th, cos th, 0), e_v = (0,0,1),  u = u0 + (iu - (nu-1)/2) du
 *   g[view][v][u], u fastest
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz, ox, oy, oz;
    int32_t nu, nv;
    double du, dv, u0, v0;
    double sad, sdd;
    int32_t n_views;
    const double *angles;
    double step; /* > 0, already resolved by the caller */
} orc_geom;

/* global t-grid: SURVEY.md §8(c) c.2 */
static double grid_R(const orc_geom *G) {
    double hx = 0.5 * (G->nx + 1) * G->dx, hy = 0.5 * (G->ny + 1) * G->dy, hz = 0.5 * (G->nz + 1) * G->dz;
    return sqrt(hx * hx + hy * hy + hz * hz) + sqrt(G->ox * G->ox + G->oy * G->oy + G->oz * G->oz);
}
void orc_grid(const orc_geom *G, double *R, double *t_min, int32_t *K) {
    double r = grid_R(G);
    *R = r;
    *t_min = G->sad - r;
    *K = (int32_t)ceil(2.0 * r / G->step);
}

static void ray_setup(const orc_geom *G, int view, int iv, int iu, double src[3], double n[3]) {
    double th = G->angles[view], c = cos(th), s = sin(th);
    double u = G->u0 + (iu - 0.5 * (G->nu - 1)) * G->du;
    double v = G->v0 + (iv - 0.5 * (G->nv - 1)) * G->dv;
    double gap = G->sdd - G->sad;
    double d[3] = {-gap * c + u * (-s), -gap * s + u * c, v};
    src[0] = G->sad * c; src[1] = G->sad * s; src[2] = 0.0;
    double e[3] = {d[0] - src[0], d[1] - src[1], d[2] - src[2]};
    double L = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
    n[0] = e[0] / L; n[1] = e[1] / L; n[2] = e[2] / L;
}

/* world point -> index coordinates X = (x-ox)/dx + (nx-1)/2 */
static void to_index(const orc_geom *G, const double p[3], double X[3]) {
    X[0] = (p[0] - G->ox) / G->dx + 0.5 * (G->nx - 1);
    X[1] = (p[1] - G->oy) / G->dy + 0.5 * (G->ny - 1);
    X[2] = (p[2] - G->oz) / G->dz + 0.5 * (G->nz - 1);
}

static double fetch(const orc_geom *G, const double *f, long ix, long iy, long iz) {
    if (ix < 0 || iy < 0 || iz < 0 || ix >= G->nx || iy >= G->ny || iz >= G->nz) return 0.0;
    return f[((size_t)iz * G->ny + iy) * G->nx + ix];
}

/* T[f](p): zero-padded trilinear interpolation at index coordinates X */
static double trilinear(const orc_geom *G, const double *f, const double X[3]) {
    double fx = floor(X[0]), fy = floor(X[1]), fz = floor(X[2]);
    long ix = (long)fx, iy = (long)fy, iz = (long)fz;
    double wx = X[0] - fx, wy = X[1] - fy, wz = X[2] - fz;
    double acc = 0.0;
    for (int c = 0; c < 2; ++c)
        for (int b = 0; b < 2; ++b)
            for (int a = 0; a < 2; ++a) {
                double w = (a ? wx : 1.0 - wx) * (b ? wy : 1.0 - wy) * (c ? wz : 1.0 - wz);
                acc += w * fetch(G, f, ix + a, iy + b, iz + c);
            }
    return acc;
}

static double forward_one(const orc_geom *G, const double *f, int view, int iv, int iu) {
    double R, t_min; int32_t K;
    orc_grid(G, &R, &t_min, &K);
    double src[3], n[3];
    ray_setup(G, view, iv, iu, src, n);
    double sum = 0.0;
    for (int32_t k = 0; k < K; ++k) {
        double t = t_min + (k + 0.5) * G->step;
        double p[3] = {src[0] + n[0] * t, src[1] + n[1] * t, src[2] + n[2] * t}, X[3];
        to_index(G, p, X);
        sum += trilinear(G, f, X);
    }
    return G->step * sum;
}

/* g = P f for every ray */
void orc_forward(const orc_geom *G, const double *f, double *g) {
    long n_rays = (long)G->n_views * G->nv * G->nu;
#pragma omp parallel for schedule(dynamic, 64)
    for (long r = 0; r < n_rays; ++r) {
        int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
        g[r] = forward_one(G, f, view, iv, iu);
    }
}

/* g[ray] for a list of flat ray indices (view*nv + iv)*nu + iu */
void orc_forward_rays(const orc_geom *G, const double *f, long n, const int64_t *rays, double *out) {
#pragma omp parallel for schedule(dynamic, 16)
    for (long i = 0; i < n; ++i) {
        long r = (long)rays[i];
        int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
        out[i] = forward_one(G, f, view, iv, iu);
    }
}

/* scatter one view of g into vol (+=).  Literal transpose of forward_one. */
static void scatter_view(const orc_geom *G, const double *g, int view, double *vol) {
    double R, t_min; int32_t K;
    orc_grid(G, &R, &t_min, &K);
    for (int iv = 0; iv < G->nv; ++iv)
        for (int iu = 0; iu < G->nu; ++iu) {
            double gr = g[((size_t)view * G->nv + iv) * G->nu + iu];
            double src[3], n[3];
            ray_setup(G, view, iv, iu, src, n);
            for (int32_t k = 0; k < K; ++k) {
                double t = t_min + (k + 0.5) * G->step;
                double p[3] = {src[0] + n[0] * t, src[1] + n[1] * t, src[2] + n[2] * t}, X[3];
                to_index(G, p, X);
                double fx = floor(X[0]), fy = floor(X[1]), fz = floor(X[2]);
                long ix = (long)fx, iy = (long)fy, iz = (long)fz;
                double wx = X[0] - fx, wy = X[1] - fy, wz = X[2] - fz;
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a) {
                            long jx = ix + a, jy = iy + b, jz = iz + c;
                            if (jx < 0 || jy < 0 || jz < 0 || jx >= G->nx || jy >= G->ny || jz >= G->nz) continue;
                            double w = (a ? wx : 1.0 - wx) * (b ? wy : 1.0 - wy) * (c ? wz : 1.0 - wz);
                            vol[((size_t)jz * G->ny + jy) * G->nx + jx] += G->step * gr * w;
                        }
            }
        }
}

/* f = P^T g, scatter form.  Views are independent: each gets a private volume, summed in view order. */
void orc_back_scatter(const orc_geom *G, const double *g, double *f) {
    size_t nvox = (size_t)G->nx * G->ny * G->nz;
    memset(f, 0, nvox * sizeof(double));
    int chunk = 8;
    double *priv = (double *)malloc((size_t)chunk * nvox * sizeof(double));
    for (int v0 = 0; v0 < G->n_views; v0 += chunk) {
        int nv_ = G->n_views - v0 < chunk ? G->n_views - v0 : chunk;
        memset(priv, 0, (size_t)nv_ * nvox * sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
        for (int j = 0; j < nv_; ++j) scatter_view(G, g, v0 + j, priv + (size_t)j * nvox);
        for (int j = 0; j < nv_; ++j)
            for (size_t i = 0; i < nvox; ++i) f[i] += priv[(size_t)j * nvox + i];
    }
    free(priv);
}

static double hat(double d) { double a = 1.0 - fabs(d); return a > 0.0 ? a : 0.0; }

/* voxel-driven gather: voxel centre c in index space, support cube [c-1,c+1]^3 */
static double gather_one(const orc_geom *G, const double *g, int jx, int jy, int jz) {
    double R, t_min; int32_t K;
    orc_grid(G, &R, &t_min, &K);
    double cidx[3] = {(double)jx, (double)jy, (double)jz};
    double total = 0.0;
    for (int view = 0; view < G->n_views; ++view) {
        double th = G->angles[view], c = cos(th), s = sin(th);
        /* project the 8 corners of the support cube: pixel-index bounding rectangle */
        double umin = 1e300, umax = -1e300, vmin = 1e300, vmax = -1e300;
        for (int cz = -1; cz <= 1; cz += 2)
            for (int cy = -1; cy <= 1; cy += 2)
                for (int cx = -1; cx <= 1; cx += 2) {
                    double x = G->ox + (jx + cx - 0.5 * (G->nx - 1)) * G->dx;
                    double y = G->oy + (jy + cy - 0.5 * (G->ny - 1)) * G->dy;
                    double z = G->oz + (jz + cz - 0.5 * (G->nz - 1)) * G->dz;
                    double D = G->sad - (x * c + y * s);
                    double tau = -x * s + y * c;
                    double us = G->sdd * tau / D, vs = G->sdd * z / D;
                    double pu = (us - G->u0) / G->du + 0.5 * (G->nu - 1);
                    double pv = (vs - G->v0) / G->dv + 0.5 * (G->nv - 1);
                    if (pu < umin) umin = pu;
                    if (pu > umax) umax = pu;
                    if (pv < vmin) vmin = pv;
                    if (pv > vmax) vmax = pv;
                }
        long iu0 = (long)ceil(umin) - 1, iu1 = (long)floor(umax) + 1; /* widened by one: harmless, hat clamps */
        long iv0 = (long)ceil(vmin) - 1, iv1 = (long)floor(vmax) + 1;
        if (iu0 < 0) iu0 = 0;
        if (iv0 < 0) iv0 = 0;
        if (iu1 > G->nu - 1) iu1 = G->nu - 1;
        if (iv1 > G->nv - 1) iv1 = G->nv - 1;
        double view_sum = 0.0;
        for (long iv = iv0; iv <= iv1; ++iv)
            for (long iu = iu0; iu <= iu1; ++iu) {
                double src[3], n[3], a[3], b[3], o[3] = {0, 0, 0}, e[3];
                ray_setup(G, view, (int)iv, (int)iu, src, n);
                /* ray in index space p(t) = a + b t */
                to_index(G, src, a);
                e[0] = src[0] + n[0]; e[1] = src[1] + n[1]; e[2] = src[2] + n[2];
                to_index(G, e, o);
                b[0] = o[0] - a[0]; b[1] = o[1] - a[1]; b[2] = o[2] - a[2];
                /* slab clip against the support cube */
                double tin = -1e300, tout = 1e300;
                int miss = 0;
                for (int ax = 0; ax < 3; ++ax) {
                    double lo = cidx[ax] - 1.0, hi = cidx[ax] + 1.0;
                    if (b[ax] == 0.0) {
                        if (a[ax] < lo || a[ax] > hi) miss = 1;
                    } else {
                        double t1 = (lo - a[ax]) / b[ax], t2 = (hi - a[ax]) / b[ax];
                        if (t1 > t2) { double tmp = t1; t1 = t2; t2 = tmp; }
                        if (t1 > tin) tin = t1;
                        if (t2 < tout) tout = t2;
                    }
                }
                if (miss || tin > tout) continue;
                long klo = (long)ceil((tin - t_min) / G->step - 0.5) - 1;  /* widened by one: harmless */
                long khi = (long)floor((tout - t_min) / G->step - 0.5) + 1;
                if (klo < 0) klo = 0;
                if (khi > K - 1) khi = K - 1;
                double gr = g[((size_t)view * G->nv + iv) * G->nu + iu];
                for (long k = klo; k <= khi; ++k) {
                    double t = t_min + (k + 0.5) * G->step;
                    double p[3] = {src[0] + n[0] * t, src[1] + n[1] * t, src[2] + n[2] * t}, X[3];
                    to_index(G, p, X);
                    view_sum += hat(X[0] - cidx[0]) * hat(X[1] - cidx[1]) * hat(X[2] - cidx[2]) * gr;
                }
            }
        total += view_sum;
    }
    return G->step * total;
}

void orc_back_gather(const orc_geom *G, const double *g, double *f) {
    long nvox = (long)G->nx * G->ny * G->nz;
#pragma omp parallel for schedule(dynamic, 64)
    for (long j = 0; j < nvox; ++j) {
        int jx = (int)(j % G->nx), jy = (int)((j / G->nx) % G->ny), jz = (int)(j / ((long)G->nx * G->ny));
        f[j] = gather_one(G, g, jx, jy, jz);
    }
}

void orc_back_gather_voxels(const orc_geom *G, const double *g, long n, const int64_t *vox, double *out) {
#pragma omp parallel for schedule(dynamic, 4)
    for (long i = 0; i < n; ++i) {
        long j = (long)vox[i];
        int jx = (int)(j % G->nx), jy = (int)((j / G->nx) % G->ny), jz = (int)(j / ((long)G->nx * G->ny));
        out[i] = gather_one(G, g, jx, jy, jz);
    }
}

/* PAPER.md:215 Eq. 3: f(x) = (dx dy dz)/(du dv) sum_theta L^3(u*) / (L0 l^2(x)) g^theta(u*),
 * u* = where the line source->x meets the imager, g(u*) by bilinear interpolation,
 * zero outside the imager. */
void orc_back_eq3(const orc_geom *G, const double *g, double *f) {
    long nvox = (long)G->nx * G->ny * G->nz;
    double pref = (G->dx * G->dy * G->dz) / (G->du * G->dv);
#pragma omp parallel for schedule(dynamic, 256)
    for (long j = 0; j < nvox; ++j) {
        int jx = (int)(j % G->nx), jy = (int)((j / G->nx) % G->ny), jz = (int)(j / ((long)G->nx * G->ny));
        double x = G->ox + (jx - 0.5 * (G->nx - 1)) * G->dx;
        double y = G->oy + (jy - 0.5 * (G->ny - 1)) * G->dy;
        double z = G->oz + (jz - 0.5 * (G->nz - 1)) * G->dz;
        double acc = 0.0;
        for (int view = 0; view < G->n_views; ++view) {
            double th = G->angles[view], c = cos(th), s = sin(th);
            double D = G->sad - (x * c + y * s), tau = -x * s + y * c;
            double us = G->sdd * tau / D, vs = G->sdd * z / D;
            double L = sqrt(G->sdd * G->sdd + us * us + vs * vs);      /* L(u*) */
            double l2 = D * D + tau * tau + z * z;                     /* l(x)^2 */
            double pu = (us - G->u0) / G->du + 0.5 * (G->nu - 1);
            double pv = (vs - G->v0) / G->dv + 0.5 * (G->nv - 1);
            double fu = floor(pu), fv = floor(pv);
            long iu = (long)fu, iv = (long)fv;
            double wu = pu - fu, wv = pv - fv, val = 0.0;
            for (int b = 0; b < 2; ++b)
                for (int a = 0; a < 2; ++a) {
                    long ju = iu + a, jv = iv + b;
                    if (ju < 0 || jv < 0 || ju >= G->nu || jv >= G->nv) continue;
                    val += (a ? wu : 1.0 - wu) * (b ? wv : 1.0 - wv) * g[((size_t)view * G->nv + jv) * G->nu + ju];
                }
            acc += L * L * L / (G->sdd * l2) * val;
        }
        f[j] = pref * acc;
    }
}

/* algorithmic samples: sum over rays of (chord through the zero-padded box [-1,n]^3 in index space)/step */
double orc_sample_count(const orc_geom *G) {
    long n_rays = (long)G->n_views * G->nv * G->nu;
    double total = 0.0;
#pragma omp parallel for reduction(+ : total) schedule(static)
    for (long r = 0; r < n_rays; ++r) {
        int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
        double src[3], n[3], a[3], e[3], o[3];
        ray_setup(G, view, iv, iu, src, n);
        to_index(G, src, a);
        e[0] = src[0] + n[0]; e[1] = src[1] + n[1]; e[2] = src[2] + n[2];
        to_index(G, e, o);
        double hi[3] = {(double)G->nx, (double)G->ny, (double)G->nz};
        double tin = -1e300, tout = 1e300;
        int miss = 0;
        for (int ax = 0; ax < 3; ++ax) {
            double b = o[ax] - a[ax];
            if (b == 0.0) { if (a[ax] < -1.0 || a[ax] > hi[ax]) miss = 1; continue; }
            double t1 = (-1.0 - a[ax]) / b, t2 = (hi[ax] - a[ax]) / b;
            if (t1 > t2) { double tmp = t1; t1 = t2; t2 = tmp; }
            if (t1 > tin) tin = t1;
            if (t2 < tout) tout = t2;
        }
        if (!miss && tout > tin) total += (tout - tin) / G->step;
    }
    return total;
}
