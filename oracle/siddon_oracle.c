/* siddon_oracle.c -- fp64 CPU oracle for the paper's OWN forward projector: Siddon's exact radiological path
 * ("each GPU thread computing the line integral of Eq. (1) along an x-ray line using Siddon's
 * ray-tracing algorithm (Siddon, 1985 ...)") and its literal transpose.
 * TEST INFRASTRUCTURE ONLY: nothing here is imported, linked or executed by the CUDA path, and it shares no
 * code with it.  SURVEY.md §8(f) NEXT-2.
 *
 * Definition (Siddon 1985, restated): the volume is piecewise constant, voxel (ix,iy,iz) filling
 * [xb + ix dx, xb + (ix+1) dx] x ... with xb = ox - nx dx / 2.  For the segment from the source S to the pixel
 * centre D, p(a) = S + a (D - S), a in [0,1]:
 *   1. the parameters a at which the ray meets every grid plane x = xb + i dx (i = 0..nx), same for y and z;
 *   2. a_min / a_max = entry / exit of the volume box (clipped to [0,1]);
 *   3. merge {a_min, a_max} and all plane parameters strictly between them, sorted;
 *   4. every consecutive pair (a_m, a_m+1) is one voxel crossing: length (a_m+1 - a_m) |D - S|, voxel = the
 *      one containing the midpoint;  g = sum length * f[voxel].
 * Written as exactly that (all plane parameters collected and sorted, no incremental traversal), so that it
 * can be checked against the description by eye.  The transpose adds g * length into the same voxels.
 *
 * Pins (tests/test_oracle_siddon.py, -m "not gpu"): for f = 1 the result is the chord of the volume box in closed
 * form; analytic ellipsoid chords (first-order convergence); a dense-sampling nearest-neighbour estimate of the
 * same path lengths; the adjoint identity; non-zeros per ray at the paper's own geometry against PAPER.md:211
 * ("approximately 4 x 10^9 non-zero elements").
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz, ox, oy, oz;
    int32_t nu, nv;
    double du, dv, u0, v0;
    double sad, sdd;
    int32_t n_views;
    const double *angles;
    double step; /* unused by Siddon: there is no step parameter */
} orc_geom;

static int cmp_double(const void *a, const void *b) {
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* source S and pixel centre D of ray (view, iv, iu): geometry of SURVEY.md §8(c) c.1 */
static void ray_ends(const orc_geom *G, int view, int iv, int iu, double S[3], double D[3]) {
    double th = G->angles[view], c = cos(th), s = sin(th);
    double u = G->u0 + (iu - 0.5 * (G->nu - 1)) * G->du;
    double v = G->v0 + (iv - 0.5 * (G->nv - 1)) * G->dv;
    double gap = G->sdd - G->sad;
    S[0] = G->sad * c; S[1] = G->sad * s; S[2] = 0.0;
    D[0] = -gap * c - u * s; D[1] = -gap * s + u * c; D[2] = v;
}

/* One ray.  mode 0: return sum length*f;  mode 1: f[voxel] += gval*length (caller serialises);  mode 2: return the
 * number of voxel crossings of positive length.  `buf` holds nx+ny+nz+5 doubles. */
static double siddon_ray(const orc_geom *G, int view, int iv, int iu, int mode, const double *f, double *fout, double gval,
                         double *buf) {
    double S[3], D[3];
    ray_ends(G, view, iv, iu, S, D);
    const double d[3] = {D[0] - S[0], D[1] - S[1], D[2] - S[2]};
    const double len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    const int n[3] = {G->nx, G->ny, G->nz};
    const double h[3] = {G->dx, G->dy, G->dz};
    const double b0[3] = {G->ox - 0.5 * G->nx * G->dx, G->oy - 0.5 * G->ny * G->dy, G->oz - 0.5 * G->nz * G->dz};
    double amin = 0.0, amax = 1.0;
    for (int a = 0; a < 3; ++a) {
        if (d[a] == 0.0) {
            if (S[a] <= b0[a] || S[a] >= b0[a] + n[a] * h[a]) return 0.0; /* parallel to and outside the slab */
            continue;
        }
        double a0 = (b0[a] - S[a]) / d[a], a1 = (b0[a] + n[a] * h[a] - S[a]) / d[a];
        double lo = a0 < a1 ? a0 : a1, hi = a0 < a1 ? a1 : a0;
        if (lo > amin) amin = lo;
        if (hi < amax) amax = hi;
    }
    if (!(amin < amax)) return 0.0;
    long m = 0;
    buf[m++] = amin;
    buf[m++] = amax;
    for (int a = 0; a < 3; ++a) {
        if (d[a] == 0.0) continue;
        for (int i = 0; i <= n[a]; ++i) {
            double al = (b0[a] + i * h[a] - S[a]) / d[a];
            if (al > amin && al < amax) buf[m++] = al;
        }
    }
    qsort(buf, (size_t)m, sizeof(double), cmp_double);
    double acc = 0.0;
    for (long j = 0; j + 1 < m; ++j) {
        double a0 = buf[j], a1 = buf[j + 1];
        if (!(a1 > a0)) continue;                       /* a plane crossing shared by two axes: zero length */
        double am = 0.5 * (a0 + a1);
        long idx[3];
        int inside = 1;
        for (int a = 0; a < 3; ++a) {
            idx[a] = (long)floor((S[a] + am * d[a] - b0[a]) / h[a]);
            if (idx[a] < 0 || idx[a] >= n[a]) inside = 0;
        }
        if (!inside) continue;                          /* cannot happen for a_min < am < a_max; kept as a guard */
        size_t lin = ((size_t)idx[2] * G->ny + idx[1]) * G->nx + idx[0];
        double l = (a1 - a0) * len;
        if (mode == 0) acc += l * f[lin];
        else if (mode == 1) fout[lin] += gval * l;
        else acc += 1.0;
    }
    return acc;
}

/* g = P_siddon f */
void orc_siddon_forward(const orc_geom *G, const double *f, double *g) {
    long n_rays = (long)G->n_views * G->nv * G->nu;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)(G->nx + G->ny + G->nz + 8));
#pragma omp for schedule(dynamic, 64)
        for (long r = 0; r < n_rays; ++r) {
            int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
            g[r] = siddon_ray(G, view, iv, iu, 0, f, 0, 0.0, buf);
        }
        free(buf);
    }
}

/* f = P_siddon^T g: the literal transpose, ray by ray (serial over rays: the scatter of PAPER.md:211) */
void orc_siddon_back(const orc_geom *G, const double *g, double *f) {
    long n_rays = (long)G->n_views * G->nv * G->nu, nvox = (long)G->nx * G->ny * G->nz;
    for (long j = 0; j < nvox; ++j) f[j] = 0.0;
    double *buf = (double *)malloc(sizeof(double) * (size_t)(G->nx + G->ny + G->nz + 8));
    for (long r = 0; r < n_rays; ++r) {
        int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
        siddon_ray(G, view, iv, iu, 1, 0, f, g[r], buf);
    }
    free(buf);
}

/* number of (ray, voxel) pairs with positive intersection length over the rays r = first, first+stride, ... */
double orc_siddon_nnz(const orc_geom *G, long first, long stride) {
    long n_rays = (long)G->n_views * G->nv * G->nu;
    double total = 0.0;
#pragma omp parallel reduction(+ : total)
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)(G->nx + G->ny + G->nz + 8));
#pragma omp for schedule(dynamic, 64)
        for (long r = first; r < n_rays; r += stride) {
            int iu = (int)(r % G->nu), iv = (int)((r / G->nu) % G->nv), view = (int)(r / ((long)G->nu * G->nv));
            total += siddon_ray(G, view, iv, iu, 2, 0, 0, 0.0, buf);
        }
        free(buf);
    }
    return total;
}
