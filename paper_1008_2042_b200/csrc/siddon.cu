// siddon.cu -- the paper's OWN projector pair: Siddon's exact radiological path,
// PAPER.md:191 ("each GPU thread computing the line integral of Eq. (1) along an x-ray line using Siddon's
// ray-tracing algorithm"), and its exact transpose ("f = P^T g").  include/cbct.h: cbct_siddon_forward,
// cbct_siddon_backproject.  The voxel model is piecewise constant: voxel (ix,iy,iz) fills
// [xb + ix dx, xb + (ix+1) dx] x ..., xb = ox - nx dx / 2, and
//     (P f)[ray] = sum over voxels  |ray ∩ voxel| f[voxel]           (no step parameter).
// One thread per ray as in the paper, but as an incremental traversal: the ray is followed from the entry face of the
// volume box to its exit face; at every step the nearest of the three next grid-plane crossings ends the current
// voxel.  What is B200-specific:
//   * the crossing parameter of plane i on axis a is evaluated afresh by ONE fused multiply-add from the integer
//     plane number, tau_a(i) = i * (1/b_a) + k_a  (tau = distance along the ray from the point at t = SAD, so |tau|
//     stays below the volume radius), never by repeated addition: no drift over the ~1000 crossings of a ray, and the
//     rounding of a crossing cancels between the two segments it separates except for (f_before - f_after);
//   * the 73 MB volume lives in the 126 MB L2; views whose rays run along x read a y-fastest copy (the 32 lanes of
//     a warp are neighbouring pixels along u, so their voxels are neighbours along the fast axis in both cases);
//   * P^T is the same traversal scattering  g * length  with fire-and-forget integer reductions (RED.ADD.S32) into
//     an int32 volume in L2: fixed point relative to max|g| as in backproject_tma.cu, so the transpose is
//     order-independent, bit-reproducible and free of the write conflicts PAPER.md:211 had to avoid; the scale and the
//     number of views per accumulation group come from a rigorous bound on the path length one voxel can collect.
// Ray set-up (entry/exit, first voxel, 1/b, k) is done in fp64 per ray; the traversal runs in fp32.
#include <cmath>

#include "common.cuh"

namespace cbct {

struct SiddonRay {
    float ib[3], k[3];          // crossing of plane p on axis a: tau = (p - p0[a]) * ib[a] + k[a]   (ib = 1/b, k = -(c - p0)/b)
    int p0[3];
    float tau, tau_end;         // current parameter (entry) and end of the segment inside the box
    int i[3], dir[3], n[3];     // current voxel, step per axis (+1 / -1 / 0), grid size
    bool hit;
};

// Entry/exit of ray (view, iv, iu) through the volume box in plane-index coordinates X_a(tau) = c_a + b_a tau
// (X_a = 0 .. n_a are the grid planes), clipped to the source-to-pixel segment.
__device__ __forceinline__ SiddonRay siddon_setup(const DevGeom &g, int view, int iv, int iu) {
    SiddonRay s;
    s.hit = false;
    const double2 cs = g.view_cs[view];
    const double u = g.u_first + iu * g.du, v = g.v_first + iv * g.dv;
    const double ex = -g.sdd * cs.x - u * cs.y, ey = -g.sdd * cs.y + u * cs.x, ez = v;      // pixel centre - source
    const double L = sqrt(ex * ex + ey * ey + ez * ez), invL = 1.0 / L;
    const double nrm[3] = {ex * invL, ey * invL, ez * invL};
    const double src[3] = {g.sad * cs.x, g.sad * cs.y, 0.0};
    const double inv_h[3] = {g.inv_dx, g.inv_dy, g.inv_dz};
    // voxel-CENTRE index coordinate is x * inv_dx + cx; the grid PLANE coordinate is that + 1/2
    const double off[3] = {g.cx + 0.5, g.cy + 0.5, g.cz + 0.5};
    s.n[0] = g.nx; s.n[1] = g.ny; s.n[2] = g.nz;
    double b[3], c[3];
    double tin = -g.sad, tout = L - g.sad;                                                  // a in [0, 1]
    int entry_axis = -1;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        b[a] = nrm[a] * inv_h[a];
        c[a] = (src[a] + nrm[a] * g.sad) * inv_h[a] + off[a];
        if (b[a] == 0.0) {
            if (c[a] <= 0.0 || c[a] >= (double)s.n[a]) return s;                            // parallel to and outside the slab
            continue;
        }
        const double t0 = (0.0 - c[a]) / b[a], t1 = ((double)s.n[a] - c[a]) / b[a];
        const double lo = fmin(t0, t1), hi = fmax(t0, t1);
        if (lo > tin) { tin = lo; entry_axis = a; }
        tout = fmin(tout, hi);
    }
    if (!(tin < tout)) return s;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        s.dir[a] = b[a] > 0.0 ? 1 : (b[a] < 0.0 ? -1 : 0);
        const double xin = c[a] + b[a] * tin, xout = c[a] + b[a] * tout;
        int i = (int)floor(xin);
        if (a == entry_axis) i = b[a] > 0.0 ? 0 : s.n[a] - 1;                               // exactly on the entry face
        s.i[a] = min(max(i, 0), s.n[a] - 1);
        // An axis whose planes the ray does not cross strictly inside (tin, tout) takes no part: this also keeps 1/b finite
        // for rays (numerically) parallel to a grid plane.  Otherwise 1/|b| <= path length, and plane numbers are counted
        // from the plane nearest to the anchor (tau = 0), p0 = round(c), so that |p' / b| ~ |tau| and the FMA stays accurate.
        const double lo = fmin(xin, xout) + 1e-9, hi = fmax(xin, xout) - 1e-9;
        if (b[a] != 0.0 && floor(hi) >= ceil(lo)) {
            s.p0[a] = (int)floor(c[a] + 0.5);
            s.ib[a] = (float)(1.0 / b[a]); s.k[a] = (float)(-(c[a] - (double)s.p0[a]) / b[a]);
        } else {
            s.dir[a] = 0; s.p0[a] = 0; s.ib[a] = 0.f; s.k[a] = 3.0e38f;                    // never the nearest crossing
        }
    }
    s.tau = (float)tin; s.tau_end = (float)tout;
    s.hit = true;
    return s;
}

// The traversal.  `visit(linear_index, length)` is called once per voxel crossing of positive or zero length.
template <class Visit>
__device__ __forceinline__ void siddon_walk(const SiddonRay &s, int sx, int sy, int sz, Visit visit) {
    int ix = s.i[0], iy = s.i[1], iz = s.i[2];
    // next plane on each axis: the upper face of the current voxel when moving up, the lower face when moving down
    // (numbered relative to p0, see siddon_setup)
    float px = (float)(ix + (s.dir[0] > 0) - s.p0[0]), py = (float)(iy + (s.dir[1] > 0) - s.p0[1]), pz = (float)(iz + (s.dir[2] > 0) - s.p0[2]);
    const float dxf = (float)s.dir[0], dyf = (float)s.dir[1], dzf = (float)s.dir[2];
    float tx = fmaf(px, s.ib[0], s.k[0]), ty = fmaf(py, s.ib[1], s.k[1]), tz = fmaf(pz, s.ib[2], s.k[2]);
    int lin = ix * sx + iy * sy + iz * sz;                                                   // n_vox < 2^31 (checked at the entry points)
    const int dsx = s.dir[0] * sx, dsy = s.dir[1] * sy, dsz = s.dir[2] * sz;
    float tau = s.tau;
    const int max_steps = s.n[0] + s.n[1] + s.n[2] + 3;                                      // a ray crosses at most that many planes
    for (int step = 0; step < max_steps; ++step) {
        const float tmin = fminf(tx, fminf(ty, tz));
        const float tnext = fminf(tmin, s.tau_end);
        visit(lin, fmaxf(tnext - tau, 0.f));
        if (!(tmin < s.tau_end)) break;                                                      // left the box (or reached the pixel)
        tau = tnext;
        if (tx <= tmin) { ix += s.dir[0]; lin += dsx; px += dxf; tx = fmaf(px, s.ib[0], s.k[0]); }
        if (ty <= tmin) { iy += s.dir[1]; lin += dsy; py += dyf; ty = fmaf(py, s.ib[1], s.k[1]); }
        if (tz <= tmin) { iz += s.dir[2]; lin += dsz; pz += dzf; tz = fmaf(pz, s.ib[2], s.k[2]); }
        if ((unsigned)ix >= (unsigned)s.n[0] || (unsigned)iy >= (unsigned)s.n[1] || (unsigned)iz >= (unsigned)s.n[2]) break;
    }
}

// pixel of this thread: 32(u) x 8(v) tiles, lanes along u
__device__ __forceinline__ bool siddon_pixel(const DevGeom &g, int &iu, int &iv, int &view) {
    iu = blockIdx.x * 32 + threadIdx.x; iv = blockIdx.y * 8 + threadIdx.y; view = blockIdx.z;
    return iu < g.nu && iv < g.nv;
}

__global__ void __launch_bounds__(256) siddon_forward_kernel(DevGeom g, const float *__restrict__ vol, const float *__restrict__ volT,
                                                             float *__restrict__ proj) {
    int iu, iv, view;
    if (!siddon_pixel(g, iu, iv, view)) return;
    const SiddonRay s = siddon_setup(g, view, iv, iu);
    float acc = 0.f;
    if (s.hit) {
        const double2 cs = g.view_cs[view];
        const bool yfast = fabs(cs.x) > fabs(cs.y);                                          // rays run along x: read vol[z][x][y]
        const float *src = yfast ? volT : vol;
        const int sx = yfast ? g.ny : 1, sy = yfast ? 1 : g.nx, sz = g.nx * g.ny;
        siddon_walk(s, sx, sy, sz, [&](int lin, float len) { acc = fmaf(len, __ldg(src + lin), acc); });
    }
    proj[((size_t)view * g.nv + iv) * g.nu + iu] = acc;
}

__global__ void __launch_bounds__(256) siddon_scatter_kernel(DevGeom g, const float *__restrict__ proj, int *__restrict__ acc_x,
                                                             int *__restrict__ acc_y, const unsigned *__restrict__ absmax_bits,
                                                             float two_qb, int view0) {
    int iu, iv, view;
    if (!siddon_pixel(g, iu, iv, view)) return;
    view += view0;
    const SiddonRay s = siddon_setup(g, view, iv, iu);
    if (!s.hit) return;
    const float amax = __uint_as_float(__ldg(absmax_bits));
    const float gs = amax > 0.f ? __ldg(proj + ((size_t)view * g.nv + iv) * g.nu + iu) * (two_qb / amax) : 0.f;
    if (gs == 0.f) return;
    const double2 cs = g.view_cs[view];
    const bool yfast = fabs(cs.x) > fabs(cs.y);
    int *dst = yfast ? acc_y : acc_x;
    const int sx = yfast ? g.ny : 1, sy = yfast ? 1 : g.nx, sz = g.nx * g.ny;
    siddon_walk(s, sx, sy, sz, [&](int lin, float len) {
        const int q = __float2int_rn(gs * len);
        if (q) atomicAdd(dst + lin, q);                                                      // result unused: RED.ADD.S32
    });
}

// Bound on the path length (mm) one voxel can collect from ONE view: (number of pixel centres its shadow can cover) x (its
// diagonal, the longest chord).  With D = depth of a point along the central ray, tau = its lateral coordinate, a point
// projects to u = SDD tau / D, v = SDD z / D.  Over one voxel tau and D each vary by at most s = sqrt(dx^2 + dy^2), z by dz,
// so the shadow is at most  Lu = s (SDD/Dmin + umax/Dmin)  by  Lv = dz SDD/Dmin + s vmax/Dmin  (umax, vmax: the largest |u|,
// |v| on the detector; Dmin = SAD - R), and an interval of length L holds at most L/pitch + 1 pixel centres.
static double siddon_weight_bound(const cbct_geometry_desc &d, double R) {
    const double dmin = d.sad - R, s = std::sqrt(d.dx * d.dx + d.dy * d.dy);
    const double umax = 0.5 * d.nu * d.du + std::fabs(d.u0), vmax = 0.5 * d.nv * d.dv + std::fabs(d.v0);
    const double lu = s * (d.sdd + umax) / dmin, lv = (d.dz * d.sdd + s * vmax) / dmin;
    return (lu / d.du + 1.0) * (lv / d.dv + 1.0) * std::sqrt(s * s + d.dz * d.dz);
}

// 2^qb units per max|g| mm; views_per_group * w * 2^qb < 2^31.  Prefer all views in one group at qb >= 18, else groups of
// views at qb = 18 (the finalize pass accumulates in fp32 between groups), else the largest qb that fits one view.
// Host arithmetic only (exported as cbct_siddon_fixed_point_plan).
bool siddon_fixed_point_plan(const cbct_geometry_desc &d, double R, int *qb_out, int *group_out, double *w_out) {
    const double w = siddon_weight_bound(d, R);
    const auto cap = [&](int bits) { return std::ldexp(1.0, 31 - bits) / w; };
    int qb = 22;
    while (qb > 18 && cap(qb) < (double)d.n_views) --qb;
    while (qb > 8 && cap(qb) < 1.0) --qb;
    if (cap(qb) < 1.0) return false;
    *qb_out = qb;
    *group_out = (int)std::fmin((double)d.n_views, std::floor(cap(qb)));
    *w_out = w;
    return true;
}

static int siddon_workspace(cbct_geometry *G) {
    if (!G->d_sd_volT) {
        CBCT_CUDA_TRY(cudaMalloc(&G->d_sd_volT, sizeof(float) * G->n_vox));
        G->workspace_bytes += sizeof(float) * G->n_vox;
    }
    if (!G->d_sd_acc) {
        int qb = 0, group = 0;
        double w = 0;
        if (!siddon_fixed_point_plan(G->desc, G->R, &qb, &group, &w)) return CBCT_E_UNSUPPORTED;
        G->sd_qb = qb; G->sd_group = group;
        CBCT_CUDA_TRY(cudaMalloc(&G->d_sd_acc, sizeof(int) * 2 * G->n_vox));
        CBCT_CUDA_TRY(cudaMalloc(&G->d_sd_absmax, sizeof(unsigned)));
        G->workspace_bytes += sizeof(int) * 2 * G->n_vox + sizeof(unsigned);
    }
    return CBCT_OK;
}

void free_siddon(cbct_geometry *G) {
    cudaFree(G->d_sd_volT); cudaFree(G->d_sd_acc); cudaFree(G->d_sd_absmax);
    G->d_sd_volT = nullptr; G->d_sd_acc = nullptr; G->d_sd_absmax = nullptr;
}

}  // namespace cbct

using namespace cbct;

// allocates the pair's workspace (the only Siddon entry point that does); idempotent
extern "C" int cbct_siddon_prepare(cbct_geometry *G) {
    if (!G) return CBCT_E_INVALID;
    if (G->n_vox > 0x7fffffffLL) return CBCT_E_UNSUPPORTED;           // 32-bit voxel indices in the traversal
    CBCT_TRY(device_supported());
    return siddon_workspace(G);
}

extern "C" int cbct_siddon_forward(const cbct_geometry *G, const float *d_vol, float *d_proj, void *stream) {
    if (!G || !d_vol || !d_proj || !G->d_sd_volT) return CBCT_E_INVALID;   // cbct_siddon_prepare first
    const DevGeom &g = G->dg;
    cudaStream_t st = as_stream(stream);
    {
        dim3 block(32, 8), grid(cdiv(g.nx, 32), cdiv(g.ny, 32), g.nz);
        transpose_vol_kernel<<<grid, block, 0, st>>>(d_vol, G->d_sd_volT, g.nx, g.ny);
        CBCT_LAUNCH_CHECK();
    }
    dim3 block(32, 8), grid(cdiv(g.nu, 32), cdiv(g.nv, 8), g.n_views);
    siddon_forward_kernel<<<grid, block, 0, st>>>(g, d_vol, G->d_sd_volT, d_proj);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int cbct_siddon_backproject(const cbct_geometry *G, const float *d_proj, float *d_vol, void *stream) {
    if (!G || !d_vol || !d_proj || !G->d_sd_acc) return CBCT_E_INVALID;     // cbct_siddon_prepare first
    const DevGeom &g = G->dg;
    cudaStream_t st = as_stream(stream);
    CBCT_CUDA_TRY(cudaMemsetAsync(G->d_sd_absmax, 0, sizeof(unsigned), st));
    absmax_kernel<<<592, 256, 0, st>>>(d_proj, (long long)G->n_rays, G->d_sd_absmax);
    CBCT_LAUNCH_CHECK();
    const float two_qb = (float)std::ldexp(1.0, G->sd_qb);
    for (int v0 = 0; v0 < g.n_views; v0 += G->sd_group) {
        const int nv_ = std::min(G->sd_group, g.n_views - v0);
        CBCT_CUDA_TRY(cudaMemsetAsync(G->d_sd_acc, 0, sizeof(int) * 2 * G->n_vox, st));
        dim3 block(32, 8), grid(cdiv(g.nu, 32), cdiv(g.nv, 8), nv_);
        siddon_scatter_kernel<<<grid, block, 0, st>>>(g, d_proj, G->d_sd_acc, G->d_sd_acc + G->n_vox, G->d_sd_absmax, two_qb, v0);
        CBCT_LAUNCH_CHECK();
        // vol (+)= (acc_x + acc_y^T) * max|g| / 2^qb : the finalize pass of backproject_tma.cu with no margins and unit step
        dim3 fb(32, 8), fg(cdiv(g.nx, 32), cdiv(g.ny, 32), g.nz);
        backproject_finalize_kernel<<<fg, fb, 0, st>>>(G->d_sd_acc, G->d_sd_acc + G->n_vox, d_vol, g.nx, g.ny, 0, 0, 0, G->d_sd_absmax,
                                                       (float)std::ldexp(1.0, -G->sd_qb), v0 > 0 ? 1 : 0, 1LL << 31, G->err, NormOut{nullptr, nullptr, nullptr});   // rigorous bound: no head-room check
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}
