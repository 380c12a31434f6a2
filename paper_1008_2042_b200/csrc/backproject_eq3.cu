// backproject_eq3.cu -- the paper's OWN backprojector, Eq. 3 (cbct_backproject_eq3 in include/cbct.h):
//   f(x) = (dx dy dz)/(du dv) * sum_theta  L^3(u*) / (L0 l^2(x)) * g^theta(u*)
// u* = where the line source -> voxel centre x meets the imager, g(u*) by bilinear interpolation of the four
// neighbouring pixels, zero outside the imager, L0 = SDD, l(x) = |x - x_S|, L(u*) = |u* - x_S|.
// It is NOT the transpose of cbct_forward: PAPER.md:506 states the adjoint condition holds "with numerical error
// less than 1%".  SURVEY.md §8(f) NEXT-1: shipped so that matched (cbct_backproject) and unmatched (this) pairs can
// be compared; CGLS in this library always uses the exact transpose.
// One thread per voxel as in the paper, lanes along x so that a warp's 32 voxels project onto
// neighbouring pixels of one detector row pair; the per-view geometry is evaluated in fp64 (40 views x 20 flops per
// voxel: 0.4 ms of fp64 at cfg 4), the interpolation and the sum in fp32.
#include "common.cuh"

namespace cbct {

__global__ void __launch_bounds__(256) backproject_eq3_kernel(DevGeom g, const float *__restrict__ proj, float *__restrict__ vol,
                                                              double ox, double oy, double oz, double inv_du, double inv_dv,
                                                              float pref) {
    const int jx = blockIdx.x * blockDim.x + threadIdx.x, jy = blockIdx.y * blockDim.y + threadIdx.y, jz = blockIdx.z;
    if (jx >= g.nx || jy >= g.ny) return;
    // voxel centre in mm: x = ox + (jx - (nx-1)/2) dx
    const double x = ox + (jx - 0.5 * (g.nx - 1)) / g.inv_dx, y = oy + (jy - 0.5 * (g.ny - 1)) / g.inv_dy;
    const double z = oz + (jz - 0.5 * (g.nz - 1)) / g.inv_dz;
    float acc = 0.f;
    for (int view = 0; view < g.n_views; ++view) {
        const double2 cs = g.view_cs[view];
        const double D = g.sad - (x * cs.x + y * cs.y), tau = -x * cs.y + y * cs.x;
        const double m = g.sdd / D, us = m * tau, vs = m * z;
        const double L2 = g.sdd * g.sdd + us * us + vs * vs, l2 = D * D + tau * tau + z * z;
        const double pu = (us - g.u_first) * inv_du, pv = (vs - g.v_first) * inv_dv;      // pixel index coordinates
        const double fu = floor(pu), fv = floor(pv);
        if (!(fu >= -1.0 && fv >= -1.0 && fu < (double)g.nu && fv < (double)g.nv)) continue;   // all four taps outside
        const int iu = (int)fu, iv = (int)fv;
        const float wu = (float)(pu - fu), wv = (float)(pv - fv);
        const float *base = proj + ((size_t)view * g.nv) * g.nu;
        const bool u0ok = iu >= 0, u1ok = iu + 1 < g.nu, v0ok = iv >= 0, v1ok = iv + 1 < g.nv;
        const float g00 = (u0ok && v0ok) ? __ldg(base + (size_t)iv * g.nu + iu) : 0.f;
        const float g10 = (u1ok && v0ok) ? __ldg(base + (size_t)iv * g.nu + iu + 1) : 0.f;
        const float g01 = (u0ok && v1ok) ? __ldg(base + (size_t)(iv + 1) * g.nu + iu) : 0.f;
        const float g11 = (u1ok && v1ok) ? __ldg(base + (size_t)(iv + 1) * g.nu + iu + 1) : 0.f;
        const float r0 = fmaf(wu, g10 - g00, g00), r1 = fmaf(wu, g11 - g01, g01);
        const float val = fmaf(wv, r1 - r0, r0);
        const float weight = (float)(L2 * sqrt(L2) / (g.sdd * l2));                           // L^3 / (L0 l^2)
        acc = fmaf(weight, val, acc);
    }
    vol[((size_t)jz * g.ny + jy) * g.nx + jx] = pref * acc;
}

}  // namespace cbct

using namespace cbct;

extern "C" int cbct_backproject_eq3(const cbct_geometry *G, const float *d_proj, float *d_vol, void *stream) {
    if (!G || !d_proj || !d_vol) return CBCT_E_INVALID;
    const DevGeom &g = G->dg;
    const cbct_geometry_desc &d = G->desc;
    dim3 block(32, 8), grid(cdiv(g.nx, 32), cdiv(g.ny, 8), g.nz);
    backproject_eq3_kernel<<<grid, block, 0, as_stream(stream)>>>(g, d_proj, d_vol, d.ox, d.oy, d.oz, 1.0 / d.du, 1.0 / d.dv,
                                                                  (float)(d.dx * d.dy * d.dz / (d.du * d.dv)));
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
