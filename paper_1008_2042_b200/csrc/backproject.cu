// backproject.cu -- f = P^T g, the exact transpose of forward.cu (include/cbct.h: cbct_backproject).
// Voxel-driven ("each GPU thread for a voxel"), but instead of the paper's approximate
// Eq. 3 every voxel gathers exactly the forward projector's samples that touch it:
//   f_j = step * sum_rays g_ray * sum_k hat(X_k - jx) hat(Y_k - jy) hat(Z_k - jz)
// (SURVEY.md §8(c) c.3).  No atomics: each output voxel is owned by one thread, so the result is
// deterministic.
#include "common.cuh"

namespace cbct {

__device__ __forceinline__ float hatf(float d) { return fmaxf(1.f - fabsf(d), 0.f); }

// ------------------------------------------------------------------------------------------------
// General path: one thread per voxel, candidate pixels from the projected support cube, k-range
// from a slab clip of each candidate ray against the support cube [j-1, j+1]^3.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) backproject_gather_kernel(DevGeom g, const float *__restrict__ proj,
                                                                 float *__restrict__ vol) {
    const int jx = blockIdx.x * blockDim.x + threadIdx.x;
    const int jy = blockIdx.y * blockDim.y + threadIdx.y;
    const int jz = blockIdx.z;
    if (jx >= g.nx || jy >= g.ny) return;
    // world coordinates of the support-cube corners: x = (X - cx)/inv_dx
    const double dx = 1.0 / g.inv_dx, dy = 1.0 / g.inv_dy, dz = 1.0 / g.inv_dz;
    const double inv_du = 1.0 / g.du, inv_dv = 1.0 / g.dv;
    const float stepf = (float)g.step;
    float total = 0.f;
    for (int view = 0; view < g.n_views; ++view) {
        const double2 cs = g.view_cs[view];
        double umin = 1e300, umax = -1e300, vmin = 1e300, vmax = -1e300;
#pragma unroll
        for (int corner = 0; corner < 8; ++corner) {
            const double x = ((jx + ((corner & 1) ? 1 : -1)) - g.cx) * dx;
            const double y = ((jy + ((corner & 2) ? 1 : -1)) - g.cy) * dy;
            const double z = ((jz + ((corner & 4) ? 1 : -1)) - g.cz) * dz;
            const double D = g.sad - (x * cs.x + y * cs.y), tau = -x * cs.y + y * cs.x;
            const double s = g.sdd / D;
            const double pu = (tau * s - g.u_first) * inv_du, pv = (z * s - g.v_first) * inv_dv;
            umin = fmin(umin, pu); umax = fmax(umax, pu);
            vmin = fmin(vmin, pv); vmax = fmax(vmax, pv);
        }
        const int iu0 = max(0, (int)ceil(umin) - 1), iu1 = min(g.nu - 1, (int)floor(umax) + 1);
        const int iv0 = max(0, (int)ceil(vmin) - 1), iv1 = min(g.nv - 1, (int)floor(vmax) + 1);
        float view_sum = 0.f;
        for (int iv = iv0; iv <= iv1; ++iv)
            for (int iu = iu0; iu <= iu1; ++iu) {
                RayF r;
                double b[3], c[3];
                ray_setup(g, view, iv, iu, r, b[0], b[1], b[2], c[0], c[1], c[2]);
                const double ctr[3] = {(double)jx, (double)jy, (double)jz};
                double tin = -1e300, tout = 1e300;
                bool miss = false;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    if (b[a] == 0.0) { miss |= (c[a] < ctr[a] - 1.0 || c[a] > ctr[a] + 1.0); continue; }
                    const double inv = 1.0 / b[a];
                    double t1 = (ctr[a] - 1.0 - c[a]) * inv, t2 = (ctr[a] + 1.0 - c[a]) * inv;
                    if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
                    tin = fmax(tin, t1); tout = fmin(tout, t2);
                }
                if (miss || tin > tout) continue;
                long long klo = (long long)ceil((tin - g.tau0) / g.step) - 1;     // widened: the hat clamps to 0
                long long khi = (long long)floor((tout - g.tau0) / g.step) + 1;
                if (klo < 0) klo = 0;
                if (khi > g.K - 1) khi = g.K - 1;
                if (khi < klo) continue;
                const float gv = __ldg(proj + ((size_t)view * g.nv + iv) * g.nu + iu);
                const float tau_base = (float)(g.tau0 + (double)klo * g.step);
                float ray_sum = 0.f;
                for (int j = 0; j <= (int)(khi - klo); ++j) {
                    const float tau = fmaf((float)j, stepf, tau_base);
                    const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
                    ray_sum += hatf(X - (float)jx) * hatf(Y - (float)jy) * hatf(Z - (float)jz);
                }
                view_sum = fmaf(ray_sum, gv, view_sum);
            }
        total += view_sum;                                  // per-view partial sums (SURVEY.md §8(c) guidance)
    }
    vol[((size_t)jz * g.ny + jy) * g.nx + jx] = total * stepf;
}

int launch_backproject(const cbct_geometry *G, const float *d_proj, float *d_vol, cudaStream_t st) {
    const DevGeom &g = G->dg;
    ProfScope prof(PROF_BACK, st);
    dim3 block(32, 4), grid(cdiv(g.nx, 32), cdiv(g.ny, 4), g.nz);
    backproject_gather_kernel<<<grid, block, 0, st>>>(g, d_proj, d_vol);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

}  // namespace cbct
