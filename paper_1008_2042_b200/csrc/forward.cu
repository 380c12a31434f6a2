// forward.cu -- g = P f (include/cbct.h: cbct_forward).
// PAPER.md:73 Eq. 1 as step * sum_k T[f](x_S + n t_k) on the global source-anchored grid
// (SURVEY.md §8(c) c.2).  One thread per detector ray ("each GPU thread computing the
// line integral ... along an x-ray line"), fixed step, software fp32 trilinear interpolation.
#include "common.cuh"

namespace cbct {

// ------------------------------------------------------------------------------------------------
// General path: volume read straight from global/L2 with bounds checks.  Used for shapes the tiled
// kernel does not take, and as the in-library cross-check of the tiled kernel (CBCT_FORWARD_IMPL=global).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float fetch0(const float *__restrict__ vol, const DevGeom &g, int ix, int iy, int iz) {
    if ((unsigned)ix >= (unsigned)g.nx || (unsigned)iy >= (unsigned)g.ny || (unsigned)iz >= (unsigned)g.nz) return 0.f;
    return __ldg(vol + ((size_t)iz * g.ny + iy) * g.nx + ix);
}

// tau-range of a ray inside the zero-padded box [-1, n]^3 (index space); false if it misses
__device__ __forceinline__ bool clip_box(const DevGeom &g, const double b[3], const double c[3], double &tin,
                                         double &tout) {
    const double hi[3] = {(double)g.nx, (double)g.ny, (double)g.nz};
    tin = -1e300; tout = 1e300;
    bool miss = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (b[a] == 0.0) { miss |= (c[a] <= -1.0 || c[a] >= hi[a]); continue; }
        const double inv = 1.0 / b[a];
        double t1 = (-1.0 - c[a]) * inv, t2 = (hi[a] - c[a]) * inv;
        if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
        tin = fmax(tin, t1); tout = fmin(tout, t2);
    }
    return !miss && tout > tin;
}

__global__ void __launch_bounds__(256) forward_global_kernel(DevGeom g, const float *__restrict__ vol,
                                                             float *__restrict__ proj) {
    const int iu = blockIdx.x * 32 + threadIdx.x, iv = blockIdx.y * 8 + threadIdx.y, view = blockIdx.z;
    if (iu >= g.nu || iv >= g.nv) return;
    RayF r;
    double b[3], c[3], tin, tout;
    ray_setup(g, view, iv, iu, r, b[0], b[1], b[2], c[0], c[1], c[2]);
    float total = 0.f;
    if (clip_box(g, b, c, tin, tout)) {
        // samples k with tau_k inside [tin, tout], widened by one on each side (T = 0 outside the box)
        long long klo = (long long)ceil((tin - g.tau0) / g.step) - 1, khi = (long long)floor((tout - g.tau0) / g.step) + 1;
        if (klo < 0) klo = 0;
        if (khi > g.K - 1) khi = g.K - 1;
        const float stepf = (float)g.step;
        for (long long k0 = klo; k0 <= khi; k0 += 32) {            // chunked partial sums
            const float tau_base = (float)(g.tau0 + (double)k0 * g.step);
            const int n = (int)min(32LL, khi - k0 + 1);
            float part = 0.f;
            for (int j = 0; j < n; ++j) {
                const float tau = fmaf((float)j, stepf, tau_base);
                const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
                const float fxf = floorf(X), fyf = floorf(Y), fzf = floorf(Z);
                const int ix = (int)fxf, iy = (int)fyf, iz = (int)fzf;
                const float wx = X - fxf, wy = Y - fyf, wz = Z - fzf;
                const float v000 = fetch0(vol, g, ix, iy, iz), v100 = fetch0(vol, g, ix + 1, iy, iz);
                const float v010 = fetch0(vol, g, ix, iy + 1, iz), v110 = fetch0(vol, g, ix + 1, iy + 1, iz);
                const float v001 = fetch0(vol, g, ix, iy, iz + 1), v101 = fetch0(vol, g, ix + 1, iy, iz + 1);
                const float v011 = fetch0(vol, g, ix, iy + 1, iz + 1), v111 = fetch0(vol, g, ix + 1, iy + 1, iz + 1);
                const float a00 = fmaf(wx, v100 - v000, v000), a10 = fmaf(wx, v110 - v010, v010);
                const float a01 = fmaf(wx, v101 - v001, v001), a11 = fmaf(wx, v111 - v011, v011);
                const float b0 = fmaf(wy, a10 - a00, a00), b1 = fmaf(wy, a11 - a01, a01);
                part += fmaf(wz, b1 - b0, b0);
            }
            total += part;
        }
        total *= stepf;
    }
    proj[((size_t)view * g.nv + iv) * g.nu + iu] = total;
}

int launch_forward(const cbct_geometry *G, const float *d_vol, float *d_proj, cudaStream_t st) {
    const DevGeom &g = G->dg;
    ProfScope prof(PROF_FORWARD, st);
    dim3 block(32, 8), grid(cdiv(g.nu, 32), cdiv(g.nv, 8), g.n_views);
    forward_global_kernel<<<grid, block, 0, st>>>(g, d_vol, d_proj);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

}  // namespace cbct
