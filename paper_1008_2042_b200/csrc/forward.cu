// forward.cu -- g = P f (include/cbct.h: cbct_forward).
// PAPER.md:73 Eq. 1 as step * sum_k T[f](x_S + n t_k) on the global source-anchored grid
// (SURVEY.md §8(c) c.2).  One thread per detector ray ("each GPU thread computing the
// line integral ... along an x-ray line"), fixed step, software fp32 trilinear interpolation.
#include <cmath>
#include <cstdlib>

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

// ------------------------------------------------------------------------------------------------
// Tiled path (the one that normally runs).  A CTA owns a 32(u) x 8(v) tile of detector pixels of one
// view and marches the global t-grid in chunks of <= FW_KC samples.  For each chunk the axis-aligned
// box of voxels that the tile's frustum segment can touch is staged in shared memory (zero-filled
// outside the volume = the zero padding of T), so every one of the 8 neighbour reads of a sample is
// an LDS: the row pitch is odd, lanes are neighbouring pixels, so for any view direction the 32 lanes
// fall in distinct banks or on the same word.  Positions are kept relative to the box origin.
// ------------------------------------------------------------------------------------------------
constexpr int FW_TU = 32, FW_TV = 8, FW_KC = 32, FW_CAP = 7168;

struct BoxI { int lx, ly, lz, ex, ey, ez; };

// box of the voxels touched by the tile between tau_a and tau_b: AABB of the 4 corner rays at both
// ends, grown by `margin` (sphere-patch bulge + rounding slack), +1 for the upper neighbour, clipped to
// [-2, n+1] (a thread only evaluates samples inside the padded box [-1, n]).
__device__ __forceinline__ BoxI chunk_box(const RayF *corner, float tau_a, float tau_b, float margin, int nx, int ny,
                                          int nz) {
    float mnx = 1e30f, mny = 1e30f, mnz = 1e30f, mxx = -1e30f, mxy = -1e30f, mxz = -1e30f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const RayF r = corner[c];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const float tau = e ? tau_b : tau_a;
            const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
            mnx = fminf(mnx, X); mxx = fmaxf(mxx, X);
            mny = fminf(mny, Y); mxy = fmaxf(mxy, Y);
            mnz = fminf(mnz, Z); mxz = fmaxf(mxz, Z);
        }
    }
    BoxI b;
    b.lx = max((int)floorf(mnx - margin), -2); b.ly = max((int)floorf(mny - margin), -2); b.lz = max((int)floorf(mnz - margin), -2);
    const int hx = min((int)floorf(mxx + margin) + 1, nx + 1), hy = min((int)floorf(mxy + margin) + 1, ny + 1),
              hz = min((int)floorf(mxz + margin) + 1, nz + 1);
    b.ex = hx - b.lx + 1; b.ey = hy - b.ly + 1; b.ez = hz - b.lz + 1;
    return b;
}

__global__ void __launch_bounds__(256) forward_tiled_kernel(DevGeom g, const float *__restrict__ vol,
                                                            float *__restrict__ proj, float margin) {
    __shared__ float box[FW_CAP];
    __shared__ RayF corner[4];
    __shared__ int s_klo, s_khi;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * FW_TU + tx;
    const int iu = blockIdx.x * FW_TU + tx, iv = blockIdx.y * FW_TV + ty, view = blockIdx.z;
    const bool valid = iu < g.nu && iv < g.nv;
    RayF r;
    double b[3], c[3], tin, tout;
    ray_setup(g, view, iv, iu, r, b[0], b[1], b[2], c[0], c[1], c[2]);   // also for pixels past the edge: tile corners
    int klo = 0x7fffffff, khi = -1;
    if (valid && clip_box(g, b, c, tin, tout)) {
        const long long a = (long long)ceil((tin - g.tau0) / g.step), e = (long long)floor((tout - g.tau0) / g.step);
        klo = (int)max(a, 0LL); khi = (int)min(e, (long long)g.K - 1);
        if (khi < klo) { klo = 0x7fffffff; khi = -1; }
    }
    if (tid == 0) { s_klo = 0x7fffffff; s_khi = -1; }
    if ((tx == 0 || tx == FW_TU - 1) && (ty == 0 || ty == FW_TV - 1)) corner[(ty ? 2 : 0) + (tx ? 1 : 0)] = r;
    __syncthreads();
    {
        const int wlo = __reduce_min_sync(0xffffffffu, klo), whi = __reduce_max_sync(0xffffffffu, khi);
        if (tx == 0) { atomicMin(&s_klo, wlo); atomicMax(&s_khi, whi); }
    }
    __syncthreads();
    const int K0 = s_klo, K1 = s_khi;
    const float stepf = (float)g.step;
    float total = 0.f;
    for (int k0 = K0; k0 <= K1;) {
        int kc = min(FW_KC, K1 - k0 + 1);
        BoxI bx;
        float tau_base;
        for (;;) {                                           // shrink the chunk until its box fits
            tau_base = (float)(g.tau0 + (double)k0 * g.step);
            bx = chunk_box(corner, tau_base, fmaf((float)(kc - 1), stepf, tau_base), margin, g.nx, g.ny, g.nz);
            if (((bx.ex | 1) * bx.ey * bx.ez <= FW_CAP) || kc == 1) break;
            kc >>= 1;
        }
        const int px = bx.ex | 1, pz = px * bx.ey;
        const bool staged = px * bx.ey * bx.ez <= FW_CAP;          // false only for tiles the host heuristic misjudged
        if (!staged) kc = min(FW_KC, K1 - k0 + 1);
        if (staged) {
            // stage the box: warp w takes rows (y,z) = w, w+8, ...; lanes run along x (coalesced in global)
            const int rows = bx.ey * bx.ez;
            for (int row = ty; row < rows; row += FW_TV) {
                const int rz = row / bx.ey, ry = row - rz * bx.ey;
                const int gy = bx.ly + ry, gz = bx.lz + rz;
                const bool rin = (unsigned)gy < (unsigned)g.ny && (unsigned)gz < (unsigned)g.nz;
                const float *src = vol + ((size_t)(rin ? gz : 0) * g.ny + (rin ? gy : 0)) * g.nx;
                float *dst = box + rz * pz + ry * px;
                for (int a = tx; a < bx.ex; a += FW_TU) {
                    const int gx = bx.lx + a;
                    dst[a] = (rin && (unsigned)gx < (unsigned)g.nx) ? __ldg(src + gx) : 0.f;
                }
            }
        }
        __syncthreads();
        const int ja = max(k0, klo), jb = min(k0 + kc - 1, khi);
        if (ja <= jb && staged) {
            const float cxl = r.cx - (float)bx.lx, cyl = r.cy - (float)bx.ly, czl = r.cz - (float)bx.lz;
            float part = 0.f;
#pragma unroll 4
            for (int j = ja; j <= jb; ++j) {
                const float tau = fmaf((float)(j - k0), stepf, tau_base);
                const float X = fmaf(r.bx, tau, cxl), Y = fmaf(r.by, tau, cyl), Z = fmaf(r.bz, tau, czl);
                const float fxf = floorf(X), fyf = floorf(Y), fzf = floorf(Z);
                const float wx = X - fxf, wy = Y - fyf, wz = Z - fzf;
                const float *p0 = box + ((int)fzf * pz + (int)fyf * px + (int)fxf);
                const float *p1 = p0 + pz;
                const float v000 = p0[0], v100 = p0[1], v010 = p0[px], v110 = p0[px + 1];
                const float v001 = p1[0], v101 = p1[1], v011 = p1[px], v111 = p1[px + 1];
                const float a00 = fmaf(wx, v100 - v000, v000), a10 = fmaf(wx, v110 - v010, v010);
                const float a01 = fmaf(wx, v101 - v001, v001), a11 = fmaf(wx, v111 - v011, v011);
                const float b0 = fmaf(wy, a10 - a00, a00), b1 = fmaf(wy, a11 - a01, a01);
                part += fmaf(wz, b1 - b0, b0);
            }
            total += part;
        } else if (ja <= jb) {
            float part = 0.f;
            for (int j = ja; j <= jb; ++j) {
                const float tau = fmaf((float)(j - k0), stepf, tau_base);
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
        __syncthreads();
        k0 += kc;
    }
    if (valid) proj[((size_t)view * g.nv + iv) * g.nu + iu] = total * stepf;
}

// can every single-sample slice of a 32x8 tile fit the shared-memory box?  (conservative, host side)
bool forward_tiled_fits(const cbct_geometry *G, float *margin_out) {
    const cbct_geometry_desc &d = G->desc;
    const double far = (d.sad + G->R) / d.sdd;                       // magnification bound inside the volume
    const double half_diag = 0.5 * std::sqrt((FW_TU * d.du) * (FW_TU * d.du) + (FW_TV * d.dv) * (FW_TV * d.dv));
    const double psi = half_diag / d.sdd;
    const double vmin = std::fmin(d.dx, std::fmin(d.dy, d.dz));
    const double bulge = (d.sad + G->R) * 0.5 * psi * psi / vmin;    // sagitta of the sphere patch, in voxels
    const double margin = bulge + 0.02;
    *margin_out = (float)margin;
    // heuristic only (the kernel re-checks every chunk and falls back to global reads for a chunk whose
    // box does not fit): one sample slice of the tile at the far end, seen at 45 degrees
    const double lat = FW_TU * d.du * far, ver = FW_TV * d.dv * far;
    const double exy = 0.71 * (lat + ver) / std::fmin(d.dx, d.dy) + 2 * margin + 4, ez = ver / d.dz + 2 * margin + 4;
    return exy * exy * ez <= 1.5 * FW_CAP && margin < 4.0;
}

int launch_forward(const cbct_geometry *G, const float *d_vol, float *d_proj, cudaStream_t st, double *d_norm, bool *fused) {
    const DevGeom &g = G->dg;
    ProfScope prof(PROF_FORWARD, st);
    dim3 block(FW_TU, FW_TV), grid(cdiv(g.nu, FW_TU), cdiv(g.nv, FW_TV), g.n_views);
    CBCT_TRY(device_error_pending(G));
    // the implementation was fixed at cbct_geometry_create (G->fw_impl): a failure here is returned, never re-routed
    if (fused) *fused = d_norm && G->fw_impl == FW_TMA;
    if (G->fw_impl == FW_TMA) return launch_forward_tma(G, d_vol, d_proj, st, d_norm);
    float margin = 0.f;
    if (G->fw_impl == FW_TILED) {
        if (!forward_tiled_fits(G, &margin)) return CBCT_E_UNSUPPORTED;
        forward_tiled_kernel<<<grid, block, 0, st>>>(g, d_vol, d_proj, margin);
    } else {
        forward_global_kernel<<<grid, block, 0, st>>>(g, d_vol, d_proj);
    }
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

}  // namespace cbct
