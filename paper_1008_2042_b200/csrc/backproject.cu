// backproject.cu -- f = P^T g, the exact transpose of forward.cu (include/cbct.h: cbct_backproject).
// Voxel-driven ("each GPU thread for a voxel"), but instead of the paper's approximate
// Eq. 3 every voxel gathers exactly the forward projector's samples that touch it:
//   f_j = step * sum_rays g_ray * sum_k hat(X_k - jx) hat(Y_k - jy) hat(Z_k - jz)
// (SURVEY.md §8(c) c.3).  No atomics: each output voxel is owned by one thread, so the result is
// deterministic.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

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

// ------------------------------------------------------------------------------------------------
// Cell-driven path (the one that normally runs).  Still output-stationary and atomic-free, but the unit
// of ownership is a CELL (the cube between 8 neighbouring voxel centres, padding cells included): a
// sample of the forward projector lies in exactly one cell and spreads to that cell's 8 corners with
// the trilinear weights, so one thread per cell evaluates each sample ONCE (the transposed lerp tree,
// 15 flops) instead of once per touched voxel (8 hat products).  A second kernel sums, for every
// voxel, the 8 corner accumulators of the 8 cells around it in a fixed order.
//   per (cell, view): candidate detector columns from the projected cell centre +- a bound,
//   per column: clip against the cell's x,y slabs in r = t/L (independent of the detector row),
//   per row: clip against the z slab, k-range of the global sample grid, then the samples.
// A sample belongs to the cell iff floor(X,Y,Z) == (ix,iy,iz), evaluated on the same fp32 X,Y,Z in
// every thread, so each sample is counted exactly once however the clipping rounds.
// Lane mapping: the 32 lanes of a warp are cells that are neighbours ALONG Z (same ix, iy): they share
// the column loop and the x,y clip exactly, and their row loops and sample counts have (nearly) equal
// trip counts, so the warp stays converged.  Projections and the per-pixel table are read through
// v-fastest (transposed) copies so that those lanes touch neighbouring addresses.
// ------------------------------------------------------------------------------------------------
constexpr float BP_EPS = 0.02f;
// The clipping arithmetic (r-slabs from the fp32 tables) and the membership test (fp32 sample positions) round
// differently; for a ray that grazes a cell face or corner a position error of 1e-5 voxel moves the crossing by
// many samples.  Clipping therefore uses the cell grown by BP_GROW voxels on every side and accepts an (almost)
// empty in-plane chord; membership is still decided by the positions alone.  (Found with the scatter kernel:
// without this, 1e-8 of the samples at cfg 4 were skipped.)
constexpr float BP_GROW = 1e-3f, BP_R_EPS = 1e-5f;

// gT[view][iu][iv] = g[view][iv][iu]
__global__ void __launch_bounds__(256) transpose_proj_kernel(const float *__restrict__ g, float *__restrict__ gT, int nu,
                                                             int nv) {
    __shared__ float tile[32][33];
    const size_t base = (size_t)blockIdx.z * nu * nv;
    const int u0 = blockIdx.x * 32, v0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int u = u0 + threadIdx.x, v = v0 + j;
        if (u < nu && v < nv) tile[j][threadIdx.x] = __ldg(g + base + (size_t)v * nu + u);
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int u = u0 + j, v = v0 + threadIdx.x;
        if (u < nu && v < nv) gT[base + (size_t)u * nv + v] = tile[threadIdx.x][j];
    }
}

template <int MAXT, int MINB, bool ZCLIP>
__global__ void __launch_bounds__(MAXT, MINB) backproject_cell_kernel(BpTables P, int nx, int ny, int nz, int nu, int nv,
                                                               int n_views, int K, int xb, const float *__restrict__ projT,
                                                               float *__restrict__ partial) {
    const int nzc = nz + 1;
    const int xr = (int)threadIdx.x / nzc, zc = (int)threadIdx.x - xr * nzc;
    const int ix = blockIdx.x * xb + xr - 1, iy = (int)blockIdx.y - 1, iz = zc - 1;
    if (xr >= xb || ix > nx - 1) return;
    const float fix = (float)ix, fiy = (float)iy, fiz = (float)iz;
    const float az = fiz - P.Kz - BP_GROW, bz = az + (1.f + 2.f * BP_GROW);
    float a000 = 0.f, a100 = 0.f, a010 = 0.f, a110 = 0.f, a001 = 0.f, a101 = 0.f, a011 = 0.f, a111 = 0.f;
    const float inv_step = P.inv_step, stepf = P.stepf, tau0f = P.tau0f;
    const float k_lo_off = -(P.t0 * P.inv_step) - P.k_eps, k_hi_off = -(P.t0 * P.inv_step) + P.k_eps;
    for (int view = 0; view < n_views; ++view) {
        const BpView V = P.views[view];
        // candidate columns: projected cell centre +- conservative half width
        const float D = fmaf(V.Dx, fix + 0.5f, fmaf(V.Dy, fiy + 0.5f, V.D0));
        const float tc = fmaf(V.Tx, fix + 0.5f, fmaf(V.Ty, fiy + 0.5f, V.T0));
        const float rD = __frcp_rn(D), rDn = __frcp_rn(D - V.hd);
        const float uc = P.sdd * tc * rD;
        const float dumax = P.sdd * rDn * fmaf(fabsf(tc) * rD, V.hd, V.hl);
        const int iu0 = max(0, (int)ceilf((uc - dumax - P.u_first) * P.inv_du - BP_EPS));
        const int iu1 = min(nu - 1, (int)floorf((uc + dumax - P.u_first) * P.inv_du + BP_EPS));
        const BpViewU *vu = P.viewu + view * nu;
        const float *pv = projT + (size_t)view * nv * nu;
        for (int iu = iu0; iu <= iu1; ++iu) {
            const float4 w0 = __ldg(reinterpret_cast<const float4 *>(vu + iu));        // Ax Ay Wx Wy
            const float rx0 = (fix - V.Kx - BP_GROW) * w0.z, rx1 = fmaf(1.f + 2.f * BP_GROW, w0.z, rx0);
            const float ry0 = (fiy - V.Ky - BP_GROW) * w0.w, ry1 = fmaf(1.f + 2.f * BP_GROW, w0.w, ry0);
            const float rin = fmaxf(fminf(rx0, rx1), fminf(ry0, ry1)), rout = fminf(fmaxf(rx0, rx1), fmaxf(ry0, ry1));
            if (!(rin < rout + BP_R_EPS) || !(rin > 0.f)) continue;
            const float2 w1 = __ldg(reinterpret_cast<const float2 *>(vu + iu) + 2);    // Gx Gy
            const float i_in = __frcp_rn(rin), i_out = __frcp_rn(rout);
            const float vzmin = fminf(az * i_in, az * i_out), vzmax = fmaxf(bz * i_in, bz * i_out);
            const int iv0 = max(0, (int)ceilf(fmaf(vzmin, P.dz_dv, -P.vfirst_dv) - BP_EPS));
            const int iv1 = min(nv - 1, (int)floorf(fmaf(vzmax, P.dz_dv, -P.vfirst_dv) + BP_EPS));
            // running pointers (v-fastest tables): one add per row instead of 64-bit index arithmetic
            const float4 *pp = P.pixT + (iu * nv + iv0);
            const float *gp = pv + (iu * nv + iv0);
            const float2 *rp = P.rows + iv0;
            if (iv0 > iv1) continue;
            // software pipeline: the three loads of row iv+1 are issued before row iv is processed
            float2 rw_n = __ldg(rp);
            float4 t_n = __ldg(pp);
            float g_n = __ldg(gp);
            for (int iv = iv0; iv <= iv1; ++iv) {
                const float2 rw = rw_n;                                                // vz, 1/vz
                const float4 t = t_n;                                                  // 1/L, q, L
                const float gval = g_n;
                const int adv = iv < iv1 ? 1 : 0;                                      // stay in range on the last row
                pp += adv; gp += adv; rp += adv;
                rw_n = __ldg(rp); t_n = __ldg(pp); g_n = __ldg(gp);
                // z clip of the k-range: only worth its instructions when rays are steep against flat cells
                float rlo = rin, rhi = rout;
                if constexpr (ZCLIP) {
                    const float rz0 = az * rw.y, rz1 = bz * rw.y;
                    rlo = fmaxf(rin, fminf(rz0, rz1)); rhi = fminf(rout, fmaxf(rz0, rz1));
                }
                const float sl = t.z * inv_step;
                const int ka = max(0, (int)ceilf(fmaf(rlo, sl, k_lo_off)));
                const int kb = min(K - 1, (int)floorf(fmaf(rhi, sl, k_hi_off)));
                if (ka > kb) continue;                                                 // also rejects rlo > rhi
                const float bx = w0.x * t.x, by = w0.y * t.x, bzz = rw.x * t.x;
                const float cx = fmaf(w1.x, t.x, fmaf(V.Fx, t.y, P.cx0));
                const float cy = fmaf(w1.y, t.x, fmaf(V.Fy, t.y, P.cy0));
                const float cz = fmaf(P.sad * rw.x, t.x, P.cz0);
                float kf = (float)ka;
                for (int k = ka; k <= kb; ++k, kf += 1.f) {
                    const float tau = fmaf(kf, stepf, tau0f);
                    // X,Y,Z depend on (view, iu, iv, k) only, so all cells agree on them; X - ix is exact
                    const float fx = fmaf(bx, tau, cx) - fix, fy = fmaf(by, tau, cy) - fiy, fz = fmaf(bzz, tau, cz) - fiz;
                    // 0 <= f < 1 on all three axes, as one unsigned compare each (negative floats have the sign bit set)
                    const bool in = __float_as_uint(fx) < 0x3f800000u && __float_as_uint(fy) < 0x3f800000u &&
                                    __float_as_uint(fz) < 0x3f800000u;
                    const float gg = in ? gval : 0.f;
                    const float g1 = gg * fz, g0 = gg - g1;
                    const float g01 = g0 * fy, g00 = g0 - g01, g11 = g1 * fy, g10 = g1 - g11;
                    const float ofx = 1.f - fx;
                    a000 = fmaf(g00, ofx, a000); a100 = fmaf(g00, fx, a100);
                    a010 = fmaf(g01, ofx, a010); a110 = fmaf(g01, fx, a110);
                    a001 = fmaf(g10, ofx, a001); a101 = fmaf(g10, fx, a101);
                    a011 = fmaf(g11, ofx, a011); a111 = fmaf(g11, fx, a111);
                }
            }
        }
    }
    // partial[corner][(iy+1)][(ix+1)][(iz+1)], z fastest: lanes write neighbouring words
    const size_t ncell = (size_t)(nx + 1) * (ny + 1) * nzc;
    const size_t ci = ((size_t)(iy + 1) * (nx + 1) + (ix + 1)) * nzc + zc;
    partial[ci] = a000; partial[ncell + ci] = a100; partial[2 * ncell + ci] = a010; partial[3 * ncell + ci] = a110;
    partial[4 * ncell + ci] = a001; partial[5 * ncell + ci] = a101; partial[6 * ncell + ci] = a011;
    partial[7 * ncell + ci] = a111;
}

// voxel (x,y,z) = step * sum over the 8 cells (x-dx, y-dy, z-dz) of their corner (dx,dy,dz) accumulator.
// The partials are z-fastest, the volume x-fastest: a CTA takes 32 x-neighbouring columns of one y, its
// warps read whole z-runs (coalesced), sum the 8 contributions in a fixed order in registers, and the
// tile is transposed through shared memory so that the volume is written with coalesced rows.
__global__ void __launch_bounds__(256) backproject_combine_kernel(const float *__restrict__ partial, float *__restrict__ vol,
                                                                  int nx, int ny, int nz, float stepf) {
    extern __shared__ float tile[];                     // [32][pitch], pitch odd
    const int pitch = nz | 1;
    const int x0 = blockIdx.x * 32, y = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nzc = nz + 1;
    const size_t ncell = (size_t)(nx + 1) * (ny + 1) * nzc;
    for (int j = warp; j < 32; j += 8) {
        const int x = x0 + j;
        if (x >= nx) break;
        for (int z = lane; z < nz; z += 32) {
            float acc = 0.f;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int dx = c & 1, dy = (c >> 1) & 1, dz = c >> 2;
                acc += __ldg(partial + (size_t)c * ncell + ((size_t)(y - dy + 1) * (nx + 1) + (x - dx + 1)) * nzc + (z - dz + 1));
            }
            tile[j * pitch + z] = acc * stepf;
        }
    }
    __syncthreads();
    const int x = x0 + lane;
    if (x < nx)
        for (int z = warp; z < nz; z += 8) vol[((size_t)z * ny + y) * nx + x] = tile[lane * pitch + z];
}

// fall-back for volumes too tall for the shared-memory tile: one thread per (x,y) column walking z
__global__ void __launch_bounds__(128) backproject_combine_simple_kernel(const float *__restrict__ partial,
                                                                         float *__restrict__ vol, int nx, int ny, int nz,
                                                                         float stepf) {
    const int x = blockIdx.x * 32 + threadIdx.x, y = blockIdx.y * 4 + threadIdx.y;
    if (x >= nx || y >= ny) return;
    const int nzc = nz + 1;
    const size_t ncell = (size_t)(nx + 1) * (ny + 1) * nzc;
    for (int z = 0; z < nz; ++z) {
        float acc = 0.f;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int dx = c & 1, dy = (c >> 1) & 1, dz = c >> 2;
            acc += __ldg(partial + (size_t)c * ncell + ((size_t)(y - dy + 1) * (nx + 1) + (x - dx + 1)) * nzc + (z - dz + 1));
        }
        vol[((size_t)z * ny + y) * nx + x] = acc * stepf;
    }
}

void free_bp_tables(cbct_geometry *G) {
    cudaFree(const_cast<BpView *>(G->bp.views));
    cudaFree(const_cast<BpViewU *>(G->bp.viewu));
    cudaFree(const_cast<float4 *>(G->bp.pixT));
    cudaFree(G->d_bp_projT);
    G->d_bp_projT = nullptr;
    cudaFree(const_cast<float2 *>(G->bp.rows));
    cudaFree(G->d_bp_partial);
    G->bp = BpTables{};
    G->d_bp_partial = nullptr;
}

static double nudge(double a, double floor_mag) {
    if (std::fabs(a) >= floor_mag) return a;
    return a < 0 ? -floor_mag : floor_mag;
}

int build_bp_tables(cbct_geometry *G) {
    if (G->bp_impl != BP_CELL) return CBCT_OK;        // tables and partial volumes of a kernel that will not run
    const cbct_geometry_desc &d = G->desc;
    const int nu = d.nu, nv = d.nv, nvw = d.n_views;
    std::vector<BpView> views(nvw);
    std::vector<BpViewU> viewu((size_t)nvw * nu);
    std::vector<float4> pix((size_t)nv * nu);   // stored v-fastest: pixT[iu][iv]
    std::vector<float2> rows(nv);
    const double cx0 = -d.ox / d.dx + 0.5 * (d.nx - 1), cy0 = -d.oy / d.dy + 0.5 * (d.ny - 1),
                 cz0 = -d.oz / d.dz + 0.5 * (d.nz - 1);
    const double u_first = d.u0 - 0.5 * (nu - 1) * d.du, v_first = d.v0 - 0.5 * (nv - 1) * d.dv;
    for (int i = 0; i < nvw; ++i) {
        const double c = std::cos(d.angles[i]), s = std::sin(d.angles[i]);
        BpView &V = views[i];
        V.Kx = (float)(d.sad * c / d.dx + cx0); V.Ky = (float)(d.sad * s / d.dy + cy0);
        V.Fx = (float)(d.sad * c / d.dx); V.Fy = (float)(d.sad * s / d.dy);
        // world x = (X - cx0) dx, y = (Y - cy0) dy
        V.Dx = (float)(-c * d.dx); V.Dy = (float)(-s * d.dy);
        V.D0 = (float)(d.sad + c * cx0 * d.dx + s * cy0 * d.dy);
        V.Tx = (float)(-s * d.dx); V.Ty = (float)(c * d.dy);
        V.T0 = (float)(s * cx0 * d.dx - c * cy0 * d.dy);
        V.hl = (float)(0.5 * (std::fabs(s) * d.dx + std::fabs(c) * d.dy));
        V.hd = (float)(0.5 * (std::fabs(c) * d.dx + std::fabs(s) * d.dy));
        for (int iu = 0; iu < nu; ++iu) {
            const double u = u_first + iu * d.du;
            BpViewU &W = viewu[(size_t)i * nu + iu];
            const double Ax = (-d.sdd * c - u * s) / d.dx, Ay = (-d.sdd * s + u * c) / d.dy;
            W.Ax = (float)Ax; W.Ay = (float)Ay;
            W.Wx = (float)(1.0 / nudge(Ax, 1e-6 * d.sdd / d.dx)); W.Wy = (float)(1.0 / nudge(Ay, 1e-6 * d.sdd / d.dy));
            W.Gx = (float)(-d.sad * u * s / d.dx); W.Gy = (float)(d.sad * u * c / d.dy);
            W.pad0 = W.pad1 = 0.f;
        }
    }
    for (int iv = 0; iv < nv; ++iv) {
        const double v = v_first + iv * d.dv, vz = v / d.dz;
        rows[iv] = make_float2((float)vz, (float)(1.0 / nudge(vz, 1e-6 * d.sdd / d.dz)));
        for (int iu = 0; iu < nu; ++iu) {
            const double u = u_first + iu * d.du;
            const double L = std::sqrt(d.sdd * d.sdd + u * u + v * v);
            const double q = (u * u + v * v) / (L * (L + d.sdd));                 // 1 - SDD/L without cancellation
            pix[(size_t)iu * nv + iv] = make_float4((float)(1.0 / L), (float)q, (float)L, 0.f);
        }
    }
    BpTables &T = G->bp;
    const size_t ncell = (size_t)(d.nx + 1) * (d.ny + 1) * (d.nz + 1);
    cudaError_t e = cudaMalloc((void **)&T.views, sizeof(BpView) * views.size());
    if (e == cudaSuccess) e = cudaMalloc((void **)&T.viewu, sizeof(BpViewU) * viewu.size());
    if (e == cudaSuccess) e = cudaMalloc((void **)&T.pixT, sizeof(float4) * pix.size());
    if (e == cudaSuccess) e = cudaMalloc((void **)&T.rows, sizeof(float2) * rows.size());
    const bool cell = true;
    if (e == cudaSuccess && cell) e = cudaMalloc((void **)&G->d_bp_partial, sizeof(float) * 8 * ncell);
    if (e == cudaSuccess && cell) e = cudaMalloc((void **)&G->d_bp_projT, sizeof(float) * G->n_rays);
    if (e == cudaSuccess) e = cudaMemcpy((void *)T.views, views.data(), sizeof(BpView) * views.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy((void *)T.viewu, viewu.data(), sizeof(BpViewU) * viewu.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy((void *)T.pixT, pix.data(), sizeof(float4) * pix.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy((void *)T.rows, rows.data(), sizeof(float2) * rows.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return set_cuda_error(e);
    T.Kz = (float)cz0; T.cx0 = (float)cx0; T.cy0 = (float)cy0; T.cz0 = (float)cz0;
    T.sdd = (float)d.sdd; T.sad = (float)d.sad; T.u_first = (float)u_first; T.inv_du = (float)(1.0 / d.du);
    T.dz_dv = (float)(d.dz / d.dv); T.vfirst_dv = (float)(v_first / d.dv);
    T.t0 = (float)(G->t_min + 0.5 * G->step); T.inv_step = (float)(1.0 / G->step);
    T.k_eps = (float)std::fmax(0.02, 4.0 * 1.2e-7 * (d.sad + G->R) / G->step);   // fp32 rounding of r*L, in samples
    T.stepf = (float)G->step; T.tau0f = (float)(G->t_min + 0.5 * G->step - d.sad);
    G->workspace_bytes += sizeof(BpView) * views.size() + sizeof(BpViewU) * viewu.size() + sizeof(float4) * pix.size() +
                          sizeof(float2) * rows.size() + (cell ? sizeof(float) * 8 * ncell + sizeof(float) * G->n_rays : 0);
    return CBCT_OK;
}

int launch_backproject(const cbct_geometry *G, const float *d_proj, float *d_vol, cudaStream_t st, double *d_norm, bool *fused) {
    const DevGeom &g = G->dg;
    ProfScope prof(PROF_BACK, st);
    CBCT_TRY(device_error_pending(G));
    // the implementation was fixed at cbct_geometry_create (G->bp_impl): scatter (backproject_tma.cu) where the geometry
    // supports it, else the cell-driven kernel below; gather = the per-voxel cross-check
    if (fused) *fused = d_norm && G->bp_impl == BP_SCATTER;
    if (G->bp_impl == BP_SCATTER) return launch_backproject_tma(G, d_proj, d_vol, st, d_norm);
    if (G->bp_impl == BP_GATHER) {
        dim3 block(32, 4), grid(cdiv(g.nx, 32), cdiv(g.ny, 4), g.nz);
        backproject_gather_kernel<<<grid, block, 0, st>>>(g, d_proj, d_vol);
        CBCT_LAUNCH_CHECK();
        return CBCT_OK;
    }
    {
        dim3 block(32, 8), grid(cdiv(g.nu, 32), cdiv(g.nv, 32), g.n_views);
        transpose_proj_kernel<<<grid, block, 0, st>>>(d_proj, G->d_bp_projT, g.nu, g.nv);
        CBCT_LAUNCH_CHECK();
    }
    {
        // block = xb x-neighbouring columns of nz+1 cells, lanes along z; xb minimises idle lanes
        const int nzc = g.nz + 1;
        int xb = 1, best_waste = 1 << 30;
        const int max_threads = 320;
        for (int c = 1; c <= 16 && c * nzc <= max_threads; ++c) {
            const int th = ((c * nzc + 31) / 32) * 32, waste = (th - c * nzc) * 1024 / th;
            if (th >= 128 && waste < best_waste) { best_waste = waste; xb = c; }
        }
        if (best_waste == (1 << 30)) xb = nzc <= 512 ? std::max(1, std::min(16, 512 / nzc)) : 1;
        if (nzc > 512) return CBCT_E_UNSUPPORTED;   // taller volumes: use CBCT_BACKPROJECT_IMPL=gather
        const int threads = ((xb * nzc + 31) / 32) * 32;
        dim3 grid(cdiv(g.nx + 1, xb), g.ny + 1);
        // z travel of the steepest ray across one cell's x,y chord, in cells: small -> skip the z clip
        const cbct_geometry_desc &d = G->desc;
        const double tan_max = (std::fabs(d.v0) + 0.5 * d.nv * d.dv) / d.sdd;
        const bool zclip = tan_max * 1.4143 * std::fmax(d.dx, d.dy) / d.dz > 0.25;
#define CBCT_BP_LAUNCH(MAXT, MINB, ZC)                                                                              \
    backproject_cell_kernel<MAXT, MINB, ZC><<<grid, threads, 0, st>>>(G->bp, g.nx, g.ny, g.nz, g.nu, g.nv, g.n_views, \
                                                                      g.K, xb, G->d_bp_projT, G->d_bp_partial)
        if (threads <= 320) { if (zclip) CBCT_BP_LAUNCH(320, 3, true); else CBCT_BP_LAUNCH(320, 3, false); }
        else { if (zclip) CBCT_BP_LAUNCH(512, 2, true); else CBCT_BP_LAUNCH(512, 2, false); }
#undef CBCT_BP_LAUNCH
        CBCT_LAUNCH_CHECK();
    }
    {
        const size_t smem = sizeof(float) * 32 * (size_t)(g.nz | 1);
        if (smem <= 48 * 1024) {
            dim3 grid(cdiv(g.nx, 32), g.ny);
            backproject_combine_kernel<<<grid, 256, smem, st>>>(G->d_bp_partial, d_vol, g.nx, g.ny, g.nz, (float)G->step);
        } else {
            dim3 block(32, 4), grid(cdiv(g.nx, 32), cdiv(g.ny, 4));
            backproject_combine_simple_kernel<<<grid, block, 0, st>>>(G->d_bp_partial, d_vol, g.nx, g.ny, g.nz, (float)G->step);
        }
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}

}  // namespace cbct
