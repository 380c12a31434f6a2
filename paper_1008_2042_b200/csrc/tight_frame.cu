// tight_frame.cu -- piecewise-linear tight frame, vector shrinkage (PAPER.md:123-127
// Eq. 2), positivity and the fused f <- [H] D^T T_mu D f.
// Boundary: edge-replicate extension in D, exact matrix transpose in D^T:
// for the symmetric filters h0, h2 the transpose is the flipped filter with edge-replicate extension
// of alpha, for the antisymmetric h1 it is the flipped filter with SIGN-FLIPPED replicate extension.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/cbct_debug.h"
#include "common.cuh"

namespace cbct {

#define TF_S 0.35355339059327373f /* sqrt(2)/4 */

// alpha_l[x] = sum_a h_l[a] f[x-a]; m1 = f[x-1], c = f[x], p1 = f[x+1]
__device__ __forceinline__ void analyse3(float m1, float c, float p1, float &o0, float &o1, float &o2) {
    const float e = 0.25f * (m1 + p1);
    o0 = fmaf(0.5f, c, e);          // h0 = 1/4 [1,2,1]
    o1 = TF_S * (p1 - m1);          // h1 = sqrt(2)/4 [1,0,-1]  -> h1[-1] f[x+1] + h1[+1] f[x-1]
    o2 = fmaf(0.5f, c, -e);         // h2 = 1/4 [-1,2,-1]
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// ------------------------------------------------------------------------------ alpha = D f
__global__ void __launch_bounds__(128) tf_decompose_kernel(const float *__restrict__ f, float *__restrict__ alpha,
                                                           int nx, int ny, int nz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y, z = blockIdx.z;
    if (x >= nx || y >= ny) return;
    float v[3][3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a)
                v[c][b][a] = __ldg(f + ((size_t)clampi(z + c - 1, 0, nz - 1) * ny + clampi(y + b - 1, 0, ny - 1)) * nx +
                                   clampi(x + a - 1, 0, nx - 1));
    float X[3][3][3];  // [l][z][y]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b) analyse3(v[c][b][0], v[c][b][1], v[c][b][2], X[0][c][b], X[1][c][b], X[2][c][b]);
    float Y[3][3][3];  // [l][m][z]
#pragma unroll
    for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int c = 0; c < 3; ++c) analyse3(X[l][c][0], X[l][c][1], X[l][c][2], Y[l][0][c], Y[l][1][c], Y[l][2][c]);
    const size_t nvox = (size_t)nx * ny * nz, idx = ((size_t)z * ny + y) * nx + x;
#pragma unroll
    for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            float o0, o1, o2;
            analyse3(Y[l][m][0], Y[l][m][1], Y[l][m][2], o0, o1, o2);
            alpha[(size_t)(l + 3 * m) * nvox + idx] = o0;
            alpha[(size_t)(l + 3 * m + 9) * nvox + idx] = o1;
            alpha[(size_t)(l + 3 * m + 18) * nvox + idx] = o2;
        }
}

// shrink factor of Eq. 2 from the squared norm of the 26 high bands
__device__ __forceinline__ float shrink_factor(float norm2, float mu) {
    if (!(norm2 > 0.f)) return 0.f;
    return fmaxf(1.f - mu * rsqrtf(norm2), 0.f);
}

// ------------------------------------------------------------------------------ T_mu, in place
__global__ void __launch_bounds__(256) tf_shrink_kernel(float *__restrict__ alpha, float mu, long long nvox) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= nvox) return;
    float a[26], n2 = 0.f;
#pragma unroll
    for (int b = 0; b < 26; ++b) { a[b] = alpha[(size_t)(b + 1) * nvox + i]; n2 = fmaf(a[b], a[b], n2); }
    // sqrt/div in IEEE form here: this entry point is the reference semantics of Eq. 2
    float fac = 0.f;
    if (n2 > 0.f) fac = fmaxf(1.f - mu / sqrtf(n2), 0.f);
#pragma unroll
    for (int b = 0; b < 26; ++b) alpha[(size_t)(b + 1) * nvox + i] = a[b] * fac;
}

// ------------------------------------------------------------------------------ f = D^T alpha
__constant__ float c_h[3][3] = {{0.25f, 0.5f, 0.25f}, {TF_S, 0.f, -TF_S}, {-0.25f, 0.5f, -0.25f}};  // h_l[a+1]

__global__ void __launch_bounds__(128) tf_reconstruct_kernel(const float *__restrict__ alpha, float *__restrict__ f,
                                                             int nx, int ny, int nz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y, z = blockIdx.z;
    if (x >= nx || y >= ny) return;
    const size_t nvox = (size_t)nx * ny * nz;
    // out(x) = sum_a h[a] * ext(alpha)(x + a); ext replicates the face value, negated for h1
    int xs[3], ys[3], zs[3];
    float sx[3], sy[3], sz[3];  // -1 where the antisymmetric extension applies
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int xa = x + a - 1, ya = y + a - 1, za = z + a - 1;
        xs[a] = clampi(xa, 0, nx - 1); sx[a] = (xa == xs[a]) ? 1.f : -1.f;
        ys[a] = clampi(ya, 0, ny - 1); sy[a] = (ya == ys[a]) ? 1.f : -1.f;
        zs[a] = clampi(za, 0, nz - 1); sz[a] = (za == zs[a]) ? 1.f : -1.f;
    }
    float acc = 0.f;
    for (int n = 0; n < 3; ++n)
        for (int m = 0; m < 3; ++m)
            for (int l = 0; l < 3; ++l) {
                const float *ab = alpha + (size_t)(l + 3 * m + 9 * n) * nvox;
                float band = 0.f;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float wz = c_h[n][c] * (n == 1 ? sz[c] : 1.f);
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const float wzy = wz * c_h[m][b] * (m == 1 ? sy[b] : 1.f);
                        const float *row = ab + ((size_t)zs[c] * ny + ys[b]) * nx;
                        float rs = 0.f;
#pragma unroll
                        for (int a = 0; a < 3; ++a) rs = fmaf(c_h[l][a] * (l == 1 ? sx[a] : 1.f), __ldg(row + xs[a]), rs);
                        band = fmaf(wzy, rs, band);
                    }
                }
                acc += band;
            }
    f[((size_t)z * ny + y) * nx + x] = acc;
}

// Separable, z-marching form of the same sum (the default; the direct kernel above reads every coefficient 27 times
// through L1 -- 6.3 ms for 1.98 GB at cfg 4 -- and is kept as a cross-check, CBCT_TF_RECONSTRUCT_IMPL=direct):
//   f = sum_n Hz_n^T [ sum_m Hy_m^T [ sum_l Hx_l^T alpha_lmn ] ]
// A CTA owns a 32(x) x 8(y) column of outputs over a z-segment and walks the coefficient planes once:
//   x-pass: warp w (10 warps = 8 rows + one halo row on each side) forms G_mn = sum_l Hx_l^T alpha_lmn for its
//           row of plane zz, 9 values, into shared memory;
//   y-pass: the 8 inner warps form P_n = sum_m Hy_m^T G_mn from the rows w-1, w, w+1;
//   z-pass: plane zz contributes h_n[0] P_n to out(zz+1), h_n[1] P_n to out(zz), h_n[2] P_n to out(zz-1), held in
//           three rolling registers; out(zz-1) is complete after plane zz and is stored.
// Boundary (exact transpose of the edge-replicate extension): a tap that falls outside
// reads the face value, negated for the antisymmetric h1; in z that is an extra sgn_n h_n[0] P_n on plane 0
// and sgn_n h_n[2] P_n on plane nz-1.  Every coefficient is read once (x 10/8 for the row halo, x (ZSEG+2)/ZSEG).
constexpr int TR_X = 32, TR_Y = 8, TR_ZSEG = 14, TR_THREADS = 32 * (TR_Y + 2);

__global__ void __launch_bounds__(TR_THREADS) tf_reconstruct_march_kernel(const float *__restrict__ alpha, float *__restrict__ f,
                                                                        int nx, int ny, int nz) {
    __shared__ float sG[9][TR_Y + 2][TR_X];                       // [m + 3n][row w][x]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int x0 = blockIdx.x * TR_X, y0 = blockIdx.y * TR_Y, za = blockIdx.z * TR_ZSEG, zb = min(za + TR_ZSEG, nz);
    const size_t nvox = (size_t)nx * ny * nz;
    const int x = min(x0 + lane, nx - 1);                         // lanes beyond the volume recompute the last column, never store
    const int yr = clampi(y0 - 1 + w, 0, ny - 1);                 // the row this warp filters in the x-pass
    const int y = y0 + w - 1;                                     // the output row of an inner warp
    const bool inner = w >= 1 && w <= TR_Y;
    const bool store_ok = inner && y < ny && x0 + lane < nx;
    // x taps: clamped column and the sign of the antisymmetric extension
    int xs[3];
    float sx[3], sy[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int xa = x + a - 1, ya = y + a - 1;
        xs[a] = clampi(xa, 0, nx - 1); sx[a] = (xa == xs[a]) ? 1.f : -1.f;
        sy[a] = (ya >= 0 && ya <= ny - 1) ? 1.f : -1.f;
    }
    float a_prev = 0.f, a_cur = 0.f, a_next = 0.f;
    for (int zz = za - 1; zz <= zb; ++zz) {                       // CTA-uniform trip count and branches
        if (zz >= 0 && zz < nz) {
            const float *plane = alpha + ((size_t)zz * ny + yr) * nx;
#pragma unroll
            for (int mn = 0; mn < 9; ++mn) {
                float acc = 0.f;
#pragma unroll
                for (int l = 0; l < 3; ++l) {
                    const float *row = plane + (size_t)(l + 3 * mn) * nvox;
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        if (l == 1 && a == 1) continue;          // h1[0] = 0
                        acc = fmaf(c_h[l][a] * (l == 1 ? sx[a] : 1.f), __ldg(row + xs[a]), acc);
                    }
                }
                sG[mn][w][lane] = acc;
            }
            __syncthreads();
            if (inner) {
                float c_next = 0.f, c_cur = 0.f, c_prev = 0.f;
#pragma unroll
                for (int n = 0; n < 3; ++n) {
                    float P = 0.f;
#pragma unroll
                    for (int m = 0; m < 3; ++m)
#pragma unroll
                        for (int b = 0; b < 3; ++b) {
                            if (m == 1 && b == 1) continue;
                            P = fmaf(c_h[m][b] * (m == 1 ? sy[b] : 1.f), sG[m + 3 * n][w + b - 1][lane], P);
                        }
                    const float sgn = n == 1 ? -1.f : 1.f;
                    c_next = fmaf(c_h[n][0], P, c_next);
                    float k_cur = c_h[n][1];
                    if (zz == 0) k_cur = fmaf(sgn, c_h[n][0], k_cur);
                    if (zz == nz - 1) k_cur = fmaf(sgn, c_h[n][2], k_cur);
                    c_cur = fmaf(k_cur, P, c_cur);
                    c_prev = fmaf(c_h[n][2], P, c_prev);
                }
                a_next += c_next; a_cur += c_cur; a_prev += c_prev;
            }
            __syncthreads();                                      // sG is rewritten for the next plane
        }
        if (store_ok && zz - 1 >= za && zz - 1 < zb) f[((size_t)(zz - 1) * ny + y) * nx + x] = a_prev;
        a_prev = a_cur; a_cur = a_next; a_next = 0.f;
    }
}

// ------------------------------------------------------------------------------ fused [H] D^T T_mu D
// Uses the tight-frame identities sum_i psi_i(a) psi_i(b) = delta_ab psi_0(a):
//   ||alpha_h||^2 = W0[f^2] - (W0 f)^2                      (a weighted local variance)
//   D^T T_mu D f  = f * W0^T s + W0^T((1 - s) * W0 f),  s = max(1 - mu/||alpha_h||, 0)
// with W0 the low-pass band operator (edge-replicate), W0^T = W0 because h0 is symmetric.
// The variance is formed on centre-subtracted data (shift invariant) to avoid fp32 cancellation.
constexpr int FT_X = 32, FT_Y = 8, FT_Z = 4;                       // output tile
constexpr int FA_X = FT_X + 4, FA_Y = FT_Y + 4, FA_Z = FT_Z + 4;   // f tile, halo 2
constexpr int FB_X = FT_X + 2, FB_Y = FT_Y + 2, FB_Z = FT_Z + 2;   // s / (1-s)m tile, halo 1

__global__ void __launch_bounds__(256) tf_fused_kernel(const float *__restrict__ fin, float *__restrict__ fout, float mu,
                                                       int clamp_nonneg, int nx, int ny, int nz) {
    __shared__ float sf[FA_Z][FA_Y][FA_X];
    __shared__ float ss[FB_Z][FB_Y][FB_X];
    __shared__ float sb[FB_Z][FB_Y][FB_X];
    const int x0 = blockIdx.x * FT_X, y0 = blockIdx.y * FT_Y, z0 = blockIdx.z * FT_Z;
    const int tid = threadIdx.x;
    for (int i = tid; i < FA_X * FA_Y * FA_Z; i += 256) {
        const int a = i % FA_X, b = (i / FA_X) % FA_Y, c = i / (FA_X * FA_Y);
        sf[c][b][a] = __ldg(fin + ((size_t)clampi(z0 + c - 2, 0, nz - 1) * ny + clampi(y0 + b - 2, 0, ny - 1)) * nx +
                            clampi(x0 + a - 2, 0, nx - 1));
    }
    __syncthreads();
    const float w3[3] = {0.25f, 0.5f, 0.25f};
    for (int i = tid; i < FB_X * FB_Y * FB_Z; i += 256) {
        const int a = i % FB_X, b = (i / FB_X) % FB_Y, c = i / (FB_X * FB_Y);
        // position in the volume, clamped: the extension of a field is its value at the clamped position
        const int px = clampi(x0 + a - 1, 0, nx - 1), py = clampi(y0 + b - 1, 0, ny - 1), pz = clampi(z0 + c - 1, 0, nz - 1);
        const int lx = px - x0 + 2, ly = py - y0 + 2, lz = pz - z0 + 2;   // centre in sf
        const float ctr = sf[lz][ly][lx];
        float m1 = 0.f, m2 = 0.f;
#pragma unroll
        for (int dz = 0; dz < 3; ++dz)
#pragma unroll
            for (int dy = 0; dy < 3; ++dy) {
                float r1 = 0.f, r2 = 0.f;
#pragma unroll
                for (int dxx = 0; dxx < 3; ++dxx) {
                    const float d = sf[lz + dz - 1][ly + dy - 1][lx + dxx - 1] - ctr;
                    r1 = fmaf(w3[dxx], d, r1);
                    r2 = fmaf(w3[dxx] * d, d, r2);
                }
                m1 = fmaf(w3[dz] * w3[dy], r1, m1);
                m2 = fmaf(w3[dz] * w3[dy], r2, m2);
            }
        const float var = fmaxf(m2 - m1 * m1, 0.f);
        const float s = shrink_factor(var, mu);
        ss[c][b][a] = s;
        sb[c][b][a] = (1.f - s) * (ctr + m1);
    }
    __syncthreads();
    for (int i = tid; i < FT_X * FT_Y * FT_Z; i += 256) {
        const int a = i % FT_X, b = (i / FT_X) % FT_Y, c = i / (FT_X * FT_Y);
        const int x = x0 + a, y = y0 + b, z = z0 + c;
        if (x >= nx || y >= ny || z >= nz) continue;
        float A = 0.f, B = 0.f;
#pragma unroll
        for (int dz = 0; dz < 3; ++dz)
#pragma unroll
            for (int dy = 0; dy < 3; ++dy) {
                float ra = 0.f, rb = 0.f;
#pragma unroll
                for (int dxx = 0; dxx < 3; ++dxx) {
                    ra = fmaf(w3[dxx], ss[c + dz][b + dy][a + dxx], ra);
                    rb = fmaf(w3[dxx], sb[c + dz][b + dy][a + dxx], rb);
                }
                A = fmaf(w3[dz] * w3[dy], ra, A);
                B = fmaf(w3[dz] * w3[dy], rb, B);
            }
        float out = fmaf(sf[c + 2][b + 2][a + 2], A, B);
        if (clamp_nonneg) out = fmaxf(out, 0.f);
        fout[((size_t)z * ny + y) * nx + x] = out;
    }
}


// ------------------------------------------------------------------------------ fused [H] D^T T_mu D, z-marching
// The same result as tf_fused_kernel with every voxel read from global memory once per CTA and no 27-tap sums: the CTA
// owns a 28(x) x (4 FM_WARPS RPT - 4)(y) column of outputs over a z-segment and walks the planes once.
//   * ||alpha_h||^2 from SEPARABLE, cancellation-free pieces.  Per axis the three filters satisfy
//     sum_l (h_l * g)^2 = h0 * g^2  (the identity above, one axis at a time), hence with X_l = h_l *x f, Y_0m = h_m *y X_0,
//     alpha_00n = h_n *z Y_00:
//       ||alpha_h||^2 = Wz[ Wy[X_1^2 + X_2^2] + Y_01^2 + Y_02^2 ] + alpha_001^2 + alpha_002^2
//     (bands with l != 0; bands with l = 0, m != 0; bands with l = m = 0, n != 0): a sum of non-negative terms built
//     from difference filters, so no local mean has to be subtracted first (what forced tf_fused_kernel's 27-tap form).
//   * x neighbours by warp shuffle (a warp = 32 consecutive columns of one row, 28 of them outputs), y neighbours
//     through shared memory (only the first / last row of a thread's RPT rows), z neighbours in rolling registers;
//   * the synthesis  out = f W0[s] + W0[(1-s) W0 f]  is three more separable [1 2 1]/4 passes with the same plumbing, one
//     plane behind the analysis; its z-pass is kept as three rolling accumulators per field (plane j adds 1/4, 1/2, 1/4
//     to the outputs j-1, j, j+1; the planes 0 and nz-1 add their clamped copy to themselves).
// Extensions are "the value at the clamped position" as in tf_fused_kernel: rows / columns / planes are LOADED at
// clamped coordinates (so the analysis fields of an outside row equal the face row's), and the synthesis passes take
// a face voxel's outside neighbour from the voxel itself.
constexpr int FM_WARPS = 8, FM_TX = 28;

// [1 2 1] and [-1 2 -1] of (m, c, p) WITHOUT the factor 1/4, and the squared antisymmetric tap 2 (p - m)^2 = 16 (h1 * g)^2:
// the normalisations (powers of two, exact) are applied once per field instead of once per pass.
__device__ __forceinline__ void fm_pass(float m, float c, float p, float &lo, float &hi, float &d2) {
    const float e = m + p, d = p - m;
    lo = fmaf(2.f, c, e);
    hi = fmaf(2.f, c, -e);
    d2 = (d + d) * d;
}
__device__ __forceinline__ float fm_low(float m, float c, float p) { return fmaf(2.f, c, m + p); }

template <int RPT>
__global__ void __launch_bounds__(FM_WARPS * 32) tf_fused_march_kernel(const float *__restrict__ fin, float *__restrict__ fout,
                                                                       float mu, int clamp_nonneg, int nx, int ny, int nz, int zseg) {
    constexpr int R = FM_WARPS * RPT;                              // rows of the CTA, R - 4 of them outputs
    __shared__ float sA0[R][32], sA1[R][32];                       // analysis: 4 X_0 and 16 (X_1^2 + X_2^2) of the rows other threads need
    __shared__ float sS0[R][32], sS1[R][32];                       // synthesis: 4 Wx[s], 4 Wx[b]
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int x0 = blockIdx.x * FM_TX, y0 = blockIdx.y * (R - 4);
    const int za = blockIdx.z * zseg, zb = min(za + zseg, nz);
    const int xl = x0 - 2 + lane, r0 = w * RPT;
    const int lane_m = max(lane - 1, 0), lane_p = min(lane + 1, 31);
    // synthesis neighbours are "the value at the clamped position": a face voxel's outside neighbour is the voxel itself
    const int slane_m = xl == 0 ? lane : lane_m, slane_p = xl == nx - 1 ? lane : lane_p;
    const int plane = nx * ny;                                     // nx ny nz < 2^31 (tf_check): 32-bit element offsets
    int rowoff[RPT];
    unsigned face_lo = 0, face_hi = 0, store = 0;                  // bit i: row i is y = 0 / y = ny - 1 / an output of this thread
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
        const int yl = y0 - 2 + r0 + i, r = r0 + i;
        rowoff[i] = clampi(yl, 0, ny - 1) * nx + clampi(xl, 0, nx - 1);
        face_lo |= (yl == 0) << i;
        face_hi |= (yl == ny - 1) << i;
        store |= (r >= 2 && r < R - 2 && yl < ny && lane >= 2 && lane < 2 + FM_TX && xl < nx) << i;
    }
    // shared rows read for the first / last row of this thread (clamped into the CTA; the face rule for the synthesis)
    const int ra_up = max(r0 - 1, 0), ra_dn = min(r0 + RPT, R - 1);
    const int rs_up = (face_lo & 1u) ? r0 : ra_up, rs_dn = ((face_hi >> (RPT - 1)) & 1u) ? r0 + RPT - 1 : ra_dn;
    float c0[RPT], c1[RPT], c2[RPT];                               // f of the planes q, q+1, q+2 (loads two steps ahead)
    float fa[RPT], fb[RPT], Ya[RPT], Yb[RPT], ta[RPT], tb[RPT];    // f, 16 Y_00, 256 t of the planes q-2, q-1
    float Sp[RPT], Sc[RPT], Bp[RPT], Bc[RPT];                      // z-pass accumulators of the outputs j-1, j
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
        c0[i] = __ldg(fin + clampi(za - 2, 0, nz - 1) * plane + rowoff[i]);
        c1[i] = __ldg(fin + clampi(za - 1, 0, nz - 1) * plane + rowoff[i]);
        c2[i] = __ldg(fin + clampi(za, 0, nz - 1) * plane + rowoff[i]);
        fa[i] = fb[i] = Ya[i] = Yb[i] = ta[i] = tb[i] = Sp[i] = Sc[i] = Bp[i] = Bc[i] = 0.f;
    }
#pragma unroll 3                                                  // the rolling registers are rings of three: no moves
    for (int q = za - 2; q <= zb + 1; ++q) {                       // CTA-uniform trip count and branches
        float fn[RPT], X0[RPT], Q1[RPT], Yn[RPT], tn[RPT], Sn[RPT], Bn[RPT];
#pragma unroll
        for (int i = 0; i < RPT; ++i) { fn[i] = c0[i]; c0[i] = c1[i]; c1[i] = c2[i]; }
        if (q + 3 <= zb + 1) {
            const float *pl = fin + clampi(q + 3, 0, nz - 1) * plane;
#pragma unroll
            for (int i = 0; i < RPT; ++i) c2[i] = __ldg(pl + rowoff[i]);
        }
        // analysis, x-pass on plane q: X0 = 4 X_0, Q1 = 16 (X_1^2 + X_2^2)
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            float hi, d2;
            fm_pass(__shfl_sync(full, fn[i], lane_m), fn[i], __shfl_sync(full, fn[i], lane_p), X0[i], hi, d2);
            Q1[i] = fmaf(hi, hi, d2);
        }
        sA0[r0][lane] = X0[0]; sA1[r0][lane] = Q1[0];
        if (RPT > 1) { sA0[r0 + RPT - 1][lane] = X0[RPT - 1]; sA1[r0 + RPT - 1][lane] = Q1[RPT - 1]; }
        __syncthreads();
        // analysis, y-pass: Yn = 16 Y_00, tn = 256 (Wy[X_1^2 + X_2^2] + Y_01^2 + Y_02^2)
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            const float X0m = i > 0 ? X0[i - 1] : sA0[ra_up][lane], X0p = i < RPT - 1 ? X0[i + 1] : sA0[ra_dn][lane];
            const float Q1m = i > 0 ? Q1[i - 1] : sA1[ra_up][lane], Q1p = i < RPT - 1 ? Q1[i + 1] : sA1[ra_dn][lane];
            float hi, d2;
            fm_pass(X0m, X0[i], X0p, Yn[i], hi, d2);
            tn[i] = fmaf(4.f, fm_low(Q1m, Q1[i], Q1p), fmaf(hi, hi, d2));      // 64 Wy[16 q] * 4 + 256 (Y_01^2 + Y_02^2)
        }
        // analysis, z-pass on plane j = q - 1 (planes q-2, q-1, q), shrink factor, then the synthesis x-pass
        const int j = q - 1;
        const bool vj = j >= 0 && j < nz && j >= za - 1 && j <= zb;
        float sx[RPT], bx[RPT];
        if (vj) {
#pragma unroll
            for (int i = 0; i < RPT; ++i) {
                float m64, hi, d2;
                fm_pass(Ya[i], Yb[i], Yn[i], m64, hi, d2);                      // 64 alpha_000, 64 alpha_002, 4096 alpha_001^2
                const float Eh = (fmaf(4.f, fm_low(ta[i], tb[i], tn[i]), fmaf(hi, hi, d2))) * (1.f / 4096.f);
                const float s = shrink_factor(Eh, mu), b = (1.f - s) * (m64 * (1.f / 64.f));
                sx[i] = fm_low(__shfl_sync(full, s, slane_m), s, __shfl_sync(full, s, slane_p));
                bx[i] = fm_low(__shfl_sync(full, b, slane_m), b, __shfl_sync(full, b, slane_p));
            }
            sS0[r0][lane] = sx[0]; sS1[r0][lane] = bx[0];
            if (RPT > 1) { sS0[r0 + RPT - 1][lane] = sx[RPT - 1]; sS1[r0 + RPT - 1][lane] = bx[RPT - 1]; }
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < RPT; ++i) { Sn[i] = 0.f; Bn[i] = 0.f; }
        if (vj) {
            // synthesis, y-pass (sxy = 16 Wy Wx[s]) and the z-pass contributions of plane j (weights 1, 2, 1 and the faces' own copy)
            const float wc = 2.f + (j == 0 ? 1.f : 0.f) + (j == nz - 1 ? 1.f : 0.f);
#pragma unroll
            for (int i = 0; i < RPT; ++i) {
                float su = i > 0 ? sx[i - 1] : sS0[rs_up][lane], sd = i < RPT - 1 ? sx[i + 1] : sS0[rs_dn][lane];
                float bu = i > 0 ? bx[i - 1] : sS1[rs_up][lane], bd = i < RPT - 1 ? bx[i + 1] : sS1[rs_dn][lane];
                if (i > 0 && ((face_lo >> i) & 1u)) { su = sx[i]; bu = bx[i]; }
                if (i < RPT - 1 && ((face_hi >> i) & 1u)) { sd = sx[i]; bd = bx[i]; }
                const float sxy = fm_low(su, sx[i], sd), bxy = fm_low(bu, bx[i], bd);
                Sp[i] += sxy; Sc[i] = fmaf(wc, sxy, Sc[i]); Sn[i] = sxy;
                Bp[i] += bxy; Bc[i] = fmaf(wc, bxy, Bc[i]); Bn[i] = bxy;
            }
        }
        // output plane q - 2 is complete: out = f W0[s] + W0[b], the accumulators carry the factor 64
        const int o = q - 2;
        if (o >= za && o < zb) {
            float *pl = fout + o * plane;
#pragma unroll
            for (int i = 0; i < RPT; ++i)
                if ((store >> i) & 1u) {
                    float out = fmaf(fa[i], Sp[i], Bp[i]) * (1.f / 64.f);
                    if (clamp_nonneg) out = fmaxf(out, 0.f);
                    pl[rowoff[i]] = out;
                }
        }
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            Sp[i] = Sc[i]; Sc[i] = Sn[i]; Bp[i] = Bc[i]; Bc[i] = Bn[i];
            Ya[i] = Yb[i]; Yb[i] = Yn[i]; ta[i] = tb[i]; tb[i] = tn[i]; fa[i] = fb[i]; fb[i] = fn[i];
        }
    }
}

}  // namespace cbct

using namespace cbct;

static int tf_check(const void *a, const void *b, int nx, int ny, int nz) {
    if (!a || !b || nx <= 0 || ny <= 0 || nz <= 0) return CBCT_E_INVALID;
    if ((long long)nx * ny * nz > (1LL << 31) - 1) return CBCT_E_INVALID;
    return device_supported();
}

extern "C" int tf_decompose(const float *d_f, float *d_alpha, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_f, d_alpha, nx, ny, nz));
    dim3 block(32, 4), grid(cdiv(nx, 32), cdiv(ny, 4), nz);
    tf_decompose_kernel<<<grid, block, 0, as_stream(stream)>>>(d_f, d_alpha, nx, ny, nz);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int tf_shrink(float *d_alpha, float mu, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_alpha, d_alpha, nx, ny, nz));
    if (!(mu >= 0.f)) return CBCT_E_INVALID;
    const long long nvox = (long long)nx * ny * nz;
    tf_shrink_kernel<<<cdiv(nvox, 256), 256, 0, as_stream(stream)>>>(d_alpha, mu, nvox);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int tf_reconstruct(const float *d_alpha, float *d_f, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_alpha, d_f, nx, ny, nz));
    dim3 grid(cdiv(nx, TR_X), cdiv(ny, TR_Y), cdiv(nz, TR_ZSEG));
    tf_reconstruct_march_kernel<<<grid, TR_THREADS, 0, as_stream(stream)>>>(d_alpha, d_f, nx, ny, nz);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// cbct_debug.h: the 27 x 27-tap cross-check of the kernel above
extern "C" int tf_reconstruct_direct(const float *d_alpha, float *d_f, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_alpha, d_f, nx, ny, nz));
    dim3 block(32, 4), grid(cdiv(nx, 32), cdiv(ny, 4), nz);
    tf_reconstruct_kernel<<<grid, block, 0, as_stream(stream)>>>(d_alpha, d_f, nx, ny, nz);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

static int launch_tf_fused_tile(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, cudaStream_t st) {
    dim3 grid(cdiv(nx, FT_X), cdiv(ny, FT_Y), cdiv(nz, FT_Z));
    tf_fused_kernel<<<grid, 256, 0, st>>>(d_in, d_out, mu, clamp_nonneg, nx, ny, nz);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

static int launch_tf_fused_march(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, cudaStream_t st) {
    const int rpt = ny > 12 ? 4 : 2, rows_out = FM_WARPS * rpt - 4;
    const int tx = cdiv(nx, FM_TX), ty = cdiv(ny, rows_out);
    // z-segments: enough CTAs for ~8 per SM, never shorter than 8 planes (a segment recomputes 4 planes of halo)
    int nseg = (int)((1184.0 + 0.5 * tx * ty) / ((double)tx * ty));
    nseg = nseg < 1 ? 1 : nseg;
    if (nseg > nz / 8) nseg = nz / 8 > 0 ? nz / 8 : 1;
    const int zseg = cdiv(nz, nseg);
    dim3 grid(tx, ty, cdiv(nz, zseg));
    if (rpt == 4) tf_fused_march_kernel<4><<<grid, FM_WARPS * 32, 0, st>>>(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, zseg);
    else tf_fused_march_kernel<2><<<grid, FM_WARPS * 32, 0, st>>>(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, zseg);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// Which kernel serves tf_apply_fused: decided once per process.  tf_fused_kernel (3-D tile, 27-tap sums) is the variant that
// has run on a B200 (round 1: 0.50 ms at 512x512x70, shared-memory bound); tf_fused_march_kernel reads every voxel once.
// As for the projectors (geometry.cu: fast_variants_ok), the newer kernel becomes the default only after it has reproduced
// the older one on the device in use: both run once on a built-in 45 x 37 x 11 volume (ragged in every tile dimension, both
// z-segment ends inside), with and without the positivity clamp, and must agree to 1e-5 of max|f|.  CBCT_TF_FUSED_IMPL =
// tile | march forces a choice (read once).  The check runs inside the first tf_apply_fused / cbct_recon_create of the
// process and synchronises the device then; no later call does.
static int g_tf_state = -1;                               // -1 undecided, 0 tile, 1 march (checked), 2 march (forced)
static std::mutex g_tf_mu;

static bool run_tf_selfcheck() {
    const int nx = 45, ny = 37, nz = 11;
    const size_t n = (size_t)nx * ny * nz;
    std::vector<float> h(n), a(n), b(n);
    unsigned lcg = 777u;
    for (auto &v : h) { lcg = lcg * 1664525u + 1013904223u; v = (float)(lcg >> 8) * (1.0f / 16777216.0f) - 0.3f; }
    float *d_in = nullptr, *d_a = nullptr, *d_b = nullptr;
    bool ok = cudaMalloc(&d_in, n * 4) == cudaSuccess && cudaMalloc(&d_a, n * 4) == cudaSuccess && cudaMalloc(&d_b, n * 4) == cudaSuccess &&
              cudaMemcpy(d_in, h.data(), n * 4, cudaMemcpyHostToDevice) == cudaSuccess;
    for (int clamp = 0; ok && clamp < 2; ++clamp) {
        const float mu = clamp ? 0.25f : 0.1f;
        ok = launch_tf_fused_tile(d_in, d_a, mu, clamp, nx, ny, nz, nullptr) == CBCT_OK &&
             launch_tf_fused_march(d_in, d_b, mu, clamp, nx, ny, nz, nullptr) == CBCT_OK && cudaDeviceSynchronize() == cudaSuccess &&
             cudaMemcpy(a.data(), d_a, n * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
             cudaMemcpy(b.data(), d_b, n * 4, cudaMemcpyDeviceToHost) == cudaSuccess;
        for (size_t i = 0; ok && i < n; ++i) ok = std::fabs(a[i] - b[i]) <= 1e-5f;      // max|f| < 1
    }
    if (!ok) (void)cudaGetLastError();
    cudaFree(d_in); cudaFree(d_a); cudaFree(d_b);
    return ok;
}

static int tf_fused_choice() {
    std::lock_guard<std::mutex> lk(g_tf_mu);
    if (g_tf_state < 0) {
        const char *e = getenv("CBCT_TF_FUSED_IMPL");
        if (e && !strcmp(e, "tile")) g_tf_state = 0;
        else if (e && !strcmp(e, "march")) g_tf_state = 2;
        else g_tf_state = run_tf_selfcheck() ? 1 : 0;
    }
    return g_tf_state;
}

namespace cbct {
void tf_fused_prepare() { (void)tf_fused_choice(); }
}

extern "C" int tf_apply_fused(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz,
                              void *stream) {
    CBCT_TRY(tf_check(d_in, d_out, nx, ny, nz));
    if (d_in == d_out || !(mu >= 0.f)) return CBCT_E_INVALID;
    return tf_fused_choice() ? launch_tf_fused_march(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, as_stream(stream))
                             : launch_tf_fused_tile(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, as_stream(stream));
}

// cbct_debug.h: each kernel on its own (cross-checks, A/B timing), and which one tf_apply_fused uses
extern "C" int tf_apply_fused_tile(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_in, d_out, nx, ny, nz));
    if (d_in == d_out || !(mu >= 0.f)) return CBCT_E_INVALID;
    return launch_tf_fused_tile(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, as_stream(stream));
}
extern "C" int tf_apply_fused_march(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, void *stream) {
    CBCT_TRY(tf_check(d_in, d_out, nx, ny, nz));
    if (d_in == d_out || !(mu >= 0.f)) return CBCT_E_INVALID;
    return launch_tf_fused_march(d_in, d_out, mu, clamp_nonneg, nx, ny, nz, as_stream(stream));
}
extern "C" const char *tf_apply_fused_describe(void) {
    if (device_supported() != CBCT_OK) return "unavailable (no sm_100 device)";
    switch (tf_fused_choice()) {
        case 1: return "tf_fused_march_kernel (self-check passed)";
        case 2: return "tf_fused_march_kernel (forced)";
        default: return getenv("CBCT_TF_FUSED_IMPL") ? "tf_fused_kernel (forced)" : "tf_fused_kernel (tf_fused_march_kernel rejected by the self-check)";
    }
}
