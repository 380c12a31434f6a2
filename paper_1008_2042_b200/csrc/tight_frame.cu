// tight_frame.cu -- piecewise-linear tight frame, vector shrinkage (PAPER.md:123-127
// Eq. 2), positivity and the fused f <- [H] D^T T_mu D f.
// Boundary: edge-replicate extension in D, exact matrix transpose in D^T:
// for the symmetric filters h0, h2 the transpose is the flipped filter with edge-replicate extension
// of alpha, for the antisymmetric h1 it is the flipped filter with SIGN-FLIPPED replicate extension.
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

extern "C" int tf_apply_fused(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz,
                              void *stream) {
    CBCT_TRY(tf_check(d_in, d_out, nx, ny, nz));
    if (d_in == d_out || !(mu >= 0.f)) return CBCT_E_INVALID;
    dim3 grid(cdiv(nx, FT_X), cdiv(ny, FT_Y), cdiv(nz, FT_Z));
    tf_fused_kernel<<<grid, 256, 0, as_stream(stream)>>>(d_in, d_out, mu, clamp_nonneg, nx, ny, nz);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
