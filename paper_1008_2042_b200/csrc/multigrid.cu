// multigrid.cu -- grid transfer operators (§2.2.3) and Algorithm A2 step 1
// (PAPER.md:165).  Readings: SURVEY.md §8(c) items 11, 20, 22.
#include "common.cuh"

namespace cbct {

// fine[i] = 3/4 coarse[i>>1] + 1/4 coarse[nearer neighbour, clamped]   (cell-centred linear)
__global__ void __launch_bounds__(256) mg_prolong_kernel(const float *__restrict__ coarse, float *__restrict__ fine,
                                                         int nxf, int nyf, int nzf, int fx, int fy, int fz) {
    const long long n = (long long)nxf * nyf * nzf;
    const int nxc = nxf / fx, nyc = nyf / fy, nzc = nzf / fz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % nxf), y = (int)((i / nxf) % nyf), z = (int)(i / ((long long)nxf * nyf));
        int xa, xb, ya, yb, za, zb;
        float wxb, wyb, wzb;
        if (fx == 2) { xa = x >> 1; xb = (x & 1) ? min(xa + 1, nxc - 1) : max(xa - 1, 0); wxb = 0.25f; } else { xa = xb = x; wxb = 0.f; }
        if (fy == 2) { ya = y >> 1; yb = (y & 1) ? min(ya + 1, nyc - 1) : max(ya - 1, 0); wyb = 0.25f; } else { ya = yb = y; wyb = 0.f; }
        if (fz == 2) { za = z >> 1; zb = (z & 1) ? min(za + 1, nzc - 1) : max(za - 1, 0); wzb = 0.25f; } else { za = zb = z; wzb = 0.f; }
        const float wxa = 1.f - wxb, wya = 1.f - wyb, wza = 1.f - wzb;
        auto at = [&](int zz, int yy, int xx) { return __ldg(coarse + ((size_t)zz * nyc + yy) * nxc + xx); };
        const float r00 = wxa * at(za, ya, xa) + wxb * at(za, ya, xb);
        const float r01 = wxa * at(za, yb, xa) + wxb * at(za, yb, xb);
        const float r10 = wxa * at(zb, ya, xa) + wxb * at(zb, ya, xb);
        const float r11 = wxa * at(zb, yb, xa) + wxb * at(zb, yb, xb);
        fine[i] = wza * (wya * r00 + wyb * r01) + wzb * (wya * r10 + wyb * r11);
    }
}

// The same operator, four fine voxels of one row per thread (float4 store), 32-bit indices, no integer division: the
// launch is (x-quads, rows, planes).  Round 1 measured the kernel above at 0.10 of the HBM roofline (64-bit div / mod per
// voxel, scalar stores); it remains the path for row lengths that are not a multiple of 4 or misaligned buffers.
template <int FX>
__device__ __forceinline__ float4 prolong_row4(const float *__restrict__ row, int q, int nxc) {
    if (FX == 2) {                                    // fine x = 4q .. 4q+3  <-  coarse 2q-1 .. 2q+2 (clamped)
        const int c = 2 * q;
        const float m = __ldg(row + max(c - 1, 0)), a = __ldg(row + c), b = __ldg(row + c + 1), p = __ldg(row + min(c + 2, nxc - 1));
        return make_float4(0.75f * a + 0.25f * m, 0.75f * a + 0.25f * b, 0.75f * b + 0.25f * a, 0.75f * b + 0.25f * p);
    }
    return __ldg(reinterpret_cast<const float4 *>(row) + q);
}
__device__ __forceinline__ float4 mix4(float wa, float4 a, float wb, float4 b) {
    return make_float4(wa * a.x + wb * b.x, wa * a.y + wb * b.y, wa * a.z + wb * b.z, wa * a.w + wb * b.w);
}
template <int FX>
__global__ void __launch_bounds__(256) mg_prolong4_kernel(const float *__restrict__ coarse, float *__restrict__ fine,
                                                          int nxf, int nyf, int nzf, int fy, int fz) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y;
    if (4 * q >= nxf || y >= nyf) return;
    const int nxc = nxf / FX, nyc = nyf / fy, nzc = nzf / fz;
    int ya, yb;
    float wyb;
    if (fy == 2) { ya = y >> 1; yb = (y & 1) ? min(ya + 1, nyc - 1) : max(ya - 1, 0); wyb = 0.25f; } else { ya = yb = y; wyb = 0.f; }
    const float wya = 1.f - wyb;
    for (int z = blockIdx.z; z < nzf; z += gridDim.z) {
        int za, zb;
        float wzb;
        if (fz == 2) { za = z >> 1; zb = (z & 1) ? min(za + 1, nzc - 1) : max(za - 1, 0); wzb = 0.25f; } else { za = zb = z; wzb = 0.f; }
        const float *pa = coarse + (size_t)za * nyc * nxc, *pb = coarse + (size_t)zb * nyc * nxc;
        float4 r = mix4(wya, prolong_row4<FX>(pa + (size_t)ya * nxc, q, nxc), wyb, prolong_row4<FX>(pa + (size_t)yb * nxc, q, nxc));
        if (fz == 2) r = mix4(1.f - wzb, r, wzb, mix4(wya, prolong_row4<FX>(pb + (size_t)ya * nxc, q, nxc), wyb,
                                                       prolong_row4<FX>(pb + (size_t)yb * nxc, q, nxc)));
        reinterpret_cast<float4 *>(fine + ((size_t)z * nyf + y) * nxf)[q] = r;
    }
}

// coarse = mean of the children, four coarse voxels of one row per thread (float4 loads of the fine rows, float4 store)
template <int FX>
__global__ void __launch_bounds__(256) mg_restrict4_kernel(const float *__restrict__ fine, float *__restrict__ coarse,
                                                           int nxf, int nyf, int nzf, int fy, int fz) {
    const int nxc = nxf / FX, nyc = nyf / fy, nzc = nzf / fz;
    const int q = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y;
    if (4 * q >= nxc || y >= nyc) return;
    const float scale = 1.f / (float)(FX * fy * fz);
    for (int z = blockIdx.z; z < nzc; z += gridDim.z) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int c = 0; c < fz; ++c)
            for (int b = 0; b < fy; ++b) {
                const float4 *row = reinterpret_cast<const float4 *>(fine + ((size_t)(z * fz + c) * nyf + (y * fy + b)) * nxf);
                if (FX == 2) {
                    const float4 u = __ldg(row + 2 * q), v = __ldg(row + 2 * q + 1);
                    acc.x += u.x + u.y; acc.y += u.z + u.w; acc.z += v.x + v.y; acc.w += v.z + v.w;
                } else {
                    const float4 u = __ldg(row + q);
                    acc.x += u.x; acc.y += u.y; acc.z += u.z; acc.w += u.w;
                }
            }
        reinterpret_cast<float4 *>(coarse + ((size_t)z * nyc + y) * nxc)[q] =
            make_float4(acc.x * scale, acc.y * scale, acc.z * scale, acc.w * scale);
    }
}

// coarse = mean of the fx*fy*fz children
__global__ void __launch_bounds__(256) mg_restrict_kernel(const float *__restrict__ fine, float *__restrict__ coarse,
                                                          int nxf, int nyf, int nzf, int fx, int fy, int fz) {
    const int nxc = nxf / fx, nyc = nyf / fy, nzc = nzf / fz;
    const long long n = (long long)nxc * nyc * nzc;
    const float scale = 1.f / (float)(fx * fy * fz);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % nxc), y = (int)((i / nxc) % nyc), z = (int)(i / ((long long)nxc * nyc));
        float acc = 0.f;
        for (int c = 0; c < fz; ++c)
            for (int b = 0; b < fy; ++b)
                for (int a = 0; a < fx; ++a)
                    acc += __ldg(fine + ((size_t)(z * fz + c) * nyf + (y * fy + b)) * nxf + (x * fx + a));
        coarse[i] = acc * scale;
    }
}

// v = f_cur + coef (f_cur - f_prev)
__global__ void __launch_bounds__(256) extrapolate_kernel(const float *__restrict__ fc, const float *__restrict__ fp,
                                                          float *__restrict__ v, float coef, long long n) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float c = fc[i];
        v[i] = fmaf(coef, c - fp[i], c);
    }
}

static int mg_check(const void *a, const void *b, int nx, int ny, int nz, int fx, int fy, int fz) {
    if (!a || !b || nx <= 0 || ny <= 0 || nz <= 0) return CBCT_E_INVALID;
    if ((fx != 1 && fx != 2) || (fy != 1 && fy != 2) || (fz != 1 && fz != 2)) return CBCT_E_INVALID;
    if (nx % fx || ny % fy || nz % fz) return CBCT_E_INVALID;
    return device_supported();
}
static inline bool aligned16(const void *a, const void *b) {
    return ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b)) & 15) == 0;
}
static inline int vec_planes(int nz) { return nz < 64 ? nz : 64; }        // blockIdx.z strides over the planes
static inline int gs_blocks(long long n) {
    long long b = (n + 255) / 256;
    if (b > 148LL * 32) b = 148LL * 32;
    return (int)(b < 1 ? 1 : b);
}

}  // namespace cbct

using namespace cbct;

extern "C" int mg_restrict(const float *d_fine, float *d_coarse, int nx_f, int ny_f, int nz_f, int fx, int fy, int fz,
                           void *stream) {
    CBCT_TRY(mg_check(d_fine, d_coarse, nx_f, ny_f, nz_f, fx, fy, fz));
    const long long n = (long long)(nx_f / fx) * (ny_f / fy) * (nz_f / fz);
    const int nxc = nx_f / fx;
    if (nxc % 4 == 0 && aligned16(d_fine, d_coarse)) {                    // rows of float4 on both sides
        dim3 block(32, 8), grid(cdiv(nxc / 4, 32), cdiv(ny_f / fy, 8), vec_planes(nz_f / fz));
        if (fx == 2) mg_restrict4_kernel<2><<<grid, block, 0, as_stream(stream)>>>(d_fine, d_coarse, nx_f, ny_f, nz_f, fy, fz);
        else mg_restrict4_kernel<1><<<grid, block, 0, as_stream(stream)>>>(d_fine, d_coarse, nx_f, ny_f, nz_f, fy, fz);
    } else {
        mg_restrict_kernel<<<gs_blocks(n), 256, 0, as_stream(stream)>>>(d_fine, d_coarse, nx_f, ny_f, nz_f, fx, fy, fz);
    }
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int mg_prolong(const float *d_coarse, float *d_fine, int nx_f, int ny_f, int nz_f, int fx, int fy, int fz,
                          void *stream) {
    CBCT_TRY(mg_check(d_coarse, d_fine, nx_f, ny_f, nz_f, fx, fy, fz));
    const long long n = (long long)nx_f * ny_f * nz_f;
    if (nx_f % 4 == 0 && aligned16(d_coarse, d_fine) && (fx == 2 || (nx_f / fx) % 4 == 0)) {
        dim3 block(32, 8), grid(cdiv(nx_f / 4, 32), cdiv(ny_f, 8), vec_planes(nz_f));
        if (fx == 2) mg_prolong4_kernel<2><<<grid, block, 0, as_stream(stream)>>>(d_coarse, d_fine, nx_f, ny_f, nz_f, fy, fz);
        else mg_prolong4_kernel<1><<<grid, block, 0, as_stream(stream)>>>(d_coarse, d_fine, nx_f, ny_f, nz_f, fy, fz);
    } else {
        mg_prolong_kernel<<<gs_blocks(n), 256, 0, as_stream(stream)>>>(d_coarse, d_fine, nx_f, ny_f, nz_f, fx, fy, fz);
    }
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int cbct_a2_extrapolate(const float *d_f_cur, const float *d_f_prev, float *d_v, float coef, int64_t n,
                                   void *stream) {
    if (!d_f_cur || !d_f_prev || !d_v || n <= 0) return CBCT_E_INVALID;
    CBCT_TRY(device_supported());
    extrapolate_kernel<<<gs_blocks(n), 256, 0, as_stream(stream)>>>(d_f_cur, d_f_prev, d_v, coef, (long long)n);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
