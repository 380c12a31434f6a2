// tma_common.cuh -- pieces shared by the two TMA-staged projector kernels (forward_tma.cu: boxes of the volume are
// LOADED into shared memory; backproject_tma.cu: boxes of accumulators are REDUCED back into global memory):
// the pixel-tile / chunk planning (which voxel box covers samples k0..k0+kc-1 of a 16x16 pixel tile), mbarrier and
// the tensor-map encoder (the mbarrier / bulk-tensor PTX wrappers are in ptx.cuh).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"

namespace cbct {

constexpr int FT_TU = 16, FT_TV = 16, FT_THREADS = 256, FT_KCMAX = 64;
constexpr float FT_MAGIC = 8388608.0f;          // 2^23: x + 2^23 rounded down has floor(x) in its low mantissa bits
constexpr unsigned FT_MAGIC_BITS = 0x4B000000u;

struct RayL { float cf, cs, cz, bf, bs, bz; };  // ray in (fast, slow, z) index coordinates: P(tau) = c + b tau

struct Box3 { int lf, ls, lz; bool fits; };

// origin of the box for samples tau_a..tau_b of the tile (AABB of the 4 corner rays at both ends grown by
// `margin`), and whether its extents (+1 for the upper neighbour) fit the fixed box (bfs x bfs x bzz)
__device__ __forceinline__ Box3 chunk_box(const RayL *corner, float tau_a, float tau_b, float margin, int bfs, int bss, int bzz) {
    float mnf = 1e30f, mns = 1e30f, mnz = 1e30f, mxf = -1e30f, mxs = -1e30f, mxz = -1e30f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const RayL r = corner[c];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const float tau = e ? tau_b : tau_a;
            const float F = fmaf(r.bf, tau, r.cf), S = fmaf(r.bs, tau, r.cs), Z = fmaf(r.bz, tau, r.cz);
            mnf = fminf(mnf, F); mxf = fmaxf(mxf, F);
            mns = fminf(mns, S); mxs = fmaxf(mxs, S);
            mnz = fminf(mnz, Z); mxz = fmaxf(mxz, Z);
        }
    }
    Box3 b;
    // TMA: the innermost start coordinate must keep the global address 16-byte aligned -> multiple of 4
    b.lf = ((int)floorf(mnf - margin)) & ~3; b.ls = (int)floorf(mns - margin); b.lz = (int)floorf(mnz - margin);
    const int hf = (int)floorf(mxf + margin) + 1, hs = (int)floorf(mxs + margin) + 1, hz = (int)floorf(mxz + margin) + 1;
    b.fits = (hf - b.lf + 1 <= bfs) && (hs - b.ls + 1 <= bss) && (hz - b.lz + 1 <= bzz);
    return b;
}

struct ChunkPlan { int kc; Box3 box; float tau_base; };

__device__ __forceinline__ ChunkPlan plan_chunk(const DevGeom &g, const RayL *corner, int k0, int K1, float margin, int bfs,
                                                int bss, int bzz) {
    ChunkPlan p;
    p.tau_base = (float)(g.tau0 + (double)k0 * g.step);
    const float stepf = (float)g.step;
    int kc = min(FT_KCMAX, K1 - k0 + 1);
    for (;;) {
        p.box = chunk_box(corner, p.tau_base, fmaf((float)(kc - 1), stepf, p.tau_base), margin, bfs, bss, bzz);
        if (p.box.fits || kc == 1) break;
        kc = (kc > 8) ? (kc * 3) >> 2 : kc - 1;            // 64, 48, 36, 27, 20, 15, 11, 8, 7, ...
    }
    p.kc = kc;
    return p;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static inline EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            (void)cudaGetLastError();
    }
    return fn;
}

// tensor map of a [n2][n1][n0] volume of 4-byte elements (n0 fastest) with a (b0, b1, b2) box; loads zero-fill
// out-of-range elements, reductions / stores skip them
static inline bool make_map(CUtensorMap *m, const void *ptr, int n0, int n1, int n2, int b0, int b1, int b2,
                            CUtensorMapDataType dtype = CU_TENSOR_MAP_DATA_TYPE_FLOAT32) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)n0, (cuuint64_t)n1, (cuuint64_t)n2};
    const cuuint64_t strides[2] = {(cuuint64_t)n0 * 4, (cuuint64_t)n0 * n1 * 4};
    const cuuint32_t box[3] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2};
    const cuuint32_t estr[3] = {1, 1, 1};
    return fn(m, dtype, 3, const_cast<void *>(ptr), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace cbct
