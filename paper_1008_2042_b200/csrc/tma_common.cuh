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

// ---- "cannot hang, cannot fault" guards of the two TMA kernels ------------------------------------------------------------
// (1) Every wait on an mbarrier is bounded by %globaltimer: on expiry the CTA raises DEV_ERR_WAIT_TIMEOUT and leaves
//     through the normal exit path (a wrong transaction count or a lost copy becomes an error status, not a hung SM).
// (2) Before a thread touches the shared-memory box of a chunk it checks that its FIRST and LAST sample of the chunk lie
//     inside the box (positions are fma(j, s, P0): monotone in j, so the two ends bound every sample between them); a
//     thread whose samples would leave the box raises DEV_ERR_*_RANGE and skips the chunk, so a planning mistake can
//     never become an out-of-range shared-memory access.
// (3) The dynamic shared-memory base is rounded up to 128 bytes in the kernel (TMA boxes need it), not assumed.
constexpr unsigned long long CBCT_WAIT_NS = 200ull * 1000ull * 1000ull;      // 0.2 s: a box copy takes microseconds

// Deliberate protocol mistakes, compiled ONLY into the host-side test build (tests/cpu_shim defines CBCT_TEST_FAULTS;
// the product build never does, CBCT_FAULT(..) is the constant 0 there): they prove that the guards above turn a wrong
// transaction count / a mis-planned box into an error status instead of a hang / an out-of-range access.
#ifdef CBCT_TEST_FAULTS
extern "C" int cbct_test_fault;      // 1: expect_tx announces 16 bytes too many; 2 / 4: forward / scatter box origin shifted; 8: head-room plan ignored; 16: packed forward stream perturbed
#define CBCT_FAULT(bit) (cbct_test_fault & (bit))
#else
#define CBCT_FAULT(bit) 0
#endif

__device__ __forceinline__ void raise_device_error(const DevErr &e, int code) {
    atomicOr(e.dev, code);
    *reinterpret_cast<volatile int *>(e.host) = code;      // mapped pinned host word: the next entry point sees it without a sync
    __threadfence_system();
}

__device__ __forceinline__ bool mbar_wait_bounded(unsigned bar, unsigned parity) {
    if (mbar_try_wait(bar, parity)) return true;
    const unsigned long long t0 = globaltimer_ns();
    for (;;) {
#pragma unroll 1
        for (int i = 0; i < 16; ++i)
            if (mbar_try_wait(bar, parity)) return true;
        if (globaltimer_ns() - t0 > CBCT_WAIT_NS) return false;
    }
}

__device__ __forceinline__ unsigned char *align128(unsigned char *p) {
    return p + ((128u - (smem_u32(p) & 127u)) & 127u);
}

// samples j = 0..n-1 at P0 + j*s: do all floors lie in [0, ext-2] (so that floor and floor+1 are inside the box)?
__device__ __forceinline__ bool run_inside(float P0, float s, int n, int ext) {
    const float Pe = fmaf((float)(n - 1), s, P0);
    const float lo = fminf(P0, Pe), hi = fmaxf(P0, Pe);
    return lo >= 0.f && hi < (float)(ext - 1);
}

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
    if (CBCT_FAULT(2 | 4)) p.box.ls += 5;                  // test build only: a box that does not cover its samples
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
