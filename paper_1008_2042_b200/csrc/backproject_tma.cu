// backproject_tma.cu -- f = P^T g, the sm_100a fast path of cbct_backproject (include/cbct.h).
// The exact transpose of forward_tma.cu, organised as its mirror image (PAPER.md:211 names the obstacle --
// write conflicts of a ray-driven scatter -- which is removed here by hardware, not by changing the operator):
//   * a CTA owns the same 16(u) x 16(v) pixel tile of one view and marches the same chunks of the global
//     t-grid, with the same fp32 sample positions and trilinear weights as the forward kernel;
//   * instead of reading 8 voxels per sample from a TMA-loaded box it ADDS g * weight to the 8 voxels of an
//     accumulator box in shared memory.  The accumulators are 32-bit FIXED POINT: shared-memory integer
//     atomics (ATOMS.ADD) run at the rate of plain shared stores on sm_100a, whereas a float atomicAdd on shared
//     memory compiles to a compare-and-swap loop (3x slower, measured).  Integer addition is associative, so
//     the result does not depend on the order of the atomics: P^T is deterministic;
//   * a finished box is added to a global int32 accumulator volume by ONE TMA tensor reduction
//     (cp.reduce.async.bulk.tensor.3d ... .add, element type s32); elements outside the volume are skipped
//     by the TMA unit, which is the transpose of the forward kernel's zero fill.  Two boxes alternate, so the
//     reduction of one chunk overlaps the scattering of the next;
//   * a last pass converts the accumulators to fp32 (x step / scale) with coalesced float4 stores.
// Fixed point: every ray value is scaled by S = 2^qb / T, T = min(max|g|, 8 rms(g)) (both reduced on the device per
// call, in a fixed order), each contribution S g w is rounded to the nearest integer by one FFMA onto 1.5 * 2^23, and
// qb is chosen at geometry-create so that the largest possible voxel sum of a view group stays below 2^30.  The
// rounding error per contribution is uniform in +-T / 2^(qb+1) (qb = 21 at the paper-size config): relative to the
// result at most ~5e-6 even for white noise (where the result itself is small by cancellation), ~1e-7 for projections.
// Rays with |g| > T (outliers of a heavy-tailed input, e.g. CGLS residuals of low-count Poisson data; none for ordinary
// projections, where max|g| < 8 rms) are left out by the scatter kernel and added by backproject_outlier_kernel with
// their own, coarser unit T 2^m / 2^qb, 2^m >= |g| / T: the same RELATIVE precision for them, and the unit of all
// other rays no longer grows with the single largest value.
#include <cmath>
#include <cstdio>
#include <cstring>

#include "tma_common.cuh"

namespace cbct {

constexpr float BT_ROUND = 12582912.0f;          // 1.5 * 2^23: x + BT_ROUND holds round(x) in its low mantissa bits, |x| < 2^22
constexpr int BT_ROUND_BITS = 0x4B400000;

// integer nearest to c = a*b (|c| < 2^22), in one FFMA + one IADD
__device__ __forceinline__ int round_mul(float a, float b) { return __float_as_int(fmaf(a, b, BT_ROUND)) - BT_ROUND_BITS; }

// max |g| as the bit pattern of a non-negative float (orders like an unsigned integer); *out zeroed before.
// The maximum is taken on the bit patterns, so an Inf or NaN anywhere in g wins (their patterns exceed every finite
// one): the scatter kernels then contribute nothing and the finalize pass multiplies by a non-finite factor, i.e. a
// non-finite input gives an all-NaN volume instead of finite garbage.
__global__ void __launch_bounds__(256) absmax_kernel(const float *__restrict__ g, long long n, unsigned *out) {
    unsigned m = 0u;
    const bool vec = (reinterpret_cast<uintptr_t>(g) & 15) == 0;          // float4 loads only from a 16-byte aligned base
    const long long n4 = vec ? n >> 2 : 0;
    const float4 *g4 = reinterpret_cast<const float4 *>(g);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
        const float4 v = __ldg(g4 + i);
        m = max(max(m, __float_as_uint(fabsf(v.x))), max(__float_as_uint(fabsf(v.y)), max(__float_as_uint(fabsf(v.z)), __float_as_uint(fabsf(v.w)))));
    }
    for (long long i = (n4 << 2) + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        m = max(m, __float_as_uint(fabsf(__ldg(g + i))));
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// Bank conflicts decide the speed of this kernel (it is bound by shared-memory wavefronts: two lanes of one
// ATOMS that fall on the same bank -- same word or not -- cost one extra wavefront each).  Lane layouts and
// box pitches were searched with a CPU model of the cfg-4 geometry that reproduces the ncu wavefront counts:
//   LM 0: a warp = 8(u) x 4(v) pixels, the lane group of row r works 2r samples ahead of row 0 (its samples are
//         one voxel further along the ray = one box row = +8 banks), box pitch = 8 (mod 32), plane pitch = 0
//         (mod 32): 2.2 wavefronts per ATOMS;
//   LM 1: a warp = 16(u) x 2(v), rows 8 apart (their samples lie in different z-planes), no skew, the forward
//         kernel's box (pitch 8, plane pitch 16 mod 32): 2.9 wavefronts per ATOMS (model) / 2.96 (ncu).
// LM 0 is the default (verified against the oracle by executing this source on the host, tests/cpu_shim, whose bank statistics
// reproduce LM 1's measured 2.96 and give 2.25 for LM 0, 2.0 with the same-cell merging of the packed stream below: ~12 ms
// predicted from LM 1's measured 17.6 ms); CBCT_BT_LANES=1 selects LM 1.
// The order in which a thread visits the samples of a chunk is free: integer sums do not depend on it.
template <int BF, int BS, int LM, bool PK>
__global__ void __launch_bounds__(FT_THREADS) backproject_scatter_kernel(DevGeom g, const __grid_constant__ CUtensorMap map_x,
                                                                         const __grid_constant__ CUtensorMap map_y,
                                                                         const float *__restrict__ proj, int *__restrict__ acc_x,
                                                                         const unsigned *__restrict__ absmax_bits, float two_qb,
                                                                         int view0, float margin, int bzz, DevErr err) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ RayL corner[4];
    __shared__ ChunkPlan plans[2];
    __shared__ int s_klo, s_khi, s_abort;
    constexpr int bfs = BF, bss = BS;
    int *buf0 = reinterpret_cast<int *>(align128(smem_raw));      // the launch reserves 128 bytes for this
    const int box_words = bfs * bss * bzz;
    const int box_elems = (box_words + 31) & ~31;          // buffer stride: keeps the second buffer 128-byte aligned

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int tu, tv;
    if constexpr (LM == 0) { tu = (warp & 1) * 8 + (lane & 7); tv = (warp >> 1) * 4 + (lane >> 3); }
    else { tu = lane & 15; tv = warp + 8 * (lane >> 4); }
    const int skew = LM == 0 ? 2 * (lane >> 3) : 0;
    const int iu = blockIdx.x * FT_TU + tu, iv = blockIdx.y * FT_TV + tv, view = g.view_order[view0 + blockIdx.z];
    const bool valid = iu < g.nu && iv < g.nv;

    const double2 cs = g.view_cs[view];
    const bool yfast = fabs(cs.x) > fabs(cs.y);             // same orientation rule as forward_tma_kernel

    RayF r;
    double b[3], c[3];
    ray_setup(g, view, iv, iu, r, b[0], b[1], b[2], c[0], c[1], c[2]);
    int klo = 0x7fffffff, khi = -1;
    if (valid) {
        const double hi[3] = {(double)g.nx, (double)g.ny, (double)g.nz};
        double tin = -1e300, tout = 1e300;
        bool miss = false;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (b[a] == 0.0) { miss |= (c[a] <= -1.0 || c[a] >= hi[a]); continue; }
            const double inv = 1.0 / b[a];
            double t1 = (-1.0 - c[a]) * inv, t2 = (hi[a] - c[a]) * inv;
            if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
            tin = fmax(tin, t1); tout = fmin(tout, t2);
        }
        if (!miss && tout > tin) {
            const long long a = (long long)ceil((tin - g.tau0) / g.step), e = (long long)floor((tout - g.tau0) / g.step);
            klo = (int)max(a, 0LL); khi = (int)min(e, (long long)g.K - 1);
            if (khi < klo) { klo = 0x7fffffff; khi = -1; }
        }
    }
    RayL rl;
    rl.cf = yfast ? r.cy : r.cx; rl.cs = yfast ? r.cx : r.cy; rl.cz = r.cz;
    rl.bf = yfast ? r.by : r.bx; rl.bs = yfast ? r.bx : r.by; rl.bz = r.bz;

    // ray value in fixed-point units: |gs| <= 2^qb
    const float amax = __uint_as_float(__ldg(absmax_bits));           // the caller passes the reference T (bt_reference_kernel)
    const float scale = (amax > 0.f && amax <= 3.0e38f) ? two_qb / amax : 0.f;      // non-finite reference: contribute nothing (finalize writes NaN)
    float gs = valid ? __ldg(proj + ((size_t)view * g.nv + iv) * g.nu + iu) * scale : 0.f;
    if (!(fabsf(gs) <= two_qb)) gs = 0.f;                   // an outlier (|g| > T): backproject_outlier_kernel adds it

    if (tid == 0) { s_klo = 0x7fffffff; s_khi = -1; s_abort = *reinterpret_cast<volatile int *>(err.dev); }
    if ((tu == 0 || tu == FT_TU - 1) && (tv == 0 || tv == FT_TV - 1)) corner[(tv ? 2 : 0) + (tu ? 1 : 0)] = rl;
    {   // both accumulator boxes start at zero
        int4 *z = reinterpret_cast<int4 *>(buf0);
        for (int i = tid; i < (2 * box_elems) >> 2; i += FT_THREADS) z[i] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    {
        const int wlo = __reduce_min_sync(0xffffffffu, klo), whi = __reduce_max_sync(0xffffffffu, khi);
        if (lane == 0) { atomicMin(&s_klo, wlo); atomicMax(&s_khi, whi); }
    }
    __syncthreads();
    const int K0 = s_klo, K1 = s_khi;
    if (K0 > K1 || s_abort) return;                           // nothing to do / an earlier CTA or call already failed
    const float stepf = (float)g.step;
    const float sF = rl.bf * stepf, sS = rl.bs * stepf, sZ = rl.bz * stepf;
    constexpr int pS = BF, pZ = BF * BS;

    if (tid == 0) plans[0] = plan_chunk(g, corner, K0, K1, margin, bfs, bss, bzz);
    __syncthreads();
    int k0 = K0, stage = 0;
    bool first = true;
    while (k0 <= K1) {
        const ChunkPlan cur = plans[stage];
        const int kn = k0 + cur.kc;
        if (tid == 0 && kn <= K1) plans[stage ^ 1] = plan_chunk(g, corner, kn, K1, margin, bfs, bss, bzz);
        const int ja = max(k0, klo), jb = min(kn - 1, khi);
        if (cur.box.fits) {
            if (ja <= jb) {
                const float tau_a = fmaf((float)(ja - k0), stepf, cur.tau_base);
                const float F0 = fmaf(rl.bf, tau_a, rl.cf - (float)cur.box.lf);
                const float S0 = fmaf(rl.bs, tau_a, rl.cs - (float)cur.box.ls);
                const float Z0 = fmaf(rl.bz, tau_a, rl.cz - (float)cur.box.lz);
                const unsigned base_r = smem_u32(buf0 + stage * box_elems);
                const float pSf = (float)pS, pZf = (float)pZ;
                const int n = jb - ja + 1;
                if (!(run_inside(F0, sF, n, bfs) && run_inside(S0, sS, n, bss) && run_inside(Z0, sZ, n, bzz))) {
                    raise_device_error(err, DEV_ERR_BT_RANGE);          // never index outside the box: skip, report
                } else if constexpr (PK) {
                    // Packed pairs (FFMA2 / FADD2 / FMUL2), two consecutive samples per pair, as in forward_tma_kernel: the
                    // positions, floors and fractions are bit-identical to the forward kernel's.  The thread starts `skew`
                    // samples ahead (kept even, so pairs never straddle the wrap-around) and visits [s0, n) then [0, s0).
                    const f32x2 sF2 = pack2(sF, sF), sS2 = pack2(sS, sS), sZ2 = pack2(sZ, sZ);
                    const f32x2 F02 = pack2(F0, F0), S02 = pack2(S0, S0), Z02 = pack2(Z0, Z0);
                    const f32x2 magic2 = pack2(FT_MAGIC, FT_MAGIC), neg_magic2 = pack2(-FT_MAGIC, -FT_MAGIC);
                    const f32x2 pS2 = pack2(pSf, pSf), pZ2 = pack2(pZf, pZf), two2 = pack2(2.f, 2.f);
                    const f32x2 gs2 = pack2(gs, gs), one2 = pack2(1.f, 1.f), round2 = pack2(BT_ROUND, BT_ROUND);
                    const int s0 = (skew < n ? skew : skew % n) & ~1;
#pragma unroll 1
                    for (int seg = 0; seg < 2; ++seg) {
                        int j = seg ? 0 : s0;
                        const int end = seg ? s0 : n;
                        f32x2 jj = pack2((float)j, (float)j + 1.f);
#pragma unroll 1
                        for (; j + 1 < end; j += 2, jj = add2(jj, two2)) {
                            const f32x2 F = fma2(jj, sF2, F02), S = fma2(jj, sS2, S02), Z = fma2(jj, sZ2, Z02);
                            const f32x2 rF = add2(add2_rd(F, magic2), neg_magic2), rS = add2(add2_rd(S, magic2), neg_magic2),
                                        rZ = add2(add2_rd(Z, magic2), neg_magic2);
                            const f32x2 wF = sub2(F, rF), wS = sub2(S, rS), wZ = sub2(Z, rZ);
                            float ia, ib;
                            unpack2(fma2(rZ, pZ2, fma2(rS, pS2, rF)), ia, ib);
                            const unsigned aA = base_r + 4u * (unsigned)__float2int_rn(ia), aB = base_r + 4u * (unsigned)__float2int_rn(ib);
                            // transposed lerp tree on both samples: split gs along z, then the slow axis, then the fast axis
                            const f32x2 g1 = mul2(gs2, wZ), g0 = sub2(gs2, g1);
                            const f32x2 g01 = mul2(g0, wS), g00 = sub2(g0, g01), g11 = mul2(g1, wS), g10 = sub2(g1, g11);
                            const f32x2 oF = sub2(one2, wF);
                            float cA, cB;
                            // Two consecutive samples are half a voxel apart: where both fall into the same cell the second
                            // one's contributions ride on the first one's reductions, and its own eight are skipped under ONE
                            // branch, which thins out the second half of the instructions (fewer lanes, fewer bank conflicts).
                            const bool same = aA == aB;
                            int vB[8];
#define CBCT_SCATTER2(I, OFF, G, W)                                                                      \
                            unpack2(fma2(G, W, round2), cA, cB);                                         \
                            vB[I] = __float_as_int(cB) - BT_ROUND_BITS;                                  \
                            red_s32_off<OFF>(aA, __float_as_int(cA) - BT_ROUND_BITS + (same ? vB[I] : 0));
                            CBCT_SCATTER2(0, 0, g00, oF) CBCT_SCATTER2(1, 4, g00, wF)
                            CBCT_SCATTER2(2, 4 * BF, g01, oF) CBCT_SCATTER2(3, 4 * BF + 4, g01, wF)
                            CBCT_SCATTER2(4, 4 * BF * BS, g10, oF) CBCT_SCATTER2(5, 4 * BF * BS + 4, g10, wF)
                            CBCT_SCATTER2(6, 4 * BF * BS + 4 * BF, g11, oF) CBCT_SCATTER2(7, 4 * BF * BS + 4 * BF + 4, g11, wF)
                            red_s32_x8_if<BF, BS>(aB, vB, !same);
#undef CBCT_SCATTER2
                        }
                        if (j < end) {                                     // odd count: the last sample of the segment alone
                            const float jf = (float)j;
                            const float F = fmaf(jf, sF, F0), S = fmaf(jf, sS, S0), Z = fmaf(jf, sZ, Z0);
                            const float rf = __fadd_rd(F, FT_MAGIC) - FT_MAGIC, rs = __fadd_rd(S, FT_MAGIC) - FT_MAGIC,
                                        rz = __fadd_rd(Z, FT_MAGIC) - FT_MAGIC;
                            const float wf = F - rf, ws = S - rs, wz = Z - rz;
                            const unsigned a0 = base_r + 4u * (unsigned)__float2int_rn(fmaf(rz, pZf, fmaf(rs, pSf, rf)));
                            const float g1 = __fmul_rn(gs, wz), g0 = gs - g1;
                            const float g01 = __fmul_rn(g0, ws), g00 = g0 - g01, g11 = __fmul_rn(g1, ws), g10 = g1 - g11;
                            const float of = 1.f - wf;
                            red_s32_off<0>(a0, round_mul(g00, of));
                            red_s32_off<4>(a0, round_mul(g00, wf));
                            red_s32_off<4 * BF>(a0, round_mul(g01, of));
                            red_s32_off<4 * BF + 4>(a0, round_mul(g01, wf));
                            red_s32_off<4 * BF * BS>(a0, round_mul(g10, of));
                            red_s32_off<4 * BF * BS + 4>(a0, round_mul(g10, wf));
                            red_s32_off<4 * BF * BS + 4 * BF>(a0, round_mul(g11, of));
                            red_s32_off<4 * BF * BS + 4 * BF + 4>(a0, round_mul(g11, wf));
                        }
                    }
                } else {
                const float nf = (float)n;
                float jf = (float)(skew < n ? skew : skew % n);        // start `skew` samples ahead, wrap around at n
#pragma unroll 2
                for (int j = 0; j < n; ++j) {
                    // identical position / floor / fraction arithmetic to forward_tma_kernel
                    const float F = fmaf(jf, sF, F0), S = fmaf(jf, sS, S0), Z = fmaf(jf, sZ, Z0);
                    const float qf = __fadd_rd(F, FT_MAGIC), qs = __fadd_rd(S, FT_MAGIC), qz = __fadd_rd(Z, FT_MAGIC);
                    const float rf = qf - FT_MAGIC, rs = qs - FT_MAGIC, rz = qz - FT_MAGIC;
                    const float wf = F - rf, ws = S - rs, wz = Z - rz;
                    const unsigned idx = (unsigned)__float2int_rn(fmaf(rz, pZf, fmaf(rs, pSf, rf)));
                    const unsigned a0 = base_r + 4u * idx;
                    // transposed lerp tree: split gs along z, then the slow axis, then the fast axis
                    const float g1 = gs * wz, g0 = gs - g1;
                    const float g01 = g0 * ws, g00 = g0 - g01, g11 = g1 * ws, g10 = g1 - g11;
                    const float of = 1.f - wf;
                    red_s32_off<0>(a0, round_mul(g00, of));
                    red_s32_off<4>(a0, round_mul(g00, wf));
                    red_s32_off<4 * BF>(a0, round_mul(g01, of));
                    red_s32_off<4 * BF + 4>(a0, round_mul(g01, wf));
                    red_s32_off<4 * BF * BS>(a0, round_mul(g10, of));
                    red_s32_off<4 * BF * BS + 4>(a0, round_mul(g10, wf));
                    red_s32_off<4 * BF * BS + 4 * BF>(a0, round_mul(g11, of));
                    red_s32_off<4 * BF * BS + 4 * BF + 4>(a0, round_mul(g11, wf));
                    jf += 1.f;
                    if (jf >= nf) jf -= nf;
                }
                }
            }
            fence_async_smem();                           // my shared-memory writes -> visible to the TMA unit
        } else if (ja <= jb) {
            // a chunk whose box does not fit even for one sample: integer atomics straight on the x-fastest volume
            for (int j = ja; j <= jb; ++j) {
                const float tau = fmaf((float)(j - k0), stepf, cur.tau_base);
                const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
                const float fxf = floorf(X), fyf = floorf(Y), fzf = floorf(Z);
                const int ix = (int)fxf, iy = (int)fyf, iz = (int)fzf;
                const float wx = X - fxf, wy = Y - fyf, wz = Z - fzf;
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) {
                    const int x = ix + (cc & 1), y = iy + ((cc >> 1) & 1), z = iz + (cc >> 2);
                    if ((unsigned)x >= (unsigned)g.nx || (unsigned)y >= (unsigned)g.ny || (unsigned)z >= (unsigned)g.nz) continue;
                    const float w = ((cc & 1) ? wx : 1.f - wx) * ((cc & 2) ? wy : 1.f - wy) * ((cc & 4) ? wz : 1.f - wz);
                    atomicAdd(acc_x + ((size_t)(z + bzz) * (g.ny + bss) + (y + bss)) * (g.nx + bfs) + (x + bfs), round_mul(gs, w));
                }
            }
        }
        if (tid == 0) bulk_wait_read0();                  // the other box's reduction (issued one chunk ago) has read it
        __syncthreads();                                  // A: everyone finished scattering into box `stage`
        if (tid == 0 && cur.box.fits) {
            // The accumulator volumes carry a low-side margin of one box (a tensor reduction may not start at a
            // negative coordinate; elements beyond the high side are skipped by the TMA unit).  A box that starts
            // below the margin, or beyond the high side, lies entirely outside the volume: nothing to add.
            const unsigned src = smem_u32(buf0 + stage * box_elems);
            const int oF = cur.box.lf + bfs, oS = cur.box.ls + bss, oZ = cur.box.lz + bzz;
            const int nF = (yfast ? g.ny : g.nx) + bfs, nS = (yfast ? g.nx : g.ny) + bss, nZ = g.nz + bzz;
            if (oF >= 0 && oS >= 0 && oZ >= 0 && oF < nF && oS < nS && oZ < nZ) {
                if (yfast) tma_reduce_add_3d(&map_y, oF, oS, oZ, src);
                else tma_reduce_add_3d(&map_x, oF, oS, oZ, src);
                bulk_commit();
            }
        }
        if (!first && kn <= K1) {                         // clear the other box for the next chunk
            int4 *z = reinterpret_cast<int4 *>(buf0 + (stage ^ 1) * box_elems);
            for (int i = tid; i < box_elems >> 2; i += FT_THREADS) z[i] = make_int4(0, 0, 0, 0);
        }
        first = false;
        __syncthreads();                                  // B: the cleared box and the next plan are visible
        k0 = kn; stage ^= 1;
    }
    if (tid == 0) bulk_wait0();                           // shared memory must outlive the last reduction
}

// T = min(max|g|, 8 rms(g)) -> ref[1] (bits); a non-finite max|g| is passed on (the volume becomes NaN)
__global__ void bt_reference_kernel(unsigned *ref, const double *sumsq, double n) {
    const float amax = __uint_as_float(ref[0]);
    float t = amax;
    if (amax <= 3.0e38f) {
        const float r8 = (float)(8.0 * sqrt(*sumsq / n));
        if (r8 > 0.f && r8 < amax) t = r8;
    }
    ref[1] = __float_as_uint(t);
}

// The rays the scatter kernel left out (|g| > T).  A warp looks at 32 rays at a time; every outlier among them is then
// sampled by the whole warp (lanes stride over the samples of the ray, same positions and weights as the scatter
// kernel's direct path) and added to the x-fastest accumulator with integer atomics, each contribution rounded to a
// multiple of 2^m units, 2^m >= |g| / T: |g S / 2^m| <= 2^qb keeps the rounding trick in range.
__global__ void __launch_bounds__(256) backproject_outlier_kernel(DevGeom g, const float *__restrict__ proj, int *__restrict__ acc_x,
                                                                  const unsigned *__restrict__ ref, float two_qb, int view0, int n_views,
                                                                  int pf, int ps, int pz) {
    const float t = __uint_as_float(__ldg(ref));
    if (!(t > 0.f && t <= 3.0e38f)) return;
    const float scale = two_qb / t;
    // ray counts fit 31 bits (cbct_geometry_create rejects larger detectors): 32-bit index arithmetic, one division per ray
    const unsigned per_view = (unsigned)g.nv * (unsigned)g.nu, n = per_view * (unsigned)n_views;
    const int lane = threadIdx.x & 31;
    const unsigned warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned base = warp0 * 32; base < n; base += n_warps * 32) {
        const unsigned i = base + lane;
        float gs = 0.f;
        int view = 0, pix = 0;
        if (i < n) {
            const unsigned vpos = i / per_view;
            view = g.view_order[view0 + (int)vpos];
            pix = (int)(i - vpos * per_view);
            gs = __ldg(proj + (size_t)view * per_view + pix) * scale;
        }
        unsigned todo = __ballot_sync(0xffffffffu, i < n && !(fabsf(gs) <= two_qb) && fabsf(gs) <= 3.0e38f);
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            const float gso = __shfl_sync(0xffffffffu, gs, src);
            const int vw = __shfl_sync(0xffffffffu, view, src), px = __shfl_sync(0xffffffffu, pix, src);
            int m = 0;
            float gq = gso;
            while (fabsf(gq) > two_qb && m < 30) { gq *= 0.5f; ++m; }
            RayF r;
            double b[3], c[3];
            ray_setup(g, vw, px / g.nu, px % g.nu, r, b[0], b[1], b[2], c[0], c[1], c[2]);
            const double hi[3] = {(double)g.nx, (double)g.ny, (double)g.nz};
            double tin = -1e300, tout = 1e300;
            bool miss = false;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (b[a] == 0.0) { miss |= (c[a] <= -1.0 || c[a] >= hi[a]); continue; }
                const double inv = 1.0 / b[a];
                double t1 = (-1.0 - c[a]) * inv, t2 = (hi[a] - c[a]) * inv;
                if (t1 > t2) { const double tt = t1; t1 = t2; t2 = tt; }
                tin = fmax(tin, t1); tout = fmin(tout, t2);
            }
            if (miss || !(tout > tin)) continue;
            const long long ka = (long long)ceil((tin - g.tau0) / g.step), ke = (long long)floor((tout - g.tau0) / g.step);
            const int klo = (int)max(ka, 0LL), khi = (int)min(ke, (long long)g.K - 1);
            for (int k = klo + lane; k <= khi; k += 32) {
                // tau exactly as the scatter kernel forms it for a chunk starting at k: base in fp64, rounded once
                const float tau = (float)(g.tau0 + (double)k * g.step);
                const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
                const float fxf = floorf(X), fyf = floorf(Y), fzf = floorf(Z);
                const int ix = (int)fxf, iy = (int)fyf, iz = (int)fzf;
                const float wx = X - fxf, wy = Y - fyf, wz = Z - fzf;
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) {
                    const int x = ix + (cc & 1), y = iy + ((cc >> 1) & 1), z = iz + (cc >> 2);
                    if ((unsigned)x >= (unsigned)g.nx || (unsigned)y >= (unsigned)g.ny || (unsigned)z >= (unsigned)g.nz) continue;
                    const float w = ((cc & 1) ? wx : 1.f - wx) * ((cc & 2) ? wy : 1.f - wy) * ((cc & 4) ? wz : 1.f - wz);
                    atomicAdd(acc_x + ((size_t)(z + pz) * (g.ny + ps) + (y + ps)) * (g.nx + pf) + (x + pf), round_mul(gq, w) * (1 << m));
                }
            }
        }
    }
}

// vol[z][y][x] (+)= (acc_x[z][y][x] + acc_y[z][x][y]) * step * T / 2^qb; 32x32 tiles, the y-fastest accumulator is
// transposed through shared memory so that every global access is a coalesced row
// (both accumulators carry a low-side margin of one box: pf x ps x pz elements, fast axis first)
__global__ void __launch_bounds__(256) backproject_finalize_kernel(const int *__restrict__ acc_x, const int *__restrict__ acc_y,
                                                                   float *__restrict__ vol, int nx, int ny, int pf, int ps, int pz,
                                                                   const unsigned *__restrict__ absmax_bits, float step_over_two_qb,
                                                                   int accumulate, long long sat_limit, DevErr err, NormOut norm) {
    __shared__ int tile[32][33];
    const size_t base = (size_t)blockIdx.z * nx * ny;
    const size_t base_x = ((size_t)(blockIdx.z + pz) * (ny + ps) + ps) * (nx + pf) + pf;     // acc_x[z+pz][ps][pf]
    const size_t base_y = ((size_t)(blockIdx.z + pz) * (nx + ps) + ps) * (ny + pf) + pf;     // acc_y[z+pz][ps][pf]
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const float k = __uint_as_float(__ldg(absmax_bits)) * step_over_two_qb;         // the fixed-point reference of the caller
    double sq = 0.0;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int y = y0 + threadIdx.x, x = x0 + j;
        if (x < nx && y < ny) tile[j][threadIdx.x] = __ldg(acc_y + base_y + (size_t)x * (ny + pf) + y);
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int x = x0 + threadIdx.x, y = y0 + j;
        if (x < nx && y < ny) {
            const size_t o = base + (size_t)y * nx + x;
            const int ax = __ldg(acc_x + base_x + (size_t)y * (nx + pf) + x), ay = tile[threadIdx.x][j];
            // head-room check: a sum that reached sat_limit (half the int32 range for cbct_backproject) means the planned
            // bound on the weight sums does not hold here; report it (a true sum below 3 x sat_limit cannot hide by wrapping)
            const long long wide = (long long)ax + (long long)ay;
            if (wide >= sat_limit || wide <= -sat_limit) {
                atomicOr(err.dev, DEV_ERR_FIXED_POINT);
                *reinterpret_cast<volatile int *>(err.host) = DEV_ERR_FIXED_POINT;
            }
            const float v = (float)wide * k, out = accumulate ? vol[o] + v : v;
            vol[o] = out;
            sq = fma((double)out, (double)out, sq);
        }
    }
    if (norm.out) {                                        // ||s||^2 of the finished volume (CGLS step 5), fixed summation order
        __shared__ double sh[8];
        __shared__ bool last;
        double tot;
        const unsigned bid = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
        if (ordered_total_at(sq, norm.partials, norm.counter, sh, &last, tot, threadIdx.y * 32 + threadIdx.x, 256, bid,
                             gridDim.x * gridDim.y * gridDim.z))
            *norm.out = tot;
    }
}

typedef void (*ScatterKernel)(DevGeom, const CUtensorMap, const CUtensorMap, const float *, int *, const unsigned *, float, int,
                              float, int, DevErr);
// two accumulator boxes (each a multiple of 128 bytes) + 128 bytes for the in-kernel alignment of the base
static size_t bt_smem_bytes(int bf, int bs, int bz) { return (size_t)2 * ((bf * bs * bz + 31) & ~31) * 4 + 128; }
constexpr size_t BT_SMEM_MAX = 101 * 1024;
static ScatterKernel scatter_kernel_ptr(int bf, int bs, int lm, bool pk) {
#define CBCT_SK(F, S, L) \
    if (bf == F && bs == S && lm == L) return pk ? backproject_scatter_kernel<F, S, L, true> : backproject_scatter_kernel<F, S, L, false>;
    CBCT_SK(24, 24, 0) CBCT_SK(40, 32, 0) CBCT_SK(40, 40, 0) CBCT_SK(56, 48, 0) CBCT_SK(56, 56, 0)      // plane pitch = 0 (mod 32)
    CBCT_SK(24, 22, 1) CBCT_SK(40, 30, 1) CBCT_SK(40, 38, 1) CBCT_SK(56, 46, 1) CBCT_SK(56, 54, 1)      // the forward kernel's boxes
#undef CBCT_SK
    return nullptr;
}

// Fixed-point plan of the scatter kernel (host arithmetic only; exported as cbct_backproject_fixed_point_plan).
// w_view is the planned bound on the sum of trilinear weights one voxel can receive from ONE view:
//   * the largest continuum density of sample points, in samples per voxel volume.  The samples are the image of the
//     lattice (iu, iv, k) under  x_S + t (d(u,v) - x_S) / L(u,v),  whose cell has the volume  du dv step t^2 SDD / L^3
//     (t^2 / L^2 from the fan, SDD / L from the incidence on the flat panel): densest at the nearest depth t_min = SAD - R
//     and for the most oblique ray, L_max;  the sum of the hat weights of a voxel is its integral (one voxel volume) times
//     that density, when the lattice is fine against the voxel (measured with the oracle: 0.91 .. 0.98 of this figure at
//     the five configs, tests/test_abi.py);
//   * times, per lattice direction whose pitch exceeds the voxel pitch, that pitch ratio (one sample can sit on the peak
//     of the hat while the mean spreads it over the pitch);
//   * times 1.25.
// Then views_per_group * w_view * 2^qb <= 2^30 with qb <= 22 (the range of the rounding trick): the plan uses HALF the
// int32 range and backproject_finalize_kernel reports any accumulator that reaches 2^30, so a geometry that breaks the
// bound by up to 3x is caught (CBCT_STATUS_FIXED_POINT_RANGE) instead of wrapping silently.
bool bt_fixed_point_plan(const cbct_geometry_desc &d, double R, double step, int *qb_out, int *group_out, double *w_view_out) {
    const double t_min = d.sad - R, far = (d.sad + R) / d.sdd;
    const double umax = std::fabs(d.u0) + 0.5 * d.nu * d.du, vmax = std::fabs(d.v0) + 0.5 * d.nv * d.dv;
    const double l_max = std::sqrt(d.sdd * d.sdd + umax * umax + vmax * vmax);
    const double mean_w = d.dx * d.dy * d.dz * l_max * l_max * l_max / (d.sdd * t_min * t_min * d.du * d.dv * step);
    const double su = std::fmax(1.0, d.du * far / std::fmin(d.dx, d.dy)), sv = std::fmax(1.0, d.dv * far / d.dz);
    const double st = std::fmax(1.0, step / std::fmin(d.dx, std::fmin(d.dy, d.dz)));
    const double w_view = 1.25 * mean_w * su * sv * st;
    int qb = 21, group = d.n_views;
    const auto cap = [&](int bits) { return std::ldexp(1.0, 30 - bits) / w_view; };
    if (cap(22) >= d.n_views) qb = 22;
    else if (cap(21) >= d.n_views) qb = 21;
    else {
        qb = 21;
        while (qb > 12 && cap(qb) < 1.0) --qb;
        if (cap(qb) < 1.0) return false;
        group = (int)std::fmin((double)d.n_views, std::floor(cap(qb)));
    }
    *qb_out = qb; *group_out = group; *w_view_out = w_view;
    return true;
}

void free_backproject_tma(cbct_geometry *G) {
    cudaFree(G->d_bt_acc);
    cudaFree(G->d_bt_absmax);
    cudaFree(G->d_bt_sumsq); cudaFree(G->d_bt_partials); cudaFree(G->d_bt_counter);
    cudaFree(G->d_bt_norm_partials); cudaFree(G->d_bt_norm_counter);
    G->d_bt_norm_partials = nullptr; G->d_bt_norm_counter = nullptr;
    G->d_bt_acc = nullptr; G->d_bt_absmax = nullptr; G->d_bt_sumsq = G->d_bt_partials = nullptr; G->d_bt_counter = nullptr; G->bt_ok = 0;
}

// decide whether the scatter path runs for this geometry; needs the forward TMA box plan (same boxes)
void plan_backproject_tma(cbct_geometry *G) {
    const cbct_geometry_desc &d = G->desc;
    G->bt_ok = 0; G->d_bt_acc = nullptr; G->d_bt_absmax = nullptr;
    G->d_bt_sumsq = G->d_bt_partials = nullptr; G->d_bt_counter = nullptr;
    G->d_bt_norm_partials = nullptr; G->d_bt_norm_counter = nullptr;
    if (!G->fw_tma_ok) return;
    // lane layout G->bt_lm (see the kernel; chosen by cbct_geometry_create): 0 = the skewed 8x4 layout, whose box is the
    // forward kernel's with the row count rounded up to a multiple of 4 (plane pitch = 0 mod 32); 1 = 16x2, forward's box
    G->bt_b = G->fw_b; G->bt_bz = G->fw_bz; G->bt_bs = G->bt_lm == 0 ? (G->fw_bs + 3) & ~3 : G->fw_bs;
    if (bt_smem_bytes(G->bt_b, G->bt_bs, G->bt_bz) > BT_SMEM_MAX) return;
    int qb = 0, group = 0;
    double w_view = 0;
    if (!bt_fixed_point_plan(d, G->R, G->step, &qb, &group, &w_view)) return;
    G->bt_qb = qb; G->bt_group = group;
    const size_t n_acc = (size_t)(d.nx + G->bt_b) * (d.ny + G->bt_bs) * (d.nz + G->bt_bz);      // x-fastest, with margins
    const size_t n_acc_y = (size_t)(d.ny + G->bt_b) * (d.nx + G->bt_bs) * (d.nz + G->bt_bz);    // y-fastest
    G->bt_acc_y_off = (n_acc + 31) & ~(size_t)31;
    G->bt_acc_elems = G->bt_acc_y_off + n_acc_y;
    if (cudaMalloc(&G->d_bt_acc, sizeof(int) * G->bt_acc_elems) != cudaSuccess ||
        cudaMalloc(&G->d_bt_absmax, 2 * sizeof(unsigned)) != cudaSuccess || cudaMalloc(&G->d_bt_sumsq, sizeof(double)) != cudaSuccess ||
        cudaMalloc(&G->d_bt_partials, sizeof(double) * kReduceBlocks) != cudaSuccess ||
        cudaMalloc(&G->d_bt_counter, sizeof(unsigned)) != cudaSuccess || cudaMemset(G->d_bt_counter, 0, sizeof(unsigned)) != cudaSuccess ||
        cudaMalloc(&G->d_bt_norm_partials, sizeof(double) * (size_t)cdiv(d.nx, 32) * cdiv(d.ny, 32) * d.nz) != cudaSuccess ||
        cudaMalloc(&G->d_bt_norm_counter, sizeof(unsigned int)) != cudaSuccess ||
        cudaMemset(G->d_bt_norm_counter, 0, sizeof(unsigned int)) != cudaSuccess) {
        (void)cudaGetLastError();
        free_backproject_tma(G);
        return;
    }
    G->workspace_bytes += sizeof(int) * G->bt_acc_elems + sizeof(unsigned);
    CUtensorMap mx, my;
    if (!make_map(&mx, G->d_bt_acc, d.nx + G->bt_b, d.ny + G->bt_bs, d.nz + G->bt_bz, G->bt_b, G->bt_bs, G->bt_bz,
                  CU_TENSOR_MAP_DATA_TYPE_INT32) ||
        !make_map(&my, G->d_bt_acc + G->bt_acc_y_off, d.ny + G->bt_b, d.nx + G->bt_bs, d.nz + G->bt_bz, G->bt_b, G->bt_bs, G->bt_bz,
                  CU_TENSOR_MAP_DATA_TYPE_INT32)) {
        free_backproject_tma(G);
        return;
    }
    std::memcpy(G->bt_map_x, &mx, sizeof(mx));
    std::memcpy(G->bt_map_y, &my, sizeof(my));
    for (int pk = 0; pk < 2; ++pk) {
        ScatterKernel k = scatter_kernel_ptr(G->bt_b, G->bt_bs, G->bt_lm, pk != 0);
        // the attribute belongs to the kernel, not to the handle: always the plan's limit, never this geometry's need
        if (!k || cudaFuncSetAttribute(reinterpret_cast<const void *>(k), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BT_SMEM_MAX) !=
                      cudaSuccess) {
            (void)cudaGetLastError();
            free_backproject_tma(G);
            return;
        }
    }
    G->bt_ok = 1;
}

int launch_backproject_tma(const cbct_geometry *G, const float *d_proj, float *d_vol, cudaStream_t st, double *d_norm) {
    if (!G->bt_ok) return CBCT_E_UNSUPPORTED;
    const DevGeom &g = G->dg;
    CUtensorMap mx, my;
    std::memcpy(&mx, G->bt_map_x, sizeof(mx));
    std::memcpy(&my, G->bt_map_y, sizeof(my));
    ScatterKernel kern = scatter_kernel_ptr(G->bt_b, G->bt_bs, G->bt_lm, G->bt_packed != 0);
    if (!kern) return CBCT_E_UNSUPPORTED;
    CBCT_CUDA_TRY(cudaMemsetAsync(G->d_bt_absmax, 0, 2 * sizeof(unsigned), st));
    absmax_kernel<<<592, 256, 0, st>>>(d_proj, (long long)G->n_rays, G->d_bt_absmax);
    CBCT_LAUNCH_CHECK();
    CBCT_TRY(launch_sumsq(d_proj, G->n_rays, G->d_bt_sumsq, G->d_bt_partials, G->d_bt_counter, st));
    bt_reference_kernel<<<1, 1, 0, st>>>(G->d_bt_absmax, G->d_bt_sumsq, (double)G->n_rays);       // T = min(max|g|, 8 rms(g))
    CBCT_LAUNCH_CHECK();
    const size_t smem = bt_smem_bytes(G->bt_b, G->bt_bs, G->bt_bz);
    // CBCT_FAULT: 0 outside the host-side test build; there, 8 = ignore the head-room plan (all views in one group)
    const int qb = G->bt_qb, group = CBCT_FAULT(8) ? g.n_views : G->bt_group;
    const float two_qb = (float)std::ldexp(1.0, qb);
    for (int v0 = 0; v0 < g.n_views; v0 += group) {          // view0 / blockIdx.z are positions in g.view_order
        const int nv_ = std::min(group, g.n_views - v0);
        CBCT_CUDA_TRY(cudaMemsetAsync(G->d_bt_acc, 0, sizeof(int) * G->bt_acc_elems, st));
        dim3 grid(cdiv(g.nu, FT_TU), cdiv(g.nv, FT_TV), nv_);
        kern<<<grid, FT_THREADS, smem, st>>>(g, mx, my, d_proj, G->d_bt_acc, G->d_bt_absmax + 1, two_qb, v0, G->fw_margin, G->bt_bz, G->err);
        CBCT_LAUNCH_CHECK();
        backproject_outlier_kernel<<<296, 256, 0, st>>>(g, d_proj, G->d_bt_acc, G->d_bt_absmax + 1, two_qb, v0, nv_, G->bt_b, G->bt_bs, G->bt_bz);
        CBCT_LAUNCH_CHECK();
        dim3 fb(32, 8), fg(cdiv(g.nx, 32), cdiv(g.ny, 32), g.nz);
        backproject_finalize_kernel<<<fg, fb, 0, st>>>(G->d_bt_acc, G->d_bt_acc + G->bt_acc_y_off, d_vol, g.nx, g.ny, G->bt_b, G->bt_bs,
                                                       G->bt_bz, G->d_bt_absmax + 1,
                                                       (float)(G->step / std::ldexp(1.0, qb)), v0 > 0 ? 1 : 0, 1LL << 30, G->err,
                                                       NormOut{v0 + nv_ >= g.n_views ? d_norm : nullptr, G->d_bt_norm_partials, G->d_bt_norm_counter});
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}

void describe_backproject_tma(const cbct_geometry *G, char *buf, size_t cap) {
    snprintf(buf, cap, "backproject_scatter_kernel<%d,%d,LM%d,%s> box %dx%dx%d qb %d views/group %d", G->bt_b, G->bt_bs, G->bt_lm,
             G->bt_packed ? "packed" : "scalar", G->bt_b, G->bt_bs, G->bt_bz, G->bt_qb, G->bt_group);
}

}  // namespace cbct
