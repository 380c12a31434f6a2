// forward_tma.cu -- g = P f, the sm_100a fast path of cbct_forward (include/cbct.h).
// Same arithmetic as forward.cu (Eq. 1 as a fixed-step sum of zero-padded trilinear
// samples); what changes is how the volume reaches the SM:
//   * a CTA owns a 16(u) x 16(v) pixel tile of one view and marches the global t-grid in chunks;
//   * for every chunk ONE thread issues a TMA tensor copy (cp.async.bulk.tensor.3d) of the fixed-size
//     voxel box that covers the tile's frustum segment; out-of-range coordinates are zero-filled by the
//     TMA unit, which IS the zero padding of T.  Two boxes are in flight (mbarrier double buffering),
//     so staging costs no instructions and overlaps the sampling of the previous chunk;
//   * views whose detector u-axis is closer to y than to x read a y-fastest copy of the volume
//     (transposed once per call), so that the 16 pixels of a half-warp always fall on neighbouring
//     words of the fastest shared-memory axis (bank-conflict free for every view direction);
//   * floor/fraction use the add-magic-number trick in round-down mode (no conversion instructions)
//     and positions are kept relative to the box origin.
#include <cmath>
#include <cstdio>
#include <cstring>

#include "tma_common.cuh"

namespace cbct {


__device__ __forceinline__ float fetch0g(const float *__restrict__ vol, const DevGeom &g, int ix, int iy, int iz) {
    if ((unsigned)ix >= (unsigned)g.nx || (unsigned)iy >= (unsigned)g.ny || (unsigned)iz >= (unsigned)g.nz) return 0.f;
    return __ldg(vol + ((size_t)iz * g.ny + iy) * g.nx + ix);
}

// BF, BS > 0: box pitches known at compile time (neighbour loads use immediate offsets); 0: run-time pitches.
// PK: the sample arithmetic on packed fp32 pairs (FFMA2 / FADD2, ptx.cuh), two consecutive samples of the ray per pair:
// positions, floors, fractions, element index and the seven lerps are all pair instructions.  Every lane is the same IEEE
// operation in the same order as the scalar path, so both variants return bit-identical projections.
template <int BF, int BS, bool PK>
__global__ void __launch_bounds__(FT_THREADS, 3) forward_tma_kernel(DevGeom g, const __grid_constant__ CUtensorMap map_x,
                                                                 const __grid_constant__ CUtensorMap map_y,
                                                                 const float *__restrict__ vol, float *__restrict__ proj,
                                                                 float margin, int bfs, int bss, int bzz, DevErr err, NormOut norm) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2];
    __shared__ RayL corner[4];
    __shared__ ChunkPlan plans[2];
    __shared__ int s_klo, s_khi, s_abort;
    float *buf0 = reinterpret_cast<float *>(align128(smem_raw));   // the launch reserves 128 bytes for this
    const int box_elems = (bfs * bss * bzz + 31) & ~31;   // buffer stride: keeps the second buffer 128-byte aligned
    const unsigned box_bytes = (unsigned)(bfs * bss * bzz) * 4u;
    const unsigned tx_bytes = box_bytes + (CBCT_FAULT(1) ? 16u : 0u);      // CBCT_FAULT: 0 outside the host-side test build

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // a warp covers 8(u) x 4(v) pixels: <= 10 columns of the fast axis, <= 2 rows, <= 2 z-planes
    const int tu = (warp & 1) * 8 + (lane & 7), tv = (warp >> 1) * 4 + (lane >> 3);
    const int iu = blockIdx.x * FT_TU + tu, iv = blockIdx.y * FT_TV + tv, view = g.view_order[blockIdx.z];
    const bool valid = iu < g.nu && iv < g.nv;

    // orientation: the detector u-axis is e_u = (-sin, cos); the fast shared-memory axis follows it
    const double2 cs = g.view_cs[view];
    const bool yfast = fabs(cs.x) > fabs(cs.y);

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

    if (tid == 0) {
        s_klo = 0x7fffffff; s_khi = -1;
        s_abort = *reinterpret_cast<volatile int *>(err.dev);      // an earlier CTA / call already failed: do nothing
        mbar_init(smem_u32(&bars[0]), 1); mbar_init(smem_u32(&bars[1]), 1);
        fence_mbar_init();
    }
    if ((tu == 0 || tu == FT_TU - 1) && (tv == 0 || tv == FT_TV - 1)) corner[(tv ? 2 : 0) + (tu ? 1 : 0)] = rl;
    __syncthreads();
    if (s_abort) return;
    {
        const int wlo = __reduce_min_sync(0xffffffffu, klo), whi = __reduce_max_sync(0xffffffffu, khi);
        if (lane == 0) { atomicMin(&s_klo, wlo); atomicMax(&s_khi, whi); }
    }
    __syncthreads();
    const int K0 = s_klo, K1 = s_khi;
    const float stepf = (float)g.step;
    const float sF = rl.bf * stepf, sS = rl.bs * stepf, sZ = rl.bz * stepf;
    const int pS = BF > 0 ? BF : bfs, pZ = BF > 0 ? BF * BS : bfs * bss;
    float total = 0.f;

    if (K0 <= K1) {
        // thread 0 plans every chunk (box origin, length), issues its TMA copy and publishes the plan
        if (tid == 0) {
            const ChunkPlan p0 = plan_chunk(g, corner, K0, K1, margin, bfs, bss, bzz);
            plans[0] = p0;
            if (p0.box.fits) {
                mbar_expect_tx(smem_u32(&bars[0]), tx_bytes);
                if (yfast) tma_load_3d(smem_u32(buf0), &map_y, p0.box.lf, p0.box.ls, p0.box.lz, smem_u32(&bars[0]));
                else tma_load_3d(smem_u32(buf0), &map_x, p0.box.lf, p0.box.ls, p0.box.lz, smem_u32(&bars[0]));
            }
        }
        __syncthreads();
        unsigned phase0 = 0, phase1 = 0;
        int k0 = K0, stage = 0;
        bool failed = false;
        while (k0 <= K1) {
            const ChunkPlan cur = plans[stage];
            const int kn = k0 + cur.kc;
            bool next_in_flight = false;                 // thread 0: a copy into the other buffer has been issued
            if (tid == 0 && kn <= K1) {                  // the other buffer and plan slot were released by the barrier below
                const ChunkPlan nx_ = plan_chunk(g, corner, kn, K1, margin, bfs, bss, bzz);
                plans[stage ^ 1] = nx_;
                if (nx_.box.fits) {
                    next_in_flight = true;
                    const unsigned bar = smem_u32(&bars[stage ^ 1]);
                    mbar_expect_tx(bar, tx_bytes);
                    const unsigned dst = smem_u32(buf0 + (stage ^ 1) * box_elems);
                    if (yfast) tma_load_3d(dst, &map_y, nx_.box.lf, nx_.box.ls, nx_.box.lz, bar);
                    else tma_load_3d(dst, &map_x, nx_.box.lf, nx_.box.ls, nx_.box.lz, bar);
                }
            }
            const int ja = max(k0, klo), jb = min(kn - 1, khi);
            if (cur.box.fits) {
                if (!mbar_wait_bounded(smem_u32(&bars[stage]), stage ? phase1 : phase0)) {
                    failed = true;                        // the box never arrived: error status, no hang
                    raise_device_error(err, DEV_ERR_WAIT_TIMEOUT);
                }
                if (stage) phase1 ^= 1; else phase0 ^= 1;
                if (ja <= jb && !failed) {
                    // local coordinates: sample j sits at F0 + (j - ja) * sF, etc.
                    const float tau_a = fmaf((float)(ja - k0), stepf, cur.tau_base);
                    const float F0 = fmaf(rl.bf, tau_a, rl.cf - (float)cur.box.lf);
                    const float S0 = fmaf(rl.bs, tau_a, rl.cs - (float)cur.box.ls);
                    const float Z0 = fmaf(rl.bz, tau_a, rl.cz - (float)cur.box.lz);
                    // byte address = base + 4*(iF + pS*iS + pZ*iZ); the element index is formed exactly in fp32
                    // (< 2^24) from the floors that the fractions need anyway, then converted once
                    const unsigned base_r = smem_u32(buf0 + stage * box_elems);
                    const float pSf = (float)pS, pZf = (float)pZ;
                    float part = 0.f, jf = 0.f;
                    const int n = jb - ja + 1;
                    if (!(run_inside(F0, sF, n, bfs) && run_inside(S0, sS, n, bss) && run_inside(Z0, sZ, n, bzz))) {
                        raise_device_error(err, DEV_ERR_FW_RANGE);      // never index outside the box: skip, report
                    } else if constexpr (PK && BF > 0) {
                        // Two samples (j, j+1) per iteration, one in each lane of a pair: positions, floors, fractions, the
                        // element index and all seven lerps are pair instructions.  The two contributions are added to `part`
                        // one after the other, so the sum is formed in the scalar stream's order.
                        const f32x2 sF2 = pack2(sF, sF), sS2 = pack2(sS, sS), sZ2 = pack2(sZ, sZ);
                        const f32x2 F02 = pack2(F0, F0), S02 = pack2(S0, S0), Z02 = pack2(Z0, Z0);
                        const f32x2 magic2 = pack2(FT_MAGIC, FT_MAGIC), neg_magic2 = pack2(-FT_MAGIC, -FT_MAGIC);
                        const f32x2 pS2 = pack2(pSf, pSf), pZ2 = pack2(pZf, pZf), two2 = pack2(2.f, 2.f);
                        f32x2 jj = pack2(0.f, 1.f);
                        int j = 0;
#pragma unroll 1
                        for (; j + 1 < n; j += 2, jj = add2(jj, two2)) {
                            const f32x2 F = fma2(jj, sF2, F02), S = fma2(jj, sS2, S02), Z = fma2(jj, sZ2, Z02);
                            const f32x2 rF = add2(add2_rd(F, magic2), neg_magic2), rS = add2(add2_rd(S, magic2), neg_magic2),
                                        rZ = add2(add2_rd(Z, magic2), neg_magic2);                 // floors, exact
                            const f32x2 wF = sub2(F, rF), wS = sub2(S, rS), wZ = sub2(Z, rZ);
                            float ia, ib;
                            unpack2(fma2(rZ, pZ2, fma2(rS, pS2, rF)), ia, ib);
                            const unsigned aA = base_r + 4u * (unsigned)__float2int_rn(ia), aB = base_r + 4u * (unsigned)__float2int_rn(ib);
                            // pairs over the two samples
                            const f32x2 v000 = pack2(lds_f32_off<0>(aA), lds_f32_off<0>(aB));
                            const f32x2 v100 = pack2(lds_f32_off<4>(aA), lds_f32_off<4>(aB));
                            const f32x2 v010 = pack2(lds_f32_off<4 * BF>(aA), lds_f32_off<4 * BF>(aB));
                            const f32x2 v110 = pack2(lds_f32_off<4 * BF + 4>(aA), lds_f32_off<4 * BF + 4>(aB));
                            const f32x2 v001 = pack2(lds_f32_off<4 * BF * BS>(aA), lds_f32_off<4 * BF * BS>(aB));
                            const f32x2 v101 = pack2(lds_f32_off<4 * BF * BS + 4>(aA), lds_f32_off<4 * BF * BS + 4>(aB));
                            const f32x2 v011 = pack2(lds_f32_off<4 * BF * BS + 4 * BF>(aA), lds_f32_off<4 * BF * BS + 4 * BF>(aB));
                            const f32x2 v111 = pack2(lds_f32_off<4 * BF * BS + 4 * BF + 4>(aA), lds_f32_off<4 * BF * BS + 4 * BF + 4>(aB));
                            const f32x2 a00 = fma2(wF, sub2(v100, v000), v000), a10 = fma2(wF, sub2(v110, v010), v010);
                            const f32x2 a01 = fma2(wF, sub2(v101, v001), v001), a11 = fma2(wF, sub2(v111, v011), v011);
                            const f32x2 b0 = fma2(wS, sub2(a10, a00), a00), b1 = fma2(wS, sub2(a11, a01), a01);
                            float cA, cB;
                            unpack2(fma2(wZ, sub2(b1, b0), b0), cA, cB);
                            part += cA;
                            part += cB;
                            if (CBCT_FAULT(16)) part += 1e-3f;      // test build only: a packed stream that is NOT the scalar one
                        }
                        if (j < n) {                                                                   // odd count: the last sample alone
                            jf = (float)j;
                            const f32x2 FS = fma2(pack2(jf, jf), pack2(sF, sS), pack2(F0, S0));
                            const float Z = fmaf(jf, sZ, Z0);
                            const f32x2 rFS = add2(add2_rd(FS, magic2), neg_magic2);
                            const float rz = __fadd_rd(Z, FT_MAGIC) - FT_MAGIC;
                            const f32x2 wFS = sub2(FS, rFS);
                            const float wz = Z - rz;
                            float rf, rs, wf, ws;
                            unpack2(rFS, rf, rs); unpack2(wFS, wf, ws);
                            const unsigned a0 = base_r + 4u * (unsigned)__float2int_rn(fmaf(rz, pZf, fmaf(rs, pSf, rf)));
                            // pairs over z: (lower plane, upper plane)
                            const f32x2 p00 = pack2(lds_f32_off<0>(a0), lds_f32_off<4 * BF * BS>(a0));
                            const f32x2 p10 = pack2(lds_f32_off<4>(a0), lds_f32_off<4 * BF * BS + 4>(a0));
                            const f32x2 p01 = pack2(lds_f32_off<4 * BF>(a0), lds_f32_off<4 * BF * BS + 4 * BF>(a0));
                            const f32x2 p11 = pack2(lds_f32_off<4 * BF + 4>(a0), lds_f32_off<4 * BF * BS + 4 * BF + 4>(a0));
                            const f32x2 wf2 = pack2(wf, wf), ws2 = pack2(ws, ws);
                            const f32x2 a0x = fma2(wf2, sub2(p10, p00), p00), a1x = fma2(wf2, sub2(p11, p01), p01);
                            float b0, b1;
                            unpack2(fma2(ws2, sub2(a1x, a0x), a0x), b0, b1);
                            part += fmaf(wz, b1 - b0, b0);
                        }
                    } else {
#pragma unroll 2
                    for (int j = 0; j < n; ++j, jf += 1.f) {
                        const float F = fmaf(jf, sF, F0), S = fmaf(jf, sS, S0), Z = fmaf(jf, sZ, Z0);
                        const float qf = __fadd_rd(F, FT_MAGIC), qs = __fadd_rd(S, FT_MAGIC), qz = __fadd_rd(Z, FT_MAGIC);
                        const float rf = qf - FT_MAGIC, rs = qs - FT_MAGIC, rz = qz - FT_MAGIC;      // floors, exact
                        const float wf = F - rf, ws = S - rs, wz = Z - rz;
                        const unsigned idx = (unsigned)__float2int_rn(fmaf(rz, pZf, fmaf(rs, pSf, rf)));
                        const unsigned a0 = base_r + 4u * idx;
                        float v000, v100, v010, v110, v001, v101, v011, v111;
                        if constexpr (BF > 0) {
                            v000 = lds_f32_off<0>(a0);                    v100 = lds_f32_off<4>(a0);
                            v010 = lds_f32_off<4 * BF>(a0);               v110 = lds_f32_off<4 * BF + 4>(a0);
                            v001 = lds_f32_off<4 * BF * BS>(a0);          v101 = lds_f32_off<4 * BF * BS + 4>(a0);
                            v011 = lds_f32_off<4 * BF * BS + 4 * BF>(a0); v111 = lds_f32_off<4 * BF * BS + 4 * BF + 4>(a0);
                        } else {
                            const unsigned a1 = a0 + 4u * pS, a2 = a0 + 4u * pZ, a3 = a2 + 4u * pS;
                            v000 = lds_f32(a0); v100 = lds_f32_off<4>(a0);
                            v010 = lds_f32(a1); v110 = lds_f32_off<4>(a1);
                            v001 = lds_f32(a2); v101 = lds_f32_off<4>(a2);
                            v011 = lds_f32(a3); v111 = lds_f32_off<4>(a3);
                        }
                        const float a00 = fmaf(wf, v100 - v000, v000), a10 = fmaf(wf, v110 - v010, v010);
                        const float a01 = fmaf(wf, v101 - v001, v001), a11 = fmaf(wf, v111 - v011, v011);
                        const float b0 = fmaf(ws, a10 - a00, a00), b1 = fmaf(ws, a11 - a01, a01);
                        part += fmaf(wz, b1 - b0, b0);
                    }
                    }
                    total += part;
                }
            } else if (ja <= jb) {
                // a chunk whose box does not fit even for one sample: read the volume directly
                float part = 0.f;
                for (int j = ja; j <= jb; ++j) {
                    const float tau = fmaf((float)(j - k0), stepf, cur.tau_base);
                    const float X = fmaf(r.bx, tau, r.cx), Y = fmaf(r.by, tau, r.cy), Z = fmaf(r.bz, tau, r.cz);
                    const float fxf = floorf(X), fyf = floorf(Y), fzf = floorf(Z);
                    const int ix = (int)fxf, iy = (int)fyf, iz = (int)fzf;
                    const float wx = X - fxf, wy = Y - fyf, wz = Z - fzf;
                    const float v000 = fetch0g(vol, g, ix, iy, iz), v100 = fetch0g(vol, g, ix + 1, iy, iz);
                    const float v010 = fetch0g(vol, g, ix, iy + 1, iz), v110 = fetch0g(vol, g, ix + 1, iy + 1, iz);
                    const float v001 = fetch0g(vol, g, ix, iy, iz + 1), v101 = fetch0g(vol, g, ix + 1, iy, iz + 1);
                    const float v011 = fetch0g(vol, g, ix, iy + 1, iz + 1), v111 = fetch0g(vol, g, ix + 1, iy + 1, iz + 1);
                    const float a00 = fmaf(wx, v100 - v000, v000), a10 = fmaf(wx, v110 - v010, v010);
                    const float a01 = fmaf(wx, v101 - v001, v001), a11 = fmaf(wx, v111 - v011, v011);
                    const float b0 = fmaf(wy, a10 - a00, a00), b1 = fmaf(wy, a11 - a01, a01);
                    part += fmaf(wz, b1 - b0, b0);
                }
                total += part;
            }
            // everyone is done with buffer `stage`; next plan is visible; did anybody give up?
            if (__syncthreads_or(failed ? 1 : 0)) {
                // leave through the normal exit path, but not while a copy into this CTA's shared memory may still land
                if (tid == 0 && next_in_flight) (void)mbar_wait_bounded(smem_u32(&bars[stage ^ 1]), (stage ^ 1) ? phase1 : phase0);
                break;
            }
            k0 = kn; stage ^= 1;
        }
    }
    const float qv = total * stepf;
    if (valid) proj[((size_t)view * g.nv + iv) * g.nu + iu] = qv;
    if (norm.out) {                                        // ||q||^2 of this launch (CGLS step 2), fixed summation order
        __shared__ double sh[8];
        __shared__ bool last;
        double tot;
        const unsigned bid = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
        if (ordered_total_at(valid ? (double)qv * qv : 0.0, norm.partials, norm.counter, sh, &last, tot, tid, FT_THREADS, bid,
                             gridDim.x * gridDim.y * gridDim.z))
            *norm.out = tot;
    }
}

// volT[z][x][y] = vol[z][y][x]
__global__ void __launch_bounds__(256) transpose_vol_kernel(const float *__restrict__ v, float *__restrict__ vT, int nx, int ny) {
    __shared__ float tile[32][33];
    const size_t base = (size_t)blockIdx.z * nx * ny;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int x = x0 + threadIdx.x, y = y0 + j;
        if (x < nx && y < ny) tile[j][threadIdx.x] = __ldg(v + base + (size_t)y * nx + x);
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int x = x0 + j, y = y0 + threadIdx.x;
        if (x < nx && y < ny) vT[base + (size_t)x * ny + y] = tile[threadIdx.x][j];
    }
}


typedef void (*TmaKernel)(DevGeom, const CUtensorMap, const CUtensorMap, const float *, float *, float, int, int, int, DevErr, NormOut);
static TmaKernel tma_kernel_ptr(int bf, int bs, bool pk) {
#define CBCT_FK(F, S) if (bf == F && bs == S) return pk ? forward_tma_kernel<F, S, true> : forward_tma_kernel<F, S, false>;
    CBCT_FK(24, 22) CBCT_FK(40, 30) CBCT_FK(40, 38) CBCT_FK(56, 46) CBCT_FK(56, 54)
#undef CBCT_FK
    return nullptr;
}

// two boxes (each a multiple of 128 bytes) + 128 bytes for the in-kernel alignment of the base
static size_t fw_tma_smem_bytes(int bf, int bs, int bz) { return (size_t)2 * ((bf * bs * bz + 31) & ~31) * 4 + 128; }
constexpr size_t FW_TMA_SMEM_MAX = 97 * 1024;        // two boxes of <= 48 KiB: two CTAs per SM

// choose the box for this geometry (once, at create); fw_tma_ok = 0 when the TMA path cannot be used
void plan_forward_tma(cbct_geometry *G) {
    const cbct_geometry_desc &d = G->desc;
    G->fw_tma_ok = 0;
    if (d.nx % 4 || d.ny % 4) return;                            // TMA global strides must be multiples of 16 bytes
    const double far = (d.sad + G->R) / d.sdd;
    const double half_diag = 0.5 * std::sqrt((FT_TU * d.du) * (FT_TU * d.du) + (FT_TV * d.dv) * (FT_TV * d.dv));
    const double psi = half_diag / d.sdd, vmin = std::fmin(d.dx, std::fmin(d.dy, d.dz));
    const double margin = (d.sad + G->R) * 0.5 * psi * psi / vmin + 0.02;      // sphere-patch sagitta + rounding slack
    if (margin > 2.0) return;
    const double vxy = std::fmin(d.dx, d.dy);
    const double wl = FT_TU * d.du * far / vxy, wv = FT_TV * d.dv * far;       // tile footprint: lateral (voxels), vertical (mm)
    const double tilt = std::fmax(std::fabs(d.v0) + 0.5 * d.nv * d.dv, 1e-9) / d.sdd;   // |tan| of the steepest ray
    const int kc_goal = 24;
    const double travel = kc_goal * G->step / vxy;
    const int bz = (int)std::ceil(wv / d.dz + kc_goal * G->step * tilt / d.dz + 2 * margin) + 2;
    int bxy = (int)std::ceil(0.7072 * (wl + travel + wv * tilt / vxy) + 2 * margin) + 4 + 3;   // +3: 4-aligned box origin
    // Bank = (F + pitch*S + pitch*rows*Z) mod 32.  A warp's 8x4 pixels span <= 10 columns F, <= 2 rows S and
    // <= 2 planes Z, so a pitch of +-8 (mod 32) and a plane pitch of 16 (mod 32) keep its 32 lanes in distinct
    // banks (or on the same word) for every view direction: pitch in {24, 40, 56}, rows = 2 (mod 4).
    const int need_f = bxy, need_s = bxy - 3;
    int bf = 0, bs = 0;
    const int menu[][2] = {{24, 22}, {40, 30}, {40, 38}, {56, 46}, {56, 54}};   // compiled instantiations
    for (auto &m : menu)
        if (m[0] >= need_f && m[1] >= need_s) { bf = m[0]; bs = m[1]; break; }
    if (!bf || bz > 32) return;
    if (fw_tma_smem_bytes(bf, bs, bz) > FW_TMA_SMEM_MAX) return;
    G->fw_b = bf; G->fw_bs = bs; G->fw_bz = bz; G->fw_margin = (float)margin;
    if (cudaMalloc(&G->d_fw_volT, sizeof(float) * G->n_vox) != cudaSuccess) { (void)cudaGetLastError(); G->d_fw_volT = nullptr; return; }
    G->workspace_bytes += sizeof(float) * G->n_vox;
    {   // ||q||^2 in the kernel's epilogue: one fp64 partial per CTA
        const size_t n_cta = (size_t)cdiv(d.nu, FT_TU) * cdiv(d.nv, FT_TV) * d.n_views;
        if (cudaMalloc(&G->d_fw_norm_partials, sizeof(double) * n_cta) != cudaSuccess ||
            cudaMalloc(&G->d_fw_norm_counter, sizeof(unsigned int)) != cudaSuccess ||
            cudaMemset(G->d_fw_norm_counter, 0, sizeof(unsigned int)) != cudaSuccess) { (void)cudaGetLastError(); return; }
        G->workspace_bytes += sizeof(double) * n_cta;
    }
    static_assert(sizeof(CUtensorMap) <= sizeof(G->fw_map_y), "tensor map storage");
    CUtensorMap m;
    if (!make_map(&m, G->d_fw_volT, d.ny, d.nx, d.nz, bf, bs, bz)) return;
    std::memcpy(G->fw_map_y, &m, sizeof(m));
    for (int pk = 0; pk < 2; ++pk) {
        const void *kern = reinterpret_cast<const void *>(tma_kernel_ptr(bf, bs, pk != 0));
        // the attribute belongs to the kernel, not to the handle: always the plan's limit, never this geometry's need
        if (!kern || cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FW_TMA_SMEM_MAX) != cudaSuccess) {
            (void)cudaGetLastError();
            return;
        }
    }
    G->fw_tma_ok = 1;
}

int launch_forward_tma(const cbct_geometry *G, const float *d_vol, float *d_proj, cudaStream_t st, double *d_norm) {
    if (!G->fw_tma_ok) return CBCT_E_UNSUPPORTED;
    if (reinterpret_cast<uintptr_t>(d_vol) & 15) return CBCT_E_INVALID;        // include/cbct.h: device pointers are 16-byte aligned
    const DevGeom &g = G->dg;
    CUtensorMap mx, my;
    if (!make_map(&mx, d_vol, g.nx, g.ny, g.nz, G->fw_b, G->fw_bs, G->fw_bz)) return CBCT_E_UNSUPPORTED;
    std::memcpy(&my, G->fw_map_y, sizeof(my));
    {
        dim3 block(32, 8), grid(cdiv(g.nx, 32), cdiv(g.ny, 32), g.nz);
        transpose_vol_kernel<<<grid, block, 0, st>>>(d_vol, G->d_fw_volT, g.nx, g.ny);
        CBCT_LAUNCH_CHECK();
    }
    const size_t smem = fw_tma_smem_bytes(G->fw_b, G->fw_bs, G->fw_bz);
    dim3 grid(cdiv(g.nu, FT_TU), cdiv(g.nv, FT_TV), g.n_views);
    TmaKernel kern = tma_kernel_ptr(G->fw_b, G->fw_bs, G->fw_packed != 0);
    if (!kern) return CBCT_E_UNSUPPORTED;
    kern<<<grid, FT_THREADS, smem, st>>>(g, mx, my, d_vol, d_proj, G->fw_margin, G->fw_b, G->fw_bs, G->fw_bz, G->err,
                                        NormOut{d_norm, G->d_fw_norm_partials, G->d_fw_norm_counter});
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// "forward_tma_kernel<40,30,packed> box 40x30x7" -- what cbct_geometry_describe reports for P
void describe_forward_tma(const cbct_geometry *G, char *buf, size_t cap) {
    snprintf(buf, cap, "forward_tma_kernel<%d,%d,%s> box %dx%dx%d", G->fw_b, G->fw_bs, G->fw_packed ? "packed" : "scalar", G->fw_b,
             G->fw_bs, G->fw_bz);
}

}  // namespace cbct
