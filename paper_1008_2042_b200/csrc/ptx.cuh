// ptx.cuh -- every line of inline PTX the library uses, in one place: shared-memory addressing, mbarriers,
// bulk-tensor (TMA) copies and reductions, shared-memory loads / integer reductions with immediate offsets.
// Kernels call these wrappers and contain no `asm` of their own.  (Classic include guard on purpose: the CPU
// test shim under tests/cpu_shim pre-defines the guard and supplies emulations with the same names, so the
// kernel sources compile unchanged for the host-side checks; nothing here knows about the shim.)
#ifndef CBCT_PTX_CUH_
#define CBCT_PTX_CUH_
#include <cuda.h>
#include <cuda_runtime.h>

namespace cbct {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- mbarrier (one CTA) --------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// One bounded poll of the barrier's phase (the instruction itself blocks for a hardware-defined time slice at most):
// true once the phase with the given parity has completed.  There is NO unbounded wait in this library: callers loop
// over this against %globaltimer (tma_common.cuh: mbar_wait_bounded) and leave through the error path on expiry.
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ---- TMA: 3-D tiled tensor copy global -> shared, tensor reduction shared -> global ------------------------
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tma_reduce_add_3d(const CUtensorMap *map, int c0, int c1, int c2, unsigned src) {
    asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map),
                 "r"(src), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- shared-memory accesses by 32-bit shared address, neighbour offsets as immediates ----------------------------
__device__ __forceinline__ float lds_f32(unsigned addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
template <int OFF>
__device__ __forceinline__ float lds_f32_off(unsigned addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(addr), "n"(OFF));
    return v;
}
__device__ __forceinline__ void red_s32(unsigned addr, int v) { asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
template <int OFF>
__device__ __forceinline__ void red_s32_off(unsigned addr, int v) {
    asm volatile("red.shared.add.s32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "r"(v) : "memory");
}

__device__ __forceinline__ void red_u64(unsigned addr, unsigned long long v) {
    asm volatile("red.shared.add.u64 [%0], %1;" ::"r"(addr), "l"(v) : "memory");
}
// the eight corner reductions of one trilinear sample (box pitches BF, BF * BS) for the lanes whose predicate holds; the
// others sit all eight instructions out under one branch
template <int BF, int BS>
__device__ __forceinline__ void red_s32_x8_if(unsigned addr, const int (&v)[8], bool pred) {
    if (pred) {
        red_s32_off<0>(addr, v[0]);                    red_s32_off<4>(addr, v[1]);
        red_s32_off<4 * BF>(addr, v[2]);               red_s32_off<4 * BF + 4>(addr, v[3]);
        red_s32_off<4 * BF * BS>(addr, v[4]);          red_s32_off<4 * BF * BS + 4>(addr, v[5]);
        red_s32_off<4 * BF * BS + 4 * BF>(addr, v[6]); red_s32_off<4 * BF * BS + 4 * BF + 4>(addr, v[7]);
    }
}

// ---- global load that bypasses L1 (micro-benchmark of the L2) ----------------------------------------------------------------
__device__ __forceinline__ float4 ldg_cg_f4(const float4 *p) {
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// ---- packed fp32 pairs (sm_100: FFMA2 / FADD2 work on two fp32 lanes of a 64-bit register pair per instruction) -----------
// Each lane is an IEEE fp32 operation with the stated rounding: results are bit-identical to the scalar instructions.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2_rd(f32x2 a, f32x2 b) { f32x2 d; asm("add.rm.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }   // towards -inf

}  // namespace cbct
#endif  // CBCT_PTX_CUH_
