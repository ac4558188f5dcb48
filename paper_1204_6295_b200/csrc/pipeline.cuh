// pipeline.cuh -- mbarrier + TMA (cp.async.bulk) primitives for the shared-memory staging pipelines (sm_100a).
//
// The streaming kernels keep NS stages of input rows/slices in flight per CTA: one elected thread arms a
// "full" mbarrier with the expected byte count and issues the bulk copies (the TMA engine moves the bytes, no
// registers are tied up and the bytes in flight do not depend on occupancy); consumers wait on the barrier's
// phase parity, read the stage from shared memory and release it through an "empty" mbarrier.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace disc {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
// make the barrier initialisation visible to the async (TMA) proxy
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Arrive that cannot be issued before `dep0` has been computed.  A consumer releases a buffer with it: shared-memory
// loads still in flight when the producer overwrites the buffer are a race (seen on B200 with a plain arrive right
// after the loads), and an arrive without a register dependency may be scheduled ahead of the instructions that
// consume the loaded values.  dep0 = (a register computed from ALL loaded values) & (a run-time zero the compiler
// cannot fold, see rt_zero()); it is added to the barrier address.
__device__ __forceinline__ void mbar_arrive_after(uint64_t* bar, uint32_t dep0) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar) + dep0) : "memory");
}
// 0 for every legal volume (n < 2^30), opaque to the compiler
__device__ __forceinline__ uint32_t rt_zero(int n) { return (uint32_t)n >> 30; }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// 1-D bulk copy global -> shared; bytes % 16 == 0, both addresses 16-byte aligned; completes on `bar`.
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// 3-D tiled TMA load (tensor map built on the host); coordinates may lie outside the tensor: out-of-bounds
// elements are zero-filled, which is exactly the zero padding the truncated-patch box sums need.
__device__ __forceinline__ void tma_load_3d(void* dst_smem, const void* tmap, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst_smem)),
        "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}

// packed fp32x2 FMA (Blackwell FFMA2): d = a * b + c on both halves
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
    unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a), rb = *reinterpret_cast<unsigned long long*>(&b),
                       rc = *reinterpret_cast<unsigned long long*>(&c), rd;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    return *reinterpret_cast<float2*>(&rd);
}

}  // namespace disc
