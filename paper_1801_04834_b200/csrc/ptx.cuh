// Inline-PTX wrappers shared by the kernels of libcobalt_b200.so (sm_100a): mbarriers, bulk copies
// (cp.async.bulk -> SASS UBLKCP), warp election, and the one integer -> float conversion of the hot path.
// Device code only; nothing here is part of the ABI and nothing is shared with oracle/.
#pragma once

#include <cstdint>

namespace cobalt {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ------------------------------------------------------------------ mbarrier
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// The waiting warp is suspended in hardware for up to the hint instead of re-issuing the test every few cycles
// (the spin otherwise takes issue slots from the arithmetic warps of the same SM sub-partition).
constexpr uint32_t kSuspendHintNs = 20000;
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}"
            : "=r"(done)
            : "r"(bar), "r"(parity), "r"(kSuspendHintNs)
            : "memory");
    } while (!done);
}
// Spin without a suspend hint: for a wait whose wake-up latency is on the critical path.
__device__ __forceinline__ void mbar_wait_spin(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}

// ------------------------------------------------------------------ bulk copies
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *dst, uint32_t src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// generic-proxy writes to shared memory -> visible to the async proxy (bulk / tensor stores, tcgen05 operand reads)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void bar_sync_named(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

// One lane of a fully converged warp; ptxas then treats the guarded region as single-threaded and emits the
// UTCHMMA / UBLKCP / UTMASTG sequence without a per-instruction ELECT loop.
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(pred));
    return pred != 0;
}

// ------------------------------------------------------------------ step a1
// One complex sample as it sits in memory (int16: re in bits 0-15, im in bits 16-31; int8: re in bits 0-7, im in
// bits 8-15; int4: re in bits 0-3, im in bits 4-7, both two's complement) -> the integer values as floats, exact.
// The ONE conversion routine of the library: the fused F-stage kernels and cobalt_debug_unpack (pin P1) both call it.
template <int BITS>
__device__ __forceinline__ float2 unpack_sample(uint32_t raw) {
    if (BITS == 16) return make_float2((float)(short)(raw & 0xffffu), (float)(short)(raw >> 16));
    if (BITS == 8) return make_float2((float)(signed char)(raw & 0xffu), (float)(signed char)((raw >> 8) & 0xffu));
    // 4-bit: sign-extend each nibble with a shift pair
    return make_float2((float)((int)(raw << 28) >> 28), (float)((int)(raw << 24) >> 28));
}

}  // namespace cobalt
