// Inline-PTX wrappers shared by the kernels of libcobalt_b200.so (sm_100a): mbarriers, bulk copies
// (cp.async.bulk -> SASS UBLKCP), warp election, the tcgen05 / TMEM wrappers, and the one integer -> float conversion of the hot path.
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
// Producer side of a named barrier (PTX ISA "bar": st.shared ...; bar.arrive in the producer, bar.sync; ld.shared in the consumer):
// counts the calling warp's threads and does not wait.  A warp blocked in bar.sync is descheduled by the hardware -- unlike an
// mbarrier wait it issues nothing while it waits.
__device__ __forceinline__ void bar_arrive_named(int id, int threads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
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

// ------------------------------------------------------------------ tcgen05 (5th-generation tensor cores, TMEM)
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, 128 x N x 16, fp16 in, fp32 accumulate.
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
// Shared-memory operand descriptor, 128-byte swizzle, descriptor version 1 (sm_100).
//   K-major operand (rows = M or N index, 64 K-elements per 128-byte row): 8-row groups sbo bytes apart; lbo unused (1).
//   MN-major operand (rows = K index, 64 M/N-elements per 128-byte row): 8-row K-groups sbo bytes apart, blocks of 64
//   M/N-elements lbo bytes apart.
__device__ __forceinline__ uint64_t make_smem_desc_lbo(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo >> 4) & 0x3FFFu) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFFu) << 32) |
           (1ull << 46) | (2ull << 61);
}
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t addr, uint32_t sbo) { return make_smem_desc_lbo(addr, 16, sbo); }
// kind::f16 instruction descriptor: D = f32, A = B = f16; A K-major (a_mn = 0) or MN-major (1), B K-major.
__device__ __forceinline__ uint32_t make_idesc(int m, int n, int neg_a, int a_mn = 0) {
    return (1u << 4) | ((uint32_t)neg_a << 13) | ((uint32_t)a_mn << 15) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, "
        "[%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

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
