// F-stage of the Cobalt correlator pipeline, hand-written for sm_100a.
//
// One fused kernel per chunk of subbands does steps a1-a7 of SURVEY.md sec 8(a) (P:L360, P:L89,
// P:L368): int16/int8 -> fp32 unpack, 16-tap polyphase FIR with history, C-point forward DFT,
// ascending-frequency channel order, delay-phase rotation * bandpass, and the transposed write of
// the channelised data in the layout the X-stage consumes (cobalt_internal.h).  A tiny fp64 kernel
// builds the per-(station, channel) rotation table first (phase angles in double precision),
// and a copy kernel carries the FIR history to the next call.
//
// fstage_kernel<C, BITS, TENSOR> is warp specialised (17 warps, one CTA per SM):
//   CTA      = 256 / C consecutive streams (subband, station, pol) x a run of 64-spectrum k-tiles,
//              walked in sub-tiles of 16 spectra.
//   warp 16  = producer: the raw integer rows of the next sub-tiles (time-contiguous, so one bulk
//              copy -- cp.async.bulk, SASS UBLKCP -- per stream and sub-tile) land in a 4-deep
//              shared-memory ring signalled on mbarriers; the first sub-tile of a CTA is the 16-row
//              warm-up taken from the carried history (or from the preceding samples).
//   warps 0-7  = FIR: thread = polyphase branch.  Transposed-form filter: every new sample is
//              converted once and added, scaled by its 16 weights, to the 16 pending outputs held
//              in registers as (re, im) pairs (packed fma.rn.f32x2: one issue slot per two FMAs);
//              the completed output goes to a double-buffered shared-memory tile.
//   warps 8-15 = FFT + rotate + transpose: thread = (spectrum, 1/16 of its channels): radix-16 pass
//              in registers, twiddle, warp-local shared-memory exchange, radix-R pass (C = 16 R),
//              rotation * bandpass from a per-CTA table, fp16 (or fp32) conversion, staged
//              transposed in shared memory and flushed as whole 32-byte sectors (TENSOR) /
//              128-byte runs (EXACT).  The (-1)^ph needed for the ascending-frequency channel order
//              (D[(j + C/2) mod C]) is folded into the FIR weights, so the reorder is free.
#include "cobalt_internal.h"

namespace cobalt {

namespace {

struct FArgs {
    const unsigned char *samples;   // [nb][S][2][N] complex integers, first subband of the chunk
    const unsigned char *hist;      // [B][S][2][15 C] complex integers
    const float *weights;           // [16][C]
    const float2 *phase;            // [nb][S][C]
    unsigned char *z;               // chunk intermediate
    long long N, n_t;
    size_t z_subband_bytes;
    int S, M, Mpad, n_kt, b0, tiles_per_seg, groups_per_subband;
};

// Packed fp32 pairs (fma.rn.f32x2 family, SASS FFMA2/FADD2/FMUL2): a complex value is one 64-bit
// register pair, so a complex add or a real-times-complex FMA costs one issue slot instead of two.
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
// v * W, W = (t.x + i t.y):  v.x (W.re, W.im) + v.y (-W.im, W.re).  The swapped, half-negated operand is a
// register-read modifier of FFMA2 (SASS .F32x2.LO_HI.NP), so a complex multiply is two issue slots.
__device__ __forceinline__ float2 cmul_tab2(float2 v, float2 t) {
    const float2 p = __fmul2_rn(make_float2(v.x, v.x), t);
    return __ffma2_rn(make_float2(-t.y, t.x), make_float2(v.y, v.y), p);
}

// Forward 4-point DFT in place: X[k] = sum_n a[n] (-i)^{nk}.
__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = csub(a1, a3);
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    const float2 t3s = make_float2(t3.y, t3.x);
    a1 = __ffma2_rn(t3s, make_float2(1.f, -1.f), t1);   // t1 - i t3
    a3 = __ffma2_rn(t3s, make_float2(-1.f, 1.f), t1);   // t1 + i t3
}

// Forward 16-point DFT in place (radix 4 x 4).  On return X[k] is at a[dft16_pos(k)].
__device__ __forceinline__ constexpr int dft16_pos(int k) { return 4 * (k & 3) + (k >> 2); }

__device__ __forceinline__ void dft16(float2 (&a)[16]) {
    // n = 4 n1 + n2, k = k1 + 4 k2:  W16^{nk} = W4^{n1 k1} W16^{n2 k1} W4^{n2 k2}
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) dft4(a[n2], a[4 + n2], a[8 + n2], a[12 + n2]);   // -> a[4 k1 + n2]
    constexpr float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    // W16^m = (cos(2 pi m/16), -sin(2 pi m/16)) for m = n2 k1
    a[4 * 1 + 1] = cmul_tab2(a[4 * 1 + 1], make_float2(c1, -s1));    // m = 1
    a[4 * 1 + 2] = cmul_tab2(a[4 * 1 + 2], make_float2(h, -h));      // m = 2
    a[4 * 1 + 3] = cmul_tab2(a[4 * 1 + 3], make_float2(s1, -c1));    // m = 3
    a[4 * 2 + 1] = cmul_tab2(a[4 * 2 + 1], make_float2(h, -h));      // m = 2
    a[4 * 2 + 2] = make_float2(a[4 * 2 + 2].y, -a[4 * 2 + 2].x);   // m = 4: -i
    a[4 * 2 + 3] = cmul_tab2(a[4 * 2 + 3], make_float2(-h, -h));     // m = 6
    a[4 * 3 + 1] = cmul_tab2(a[4 * 3 + 1], make_float2(s1, -c1));    // m = 3
    a[4 * 3 + 2] = cmul_tab2(a[4 * 3 + 2], make_float2(-h, -h));     // m = 6
    a[4 * 3 + 3] = cmul_tab2(a[4 * 3 + 3], make_float2(-c1, s1));    // m = 9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4(a[4 * k1], a[4 * k1 + 1], a[4 * k1 + 2], a[4 * k1 + 3]);   // -> a[4 k1 + k2]
}

// ------------------------------------------------------------------ mbarrier / bulk-copy helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
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
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void bar_sync_named(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

// Thread roles: warps 0-7 FIR, warps 8-15 / 16-23 the two FFT groups, warp 24 the producer.
constexpr int kFirThreads = 256, kFftGroup = 256, kFftGroups = 2;
constexpr int kProducerWarp = (kFirThreads + kFftGroups * kFftGroup) / 32;
constexpr int kFThreads = kFirThreads + kFftGroups * kFftGroup + 32;
constexpr int kRawStages = 3;      // ring of raw sub-tiles (bulk copies in flight)
constexpr int kYBufs = 3;          // ring of FIR-output sub-tiles

template <int C, int BITS, bool TENSOR>
struct FShape {
    static constexpr int SB = BITS == 16 ? 4 : 2;          // bytes per complex sample
    static constexpr int SPC = 256 / C;                    // streams per CTA
    static constexpr int R = C / 16;                       // threads per spectrum in the FFT
    // FIR-output tile [16 spectra][SPC streams][YS] float2; branch ph sits at ph + (ph >> 4) so that the
    // radix-16 pass, the in-place exchange and the radix-R pass are all free of bank conflicts
    static constexpr int YS = C + R;
    static constexpr int RAW_STAGE = kSubTile * 256 * SB;  // bytes: [SPC][16 rows][C] samples
    static constexpr int Y_BUF = kSubTile * SPC * YS * 8;  // bytes
    // staging of the transposed output, one per FFT group: TENSOR: 32 spectra of (re | im << 16) words
    // + 2 pad words per (stream, channel) row; EXACT: 16 spectra of float2 + 1 pad
    static constexpr int STG_ROW = TENSOR ? 34 * 4 : 17 * 8;
    static constexpr int STG = 256 * STG_ROW;
    static constexpr int OFF_BAR = 0;                      // 2 kRawStages + 2 kYBufs mbarriers
    static constexpr int OFF_RAW = 128;
    static constexpr int OFF_Y = OFF_RAW + kRawStages * RAW_STAGE;
    static constexpr int OFF_STG = OFF_Y + kYBufs * Y_BUF;
    static constexpr int OFF_WTAB = OFF_STG + kFftGroups * STG;   // [SPC][C] float2: rotation * bandpass
    static constexpr int OFF_TW = OFF_WTAB + 256 * 8;      // [16][R] float2 W_C^{r k1}
    static constexpr int TOTAL = OFF_TW + (R > 1 ? R * 16 * 8 : 0);
    static_assert(TOTAL <= 227 * 1024, "shared memory budget");
};

template <int BITS>
__device__ __forceinline__ float2 unpack_sample(uint32_t raw) {
    // Step a1: the two's-complement integer value as a float, exact.
    if (BITS == 16) return make_float2((float)(short)(raw & 0xffffu), (float)(short)(raw >> 16));
    return make_float2((float)(signed char)(raw & 0xffu), (float)(signed char)((raw >> 8) & 0xffu));
}

template <int C, int BITS, bool TENSOR>
__global__ void __launch_bounds__(kFThreads, 1) fstage_kernel(const FArgs a) {
    using Sh = FShape<C, BITS, TENSOR>;
    constexpr int SB = Sh::SB, SPC = Sh::SPC, R = Sh::R, YS = Sh::YS;
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_raw_full = sbase + Sh::OFF_BAR;                 // [kRawStages]
    const uint32_t bar_raw_empty = bar_raw_full + 8 * kRawStages;      // [kRawStages]
    const uint32_t bar_y_full = bar_raw_empty + 8 * kRawStages;        // [kYBufs]
    const uint32_t bar_y_empty = bar_y_full + 8 * kYBufs;              // [kYBufs]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int grp = blockIdx.x;                          // stream group within the chunk
    const int bl = grp / a.groups_per_subband;
    const int m0 = (grp - bl * a.groups_per_subband) * SPC;
    const int n_valid = min(SPC, a.M - m0);              // streams of this CTA that exist
    const int kt0 = blockIdx.y * a.tiles_per_seg;
    const int kt1 = min(kt0 + a.tiles_per_seg, a.n_kt);
    const int n_sub = (kt1 - kt0) * (kKTile / kSubTile);
    const long long t0 = (long long)kt0 * kKTile;

    if (tid == 0) {
        for (int s = 0; s < kRawStages; ++s) {
            mbar_init(bar_raw_full + 8 * s, 1);
            mbar_init(bar_raw_empty + 8 * s, kFirThreads / 32);
        }
        for (int b = 0; b < kYBufs; ++b) {
            mbar_init(bar_y_full + 8 * b, kFirThreads / 32);
            mbar_init(bar_y_empty + 8 * b, kFftGroup / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {   // rotation * bandpass of the CTA's streams (station = m >> 1) and the inter-pass twiddles
        float2 *wtab = reinterpret_cast<float2 *>(smem + Sh::OFF_WTAB);
        for (int i = tid; i < 256; i += kFThreads) {
            const int sl = i / C, j = i - sl * C;
            const int m = min(m0 + sl, a.M - 1);
            wtab[i] = a.phase[((size_t)bl * a.S + (m >> 1)) * C + j];
        }
        if (R > 1) {
            float2 *tw = reinterpret_cast<float2 *>(smem + Sh::OFF_TW);
            for (int i = tid; i < R * 16; i += kFThreads) {
                float sn, cs;
                sincospif(-2.0f * (float)((i / R) * (i % R)) / (float)C, &sn, &cs);   // entry [k1][r]
                tw[i] = make_float2(cs, sn);
            }
        }
    }
    __syncthreads();

    if (warp == kProducerWarp) {
        // ------------------------------------------------------------------ producer
        for (int j = 0; j <= n_sub; ++j) {
            const int s = j % kRawStages;
            const uint32_t ph = (uint32_t)(j / kRawStages) & 1u;
            mbar_wait(bar_raw_empty + 8 * s, ph ^ 1u);
            const long long tb = t0 - kSubTile + (long long)j * kSubTile;     // first row of the sub-tile
            const uint32_t full = bar_raw_full + 8 * s;
            uint32_t tx = 0;
            for (int sl = 0; sl < n_valid; ++sl) {
                const size_t stream = (size_t)bl * a.M + (m0 + sl);
                const uint32_t dst0 = sbase + Sh::OFF_RAW + s * Sh::RAW_STAGE + sl * (kSubTile * C * SB);
#pragma unroll
                for (int part = 0; part < 2; ++part) {
                    // part 0: rows from the carried history (t < 0); part 1: rows of this call's block
                    long long lo, hi;
                    const unsigned char *src;
                    if (part == 0) {
                        lo = max(tb, -(long long)(kTaps - 1));
                        hi = min(tb + kSubTile, 0ll);
                        src = a.hist + (((size_t)(a.b0 + bl) * a.M + (m0 + sl)) * (kTaps - 1) + (size_t)(lo + kTaps - 1)) * C * SB;
                    } else {
                        lo = max(tb, 0ll);
                        hi = min(tb + kSubTile, a.n_t);
                        src = a.samples + (stream * (size_t)a.N + (size_t)lo * C) * SB;
                    }
                    if (hi <= lo) continue;
                    const uint32_t bytes = (uint32_t)(hi - lo) * C * SB;
                    const uint32_t dst = dst0 + (uint32_t)(lo - tb) * C * SB;
                    if ((reinterpret_cast<uintptr_t>(src) & 15u) == 0) {
                        if (lane == 0) bulk_g2s(dst, src, bytes, full);
                        tx += bytes;
                    } else {   // stream not 16-byte aligned (odd N): element-wise copy by the warp
                        for (uint32_t e = lane * SB; e < bytes; e += 32 * SB) {
                            if (SB == 4) {
                                const uint32_t v = __ldg(reinterpret_cast<const uint32_t *>(src + e));
                                asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + e), "r"(v) : "memory");
                            } else {
                                const unsigned short v = __ldg(reinterpret_cast<const unsigned short *>(src + e));
                                asm volatile("st.shared.b16 [%0], %1;" ::"r"(dst + e), "h"(v) : "memory");
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_expect_tx(full, tx);
        }
    } else if (warp < kFirThreads / 32) {
        // ------------------------------------------------------------------ FIR (steps a1, a2)
        const int sl = tid / C, ph = tid - sl * C;
        float wk[kTaps];
        {
            const float sgn = (ph & 1) ? -1.f : 1.f;      // (-1)^ph: channel j <- DFT bin (j + C/2) mod C
#pragma unroll
            for (int k = 0; k < kTaps; ++k) wk[k] = a.weights[k * C + ph] * sgn;
        }
        float2 acc[kTaps];                                // outputs still collecting taps (garbage until warmed up)
#pragma unroll
        for (int k = 0; k < kTaps; ++k) acc[k] = make_float2(0.f, 0.f);
        const uint32_t raw_thread = sbase + Sh::OFF_RAW + sl * (kSubTile * C * SB) + ph * SB;
        float2 *ybuf = reinterpret_cast<float2 *>(smem + Sh::OFF_Y) + sl * YS + ph + (ph >> 4);

        for (int j = 0; j <= n_sub; ++j) {
            const int s = j % kRawStages;
            mbar_wait(bar_raw_full + 8 * s, (uint32_t)(j / kRawStages) & 1u);
            const int jj = j - 1;                         // real sub-tile index (j = 0 is the warm-up)
            const int yb = jj % kYBufs;
            const uint32_t raw = raw_thread + s * Sh::RAW_STAGE;
            // The warm-up sub-tile (jj < 0) also stores: into buffer 0, which nobody reads before the first real
            // sub-tile has overwritten it and signalled y_full.
            if (jj >= 0) mbar_wait(bar_y_empty + 8 * yb, ((uint32_t)(jj / kYBufs) & 1u) ^ 1u);
            float2 *yrow = ybuf + (size_t)(jj >= 0 ? yb : 0) * (Sh::Y_BUF / 8);
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                uint32_t rw[kSubTile / 2];                // 8 raw words per batch: one shared-memory latency, not 8
#pragma unroll
                for (int i = 0; i < kSubTile / 2; ++i) {
                    const uint32_t addr = raw + (half * 8 + i) * C * SB;
                    if (SB == 4) asm volatile("ld.shared.b32 %0, [%1];" : "=r"(rw[i]) : "r"(addr));
                    else {
                        unsigned short h;
                        asm volatile("ld.shared.b16 %0, [%1];" : "=h"(h) : "r"(addr));
                        rw[i] = h;
                    }
                }
#pragma unroll
                for (int ii = 0; ii < kSubTile / 2; ++ii) {
                    const int i = half * 8 + ii;
                    const float2 x = unpack_sample<BITS>(rw[ii]);
                    // sample u contributes w[k] x[u] to output u + k (slot (u + k) mod 16); output u is then complete
#pragma unroll
                    for (int k = 0; k < kTaps - 1; ++k)
                        acc[(i + k) & 15] = __ffma2_rn(make_float2(wk[k], wk[k]), x, acc[(i + k) & 15]);
                    yrow[i * (SPC * YS)] = acc[i];
                    acc[(i + 15) & 15] = __fmul2_rn(make_float2(wk[15], wk[15]), x);   // first tap of output u + 15
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_raw_empty + 8 * s);
                if (jj >= 0) mbar_arrive(bar_y_full + 8 * yb);
            }
        }
    } else {
        // ------------------------------------------------------------------ FFT, rotate, transpose (steps a3-a7)
        // Group g takes the pairs of sub-tiles (32 spectra = half a k-tile) pp = g, g + 2, ...
        const int g = (tid - kFirThreads) / kFftGroup;
        const int ft = (tid - kFirThreads) % kFftGroup;   // 0..255
        const int tl = ft >> 4;                           // spectrum of the sub-tile
        const int sl = (ft & 15) / R, r = (ft & 15) % R;  // stream of the CTA, residue of the channel index
        float2 *ybase = reinterpret_cast<float2 *>(smem + Sh::OFF_Y) + (tl * SPC + sl) * YS;
        const float2 *wtab = reinterpret_cast<const float2 *>(smem + Sh::OFF_WTAB) + sl * C;
        const float2 *twr = reinterpret_cast<const float2 *>(smem + Sh::OFF_TW) + r;   // W_C^{r k1} at [k1 * R]
        unsigned char *stg = smem + Sh::OFF_STG + g * Sh::STG;
        unsigned char *zsub = a.z + (size_t)bl * a.z_subband_bytes;
        // flush items of this thread (TENSOR): staging row it * 64 + (ft >> 2) = (stream, channel), 8 spectra
        // tg = ft & 3.  Row (channel c, k-tile kt, plane, input m) of z starts at ((c n_kt + kt) 2 Mpad + m) 128;
        // the 16-byte chunk q of that row sits at q ^ (m & 7) (cobalt_internal.h), q = 4 (sub >> 1) + tg.
        const size_t plane_stride = (size_t)a.Mpad * 128;
        size_t fl_off[4];
        bool fl_ok[4];
#pragma unroll
        for (int it = 0; it < 4; ++it) {
            const int row = it * (kFftGroup / 4) + (ft >> 2);
            const int fsl = row / C, fc = row - fsl * C, fm = m0 + fsl;
            fl_ok[it] = fm < a.M;
            fl_off[it] = ((size_t)fc * a.n_kt * 2 * a.Mpad + fm) * 128 + ((((ft & 3) ^ (fm & 3)) << 4) | (fm & 4) << 4);
        }

        for (int pp = g; pp < n_sub / 2; pp += kFftGroups) {
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
                const int jj = 2 * pp + h;
                const int yb = jj % kYBufs;
                const int kt = kt0 + (jj >> 2), sub = jj & 3;
                const long long t_base = (long long)kt * kKTile + sub * kSubTile;
                float2 *y = ybase + (size_t)yb * (Sh::Y_BUF / 8);
                mbar_wait(bar_y_full + 8 * yb, (uint32_t)(jj / kYBufs) & 1u);
                float2 o[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) o[q] = y[r + R * q + ((r + R * q) >> 4)];
                dft16(o);                                 // X[k] at o[dft16_pos(k)]
                if (R == 16) {
                    // twiddle, exchange in place (each thread rewrites the 16 slots it read), radix-16 pass
#pragma unroll
                    for (int k = 0; k < 16; ++k)
                        y[r + 17 * k] = k ? cmul_tab2(o[dft16_pos(k)], twr[k * R]) : o[0];   // A[r][k1] W_C^{r k1}
                    __syncwarp();
#pragma unroll
                    for (int r2 = 0; r2 < 16; ++r2) o[r2] = y[r2 + 17 * r];
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_y_empty + 8 * yb);
                    dft16(o);                             // channel r + 16 k2 at o[dft16_pos(k2)]
                } else if (R == 4) {
#pragma unroll
                    for (int k = 0; k < 16; ++k)
                        y[r + 4 * k + (k >> 2)] = k ? cmul_tab2(o[dft16_pos(k)], twr[k * R]) : o[0];
                    __syncwarp();
#pragma unroll
                    for (int a4 = 0; a4 < 4; ++a4) {
                        const int k1 = 4 * r + a4;         // channel k1 + 16 k2 at o[4 a4 + k2]
#pragma unroll
                        for (int r2 = 0; r2 < 4; ++r2) o[4 * a4 + r2] = y[4 * k1 + r2 + r];
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_y_empty + 8 * yb);
#pragma unroll
                    for (int a4 = 0; a4 < 4; ++a4) dft4(o[4 * a4], o[4 * a4 + 1], o[4 * a4 + 2], o[4 * a4 + 3]);
                } else {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_y_empty + 8 * yb);
                }
                // steps a5-a7: rotate * bandpass, convert, stage transposed.  Spectra t >= n_t (padding of
                // the last k-tile) are staged as exact zeros: the rotation table is replaced by zero.
                const bool live = t_base + tl < a.n_t;
                const int ts = TENSOR ? h * kSubTile + tl : tl;   // spectrum slot in the staging row
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    int j, oi;                            // channel index, register holding it
                    if (R == 16) { j = r + 16 * i; oi = dft16_pos(i); }
                    else if (R == 4) { j = 4 * r + (i >> 2) + 16 * (i & 3); oi = i; }
                    else { j = i; oi = dft16_pos(i); }
                    float2 zz = cmul_tab2(o[oi], wtab[j]);
                    if (TENSOR) {
                        uint32_t hv;
                        {
                            const __half2 t2 = __floats2half2_rn(zz.x, zz.y);
                            hv = *reinterpret_cast<const uint32_t *>(&t2);
                        }
                        if (!live) hv = 0u;
                        *reinterpret_cast<uint32_t *>(stg + (sl * C + j) * Sh::STG_ROW + ts * 4) = hv;
                    } else {
                        if (!live) zz = make_float2(0.f, 0.f);
                        *reinterpret_cast<float2 *>(stg + (sl * C + j) * Sh::STG_ROW + ts * 8) = zz;
                    }
                }
                if (TENSOR && h == 0) continue;           // flush every 32 spectra
                bar_sync_named(1 + g, kFftGroup);         // staging complete
                if (TENSOR) {
                    // item = (row = (stream, channel), tg = 8 spectra): 8 words (re | im << 16) -> one 16-byte
                    // chunk per plane; 4 consecutive lanes write one 64-byte run of a 128-byte row
                    unsigned char *zkt = zsub + (size_t)kt * 2 * plane_stride;
                    const size_t half = (size_t)(sub >> 1) << 6;   // which 64 bytes of the row these 32 spectra are
#pragma unroll
                    for (int it = 0; it < 4; ++it) {
                        if (!fl_ok[it]) continue;
                        const unsigned char *src = stg + (it * (kFftGroup / 4) + (ft >> 2)) * Sh::STG_ROW + (ft & 3) * 32;
                        uint32_t w[8];
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const uint2 v = *reinterpret_cast<const uint2 *>(src + i * 8);
                            w[2 * i] = v.x;
                            w[2 * i + 1] = v.y;
                        }
                        uint4 re, im;
                        re.x = __byte_perm(w[0], w[1], 0x5410);
                        re.y = __byte_perm(w[2], w[3], 0x5410);
                        re.z = __byte_perm(w[4], w[5], 0x5410);
                        re.w = __byte_perm(w[6], w[7], 0x5410);
                        im.x = __byte_perm(w[0], w[1], 0x7632);
                        im.y = __byte_perm(w[2], w[3], 0x7632);
                        im.z = __byte_perm(w[4], w[5], 0x7632);
                        im.w = __byte_perm(w[6], w[7], 0x7632);
                        unsigned char *rowp = zkt + (fl_off[it] ^ half);
                        *reinterpret_cast<uint4 *>(rowp) = re;
                        *reinterpret_cast<uint4 *>(rowp + plane_stride) = im;
                    }
                } else {
                    const int fsl = ft / C, fc = ft - fsl * C;    // this thread owns staging row ft = (stream, channel)
                    const int fm = m0 + fsl;
                    if (fm < a.M) {
                        float2 *dst = reinterpret_cast<float2 *>(zsub) + ((size_t)fc * a.M + fm) * a.n_t + t_base;
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (t_base + i < a.n_t) dst[i] = *reinterpret_cast<const float2 *>(stg + ft * Sh::STG_ROW + i * 8);
                    }
                }
                bar_sync_named(1 + g, kFftGroup);         // staging drained
            }
        }
    }
}

// "we compute the channel-dependent phase angles in double precision".  One entry per
// (subband of the chunk, station, channel): s b[j] exp(-2 pi i frac(f[s][j] tau_a)), f per reading A6.
//
// s is the power-of-two scale of the fp16 intermediate (TENSOR mode; 1 otherwise): with
// e = ceil(log2(max_j |b_j| * amp_max / 32768)) and s = 2^-e, full-scale input cannot overflow fp16
// (|z s| <= 32768) and tiny bandpass weights cannot push z into the fp16 subnormals.  The X-stage
// epilogue multiplies the visibilities by 1/s^2; both factors are exact.  Every block derives the
// same s from the same C weights; block 0 publishes {s, 1/s, 1/s^2} for the X-stage.
__global__ void phase_table_kernel(const double *__restrict__ delays, const float *__restrict__ bandpass,
                                   const double *__restrict__ f_sb, int b0, int nb, int S, int C, double f_s,
                                   float amp_max, int tensor, float *__restrict__ scale_out,
                                   float2 *__restrict__ out) {
    __shared__ float s_max[32];
    __shared__ float s_scale;
    float bm = 0.f;
    for (int j = threadIdx.x; j < C; j += blockDim.x) bm = fmaxf(bm, fabsf(bandpass[j]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bm = fmaxf(bm, __shfl_xor_sync(0xffffffffu, bm, o));
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = bm;
    __syncthreads();
    if (threadIdx.x == 0) {
        float m = 0.f;
        for (int w = 0; w < (int)((blockDim.x + 31) >> 5); ++w) m = fmaxf(m, s_max[w]);
        int e = 0;
        if (tensor && m > 0.f && m < 3.0e38f) {
            e = (int)ceilf(log2f(m * amp_max / 32768.f));
            e = max(-40, min(40, e));
        }
        s_scale = scalbnf(1.f, -e);
        if (blockIdx.x == 0) {
            scale_out[0] = scalbnf(1.f, -e);
            scale_out[1] = scalbnf(1.f, e);
            scale_out[2] = scalbnf(1.f, 2 * e);
        }
    }
    __syncthreads();
    const double sc = (double)s_scale;
    const long long total = (long long)nb * S * C;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(idx % C);
        const int s = (int)((idx / C) % S);
        const int bl = (int)(idx / ((long long)C * S));
        const double f = f_sb[b0 + bl] + ((double)j - 0.5 * (double)C) * f_s / (double)C;
        const double cyc = f * delays[s];
        const double frac = cyc - floor(cyc);
        double sn, cs;
        sincospi(-2.0 * frac, &sn, &cs);
        const double b = (double)bandpass[j] * sc;
        out[idx] = make_float2((float)(b * cs), (float)(b * sn));
    }
}

__global__ void unit_scale_kernel(float *scale_out) {
    if (threadIdx.x < 3) scale_out[threadIdx.x] = 1.f;
}

// P:L360 "We carry FIR filter history samples across to the next block": new history = the last
// 15 C consumed samples of (old history ++ block); raw integers, so the carry is bit-exact.
template <typename W>
__global__ void history_kernel(const W *__restrict__ samples, const W *__restrict__ hist_old, W *__restrict__ hist_new,
                               long long streams, long long stream0, long long N, long long N_u, int HC) {
    const long long total = streams * HC;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long st = idx / HC;
        const int i = (int)(idx - st * HC);
        const long long src = N_u - HC + i;
        const long long h = (stream0 + st) * HC;
        hist_new[h + i] = src >= 0 ? samples[st * N + src] : hist_old[h + (HC + src)];
    }
}

template <typename I>
__global__ void unpack_kernel(const I *__restrict__ in, long long n, float *__restrict__ out) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x)
        out[idx] = (float)in[idx];
}

template <int C, int BITS, bool TENSOR>
cudaError_t launch_f(const cobalt_plan_s *p, cudaStream_t st, const FArgs &a, int nb) {
    using Sh = FShape<C, BITS, TENSOR>;
    auto kern = fstage_kernel<C, BITS, TENSOR>;
    const size_t smem = Sh::TOTAL;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    FArgs args = a;
    // One CTA per SM: enough CTAs for >= 8 waves when the chunk allows, as few time segments as
    // possible (each segment re-reads its 16 warm-up rows).
    args.groups_per_subband = (p->M + Sh::SPC - 1) / Sh::SPC;
    const long long groups = (long long)nb * args.groups_per_subband;
    const long long want = (long long)p->sm_count * 8;
    int n_seg = (int)((want + groups - 1) / groups);
    if (n_seg < 1) n_seg = 1;
    const int max_seg = (p->n_kt + 3) / 4;            // at least 4 k-tiles (256 spectra) per segment
    if (n_seg > max_seg) n_seg = max_seg;
    args.tiles_per_seg = (p->n_kt + n_seg - 1) / n_seg;
    n_seg = (p->n_kt + args.tiles_per_seg - 1) / args.tiles_per_seg;
    dim3 grid((unsigned)groups, (unsigned)n_seg);
    kern<<<grid, kFThreads, smem, st>>>(args);
    return cudaGetLastError();
}

template <int C>
cudaError_t launch_f_c(const cobalt_plan_s *p, cudaStream_t st, const FArgs &a, int nb) {
    const bool tensor = p->mode == COBALT_MODE_TENSOR_FP16;
    if (p->bits == 16) return tensor ? launch_f<C, 16, true>(p, st, a, nb) : launch_f<C, 16, false>(p, st, a, nb);
    return tensor ? launch_f<C, 8, true>(p, st, a, nb) : launch_f<C, 8, false>(p, st, a, nb);
}

}  // namespace

cudaError_t launch_phase_table(const cobalt_plan_s *p, cudaStream_t st, const double *d_delays,
                               const float *d_bandpass, int b0, int nb) {
    const long long total = (long long)nb * p->S * p->C;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 4096) blocks = 4096;
    phase_table_kernel<<<(unsigned)blocks, threads, 0, st>>>(d_delays, d_bandpass, p->d_f_sb, b0, nb, p->S, p->C,
                                                             p->f_s, p->amp_max, p->mode == COBALT_MODE_TENSOR_FP16 ? 1 : 0,
                                                             p->d_scale, p->d_phase);
    return cudaGetLastError();
}

cudaError_t launch_set_unit_scale(const cobalt_plan_s *p, cudaStream_t st) {
    unit_scale_kernel<<<1, 32, 0, st>>>(p->d_scale);
    return cudaGetLastError();
}

cudaError_t launch_fstage(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb) {
    FArgs a;
    a.samples = static_cast<const unsigned char *>(samples_b0);
    a.hist = static_cast<const unsigned char *>(p->d_hist[p->hist_cur]);
    a.weights = p->d_weights;
    a.phase = p->d_phase;
    a.z = static_cast<unsigned char *>(p->d_z);
    a.N = p->N;
    a.n_t = p->n_t;
    a.z_subband_bytes = p->z_subband_bytes;
    a.S = p->S;
    a.M = p->M;
    a.Mpad = p->Mpad;
    a.n_kt = p->n_kt;
    a.b0 = b0;
    a.tiles_per_seg = p->n_kt;
    switch (p->C) {
        case 16: return launch_f_c<16>(p, st, a, nb);
        case 64: return launch_f_c<64>(p, st, a, nb);
        case 256: return launch_f_c<256>(p, st, a, nb);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_history_update(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb) {
    const long long streams = (long long)nb * p->M, stream0 = (long long)b0 * p->M;
    const int HC = (kTaps - 1) * p->C;
    const long long total = streams * HC;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 65535) blocks = 65535;
    const void *ho = p->d_hist[p->hist_cur];
    void *hn = p->d_hist[p->hist_cur ^ 1];
    if (p->bits == 16)
        history_kernel<unsigned int><<<(unsigned)blocks, threads, 0, st>>>(
            static_cast<const unsigned int *>(samples_b0), static_cast<const unsigned int *>(ho),
            static_cast<unsigned int *>(hn), streams, stream0, p->N, p->N_u, HC);
    else
        history_kernel<unsigned short><<<(unsigned)blocks, threads, 0, st>>>(
            static_cast<const unsigned short *>(samples_b0), static_cast<const unsigned short *>(ho),
            static_cast<unsigned short *>(hn), streams, stream0, p->N, p->N_u, HC);
    return cudaGetLastError();
}

cudaError_t launch_unpack(cudaStream_t st, int bits, const void *d_in, long long n, float *d_out) {
    if (n <= 0) return cudaSuccess;
    const int threads = 256;
    long long blocks = (n + threads - 1) / threads;
    if (blocks > 65535) blocks = 65535;
    if (bits == 16) unpack_kernel<short><<<(unsigned)blocks, threads, 0, st>>>(static_cast<const short *>(d_in), n, d_out);
    else unpack_kernel<signed char><<<(unsigned)blocks, threads, 0, st>>>(static_cast<const signed char *>(d_in), n, d_out);
    return cudaGetLastError();
}

}  // namespace cobalt
