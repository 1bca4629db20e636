// F-stage of the Cobalt correlator pipeline, hand-written for sm_100a.
//
// One fused kernel per chunk of subbands does steps a1-a4 and a7 of SURVEY.md sec 8(a): int16/int8 -> fp32
// unpack, 16-tap polyphase FIR with history, C-point forward DFT, ascending-frequency channel order, and the transposed write
// of the channelised data in the layout the X-stage consumes (cobalt_internal.h).  The delay-phase rotation and the bandpass
// (a5, a6) are constants per (input, channel) within a call: the fp64 phase_table_kernel below builds them and the
// X-stage multiplies every visibility by w_i conj(w_k) -- the same product as rotating every sample, once per visibility
// instead of once per sample.  Only the time-varying part of cobalt_process_interp (reading A21) is applied here, per sample.
// A copy kernel carries the FIR history to the next call.
//
// fstage_kernel<C, BITS, TENSOR, INTERP> is warp specialised (18 warps, one persistent CTA per SM):
//   unit     = 256 / C consecutive streams (subband, station, pol) x a run of 64-spectrum k-tiles,
//              walked in sub-tiles of 16 spectra; for C = 256 the two polarisations of a station one after the other.
//              A CTA takes the units b, b + gridDim.x, ... back to back: every role walks the same list with running ring
//              positions, so the producer already fetches the next unit while the FFT warps finish the current one.
//   warp 16  = producer: the raw integer rows of the next sub-tiles (time-contiguous, so one bulk
//              copy -- cp.async.bulk, SASS UBLKCP -- per stream and sub-tile, starting at the station's coarse sample
//              offset, reading A25) land in a 3-deep shared-memory ring signalled on mbarriers; the first sub-tile of a CTA
//              is the 16-row warm-up taken from the carried history (or from the preceding samples).
//   warps 0-7  = FIR: thread = polyphase branch.  Transposed-form filter: every new sample is
//              converted once and added, scaled by its 16 weights, to the 16 pending outputs held
//              in registers as (re, im) pairs (packed fma.rn.f32x2: one issue slot per two FMAs);
//              the completed output goes to a 3-deep ring of shared-memory tiles.  The weights carry (-1)^ph (the
//              ascending-frequency channel order D[(j + C/2) mod C] for free) and the power-of-two scale of the fp16
//              intermediate (exact).
//              The FIR -> FFT hand-over uses hardware named barriers (a waiting warp issues nothing).
//   warps 8-15 = FFT + transpose, two teams of four warps on alternate sub-tiles: thread = (two spectra, 1/16 of their
//              channels): radix-16 pass in registers, twiddle, warp-local shared-memory exchange, radix-R pass (C = 16 R),
//              [INTERP: exp(-2 pi i t step)], fp16 (or fp32) conversion, staged transposed in shared memory.  Spectra beyond
//              n_t, rows beyond 2S and lost tiles (valid-sample flags, reading A24) leave as exact zeros.
//   warp 17  = issues the 5-D tensor stores (cp.async.bulk.tensor, SASS UTMASTG) of the staged tiles.
#include "cobalt_internal.h"
#include "ptx.cuh"

#include <type_traits>

namespace cobalt {

namespace {

struct FArgs {
    const unsigned char *samples;   // [nb][S][2][N] complex integers, first subband of the chunk
    const unsigned char *hist;      // [B][S][2][15 C] complex integers
    const float *weights;           // [16][C]
    const float *dstep;             // [nb][S][C] phase step per spectrum in cycles (time-varying delay), or nullptr
    float zscale;                   // power-of-two scale s of the fp16 intermediate (1 in EXACT mode), folded into the FIR weights
    const unsigned char *valid;     // [B][S][n_kt] valid-sample flags per 64-spectrum tile (reading A24), or nullptr
    const int *coarse;              // [S] first sample of each station's block (reading A25), or nullptr
    unsigned char *z;               // chunk intermediate
    long long N, n_t;               // N = stream stride of `samples`
    size_t z_subband_bytes;
    int S, M, Mpad, n_kt, b0, tiles_per_seg, groups_per_subband;
    int n_groups, n_seg;            // work units of a launch = (stream group, time segment) pairs, n_groups * n_seg of them
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

// Time-varying delay (reading A21): exp(-2 pi i frac(t step)) for the spectra t and t + 1, step in cycles per spectrum
// (from the fp64 phase_table_kernel); the factor itself in fp32.  The static part of the rotation (the delay at the
// first spectrum, bandpass, phase offsets) is applied to the visibilities by the X-stage.
__device__ __forceinline__ void interp_factors(float step, long long t, float2 &w0, float2 &w1) {
    float p0 = step * (float)t;
    p0 -= rintf(p0);
    float p1 = p0 + step;
    p1 -= rintf(p1);
    float s0, c0, s1, c1;
    __sincosf(-6.283185307179586f * p0, &s0, &c0);
    __sincosf(-6.283185307179586f * p1, &s1, &c1);
    w0 = make_float2(c0, s0);
    w1 = make_float2(c1, s1);
}

// v * (c + i s) for compile-time c, s.  IMM: v c + (-v.y, v.x) s -- both constants enter as broadcast scalars (immediates of
// FMUL2 / FFMA2) and the swapped, half-negated v is a register-read modifier, so no constant pair is ever built in registers
// (the pair form cost 76 MOVs per FFT-loop iteration of the C = 256 kernel: 4.15 -> 3.93 ms per launch).  Same products, same
// rounding as the pair form cmul_tab2, which the C = 64 and C = 16 kernels keep (there the immediate form measured 1-3 % slower).
template <bool IMM>
__device__ __forceinline__ float2 cmul_const(float2 v, float c, float s) {
    if (!IMM) return cmul_tab2(v, make_float2(c, s));
    const float2 p = __fmul2_rn(v, make_float2(c, c));
    return __ffma2_rn(make_float2(-v.y, v.x), make_float2(s, s), p);
}

// Forward 4-point DFT in place: X[k] = sum_n a[n] (-i)^{nk}.
template <bool IMM>
__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = csub(a1, a3);
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    const float2 t3s = make_float2(t3.y, t3.x);
    if (IMM) a1 = __ffma2_rn(make_float2(-t3.y, t3.x), make_float2(-1.f, -1.f), t1);   // t1 - i t3: (i t3) as an operand modifier
    else a1 = __ffma2_rn(t3s, make_float2(1.f, -1.f), t1);
    a3 = __ffma2_rn(t3s, make_float2(-1.f, 1.f), t1);   // t1 + i t3
}

// Forward 16-point DFT in place (radix 4 x 4).  On return X[k] is at a[dft16_pos(k)].
__device__ __forceinline__ constexpr int dft16_pos(int k) { return 4 * (k & 3) + (k >> 2); }

template <bool IMM>
__device__ __forceinline__ void dft16(float2 (&a)[16]) {
    // n = 4 n1 + n2, k = k1 + 4 k2:  W16^{nk} = W4^{n1 k1} W16^{n2 k1} W4^{n2 k2}
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) dft4<IMM>(a[n2], a[4 + n2], a[8 + n2], a[12 + n2]);   // -> a[4 k1 + n2]
    constexpr float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    // W16^m = (cos(2 pi m/16), -sin(2 pi m/16)) for m = n2 k1
    a[4 * 1 + 1] = cmul_const<IMM>(a[4 * 1 + 1], c1, -s1);    // m = 1
    a[4 * 1 + 2] = cmul_const<IMM>(a[4 * 1 + 2], h, -h);      // m = 2
    a[4 * 1 + 3] = cmul_const<IMM>(a[4 * 1 + 3], s1, -c1);    // m = 3
    a[4 * 2 + 1] = cmul_const<IMM>(a[4 * 2 + 1], h, -h);      // m = 2
    if (IMM) a[4 * 2 + 2] = __fmul2_rn(make_float2(-a[4 * 2 + 2].y, a[4 * 2 + 2].x), make_float2(-1.f, -1.f));   // m = 4: -i
    else a[4 * 2 + 2] = make_float2(a[4 * 2 + 2].y, -a[4 * 2 + 2].x);
    a[4 * 2 + 3] = cmul_const<IMM>(a[4 * 2 + 3], -h, -h);     // m = 6
    a[4 * 3 + 1] = cmul_const<IMM>(a[4 * 3 + 1], s1, -c1);    // m = 3
    a[4 * 3 + 2] = cmul_const<IMM>(a[4 * 3 + 2], -h, -h);     // m = 6
    a[4 * 3 + 3] = cmul_const<IMM>(a[4 * 3 + 3], -c1, s1);    // m = 9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4<IMM>(a[4 * k1], a[4 * k1 + 1], a[4 * k1 + 2], a[4 * k1 + 3]);   // -> a[4 k1 + k2]
}

// Thread roles: warps 0-7 FIR, warps 8-15 FFT (two teams of four warps taking alternate sub-tiles), warp 16 the
// bulk-copy producer, warp 17 the tensor-store issuer.
constexpr int kFirThreads = 256, kFftThreads = 256, kFftTeam = 128, kFftTeams = 2;
constexpr int kProducerWarp = (kFirThreads + kFftThreads) / 32;
constexpr int kStoreWarp = kProducerWarp + 1;
constexpr int kFThreads = kFirThreads + kFftThreads + 64;
constexpr int kRawStages = 3;      // ring of raw sub-tiles (bulk copies in flight)
constexpr int kYBufs = 3;          // ring of FIR-output sub-tiles
constexpr int kStgTile = 32;       // spectra per staged output tile (= one tensor store per box)
constexpr int kStgBufs = 2;
// Named (hardware) barriers for the FIR -> FFT hand-over of the y ring: a warp waiting in bar.sync issues nothing, a warp polling
// an mbarrier does (barrier 0 is __syncthreads).  The single-warp waits (producer, store issuer) stay on mbarriers: moving them to
// named barriers as well measured slower (4.19 / 4.24 ms against 4.15 ms per 61-subband launch).
// One barrier per (y buffer, consuming FFT team): the two teams are not paced against each other (EXACT mode has no staging
// that couples them), and a team that runs ahead must not complete the barrier generation meant for the other one.
constexpr int kBarYFull = 1, kBarYEmpty = kBarYFull + kYBufs * kFftTeams;
static_assert(kBarYEmpty + kYBufs * kFftTeams <= 16, "named barriers");

template <int C, int BITS, bool TENSOR, bool INTERP = false>
struct FShape {
    static constexpr int SB = BITS == 16 ? 4 : 2;          // bytes per complex sample
    static constexpr int SPC = 256 / C;                    // streams per CTA
    static constexpr int R = C / 16;                       // threads per spectrum in the FFT
    // C = 256: a CTA works through the two polarisations of one station back to back (same rotation table and FIR
    // weights), so that the pipeline fills and drains once per two streams
    static constexpr int IPC = C == 256 ? 2 : 1;           // items (groups of SPC streams) per CTA
    // FIR-output tile [16 spectra][SPC streams][YS] float2.
    //   C = 256: branch ph = r + 16 q sits at 18 r + q, so that the FFT thread r reads its 16 inputs, and rewrites
    //            them in the in-place exchange, as 16-byte pairs, conflict free; the FIR lanes are permuted to match.
    //   C < 256: branch ph sits at ph + (ph >> 4).
    static constexpr int YS = R == 16 ? 16 * 18 : C + R;
    static constexpr int RAW_STAGE = kSubTile * 256 * SB;  // bytes: [SPC][16 rows][C] samples
    // One spectrum of the tile = SPC * YS float2; for C = 64 two pad elements make the stride of a spectrum PAIR
    // 4 (mod 16) eight-byte words, so that the four pairs of an FFT half-warp (lane = (pair, residue r)) hit
    // distinct banks in every load and store of the exchange (without them: 4-way conflicts, LSU pipe 91 % busy).
    static constexpr int TS = SPC * YS + (R == 4 ? 2 : 0);
    static constexpr int Y_BUF = kSubTile * TS * 8;        // bytes
    // TENSOR: staged output tile = kStgTile spectra of every (stream, channel) of the CTA as fp16 planes, laid out
    // as the shared-memory side of the tensor store: boxes of [SPB streams][2 planes][C channels][32 spectra]
    // (64-byte rows), 64-byte swizzled.
    static constexpr int SPB = SPC < 4 ? SPC : 4;          // streams per store box
    static constexpr int BOXES = SPC / SPB;
    static constexpr int BOX_BYTES = SPB * 2 * C * kStgTile * 2;
    static constexpr int STG = TENSOR ? BOXES * BOX_BYTES : 0;   // 32 KB
    static constexpr int OFF_BAR = 0;                      // mbarriers
    static constexpr int OFF_STG = 1024;                   // 1024-byte aligned (swizzle pattern)
    static constexpr int OFF_RAW = OFF_STG + kStgBufs * STG;
    static constexpr int OFF_Y = OFF_RAW + kRawStages * RAW_STAGE;
    // per-thread tables, one row of 16 float2 per (stream, residue r) at a pitch of 144 bytes (16-byte loads of
    // consecutive rows then hit distinct banks)
    static constexpr int TAB_ROW = 144;
    static constexpr int OFF_TW = OFF_Y + kYBufs * Y_BUF;        // [R] rows: W_C^{r k1}
    static constexpr int OFF_STEP = OFF_TW + (R > 1 ? R * TAB_ROW : 0);   // INTERP: [SPC][R] rows of 16 floats, pitch 80 bytes
    static constexpr int STEP_ROW = 80;
    static constexpr int TOTAL = OFF_STEP + (INTERP ? 16 * STEP_ROW : 0);
    static_assert(TOTAL <= 227 * 1024, "shared memory budget");
};

__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    const __half2 t = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const uint32_t *>(&t);
}

// channel index held in register slot i of FFT thread r after the last pass, and the register holding it
template <int R>
__device__ __forceinline__ constexpr int out_channel(int r, int i) {
    return R == 16 ? r + 16 * i : R == 4 ? 4 * r + (i >> 2) + 16 * (i & 3) : i;
}
template <int R>
__device__ __forceinline__ constexpr int out_reg(int i) {
    return R == 4 ? i : dft16_pos(i);
}

// One work unit of a launch: a group of 256 / C consecutive streams (for C = 256: both polarisations of a station, one after the
// other) over one time segment.  CTAs are persistent: CTA b takes the units b, b + gridDim.x, ... back to back, so that the
// producer already fetches the next unit while the FFT warps finish the current one (no pipeline fill / drain, no CTA launch
// between units); every role walks the same unit list and keeps the same running ring positions.
struct FUnit {
    int bl, m0, n_items, kt0, n_sub;
    long long t0;
};
template <int SPC, int IPC>
__device__ __forceinline__ FUnit decode_unit(const FArgs &a, int u) {
    FUnit w;
    const int grp = u % a.n_groups, seg = u / a.n_groups;
    w.bl = grp / a.groups_per_subband;
    w.m0 = (grp - w.bl * a.groups_per_subband) * SPC * IPC;            // first stream of the unit
    w.n_items = min(IPC, (a.M - w.m0 + SPC - 1) / SPC);                // items of the unit that exist
    w.kt0 = seg * a.tiles_per_seg;
    const int kt1 = min(w.kt0 + a.tiles_per_seg, a.n_kt);
    w.n_sub = (kt1 - w.kt0) * (kKTile / kSubTile);
    w.t0 = (long long)w.kt0 * kKTile;
    return w;
}

// INTERP (reading A21): the delay of spectrum t is tau_b + (tau_e - tau_b) t / n_t.
// The table holds the rotation for tau_b; a second table holds the phase step per spectrum f (tau_e - tau_b) / n_t in
// cycles (computed in fp64), and the per-spectrum factor exp(-2 pi i frac(t step)) is formed in fp32 ("sin/cos and
// complex multiply in single precision").
template <int C, int BITS, bool TENSOR, bool INTERP>
__global__ void __launch_bounds__(kFThreads, 1) fstage_kernel(const FArgs a, const __grid_constant__ CUtensorMap zmap) {
    using Sh = FShape<C, BITS, TENSOR, INTERP>;
    constexpr int SB = Sh::SB, SPC = Sh::SPC, R = Sh::R, YS = Sh::YS;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_raw_full = sbase + Sh::OFF_BAR;                 // [kRawStages]
    const uint32_t bar_stg_empty = bar_raw_full + 8 * kRawStages;      // [kStgBufs]
    const uint32_t bar_raw_empty = bar_stg_empty + 8 * kStgBufs;       // [kRawStages]
    const uint32_t bar_stg_full = bar_raw_empty + 8 * kRawStages;      // [kStgBufs]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int IPC = Sh::IPC;
    const int n_units = a.n_groups * a.n_seg;
    const FUnit first = decode_unit<SPC, IPC>(a, blockIdx.x);            // INTERP: the CTA's only unit (grid = units)

    if (tid == 0) {
        for (int s = 0; s < kRawStages; ++s) mbar_init(bar_raw_full + 8 * s, 1);
        for (int b = 0; b < kStgBufs; ++b) mbar_init(bar_stg_empty + 8 * b, 1);
        for (int s = 0; s < kRawStages; ++s) mbar_init(bar_raw_empty + 8 * s, kFirThreads / 32);
        for (int b = 0; b < kStgBufs; ++b) mbar_init(bar_stg_full + 8 * b, kFftThreads / 32);
        mbar_fence_init();
    }
    {   // per-CTA tables: the phase step per spectrum of the CTA's streams (INTERP) in the FFT threads' register order, and
        // the inter-pass twiddles
        if (INTERP) {
            for (int idx = tid; idx < 256; idx += kFThreads) {
                const int sl = idx / C, rr = (idx % C) / 16, i = idx % 16;
                const int m = first.m0 + sl;
                reinterpret_cast<float *>(smem + Sh::OFF_STEP + (idx >> 4) * Sh::STEP_ROW)[i] =
                    m < a.M ? a.dstep[((size_t)first.bl * a.S + (m >> 1)) * C + out_channel<R>(rr, i)] : 0.f;
            }
        }
        if (R > 1) {
            for (int idx = tid; idx < R * 16; idx += kFThreads) {
                float sn, cs;
                sincospif(-2.0f * (float)((idx / 16) * (idx % 16)) / (float)C, &sn, &cs);   // entry [r][k1]
                reinterpret_cast<float2 *>(smem + Sh::OFF_TW + (idx >> 4) * Sh::TAB_ROW)[idx & 15] = make_float2(cs, sn);
            }
        }
    }
    __syncthreads();

    if (warp == kProducerWarp) {
        // ------------------------------------------------------------------ producer
        uint32_t base_raw = 0;                                   // raw sub-tiles of the units before this one
        for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const FUnit w = decode_unit<SPC, IPC>(a, u);
        const int bl = w.bl, m0 = w.m0, n_items = w.n_items, n_sub = w.n_sub;
        const long long t0 = w.t0;
        for (int item = 0; item < n_items; ++item)
        for (int j = 0; j <= n_sub; ++j) {
            const int mi = m0 + item * SPC, n_valid = min(SPC, a.M - mi);
            const uint32_t jg = base_raw + (uint32_t)(item * (n_sub + 1) + j);   // position in the ring, over all units and items
            const int s = (int)(jg % kRawStages);
            mbar_wait(bar_raw_empty + 8 * s, ((jg / kRawStages) & 1u) ^ 1u);
            const long long tb = t0 - kSubTile + (long long)j * kSubTile;     // first row of the sub-tile
            const uint32_t full = bar_raw_full + 8 * s;
            uint32_t tx = 0;
            for (int sl = 0; sl < n_valid; ++sl) {
                const size_t stream = (size_t)bl * a.M + (mi + sl);
                const uint32_t dst0 = sbase + Sh::OFF_RAW + s * Sh::RAW_STAGE + sl * (kSubTile * C * SB);
#pragma unroll
                for (int part = 0; part < 2; ++part) {
                    // part 0: rows from the carried history (t < 0); part 1: rows of this call's block
                    long long lo, hi;
                    const unsigned char *src;
                    if (part == 0) {
                        lo = max(tb, -(long long)(kTaps - 1));
                        hi = min(tb + kSubTile, 0ll);
                        src = a.hist + (((size_t)(a.b0 + bl) * a.M + (mi + sl)) * (kTaps - 1) + (size_t)(lo + kTaps - 1)) * C * SB;
                    } else {
                        lo = max(tb, 0ll);
                        hi = min(tb + kSubTile, a.n_t);
                        src = a.samples + (stream * (size_t)a.N + (size_t)(a.coarse ? a.coarse[(mi + sl) >> 1] : 0) + (size_t)lo * C) * SB;
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
        base_raw += (uint32_t)(n_items * (n_sub + 1));
        }
    } else if (warp == kStoreWarp) {
        // ------------------------------------------------------------------ tensor-store issuer (step a7)
        // One staged tile = 32 spectra of every (stream, channel) of the CTA.  Row (channel c, k-tile kt, row group
        // m / 8, plane, m % 8) of z is 128 bytes = 64 spectra whose 16-byte chunk q sits at q ^ (m & 7) (cobalt_internal.h;
        // tensor-map coordinates: spectrum, channel, 2 (m / 8) + plane, m % 8, k-tile):
        // the 32 spectra of a tile are therefore the 64-byte half (tile & 1) ^ ((m >> 2) & 1) of the row, permuted
        // inside by m & 3 (done by the FFT threads); m >> 2 is the same for the <= 4 streams of a box.
        if (TENSOR) {
            const bool leader = elect_one();
            uint32_t stg_count = 0;
            for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
            const FUnit w = decode_unit<SPC, IPC>(a, u);
            const int bl = w.bl, m0 = w.m0, n_items = w.n_items, n_sub = w.n_sub, kt0 = w.kt0;
            for (int item = 0; item < n_items; ++item)
            for (int tile = 0; tile < n_sub / 2; ++tile) {
                const int sbuf = tile & 1;
                mbar_wait(bar_stg_full + 8 * sbuf, (stg_count >> 1) & 1u);
                if (leader) {
                    const int kt = kt0 + (tile >> 1);
#pragma unroll
                    for (int b = 0; b < Sh::BOXES; ++b) {
                        const int mb = m0 + item * SPC + b * Sh::SPB;
                        if (mb >= a.Mpad) break;
                        const int c0 = 32 * ((tile & 1) ^ ((mb >> 2) & 1));
                        asm volatile(
                            "cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];" ::"l"(&zmap),
                            "r"(sbase + Sh::OFF_STG + sbuf * Sh::STG + b * Sh::BOX_BYTES), "r"(c0), "r"(bl * C), "r"(2 * (mb >> 3)), "r"(mb & 7), "r"(kt)
                            : "memory");
                    }
                    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory has been read
                    mbar_arrive(bar_stg_empty + 8 * sbuf);
                }
                __syncwarp();
                ++stg_count;
            }
            }
            if (leader) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        }
    } else if (warp < kFirThreads / 32) {
        // ------------------------------------------------------------------ FIR (steps a1, a2)
        int sl, ph;
        if (R == 16) {   // lane permutation matching the 18 r + q tile (see FShape)
            sl = 0;
            ph = (lane >> 1) + 16 * (2 * warp + (lane & 1));
        } else {
            sl = tid / C;
            ph = tid - sl * C;
        }
        float wk[kTaps];
        {
            // (-1)^ph: channel j <- DFT bin (j + C/2) mod C; zscale: the power-of-two scale of the fp16 intermediate (exact)
            const float sgn = ((ph & 1) ? -1.f : 1.f) * a.zscale;
#pragma unroll
            for (int k = 0; k < kTaps; ++k) wk[k] = a.weights[k * C + ph] * sgn;
        }
        float2 acc[kTaps];                                // outputs still collecting taps (garbage until warmed up)
#pragma unroll
        for (int k = 0; k < kTaps; ++k) acc[k] = make_float2(0.f, 0.f);
        const uint32_t raw_thread = sbase + Sh::OFF_RAW + sl * (kSubTile * C * SB) + ph * SB;
        float2 *ybuf = reinterpret_cast<float2 *>(smem + Sh::OFF_Y) + sl * YS + (R == 16 ? 18 * (ph & 15) + (ph >> 4) : ph + (ph >> 4));

        uint32_t base_raw = 0, base_y = 0;
        for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const FUnit w = decode_unit<SPC, IPC>(a, u);
        const int n_items = w.n_items, n_sub = w.n_sub;
        for (int item = 0; item < n_items; ++item)
        for (int j = 0; j <= n_sub; ++j) {
            const uint32_t jg = base_raw + (uint32_t)(item * (n_sub + 1) + j);
            const int s = (int)(jg % kRawStages);
            mbar_wait(bar_raw_full + 8 * s, (jg / kRawStages) & 1u);
            const int jj = j - 1;                         // real sub-tile index (j = 0 is the warm-up)
            const uint32_t jjg = base_y + (uint32_t)(item * n_sub + jj);   // (unused for the warm-up)
            const int yb = (int)(jjg % kYBufs);
            const uint32_t raw = raw_thread + s * Sh::RAW_STAGE;
            // The warm-up sub-tile (jj < 0) stores nothing: its 16 samples only re-initialise the pending outputs (every
            // slot gets its first tap from one of them), also when the accumulators still hold the previous item's sums.
            // FIR -> FFT hand-over of the y ring through NAMED barriers (ids kBarYFull.., kBarYEmpty..; the 256 FIR threads
            // and the 128 threads of the consuming team): a warp waiting in bar.sync issues nothing, where the eight FIR warps
            // polling an mbarrier took 8 % of the kernel's issue slots from the FFT warps they were waiting for.
            if (jj >= 0 && jjg >= (uint32_t)kYBufs) bar_sync_named(kBarYEmpty + kFftTeams * yb + (int)((jjg - kYBufs) & 1u), kFirThreads + kFftTeam);
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
                    if (jj >= 0) yrow[i * Sh::TS] = acc[i];
                    acc[(i + 15) & 15] = __fmul2_rn(make_float2(wk[15], wk[15]), x);   // first tap of output u + 15
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_raw_empty + 8 * s);
            if (jj >= 0) {
                __threadfence_block();
                bar_arrive_named(kBarYFull + kFftTeams * yb + (int)(jjg & 1u), kFirThreads + kFftTeam);
            }
        }
        base_raw += (uint32_t)(n_items * (n_sub + 1));
        base_y += (uint32_t)(n_items * n_sub);
        }
    } else {
        // ------------------------------------------------------------------ FFT, rotate, transpose (steps a3-a7)
        // Team tm takes the sub-tiles jj = tm, tm + 2, ...; a thread owns TWO consecutive spectra (so that the fp16
        // values of spectra t, t + 1 leave as one 32-bit word and every table load serves both) and 16 channels.
        const int tm = (tid - kFirThreads) / kFftTeam;
        const int ft = (tid - kFirThreads) % kFftTeam;    // 0..127
        int tp, sl, r;                                    // spectrum pair of the sub-tile, stream of the CTA, channel residue
        if (R == 4) {   // warp = 8 pairs x 1 stream x 4 residues: conflict-free staging (see FShape / store issuer)
            tp = (ft & 31) >> 2;
            sl = ft >> 5;
            r = ft & 3;
        } else {
            tp = ft >> 4;
            sl = (ft & 15) / R;
            r = (ft & 15) % R;
        }
        float2 *ybase = reinterpret_cast<float2 *>(smem + Sh::OFF_Y) + 2 * tp * Sh::TS + sl * YS;
        const float *steps = reinterpret_cast<const float *>(smem + Sh::OFF_STEP + (sl * R + r) * Sh::STEP_ROW);
        const float4 *tw4 = reinterpret_cast<const float4 *>(smem + Sh::OFF_TW + r * Sh::TAB_ROW);
        // staging word of (channel c, plane, pair p of the tile): box b = sl / SPB, then [stream][plane][channel][64 B],
        // the 16-byte chunk (p >> 2) stored at (p >> 2) ^ (m & 3), 64-byte swizzled like the tensor store reads it
        const uint32_t stg_thread = (uint32_t)((sl / Sh::SPB) * Sh::BOX_BYTES + (sl % Sh::SPB) * (2 * C * 64));
        uint32_t base_y = 0;
        for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const FUnit w = decode_unit<SPC, IPC>(a, u);
        const int bl = w.bl, m0 = w.m0, n_items = w.n_items, n_sub = w.n_sub, kt0 = w.kt0;
        unsigned char *zsub = a.z + (size_t)bl * a.z_subband_bytes;

        for (int item = 0; item < n_items; ++item)
        for (int jj = tm; jj < n_sub; jj += kFftTeams) {
            const int m = m0 + item * SPC + sl;
            const uint32_t jjg = base_y + (uint32_t)(item * n_sub + jj);   // n_sub is a multiple of 4: team and staging parities carry over
            const int yb = (int)(jjg % kYBufs);
            const int kt = kt0 + (jj >> 2), sub = jj & 3;
            const long long t_spec = (long long)kt * kKTile + sub * kSubTile + 2 * tp;   // first of the two spectra
            float2 *y0 = ybase + (size_t)yb * (Sh::Y_BUF / 8);
            float2 *y1 = y0 + Sh::TS;
            __syncwarp();                                 // bar.sync is warp-aligned: reconverge after the previous sub-tile's stores
            bar_sync_named(kBarYFull + kFftTeams * yb + tm, kFirThreads + kFftTeam);
            float2 o0[16], o1[16];
            if (R == 16) {
#pragma unroll
                for (int q = 0; q < 16; q += 2) {
                    const float4 v0 = *reinterpret_cast<const float4 *>(y0 + 18 * r + q);
                    const float4 v1 = *reinterpret_cast<const float4 *>(y1 + 18 * r + q);
                    o0[q] = make_float2(v0.x, v0.y);
                    o0[q + 1] = make_float2(v0.z, v0.w);
                    o1[q] = make_float2(v1.x, v1.y);
                    o1[q + 1] = make_float2(v1.z, v1.w);
                }
            } else {
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    o0[q] = y0[r + R * q + ((r + R * q) >> 4)];
                    o1[q] = y1[r + R * q + ((r + R * q) >> 4)];
                }
            }
            dft16<R == 16>(o0);                           // X[k] at o[dft16_pos(k)]
            dft16<R == 16>(o1);
            if (R == 16) {
                // twiddle, exchange in place (each thread rewrites the 16 slots it read), radix-16 pass
#pragma unroll
                for (int k = 0; k < 16; k += 2) {
                    const float4 w = tw4[k >> 1];           // W_C^{r k}, W_C^{r (k + 1)}
                    const float2 a0 = k ? cmul_tab2(o0[dft16_pos(k)], make_float2(w.x, w.y)) : o0[0];
                    const float2 a1 = k ? cmul_tab2(o1[dft16_pos(k)], make_float2(w.x, w.y)) : o1[0];
                    const float2 b0 = cmul_tab2(o0[dft16_pos(k + 1)], make_float2(w.z, w.w));
                    const float2 b1 = cmul_tab2(o1[dft16_pos(k + 1)], make_float2(w.z, w.w));
                    *reinterpret_cast<float4 *>(y0 + 18 * r + k) = make_float4(a0.x, a0.y, b0.x, b0.y);
                    *reinterpret_cast<float4 *>(y1 + 18 * r + k) = make_float4(a1.x, a1.y, b1.x, b1.y);
                }
                __syncwarp();
#pragma unroll
                for (int r2 = 0; r2 < 16; ++r2) {
                    o0[r2] = y0[18 * r2 + r];
                    o1[r2] = y1[18 * r2 + r];
                }
                __syncwarp();
                bar_arrive_named(kBarYEmpty + kFftTeams * yb + tm, kFirThreads + kFftTeam);
                dft16<true>(o0);                          // channel r + 16 k2 at o[dft16_pos(k2)]
                dft16<true>(o1);
            } else if (R == 4) {
#pragma unroll
                for (int k = 0; k < 16; k += 2) {
                    const float4 w = tw4[k >> 1];
                    y0[r + 4 * k + (k >> 2)] = k ? cmul_tab2(o0[dft16_pos(k)], make_float2(w.x, w.y)) : o0[0];
                    y1[r + 4 * k + (k >> 2)] = k ? cmul_tab2(o1[dft16_pos(k)], make_float2(w.x, w.y)) : o1[0];
                    y0[r + 4 * (k + 1) + ((k + 1) >> 2)] = cmul_tab2(o0[dft16_pos(k + 1)], make_float2(w.z, w.w));
                    y1[r + 4 * (k + 1) + ((k + 1) >> 2)] = cmul_tab2(o1[dft16_pos(k + 1)], make_float2(w.z, w.w));
                }
                __syncwarp();
#pragma unroll
                for (int a4 = 0; a4 < 4; ++a4) {
                    const int k1 = 4 * r + a4;             // channel k1 + 16 k2 at o[4 a4 + k2]
#pragma unroll
                    for (int r2 = 0; r2 < 4; ++r2) {
                        o0[4 * a4 + r2] = y0[4 * k1 + r2 + r];
                        o1[4 * a4 + r2] = y1[4 * k1 + r2 + r];
                    }
                }
                __syncwarp();
                bar_arrive_named(kBarYEmpty + kFftTeams * yb + tm, kFirThreads + kFftTeam);
#pragma unroll
                for (int a4 = 0; a4 < 4; ++a4) {
                    dft4<false>(o0[4 * a4], o0[4 * a4 + 1], o0[4 * a4 + 2], o0[4 * a4 + 3]);
                    dft4<false>(o1[4 * a4], o1[4 * a4 + 1], o1[4 * a4 + 2], o1[4 * a4 + 3]);
                }
            } else {
                __syncwarp();
                bar_arrive_named(kBarYEmpty + kFftTeams * yb + tm, kFirThreads + kFftTeam);
            }
            // steps a5-a7.  The static rotation * bandpass (a5, a6) is a per-(input, channel) constant and is applied to the
            // visibilities by the X-stage (V_ik <- w_i conj(w_k) V_ik, the same product); here only the time-varying part of
            // cobalt_process_interp, then the conversion and the transposed staging (a7).  Spectra t >= n_t (padding of the last
            // k-tile), rows m >= 2S and lost tiles (valid-sample flags, reading A24) leave as exact zeros.
            const bool live0 = t_spec < a.n_t, live1 = t_spec + 1 < a.n_t;
            const bool lost = m >= a.M || (a.valid && a.valid[((size_t)(a.b0 + bl) * a.S + (m >> 1)) * a.n_kt + kt] == 0);
            if (TENSOR) {
                const uint32_t tile = jjg >> 1;
                const int sbuf = (int)(tile & 1u);
                const int p = 8 * (jj & 1) + tp;          // pair of spectra within the 32-spectrum tile
                const uint32_t msk = !live0 || lost ? 0u : live1 ? 0xffffffffu : 0x0000ffffu;   // n_t odd: last pair is half live
                mbar_wait(bar_stg_empty + 8 * sbuf, ((tile >> 1) & 1u) ^ 1u);
                unsigned char *stg = smem + Sh::OFF_STG + sbuf * Sh::STG + stg_thread;
                // byte offset of (channel j, plane re, this pair) in the box: 64 j + 16 ((p >> 2) ^ (m & 3)) + 4 (p & 3), then
                // the store's 64-byte swizzle (bits 4-5 ^= bits 7-8).  Bits 7-8 come from 64 j only, and j = (part fixed by
                // r) + (part fixed by the register slot i), so the r part is folded in once and the i part is a constant.
                const uint32_t rbits = R == 16 ? (uint32_t)(r >> 1) & 3u : R == 4 ? (uint32_t)(r & 1) << 1 : 0u;
                const uint32_t base = (uint32_t)out_channel<R>(r, 0) * 64 + (uint32_t)(((((p >> 2) ^ (m & 3)) << 4) | ((p & 3) << 2)) ^ (rbits << 4));
                // the slot part of the swizzle flips bits 4-5 by a compile-time constant: one base address per value
                unsigned char *stg_v[4];
#pragma unroll
                for (int v = 0; v < 4; ++v) stg_v[v] = stg + (base ^ (uint32_t)(v << 4));
                // almost every tile is fully live: the padding mask is applied only where a lane of the warp needs it
                auto stage = [&](auto masked) {
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const int oi = out_reg<R>(i);
                        const int dj = out_channel<R>(0, i);                     // compile-time part of the channel index
                        const int ibits = R == 16 ? 0 : R == 4 ? (i >> 3) & 1 : (i >> 1) & 3;
                        float2 z0 = o0[oi], z1 = o1[oi];
                        if (INTERP) {
                            float2 w0, w1;
                            interp_factors(steps[i], t_spec, w0, w1);
                            z0 = cmul_tab2(z0, w0);
                            z1 = cmul_tab2(z1, w1);
                        }
                        const uint32_t re = pack_half2(z0.x, z1.x), im = pack_half2(z0.y, z1.y);
                        *reinterpret_cast<uint32_t *>(stg_v[ibits] + dj * 64) = decltype(masked)::value ? re & msk : re;
                        *reinterpret_cast<uint32_t *>(stg_v[ibits] + dj * 64 + C * 64) = decltype(masked)::value ? im & msk : im;
                    }
                };
                if (__all_sync(0xffffffffu, msk == 0xffffffffu)) stage(std::false_type{});
                else stage(std::true_type{});
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the store
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_stg_full + 8 * sbuf);
            } else {
                // EXACT mode (parity instrument): fp32 values straight to z [C][M][n_t]
                if (m < a.M) {
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const int j = out_channel<R>(r, i), oi = out_reg<R>(i);
                        float2 z0 = o0[oi], z1 = o1[oi];
                        if (INTERP) {
                            float2 w0, w1;
                            interp_factors(steps[i], t_spec, w0, w1);
                            z0 = cmul_tab2(z0, w0);
                            z1 = cmul_tab2(z1, w1);
                        }
                        if (lost) z0 = z1 = make_float2(0.f, 0.f);
                        float2 *dst = reinterpret_cast<float2 *>(zsub) + ((size_t)j * a.M + m) * a.n_t + t_spec;
                        if (live0) dst[0] = z0;
                        if (live1) dst[1] = z1;
                    }
                }
            }
        }
        base_y += (uint32_t)(n_items * n_sub);
        }
    }
}

// "we compute the channel-dependent phase angles in double precision".  One entry per (subband, station,
// channel): w = b[j] exp(-2 pi i frac(f[s][j] tau_a)), f per reading A6; fp64 up to the final rounding.  The X-stage
// applies w_i conj(w_k) to the visibility of baseline (i, k) -- the same product as rotating every sample (a5, a6).
// delays_end != nullptr (reading A21): also the phase step per spectrum f (tau_e - tau_b) / n_t in cycles, for the
// time-varying part the F-stage applies.
__global__ void phase_table_kernel(const double *__restrict__ delays, const float *__restrict__ bandpass,
                                   const double *__restrict__ f_sb, int b0, int nb, int S, int C, double f_s,
                                   float2 *__restrict__ out, const double *__restrict__ delays_end, double inv_n_t,
                                   float *__restrict__ step_out) {
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
        const double b = bandpass ? (double)bandpass[j] : 1.0;      // nullptr: pure phase (the beamformer applies b[j] itself)
        const long long o = (long long)b0 * S * C + idx;      // tables are indexed by the subband of the plan
        out[o] = make_float2((float)(b * cs), (float)(b * sn));
        if (delays_end) step_out[o] = (float)(f * (delays_end[s] - delays[s]) * inv_n_t);
    }
}

// P:L360 "We carry FIR filter history samples across to the next block": new history = the last
// 15 C consumed samples of (old history ++ block); raw integers, so the carry is bit-exact.
template <typename W>
__global__ void history_kernel(const W *__restrict__ samples, const W *__restrict__ hist_old, W *__restrict__ hist_new,
                               long long streams, long long stream0, long long N, long long N_u, int HC,
                               const int *__restrict__ coarse, int S) {
    const long long total = streams * HC;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long st = idx / HC;
        const int i = (int)(idx - st * HC);
        const long long src = N_u - HC + i;
        const long long h = (stream0 + st) * HC;
        const long long off = coarse ? coarse[(st % (2 * S)) >> 1] : 0;   // reading A25: the block starts at this sample
        hist_new[h + i] = src >= 0 ? samples[st * N + off + src] : hist_old[h + (HC + src)];
    }
}

// Same carry for the common case (block at least 15 C samples long, every stream 16-byte aligned): 16-byte copies.
__global__ void history_vec_kernel(const uint4 *__restrict__ samples, uint4 *__restrict__ hist_new, long long streams,
                                   long long stream0, long long stream_vecs, long long first_vec, int hist_vecs) {
    const long long total = streams * hist_vecs;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long st = idx / hist_vecs;
        const int i = (int)(idx - st * hist_vecs);
        hist_new[(stream0 + st) * hist_vecs + i] = __ldg(samples + st * stream_vecs + first_vec + i);
    }
}

// cobalt_debug_unpack (pin P1): step a1 alone, through the SAME unpack_sample<BITS> the fused kernel applies to the
// packed complex samples it reads from shared memory (ptx.cuh).  n components = n / 2 complex samples (+ one odd
// component, taken as the low half of a word whose high half is zero).
template <int BITS>
__global__ void unpack_kernel(const unsigned char *__restrict__ in, long long n, float *__restrict__ out) {
    if (BITS == 4) {                                   // n bytes = n complex samples -> 2 n floats (reading A27)
        for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n; idx += (long long)gridDim.x * blockDim.x) {
            const float2 v = unpack_sample<4>(in[idx]);
            out[2 * idx] = v.x;
            out[2 * idx + 1] = v.y;
        }
        return;
    }
    constexpr int SB = BITS == 16 ? 4 : 2;             // bytes per complex sample
    const long long pairs = n / 2;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < pairs + (n & 1);
         idx += (long long)gridDim.x * blockDim.x) {
        uint32_t raw;
        if (idx < pairs) raw = SB == 4 ? *reinterpret_cast<const uint32_t *>(in + idx * 4) : *reinterpret_cast<const unsigned short *>(in + idx * 2);
        else raw = SB == 4 ? *reinterpret_cast<const unsigned short *>(in + idx * 4) : in[idx * 2];
        const float2 v = unpack_sample<BITS>(raw);
        out[2 * idx] = v.x;
        if (idx < pairs) out[2 * idx + 1] = v.y;
    }
}

template <int C, int BITS, bool TENSOR, bool INTERP>
cudaError_t launch_f(const cobalt_plan_s *p, cudaStream_t st, const FArgs &a, int nb) {
    using Sh = FShape<C, BITS, TENSOR, INTERP>;
    auto kern = fstage_kernel<C, BITS, TENSOR, INTERP>;
    const size_t smem = Sh::TOTAL;
    static_assert(Sh::SPB == kStoreBoxStreams(C), "plan.cu builds the tensor map with the same box");
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    FArgs args = a;
    // One CTA per SM: enough CTAs for >= 8 waves when the chunk allows, as few time segments as
    // possible (each segment re-reads its 16 warm-up rows).
    args.groups_per_subband = (p->M + Sh::SPC * Sh::IPC - 1) / (Sh::SPC * Sh::IPC);
    const long long groups = (long long)nb * args.groups_per_subband;
    const long long want = (long long)p->sm_count * 8;
    int n_seg = (int)((want + groups - 1) / groups);
    if (n_seg < 1) n_seg = 1;
    const int max_seg = (p->n_kt + 3) / 4;            // at least 4 k-tiles (256 spectra) per segment
    if (n_seg > max_seg) n_seg = max_seg;
    args.tiles_per_seg = (p->n_kt + n_seg - 1) / n_seg;
    n_seg = (p->n_kt + args.tiles_per_seg - 1) / args.tiles_per_seg;
    args.n_groups = (int)groups;
    args.n_seg = n_seg;
    // Persistent CTAs, one per SM, each walking its units back to back (decode_unit).  The time-varying-delay instantiation
    // keeps a per-CTA table of its unit's phase steps: one unit per CTA there.
    const long long units = groups * n_seg;
    const unsigned grid = INTERP ? (unsigned)units : (unsigned)(units < p->sm_count ? units : p->sm_count);
    kern<<<grid, kFThreads, smem, st>>>(args, p->zmap);
    return cudaGetLastError();
}

template <int C>
cudaError_t launch_f_c(const cobalt_plan_s *p, cudaStream_t st, const FArgs &a, int nb) {
    const bool tensor = p->mode == COBALT_MODE_TENSOR_FP16;
    if (a.dstep) {
        if (p->bits == 16) return tensor ? launch_f<C, 16, true, true>(p, st, a, nb) : launch_f<C, 16, false, true>(p, st, a, nb);
        return tensor ? launch_f<C, 8, true, true>(p, st, a, nb) : launch_f<C, 8, false, true>(p, st, a, nb);
    }
    if (p->bits == 16) return tensor ? launch_f<C, 16, true, false>(p, st, a, nb) : launch_f<C, 16, false, false>(p, st, a, nb);
    return tensor ? launch_f<C, 8, true, false>(p, st, a, nb) : launch_f<C, 8, false, false>(p, st, a, nb);
}

}  // namespace

cudaError_t launch_phase_table(const cobalt_plan_s *p, cudaStream_t st, const double *d_delays,
                               const float *d_bandpass, int b0, int nb, const double *d_delays_end) {
    const long long total = (long long)nb * p->S * p->C;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 4096) blocks = 4096;
    phase_table_kernel<<<(unsigned)blocks, threads, 0, st>>>(d_delays, d_bandpass, p->d_f_sb, b0, nb, p->S, p->C, p->f_s, p->d_phase,
                                                             d_delays_end, 1.0 / (double)p->n_t, p->d_dstep);
    return cudaGetLastError();
}

cudaError_t launch_fstage(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb, const FCall &call) {
    FArgs a;
    a.samples = static_cast<const unsigned char *>(samples_b0);
    a.hist = static_cast<const unsigned char *>(p->d_hist[p->hist_cur]);
    a.weights = p->d_weights;
    a.dstep = call.delays_end ? p->d_dstep + (size_t)b0 * p->S * p->C : nullptr;
    a.zscale = p->zscale;
    a.valid = call.valid;
    a.coarse = call.coarse;
    a.z = static_cast<unsigned char *>(p->d_z);
    a.N = call.n_in;
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

cudaError_t launch_history_update(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb, const FCall &call) {
    const long long streams = (long long)nb * p->M, stream0 = (long long)b0 * p->M;
    const int HC = (kTaps - 1) * p->C;
    const long long total = streams * HC;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 65535) blocks = 65535;
    const void *ho = p->d_hist[p->hist_cur];
    // a block of at least 15 C samples replaces the whole history from the samples alone: written in place (the F-stage of this
    // chunk, earlier in the stream, was the last reader); shorter blocks (reading R3) mix old and new and go to the other buffer
    void *hn = p->d_hist[history_in_place(p) ? p->hist_cur : p->hist_cur ^ 1];
    const size_t sb = sample_bytes(p->bits);
    const long long N = call.n_in;
    if (!call.coarse && p->N_u >= HC && (N * sb) % 16 == 0 && ((p->N_u - HC) * sb) % 16 == 0 && (HC * sb) % 16 == 0 &&
        (reinterpret_cast<uintptr_t>(samples_b0) & 15u) == 0) {
        const int hist_vecs = (int)(HC * sb / 16);
        long long vb = (streams * hist_vecs + threads - 1) / threads;
        if (vb > 65535) vb = 65535;
        history_vec_kernel<<<(unsigned)vb, threads, 0, st>>>(static_cast<const uint4 *>(samples_b0), static_cast<uint4 *>(hn), streams,
                                                          stream0, (long long)(N * sb / 16), (long long)((p->N_u - HC) * sb / 16), hist_vecs);
        return cudaGetLastError();
    }
    if (p->bits == 16)
        history_kernel<unsigned int><<<(unsigned)blocks, threads, 0, st>>>(
            static_cast<const unsigned int *>(samples_b0), static_cast<const unsigned int *>(ho),
            static_cast<unsigned int *>(hn), streams, stream0, N, p->N_u, HC, call.coarse, p->S);
    else
        history_kernel<unsigned short><<<(unsigned)blocks, threads, 0, st>>>(
            static_cast<const unsigned short *>(samples_b0), static_cast<const unsigned short *>(ho),
            static_cast<unsigned short *>(hn), streams, stream0, N, p->N_u, HC, call.coarse, p->S);
    return cudaGetLastError();
}

cudaError_t launch_unpack(cudaStream_t st, int bits, const void *d_in, long long n, float *d_out) {
    if (n <= 0) return cudaSuccess;
    const int threads = 256;
    long long blocks = ((n + 1) / 2 + threads - 1) / threads;
    if (blocks > 65535) blocks = 65535;
    const unsigned char *in = static_cast<const unsigned char *>(d_in);
    if (bits == 16) unpack_kernel<16><<<(unsigned)blocks, threads, 0, st>>>(in, n, d_out);
    else if (bits == 8) unpack_kernel<8><<<(unsigned)blocks, threads, 0, st>>>(in, n, d_out);
    else unpack_kernel<4><<<(unsigned)blocks, threads, 0, st>>>(in, n, d_out);
    return cudaGetLastError();
}

}  // namespace cobalt
