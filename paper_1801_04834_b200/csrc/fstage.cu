// F-stage of the Cobalt correlator pipeline, hand-written for sm_100a.
//
// One fused kernel per chunk of subbands does steps a1-a7 of SURVEY.md sec 8(a) (P:L360, P:L89,
// P:L368): int16/int8 -> fp32 unpack, 16-tap polyphase FIR with history, C-point forward DFT,
// ascending-frequency channel order, delay-phase rotation * bandpass, and the transposed write of
// the channelised data in the layout the X-stage consumes (cobalt_internal.h).  A tiny fp64 kernel
// builds the per-(station, channel) rotation table first (phase angles in double precision),
// and a copy kernel carries the FIR history to the next call.
//
// Work decomposition of fstage_kernel<C, BITS, TENSOR>:
//   CTA  = one stream (subband, station, pol) x a run of 64-spectrum k-tiles.
//   FIR  : thread ph owns polyphase branch ph; its 16 weights and a 15-sample sliding window stay
//          in registers while the CTA marches through time, so every input sample is loaded from
//          global memory once per CTA (4-byte coalesced loads: a warp reads 128 contiguous bytes).
//   FFT  : every 16 spectra the FIR outputs cross shared memory once; C = 16 R points are done as a
//          radix-16 pass in registers, a twiddle, a conflict-free shared-memory exchange and a
//          radix-R pass, R threads per spectrum.  The (-1)^ph needed for the ascending-frequency
//          channel order (D[(j + C/2) mod C]) is folded into the FIR weights, so the reorder is free.
//   out  : rotation*bandpass from a per-CTA table, fp16 (or fp32) conversion, staged in shared
//          memory for 64 spectra and flushed as whole 128-byte lines (TENSOR) / 128-byte runs (EXACT).
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
    int S, M, Mpad, n_kt, b0, tiles_per_seg;
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// Forward 4-point DFT in place: X[k] = sum_n a[n] (-i)^{nk}.
__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    float2 t0 = make_float2(a0.x + a2.x, a0.y + a2.y);
    float2 t1 = make_float2(a0.x - a2.x, a0.y - a2.y);
    float2 t2 = make_float2(a1.x + a3.x, a1.y + a3.y);
    float2 t3 = make_float2(a1.x - a3.x, a1.y - a3.y);
    a0 = make_float2(t0.x + t2.x, t0.y + t2.y);
    a2 = make_float2(t0.x - t2.x, t0.y - t2.y);
    a1 = make_float2(t1.x + t3.y, t1.y - t3.x);   // t1 - i t3
    a3 = make_float2(t1.x - t3.y, t1.y + t3.x);   // t1 + i t3
}

// Forward 16-point DFT in place (radix 4 x 4).  On return X[k] is at a[dft16_pos(k)].
__device__ __forceinline__ constexpr int dft16_pos(int k) { return 4 * (k & 3) + (k >> 2); }

__device__ __forceinline__ void dft16(float2 (&a)[16]) {
    // n = 4 n1 + n2, k = k1 + 4 k2:  W16^{nk} = W4^{n1 k1} W16^{n2 k1} W4^{n2 k2}
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) dft4(a[n2], a[4 + n2], a[8 + n2], a[12 + n2]);   // -> a[4 k1 + n2]
    constexpr float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    // W16^m = (cos(2 pi m/16), -sin(2 pi m/16)) for m = n2 k1
    a[4 * 1 + 1] = cmul(a[4 * 1 + 1], make_float2(c1, -s1));    // m = 1
    a[4 * 1 + 2] = cmul(a[4 * 1 + 2], make_float2(h, -h));      // m = 2
    a[4 * 1 + 3] = cmul(a[4 * 1 + 3], make_float2(s1, -c1));    // m = 3
    a[4 * 2 + 1] = cmul(a[4 * 2 + 1], make_float2(h, -h));      // m = 2
    a[4 * 2 + 2] = make_float2(a[4 * 2 + 2].y, -a[4 * 2 + 2].x);   // m = 4: -i
    a[4 * 2 + 3] = cmul(a[4 * 2 + 3], make_float2(-h, -h));     // m = 6
    a[4 * 3 + 1] = cmul(a[4 * 3 + 1], make_float2(s1, -c1));    // m = 3
    a[4 * 3 + 2] = cmul(a[4 * 3 + 2], make_float2(-h, -h));     // m = 6
    a[4 * 3 + 3] = cmul(a[4 * 3 + 3], make_float2(-c1, s1));    // m = 9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4(a[4 * k1], a[4 * k1 + 1], a[4 * k1 + 2], a[4 * k1 + 3]);   // -> a[4 k1 + k2]
}

// Step a1: the integer value as a float, bit-exact; `t` may address the carried history
// (t < 0), the block (0 <= t < n_t) or the zero padding beyond the consumed samples.
template <int BITS>
__device__ __forceinline__ float2 load_sample(const unsigned char *xs, const unsigned char *hs, long long t, int ph,
                                              int C, long long n_t) {
    constexpr int SB = BITS == 16 ? 4 : 2;
    const unsigned char *p;
    if (t < 0) p = hs + ((long long)(kTaps - 1 + t) * C + ph) * SB;
    else if (t < n_t) p = xs + (t * C + ph) * SB;
    else return make_float2(0.f, 0.f);
    if (BITS == 16) {
        unsigned int w = __ldg(reinterpret_cast<const unsigned int *>(p));
        return make_float2((float)(short)(w & 0xffffu), (float)(short)(w >> 16));
    } else {
        unsigned short w = __ldg(reinterpret_cast<const unsigned short *>(p));
        return make_float2((float)(signed char)(w & 0xffu), (float)(signed char)(w >> 8));
    }
}

template <int C>
struct FShape {
    static constexpr int NT = C < 32 ? 32 : C;     // threads per CTA
    static constexpr int R = C / 16;               // threads per spectrum in the FFT
    static constexpr int EX_T = R == 16 ? 272 : (R == 4 ? 68 : 16);   // exchange elements per spectrum
    static constexpr int XCH = (kSubTile * C > kSubTile * EX_T) ? kSubTile * C : kSubTile * EX_T;   // float2
    static constexpr int STG16 = 264;              // bytes per channel of the fp16 staging (2 x 128 + pad)
    static constexpr int STG32 = 17;               // float2 per channel of the fp32 staging (16 + pad)
    static constexpr size_t smem(bool tensor) {
        return (size_t)XCH * 8 + (size_t)C * 8 * 2 + (tensor ? (size_t)C * STG16 : (size_t)C * STG32 * 8);
    }
};

template <int C, int BITS, bool TENSOR>
__global__ void __launch_bounds__(FShape<C>::NT) fstage_kernel(FArgs a) {
    using Sh = FShape<C>;
    constexpr int NT = Sh::NT, R = Sh::R, SB = BITS == 16 ? 4 : 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *xch = reinterpret_cast<float2 *>(smem_raw);            // FIR->FFT tile, reused as exchange
    float2 *tw = xch + Sh::XCH;                                    // W_C^m
    float2 *wtab = tw + C;                                         // rotation * bandpass of this station
    unsigned char *stg = reinterpret_cast<unsigned char *>(wtab + C);

    const int tid = threadIdx.x;
    const bool active = tid < C;
    const int stream = blockIdx.x;                 // within the chunk: bl * M + m
    const int bl = stream / a.M, m = stream - bl * a.M;
    const int kt0 = blockIdx.y * a.tiles_per_seg;
    const int kt1 = min(kt0 + a.tiles_per_seg, a.n_kt);
    const unsigned char *xs = a.samples + ((size_t)bl * a.M + m) * (size_t)a.N * SB;
    const unsigned char *hs = a.hist + ((size_t)(a.b0 + bl) * a.M + m) * (size_t)(kTaps - 1) * C * SB;
    unsigned char *zsub = a.z + (size_t)bl * a.z_subband_bytes;

    for (int i = tid; i < C; i += NT) {
        float sn, cs;
        sincospif(-2.0f * (float)i / (float)C, &sn, &cs);
        tw[i] = make_float2(cs, sn);
        wtab[i] = a.phase[((size_t)bl * a.S + (m >> 1)) * C + i];
    }

    // FIR state: weights of branch ph = tid (with the (-1)^ph of the channel reorder) and the window.
    float wk[kTaps];
    float2 win[kTaps - 1];
    if (active) {
        const float sgn = (tid & 1) ? -1.f : 1.f;
#pragma unroll
        for (int k = 0; k < kTaps; ++k) wk[k] = a.weights[k * C + tid] * sgn;
#pragma unroll
        for (int i = 0; i < kTaps - 1; ++i)
            win[i] = load_sample<BITS>(xs, hs, (long long)kt0 * kKTile - (kTaps - 1) + i, tid, C, a.n_t);
    }
    __syncthreads();

    for (int kt = kt0; kt < kt1; ++kt) {
#pragma unroll 1
        for (int sub = 0; sub < kKTile / kSubTile; ++sub) {
            const long long t_base = (long long)kt * kKTile + sub * kSubTile;
            if (active) {
                float2 xn[kSubTile];
#pragma unroll
                for (int i = 0; i < kSubTile; ++i) xn[i] = load_sample<BITS>(xs, hs, t_base + i, tid, C, a.n_t);
#pragma unroll
                for (int i = 0; i < kSubTile; ++i) {
                    float re = 0.f, im = 0.f;
#pragma unroll
                    for (int k = 0; k < kTaps; ++k) {       // y[t] = sum_k w[k] x[t - k]
                        const int src = i - k;
                        const float2 v = src >= 0 ? xn[src] : win[kTaps - 1 + src];
                        re = fmaf(wk[k], v.x, re);
                        im = fmaf(wk[k], v.y, im);
                    }
                    if (t_base + i >= a.n_t) re = im = 0.f;  // padding spectra are exact zeros
                    xch[i * C + tid] = make_float2(re, im);
                }
#pragma unroll
                for (int i = 0; i < kTaps - 1; ++i) win[i] = xn[i + 1];
            }
            __syncthreads();   // (A) FIR tile complete

            float2 o[16];      // 16 channels of spectrum tl
            const int tl = tid / R, r = tid % R;
            if (active) {
                float2 v[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) v[q] = xch[tl * C + r + R * q];
                dft16(v);
                if (R == 1) {
#pragma unroll
                    for (int k = 0; k < 16; ++k) o[k] = v[dft16_pos(k)];
                } else {
#pragma unroll
                    for (int k = 1; k < 16; ++k) v[dft16_pos(k)] = cmul(v[dft16_pos(k)], tw[r * k]);
#pragma unroll
                    for (int k = 0; k < 16; ++k) o[k] = v[dft16_pos(k)];   // o[k1] = A[r][k1] W_C^{r k1}
                }
            }
            if (R > 1) {
                __syncthreads();   // (B) everyone has read the FIR tile; reuse it as the exchange
                if (active) {
                    if (R == 16) {
#pragma unroll
                        for (int k = 0; k < 16; ++k) xch[tl * Sh::EX_T + r * 17 + k] = o[k];
                    } else {
#pragma unroll
                        for (int k = 0; k < 16; ++k) xch[tl * Sh::EX_T + k * 4 + r + (k >> 2)] = o[k];
                    }
                }
                __syncthreads();   // (C)
                if (active) {
                    if (R == 16) {
                        float2 v[16];
#pragma unroll
                        for (int r2 = 0; r2 < 16; ++r2) v[r2] = xch[tl * Sh::EX_T + r2 * 17 + r];
                        dft16(v);
#pragma unroll
                        for (int k2 = 0; k2 < 16; ++k2) o[k2] = v[dft16_pos(k2)];   // channel r + 16 k2
                    } else {
#pragma unroll
                        for (int a4 = 0; a4 < 4; ++a4) {
                            const int k1 = 4 * r + a4;
                            float2 c0 = xch[tl * Sh::EX_T + k1 * 4 + 0 + r];
                            float2 c1 = xch[tl * Sh::EX_T + k1 * 4 + 1 + r];
                            float2 c2 = xch[tl * Sh::EX_T + k1 * 4 + 2 + r];
                            float2 c3 = xch[tl * Sh::EX_T + k1 * 4 + 3 + r];
                            dft4(c0, c1, c2, c3);
                            o[a4 * 4 + 0] = c0;   // channel k1 + 16 k2
                            o[a4 * 4 + 1] = c1;
                            o[a4 * 4 + 2] = c2;
                            o[a4 * 4 + 3] = c3;
                        }
                    }
                }
            }
            // steps a5-a7: rotate * bandpass, convert, stage transposed
            if (active) {
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    int j;
                    if (R == 16) j = r + 16 * i;
                    else if (R == 4) j = 4 * r + (i >> 2) + 16 * (i & 3);
                    else j = i;
                    const float2 zz = cmul(o[i], wtab[j]);
                    if (TENSOR) {
                        const int tt = sub * kSubTile + tl;
                        *reinterpret_cast<__half *>(stg + j * Sh::STG16 + tt * 2) = __float2half_rn(zz.x);
                        *reinterpret_cast<__half *>(stg + j * Sh::STG16 + 128 + tt * 2) = __float2half_rn(zz.y);
                    } else {
                        reinterpret_cast<float2 *>(stg)[j * Sh::STG32 + tl] = zz;
                    }
                }
            }
            __syncthreads();   // (D) staging written, exchange reads done
            if (TENSOR) {
                if (sub == kKTile / kSubTile - 1) {
                    // whole 128-byte lines: (channel, plane) rows of this stream, chunks pre-swizzled
                    for (int idx = tid; idx < C * 16; idx += NT) {
                        const int q = idx & 7, plane = (idx >> 3) & 1, c = idx >> 4;
                        const uint2 lo = *reinterpret_cast<const uint2 *>(stg + c * Sh::STG16 + plane * 128 + q * 16);
                        const uint2 hi = *reinterpret_cast<const uint2 *>(stg + c * Sh::STG16 + plane * 128 + q * 16 + 8);
                        unsigned char *dst = zsub + ((((size_t)c * a.n_kt + kt) * 2 + plane) * a.Mpad + m) * 128 +
                                             ((q ^ (m & 7)) << 4);
                        *reinterpret_cast<uint4 *>(dst) = make_uint4(lo.x, lo.y, hi.x, hi.y);
                    }
                }
            } else {
                float2 *z32 = reinterpret_cast<float2 *>(zsub);
                for (int idx = tid; idx < C * kSubTile; idx += NT) {
                    const int t16 = idx & 15, c = idx >> 4;
                    const long long t = t_base + t16;
                    if (t < a.n_t) z32[((size_t)c * a.M + m) * a.n_t + t] = reinterpret_cast<float2 *>(stg)[c * Sh::STG32 + t16];
                }
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
    using Sh = FShape<C>;
    auto kern = fstage_kernel<C, BITS, TENSOR>;
    const size_t smem = Sh::smem(TENSOR);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    FArgs args = a;
    // Enough CTAs for several waves, as few segments as possible (each segment re-reads 15 rows).
    const long long streams = (long long)nb * p->M;
    const long long want = (long long)p->sm_count * 16;
    int n_seg = (int)((want + streams - 1) / streams);
    if (n_seg < 1) n_seg = 1;
    if (n_seg > p->n_kt) n_seg = p->n_kt;
    args.tiles_per_seg = (p->n_kt + n_seg - 1) / n_seg;
    n_seg = (p->n_kt + args.tiles_per_seg - 1) / args.tiles_per_seg;
    dim3 grid((unsigned)streams, (unsigned)n_seg);
    kern<<<grid, Sh::NT, smem, st>>>(args);
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
