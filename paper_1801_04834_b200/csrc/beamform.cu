// Beamformer pipeline of SURVEY.md sec 8(f) row 4 (readings A28-A32 of DESIGN.md), at the channel
// resolution of the plan: "Coherent beamforming first adjusts the beam direction with a phase shift and sums over antenna
// fields, then optionally computes Stokes parameters, while incoherent beamforming first computes Stokes parameters and
// then sums over antenna fields."  Input is the channelised intermediate z of the F-stage (steps a1-a4, a7).  Feeding the
// beamformer from the correlator's 16-tap channeliser is a READING (A28), not the paper's design: P:L366 says the
// beamformer "cannot share initial steps with the correlator" (it runs its own 256-channel PPF), and the sentence "Both beam
// types have the first four kernels in common" is about coherent versus incoherent beams.  Delay compensation,
// bandpass and the per-input phase offsets (a5, a6, A22)
// are constants per (input, channel) within a call and are folded into the beam weights.
//
// bf_tc_kernel (TENSOR_FP16 mode): the coherent sum
//     Y[b][p][t] = sum_a W[b][a][p] z[a][p][t],   W = exp(-2 pi i frac(f_j tau_{b,a})) w_a[j] exp(-i phi_{a,p})
// of one (subband, channel) is a dense contraction over the 2S inputs: on tcgen05 as the real GEMM
//     D[t][n] = sum_kappa Z^T[t][kappa] W'[n][kappa],   kappa = (input m = 2a + p', plane re | im),  n = (beam, pol, re | im)
//   A = Z^T straight from the F-stage's layout: the [8 rows][64 spectra] 128-byte-swizzled atoms of z (cobalt_internal.h)
//       ARE the canonical MN-major operand (M = spectrum contiguous, K = rows); one instruction takes M = 128 spectra
//       (two k-tiles, LBO apart) x K = 16 (the re atom and the im atom of one 8-row group, SBO = 1024 apart);
//   B = W' built per job in shared memory, K-major, from the fp64 beam phase ("The beamforming kernel operates in
//       a similar way"), the fp64 phase table of the station delays and the phase offsets; row (b, p, re) holds
//       (Wr | -Wi) on the inputs of polarisation p and zeros on the other polarisation, row (b, p, im) holds (Wi | Wr);
//   D = fp32 in TMEM, lane = spectrum, column = (beam, pol, re | im): an epilogue thread owns one spectrum and finds
//       (Xr, Xi, Yr, Yi) of a beam in four adjacent columns, so complex voltages leave as coalesced float2 stores and the
//       Stokes parameters (A29) are formed in registers; time integration (A30) is a shuffle reduction over t_int lanes.
// Persistent CTAs; job = (subband, channel, block of <= 64 beams), walked in blocks of 128 spectra with two accumulator
// sets, so that the MMAs of one block overlap the epilogue of the previous one.  Warp 0 = bulk-copy producer (one copy per
// 128-spectrum block: the two k-tiles are contiguous), warp 1 = MMA issuer, warps 4-19 = weights + epilogue.
//
// bf_simt_kernel (EXACT_FP32 mode): the same sums with fp32 FMAs from the fp32 intermediate (parity instrument, not tuned).
// incoherent_kernel: sum over stations of the per-station Stokes parameters (A31), reading z once (HBM bound).
#include "cobalt_internal.h"
#include "ptx.cuh"

namespace cobalt {

namespace {

constexpr int kBfFirstEpiWarp = 4, kBfEpiWarps = 16, kBfEpiSub = kBfEpiWarps / 4;
constexpr int kBfThreads = 32 * (kBfFirstEpiWarp + kBfEpiWarps);
constexpr int kBfEpiThreads = 32 * kBfEpiWarps;
constexpr int kBfAccStride = 256;              // TMEM columns between the two accumulator sets

struct BfArgs {
    const unsigned char *z;
    size_t z_subband_bytes;
    const float2 *phase, *poff;     // [B][S][C] exp(-2 pi i frac(f tau_a)) (no bandpass), [2S] or nullptr
    const double *f_sb;             // [B]
    const double *beam_delays;      // [n_beams][S]
    const float *bandpass;          // [C]
    void *out;                      // subband b0 of the output (layout per product, reading A32)
    double f_s;
    long long n_t, n_out;
    int S, M, Mpad, C, n_kt, n_tb, b0, nb;
    int n_beams, bpb, n_bb, N;      // beams per block, beam blocks, N = 4 bpb accumulator columns
    int product, n_stokes, t_int, lg_t_int;
    float inv_s;                    // 1 / s, s = power-of-two scale of the fp16 intermediate
    int stages;
    uint32_t stage_bytes, w_bytes, kt_bytes;
    int total_jobs;
};

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// W[b][a][p] of one (subband, channel): the beam phase in fp64 up to the final rounding, times the station's
// delay-compensation factor from the fp64 phase table, times the phase offset of the input (A22).
// (Args = BfArgs or BfSimtArgs: one routine for the tensor and the fp32 kernel)
template <class Args>
__device__ __forceinline__ void beam_weight(const Args &a, double f, int sb, int c, int beam, int st, float2 &wx, float2 &wy) {
    const double cyc = f * a.beam_delays[(size_t)beam * a.S + st];
    const double frac = cyc - floor(cyc);
    float sn, cs;
    sincospif(-2.0f * (float)frac, &sn, &cs);
    const float2 w = cmulf(make_float2(cs, sn), a.phase[((size_t)sb * a.S + st) * a.C + c]);
    wx = a.poff ? cmulf(w, a.poff[2 * st]) : w;
    wy = a.poff ? cmulf(w, a.poff[2 * st + 1]) : w;
}

// Stokes parameters of (X, Y) (reading A29): I, Q, U, V.
__device__ __forceinline__ void stokes4(float xr, float xi, float yr, float yi, float &I, float &Q, float &U, float &V) {
    const float px = xr * xr + xi * xi, py = yr * yr + yi * yi;
    I = px + py;
    Q = px - py;
    U = 2.f * (xr * yr + xi * yi);
    V = 2.f * (xi * yr - xr * yi);
}

// ---- epilogue of one 128-spectrum accumulator block, per warp: lane = spectrum, 16-column chunks = 4 beams x (Xr, Xi, Yr, Yi)
struct BfEpi {
    float vs, ps;                 // scale of a voltage (b_j / s) and of a power
    int lg;                       // t_int = 2^lg
    long long t, n_t, n_out;      // this lane's spectrum
    size_t cv_pol, st_k, st_beam; // output strides: polarisation (voltages); Stokes parameter, beam (Stokes)
    float2 *o_cv;                 // voltages: element (first beam of the block, X, channel, t)
    float *o_st;                  // Stokes: element (first beam of the block, I, channel, t >> lg)
    uint32_t taddr;               // TMEM address of column 0 of this warp's lanes
    int n_chunks, sub, lane, beams_left;
};

__device__ __forceinline__ void epilogue_voltages(const BfEpi &ep) {
    const bool live = ep.t < ep.n_t;
    for (int c16 = ep.sub; c16 < ep.n_chunks; c16 += kBfEpiSub) {
        uint32_t x[16];
        tmem_ld16(ep.taddr + 16 * c16, x);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (live && 4 * c16 + e < ep.beams_left) {
                float2 *o = ep.o_cv + (size_t)(4 * c16 + e) * 2 * ep.cv_pol;
                o[0] = make_float2(__uint_as_float(x[4 * e]) * ep.vs, __uint_as_float(x[4 * e + 1]) * ep.vs);
                o[ep.cv_pol] = make_float2(__uint_as_float(x[4 * e + 2]) * ep.vs, __uint_as_float(x[4 * e + 3]) * ep.vs);
            }
        }
    }
}

// Sum of v[] over the 2^LGW lanes of a group (reading A30).  While a lane still holds more than one value a step halves
// the array instead of duplicating the sums (the lanes with the offset bit clear keep the lower half, the others the upper
// half): V - 1 shuffles for V values instead of V LGW.  On return a lane holds max(1, V >> LGW) sums: the original indices
// base + j, base = sum over the halving steps i of bit_i(lane) (V >> (i + 1)).
template <int V, int LGW>
__device__ __forceinline__ int reduce_lanes(float (&v)[V], int lane) {
    int base = 0;
    int n = V;
#pragma unroll
    for (int i = 0; i < LGW; ++i) {
        const int off = 1 << i;
        if (n > 1) {
            const int h = n >> 1;
            const bool up = (lane & off) != 0;
#pragma unroll
            for (int j = 0; j < V / 2; ++j) {
                if (j < h) {
                    const float send = up ? v[j] : v[h + j];
                    const float keep = up ? v[h + j] : v[j];
                    v[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
                }
            }
            if (up) base += h;
            n = h;
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
        }
    }
    return base;
}

template <int NS, int LGW>
__device__ __forceinline__ void epilogue_stokes(const BfEpi &ep) {
    constexpr int V = 4 * NS;                         // values of a chunk per lane: index e NS + k (beam e, parameter k)
    constexpr int HALVINGS = LGW < (NS == 1 ? 2 : 4) ? LGW : (NS == 1 ? 2 : 4);
    constexpr int R = V >> HALVINGS;                  // sums a lane holds after the reduction
    // lanes whose bits [HALVINGS, LGW) are zero write (the others hold duplicates)
    const bool writer = ((ep.lane >> HALVINGS) & ((1 << (LGW - HALVINGS)) - 1)) == 0 && (ep.t >> ep.lg) < ep.n_out;
    for (int c16 = ep.sub; c16 < ep.n_chunks; c16 += kBfEpiSub) {
        uint32_t x[16];
        tmem_ld16(ep.taddr + 16 * c16, x);
        tmem_ld_wait();
        float v[V];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float xr = __uint_as_float(x[4 * e]), xi = __uint_as_float(x[4 * e + 1]);
            const float yr = __uint_as_float(x[4 * e + 2]), yi = __uint_as_float(x[4 * e + 3]);
            if (NS == 4) {
                float I, Q, U, W;
                stokes4(xr, xi, yr, yi, I, Q, U, W);
                v[4 * e] = I * ep.ps;
                v[4 * e + 1] = Q * ep.ps;
                v[4 * e + 2] = U * ep.ps;
                v[4 * e + 3] = W * ep.ps;
            } else {
                v[e] = fmaf(xr, xr, fmaf(xi, xi, fmaf(yr, yr, yi * yi))) * ep.ps;
            }
        }
        const int base = reduce_lanes<V, LGW>(v, ep.lane);
        if (writer) {
#pragma unroll
            for (int j = 0; j < R; ++j) {
                const int idx = base + j, e = idx / NS, k = idx % NS;
                if (4 * c16 + e < ep.beams_left) {
                    float *o = ep.o_st + (size_t)(4 * c16 + e) * ep.st_beam + (size_t)k * ep.st_k;
                    if (ep.lg > 5) atomicAdd(o, v[j]);      // t_int = 64, 128: two or four warps per output sample
                    else *o = v[j];
                }
            }
        }
    }
}

template <int NS>
__device__ __forceinline__ void epilogue_stokes_lg(const BfEpi &ep) {
    switch (ep.lg < 5 ? ep.lg : 5) {
        case 0: epilogue_stokes<NS, 0>(ep); break;
        case 1: epilogue_stokes<NS, 1>(ep); break;
        case 2: epilogue_stokes<NS, 2>(ep); break;
        case 3: epilogue_stokes<NS, 3>(ep); break;
        case 4: epilogue_stokes<NS, 4>(ep); break;
        default: epilogue_stokes<NS, 5>(ep); break;
    }
}

__global__ void __launch_bounds__(kBfThreads, 1) bf_tc_kernel(const BfArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *sm = smem_raw + (base - smem_u32(smem_raw));
    // barriers: full[s] at 8 s, empty[s] at 8 (8 + s), tmem_full[2], tmem_empty[2], w_ready, TMEM base slot
    const uint32_t bar_full = base, bar_empty = base + 64, tmem_full = base + 128, tmem_empty = base + 144, w_ready = base + 160;
    const uint32_t tmem_slot = base + 176;
    const uint32_t w_base = base + 1024;
    const uint32_t stage_base = w_base + a.w_bytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_ks = a.Mpad >> 3;                       // k-steps of 16 (one 8-row group, both planes)

    if (threadIdx.x == 0) {
        for (int s = 0; s < a.stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tmem_full + 8 * b, 1);
            mbar_init(tmem_empty + 8 * b, kBfEpiWarps);
        }
        mbar_init(w_ready, 1);
        mbar_fence_init();
    }
    if (warp == 1) {
        // All 512 columns (two accumulator sets of up to 256).  Residency assumption: one CTA of this kernel per SM owns the
        // SM's whole TMEM.  __launch_bounds__(.., 1) does not enforce that -- with a small Mpad the shared memory would let a
        // second CTA in, and a second plan's bf_tc_kernel / xstage_tc_kernel on another stream can land on the same SM.  Such
        // a CTA blocks in tcgen05.alloc until this one exits (it never deadlocks: every CTA frees its columns before it
        // returns and needs no other CTA to make progress), i.e. a correlator plan and a beamformer plan running on two
        // streams take turns on an SM instead of sharing it.
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        if (elect_one()) {
            uint32_t it = 0;
            for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x) {
                const int prob = jid / a.n_bb;
                const int bl = prob / a.C, c = prob - bl * a.C;
                const unsigned char *src = a.z + (size_t)bl * a.z_subband_bytes + (size_t)c * a.n_kt * a.kt_bytes;
                for (int tb = 0; tb < a.n_tb; ++tb, ++it) {
                    const int s = it % a.stages;
                    mbar_wait(bar_empty + 8 * s, ((it / a.stages) & 1u) ^ 1u);
                    // the last block of an odd number of k-tiles brings one k-tile; the other half of the stage keeps stale
                    // data, which only reaches accumulator rows t >= n_t (never stored)
                    const uint32_t bytes = (uint32_t)min(2, a.n_kt - 2 * tb) * a.kt_bytes;
                    mbar_arrive_expect_tx(bar_full + 8 * s, bytes);
                    bulk_g2s(stage_base + (uint32_t)s * a.stage_bytes, src + (size_t)(2 * tb) * a.kt_bytes, bytes, bar_full + 8 * s);
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        if (elect_one()) {
            const uint32_t idesc = make_idesc(kBfTBlock, a.N, 0, /*a_mn=*/1);
            uint32_t it = 0, job = 0;
            for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x, ++job) {
                mbar_wait_spin(w_ready, job & 1u);          // this job's W' is in shared memory
                tc_fence_after();
                for (int tb = 0; tb < a.n_tb; ++tb, ++it) {
                    const int s = it % a.stages;
                    const uint32_t buf = it & 1u;
                    mbar_wait_spin(bar_full + 8 * s, (it / a.stages) & 1u);      // one thread: spinning costs nothing, the
                    mbar_wait_spin(tmem_empty + 8 * buf, ((it >> 1) & 1u) ^ 1u);  // suspended wait's wake-up latency would
                    tc_fence_after();
                    const uint32_t d = tmem_base + buf * kBfAccStride;
                    const uint32_t st_addr = stage_base + (uint32_t)s * a.stage_bytes;
                    for (int g = 0; g < n_ks; ++g) {
                        // A: MN-major, the re atom and the im atom of row group g (1024 apart), two k-tiles (kt_bytes apart)
                        const uint64_t ad = make_smem_desc_lbo(st_addr + (uint32_t)g * 2048, a.kt_bytes, 1024);
                        // B: K-major W', K-atom g / 4 (N rows of 128 bytes each), 32 bytes per k-step inside it
                        const uint64_t bd = make_smem_desc(w_base + (uint32_t)(g >> 2) * (uint32_t)a.N * 128 + (uint32_t)(g & 3) * 32, 1024);
                        tc_mma(d, ad, bd, idesc, g ? 1u : 0u);
                    }
                    tc_commit(bar_empty + 8 * s);
                    tc_commit(tmem_full + 8 * buf);
                }
            }
        }
    } else if (warp >= kBfFirstEpiWarp) {
        // ------------------------------------------------------------------ weights + epilogue
        const int et = threadIdx.x - 32 * kBfFirstEpiWarp;
        const int wq = warp & 3, sub = (warp - kBfFirstEpiWarp) >> 2;     // TMEM lane quarter; every kBfEpiSub-th 16-column chunk
        const int ns = a.n_stokes;
        uint32_t it = 0;
        for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x) {
            const int prob = jid / a.n_bb, bb = jid - prob * a.n_bb;
            const int bl = prob / a.C, c = prob - bl * a.C;
            const int sb = a.b0 + bl;
            // ---- W' of this job.  The previous job's MMAs have completed: its last tmem_full has been waited for below.
            {
                const double f = a.f_sb[sb] + ((double)c - 0.5 * (double)a.C) * a.f_s / (double)a.C;
                for (int item = et; item < a.bpb * n_ks; item += kBfEpiThreads) {
                    const int g = item % n_ks, b_loc = item / n_ks;
                    const int beam = bb * a.bpb + b_loc;
                    float wr[8], wi[8];                       // index r8 = 2 q + p: input 8 g + r8 = station 4 g + q, pol p
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int st = 4 * g + q;
                        float2 wx = make_float2(0.f, 0.f), wy = wx;
                        if (beam < a.n_beams && st < a.S) beam_weight(a, f, sb, c, beam, st, wx, wy);
                        wr[2 * q] = wx.x;
                        wi[2 * q] = wx.y;
                        wr[2 * q + 1] = wy.x;
                        wi[2 * q + 1] = wy.y;
                    }
                    const uint32_t atom = w_base + (uint32_t)(g >> 2) * (uint32_t)a.N * 128;
#pragma unroll
                    for (int p = 0; p < 2; ++p)
#pragma unroll
                        for (int ri = 0; ri < 2; ++ri)
#pragma unroll
                            for (int pl = 0; pl < 2; ++pl) {
                                // row (b, p, re): (Wr | -Wi);  row (b, p, im): (Wi | Wr); zeros on the other polarisation
                                uint32_t v[4];
#pragma unroll
                                for (int q = 0; q < 4; ++q) {
                                    const float x = ri == 0 ? (pl == 0 ? wr[2 * q + p] : -wi[2 * q + p]) : (pl == 0 ? wi[2 * q + p] : wr[2 * q + p]);
                                    const unsigned short h = __half_as_ushort(__float2half_rn(x));
                                    v[q] = p == 0 ? (uint32_t)h : (uint32_t)h << 16;   // element r8 = 2 q + p of the 16-byte chunk
                                }
                                const int n = 4 * b_loc + 2 * p + ri;
                                const uint32_t addr = atom + (uint32_t)(n >> 3) * 1024 + (uint32_t)(n & 7) * 128 +
                                                      (uint32_t)(((2 * (g & 3) + pl) ^ (n & 7)) << 4);
                                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
                            }
                }
                fence_async_smem();                           // generic-proxy writes -> visible to the tensor core's reads
                bar_sync_named(1, kBfEpiThreads);
                if (et == 0) mbar_arrive(w_ready);
            }
            BfEpi ep;
            ep.vs = a.bandpass[c] * a.inv_s;
            ep.ps = ep.vs * ep.vs;
            ep.lg = a.lg_t_int;
            ep.n_t = a.n_t;
            ep.n_out = a.n_out;
            ep.cv_pol = (size_t)a.C * a.n_t;
            ep.st_k = (size_t)a.C * a.n_out;
            ep.st_beam = (size_t)ns * ep.st_k;
            ep.n_chunks = a.N >> 4;
            ep.sub = sub;
            ep.lane = lane;
            const int beam0 = bb * a.bpb;
            ep.beams_left = a.n_beams - beam0;
            float2 *cv_job = static_cast<float2 *>(a.out) + ((size_t)bl * a.n_beams + beam0) * 2 * ep.cv_pol + (size_t)c * a.n_t;
            float *st_job = static_cast<float *>(a.out) + ((size_t)bl * a.n_beams + beam0) * ep.st_beam + (size_t)c * a.n_out;
            for (int tb = 0; tb < a.n_tb; ++tb, ++it) {
                const uint32_t buf = it & 1u;
                mbar_wait_spin(tmem_full + 8 * buf, (it >> 1) & 1u);
                tc_fence_after();
                ep.t = (long long)tb * kBfTBlock + 32 * wq + lane;
                ep.taddr = tmem_base + ((uint32_t)(32 * wq) << 16) + buf * kBfAccStride;
                ep.o_cv = cv_job + ep.t;
                ep.o_st = st_job + (ep.t >> ep.lg);
                if (a.product == COBALT_BF_COHERENT_VOLTAGES) epilogue_voltages(ep);
                else if (ns == 1) epilogue_stokes_lg<1>(ep);
                else epilogue_stokes_lg<4>(ep);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tmem_empty + 8 * buf);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}

// ---------------------------------------------------------------------------------------------------------------
// EXACT_FP32: coherent beams from the fp32 intermediate [C][M][n_t] float2.  One block = (subband, channel, 128 spectra,
// block of beams); thread = spectrum.  Weights of the block's beams in shared memory.
struct BfSimtArgs {
    const float2 *z;
    size_t z_subband_elems;
    const float2 *phase, *poff;
    const double *f_sb, *beam_delays;
    const float *bandpass;
    void *out;
    double f_s;
    long long n_t, n_out;
    int S, M, C, b0, n_beams, bpb, product, n_stokes, t_int;
};

__global__ void __launch_bounds__(kBfTBlock) bf_simt_kernel(const BfSimtArgs a) {
    extern __shared__ float2 sw[];                         // [bpb][M] weights, then [4][128] floats for the integration
    float *red = reinterpret_cast<float *>(sw + (size_t)a.bpb * a.M);
    const int c = blockIdx.x % a.C, bl = blockIdx.x / a.C, sb = a.b0 + bl;
    const int bb = blockIdx.z;
    const long long t = (long long)blockIdx.y * kBfTBlock + threadIdx.x;
    const double f = a.f_sb[sb] + ((double)c - 0.5 * (double)a.C) * a.f_s / (double)a.C;
    for (int item = threadIdx.x; item < a.bpb * a.S; item += kBfTBlock) {
        const int st = item % a.S, b_loc = item / a.S, beam = bb * a.bpb + b_loc;
        float2 wx = make_float2(0.f, 0.f), wy = wx;
        if (beam < a.n_beams) beam_weight(a, f, sb, c, beam, st, wx, wy);
        sw[(size_t)b_loc * a.M + 2 * st] = wx;
        sw[(size_t)b_loc * a.M + 2 * st + 1] = wy;
    }
    __syncthreads();
    const float bp = a.bandpass[c];
    const float2 *zc = a.z + (size_t)bl * a.z_subband_elems + (size_t)c * a.M * a.n_t;
    const int ns = a.n_stokes;
    for (int b_loc = 0; b_loc < a.bpb; ++b_loc) {
        const int beam = bb * a.bpb + b_loc;
        if (beam >= a.n_beams) break;
        float2 X = make_float2(0.f, 0.f), Y = X;
        if (t < a.n_t)
            for (int st = 0; st < a.S; ++st) {
                const float2 zx = zc[(size_t)(2 * st) * a.n_t + t], zy = zc[(size_t)(2 * st + 1) * a.n_t + t];
                const float2 wx = sw[(size_t)b_loc * a.M + 2 * st], wy = sw[(size_t)b_loc * a.M + 2 * st + 1];
                X.x = fmaf(wx.x, zx.x, fmaf(-wx.y, zx.y, X.x));
                X.y = fmaf(wx.x, zx.y, fmaf(wx.y, zx.x, X.y));
                Y.x = fmaf(wy.x, zy.x, fmaf(-wy.y, zy.y, Y.x));
                Y.y = fmaf(wy.x, zy.y, fmaf(wy.y, zy.x, Y.y));
            }
        X = make_float2(X.x * bp, X.y * bp);
        Y = make_float2(Y.x * bp, Y.y * bp);
        if (a.product == COBALT_BF_COHERENT_VOLTAGES) {
            if (t < a.n_t) {
                float2 *o = static_cast<float2 *>(a.out) + ((((size_t)bl * a.n_beams + beam) * 2) * a.C + c) * a.n_t + t;
                o[0] = X;
                o[(size_t)a.C * a.n_t] = Y;
            }
        } else {
            float sv[4];
            stokes4(X.x, X.y, Y.x, Y.y, sv[0], sv[1], sv[2], sv[3]);
            for (int k = 0; k < ns; ++k) red[k * kBfTBlock + threadIdx.x] = sv[k];
            __syncthreads();
            const int n_u = kBfTBlock / a.t_int;
            for (int w = threadIdx.x; w < n_u * ns; w += kBfTBlock) {
                const int k = w / n_u, ul = w % n_u;
                float s = 0.f;
                for (int i = 0; i < a.t_int; ++i) s += red[k * kBfTBlock + ul * a.t_int + i];
                const long long u = (long long)blockIdx.y * n_u + ul;
                if (u < a.n_out) static_cast<float *>(a.out)[((((size_t)bl * a.n_beams + beam) * ns + k) * a.C + c) * a.n_out + u] = s;
            }
            __syncthreads();
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Incoherent Stokes (reading A31): S_k[c][u] = sum over the t_int spectra of u, over stations a, of stokes_k(z_{a,X}, z_{a,Y}),
// z = w_a[j] F rotated like everywhere else: |w| = b_j for both polarisations of a station, so I and Q take b_j^2 and U, V
// take the relative phase offset exp(-i (phi_X - phi_Y)) of the station (A22).  One block = (subband, channel, 128 spectra).
struct IncArgs {
    const unsigned char *z;        // TENSOR: fp16 planes; EXACT: float2 [C][M][n_t]
    size_t z_subband_bytes;
    const float2 *poff;
    const float *bandpass;
    float *out;                    // [nb][n_stokes][C][n_out]
    long long n_t, n_out;
    int S, M, Mpad, C, n_kt, n_stokes, t_int, tensor;
    float inv_s;
};

__global__ void __launch_bounds__(kBfTBlock) incoherent_kernel(const IncArgs a) {
    __shared__ float red[4][kBfTBlock];
    const int c = blockIdx.x % a.C, bl = blockIdx.x / a.C;
    const long long t = (long long)blockIdx.y * kBfTBlock + threadIdx.x;
    const int kt = (int)(t / kKTile), tt = (int)(t % kKTile);
    float I = 0.f, Q = 0.f, U = 0.f, V = 0.f;
    if (t < a.n_t) {
        const unsigned char *zb = a.z + (size_t)bl * a.z_subband_bytes;
        for (int st = 0; st < a.S; ++st) {
            float2 x, y;
            if (a.tensor) {
                const int m0 = 2 * st, m1 = m0 + 1;      // both rows sit in the same 8-row group
                const unsigned char *grp = zb + (((size_t)c * a.n_kt + kt) * (a.Mpad >> 3) + (m0 >> 3)) * 2048;
                const uint32_t o0 = (uint32_t)(m0 & 7) * 128 + ((((tt >> 3) ^ (m0 & 7)) << 4) | ((tt & 7) << 1));
                const uint32_t o1 = (uint32_t)(m1 & 7) * 128 + ((((tt >> 3) ^ (m1 & 7)) << 4) | ((tt & 7) << 1));
                x = make_float2(__half2float(*reinterpret_cast<const __half *>(grp + o0)), __half2float(*reinterpret_cast<const __half *>(grp + 1024 + o0)));
                y = make_float2(__half2float(*reinterpret_cast<const __half *>(grp + o1)), __half2float(*reinterpret_cast<const __half *>(grp + 1024 + o1)));
            } else {
                const float2 *zc = reinterpret_cast<const float2 *>(zb) + (size_t)c * a.M * a.n_t;
                x = zc[(size_t)(2 * st) * a.n_t + t];
                y = zc[(size_t)(2 * st + 1) * a.n_t + t];
            }
            if (a.poff) {
                x = cmulf(x, a.poff[2 * st]);
                y = cmulf(y, a.poff[2 * st + 1]);
            }
            float i_, q_, u_, v_;
            stokes4(x.x, x.y, y.x, y.y, i_, q_, u_, v_);
            I += i_;
            Q += q_;
            U += u_;
            V += v_;
        }
    }
    const float bp = a.bandpass[c] * a.inv_s, ps = bp * bp;
    red[0][threadIdx.x] = I * ps;
    red[1][threadIdx.x] = Q * ps;
    red[2][threadIdx.x] = U * ps;
    red[3][threadIdx.x] = V * ps;
    __syncthreads();
    const int n_u = kBfTBlock / a.t_int;
    for (int w = threadIdx.x; w < n_u * a.n_stokes; w += kBfTBlock) {
        const int k = w / n_u, ul = w % n_u;
        float s = 0.f;
        for (int i = 0; i < a.t_int; ++i) s += red[k][ul * a.t_int + i];
        const long long u = (long long)blockIdx.y * n_u + ul;
        if (u < a.n_out) a.out[(((size_t)bl * a.n_stokes + k) * a.C + c) * a.n_out + u] = s;
    }
}

}  // namespace

// Shared-memory plan of bf_tc_kernel for this plan's Mpad: accumulator columns N (4 per beam) such that W' and two stages fit.
// Returns false when not even 4 beams fit (too many stations for one CTA's shared memory).
bool bf_tc_shape(const cobalt_plan_s *p, int n_beams, int &bpb, int &stages, size_t &w_bytes, size_t &stage_bytes, size_t &smem) {
    const size_t budget = (size_t)227 * 1024 - 2048;            // alignment slack + barriers
    stage_bytes = (size_t)2 * p->Mpad * 256;
    const size_t k_atoms = ((size_t)2 * p->Mpad + 63) / 64;
    if (budget < 2 * stage_bytes + k_atoms * 16 * 128) return false;
    int n_max = (int)((budget - 2 * stage_bytes) / (k_atoms * 128)) / 16 * 16;
    if (n_max > 256) n_max = 256;
    if (n_max < 16) return false;
    const int bpb_max = n_max / 4;
    const int n_bb = (n_beams + bpb_max - 1) / bpb_max;
    bpb = ((n_beams + n_bb - 1) / n_bb + 3) / 4 * 4;            // even split, N = 4 bpb a multiple of 16
    w_bytes = k_atoms * (size_t)(4 * bpb) * 128;
    stages = (int)((budget - w_bytes) / stage_bytes);
    if (stages > 4) stages = 4;
    smem = 2048 + w_bytes + (size_t)stages * stage_bytes;
    return stages >= 2;
}

cudaError_t launch_beamform(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int b0, int nb, const BfCall &bc) {
    const long long n_out = p->n_t / bc.t_int;
    const bool tensor = p->mode == COBALT_MODE_TENSOR_FP16;
    const int n_tb = (int)((p->n_t + kBfTBlock - 1) / kBfTBlock);
    if (bc.product == COBALT_BF_INCOHERENT_STOKES) {
        IncArgs a;
        a.z = static_cast<const unsigned char *>(d_z);
        a.z_subband_bytes = p->z_subband_bytes;
        a.poff = p->d_poff;
        a.bandpass = bc.bandpass;
        a.out = static_cast<float *>(bc.out);
        a.n_t = p->n_t;
        a.n_out = n_out;
        a.S = p->S;
        a.M = p->M;
        a.Mpad = p->Mpad;
        a.C = p->C;
        a.n_kt = p->n_kt;
        a.n_stokes = bc.n_stokes;
        a.t_int = bc.t_int;
        a.tensor = tensor ? 1 : 0;
        a.inv_s = 1.f / p->zscale;
        incoherent_kernel<<<dim3((unsigned)(nb * p->C), (unsigned)n_tb), kBfTBlock, 0, st>>>(a);
        return cudaGetLastError();
    }
    if (!tensor) {
        BfSimtArgs a;
        a.z = static_cast<const float2 *>(d_z);
        a.z_subband_elems = p->z_subband_bytes / sizeof(float2);
        a.phase = p->d_phase;
        a.poff = p->d_poff;
        a.f_sb = p->d_f_sb;
        a.beam_delays = bc.beam_delays;
        a.bandpass = bc.bandpass;
        a.out = bc.out;
        a.f_s = p->f_s;
        a.n_t = p->n_t;
        a.n_out = n_out;
        a.S = p->S;
        a.M = p->M;
        a.C = p->C;
        a.b0 = b0;
        a.n_beams = bc.n_beams;
        int bpb = (int)(((size_t)200 * 1024) / ((size_t)p->M * sizeof(float2)));
        if (bpb < 1) return cudaErrorInvalidConfiguration;
        if (bpb > bc.n_beams) bpb = bc.n_beams;
        a.bpb = bpb;
        a.product = bc.product;
        a.n_stokes = bc.n_stokes;
        a.t_int = bc.t_int;
        const size_t smem = (size_t)bpb * p->M * sizeof(float2) + 4 * kBfTBlock * sizeof(float);
        cudaError_t e = cudaFuncSetAttribute(bf_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        bf_simt_kernel<<<dim3((unsigned)(nb * p->C), (unsigned)n_tb, (unsigned)((bc.n_beams + bpb - 1) / bpb)), kBfTBlock, smem, st>>>(a);
        return cudaGetLastError();
    }
    BfArgs a;
    int bpb = 0, stages = 0;
    size_t w_bytes = 0, stage_bytes = 0, smem = 0;
    if (!bf_tc_shape(p, bc.n_beams, bpb, stages, w_bytes, stage_bytes, smem)) return cudaErrorInvalidConfiguration;
    a.z = static_cast<const unsigned char *>(d_z);
    a.z_subband_bytes = p->z_subband_bytes;
    a.phase = p->d_phase;
    a.poff = p->d_poff;
    a.f_sb = p->d_f_sb;
    a.beam_delays = bc.beam_delays;
    a.bandpass = bc.bandpass;
    a.out = bc.out;
    a.f_s = p->f_s;
    a.n_t = p->n_t;
    a.n_out = n_out;
    a.S = p->S;
    a.M = p->M;
    a.Mpad = p->Mpad;
    a.C = p->C;
    a.n_kt = p->n_kt;
    a.n_tb = (p->n_kt + 1) / 2;
    a.b0 = b0;
    a.nb = nb;
    a.n_beams = bc.n_beams;
    a.bpb = bpb;
    a.n_bb = (bc.n_beams + bpb - 1) / bpb;
    a.N = 4 * bpb;
    a.product = bc.product;
    a.n_stokes = bc.n_stokes;
    a.t_int = bc.t_int;
    a.lg_t_int = 0;
    while ((1 << a.lg_t_int) < bc.t_int) ++a.lg_t_int;
    a.inv_s = 1.f / p->zscale;
    a.stages = stages;
    a.stage_bytes = (uint32_t)stage_bytes;
    a.w_bytes = (uint32_t)w_bytes;
    a.kt_bytes = (uint32_t)p->Mpad * 256;
    a.total_jobs = nb * p->C * a.n_bb;
    cudaError_t e = cudaFuncSetAttribute(bf_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int grid = a.total_jobs < p->sm_count ? a.total_jobs : p->sm_count;
    bf_tc_kernel<<<grid, kBfThreads, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace cobalt
