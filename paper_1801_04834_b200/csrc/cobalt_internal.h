// Internal declarations shared by the CUDA translation units of libcobalt_b200.so.
// Nothing here is part of the ABI (see include/cobalt.h) and nothing here is shared with oracle/.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>

#include <cstdint>
#include <string>
#include <vector>

#include "cobalt.h"

namespace cobalt {

constexpr int kTaps = 16;          // P:L360 FIR filter; BASELINE.json: 16-tap
constexpr int kSubTile = 16;       // spectra per FIR->FFT hand-over
constexpr int kKTile = 64;         // spectra per X-stage K tile (= one 128-byte fp16 row)
constexpr int kMaxMmaGroups = 2;   // MMA groups per X-stage job
constexpr int kBfTBlock = 2 * kKTile;   // beamformer: spectra per accumulator block (M of the instruction) and per CTA of its SIMT kernels
constexpr int kMaxGridYZ = 65535;  // CUDA's limit on gridDim.y / gridDim.z
constexpr int kStoreTile = 32;     // spectra per F-stage tensor store (half a k-tile row)
// streams (rows m) per F-stage tensor-store box: the CTA's 256 / C streams, at most 4 (all with the same m >> 2)
constexpr int kStoreBoxStreams(int C) { return 256 / C < 4 ? 256 / C : 4; }

// ---------------------------------------------------------------------------------------------
// Layout of the channelised intermediate ("z", step a7, "transposes data on write-back").
//
// TENSOR_FP16: per subband  [C][n_kt][Mpad/8 row groups][2 planes (re, im)][8 rows][64 t] fp16,
//   rows = inputs (2*station + pol) padded with zero rows to Mpad = round_up(2S, 16).  A row is 128 bytes
//   (64 spectra); the 16-byte chunk q (8 spectra) of row m sits at chunk q ^ (m & 7) of that row, i.e. every
//   [8 rows][128 B] block is one atom of the 128-byte-swizzled K-major shared-memory image the tcgen05
//   descriptors expect.  The two planes alternate atom by atom, so the same bytes can be read two ways:
//     one plane   = atoms 2048 bytes apart (descriptor SBO = 2048; the im plane starts 1024 bytes in);
//     both planes = atoms 1024 bytes apart (SBO = 1024): rows in the order re 0-7, im 0-7, re 8-15, ...
//   (the X-stage uses the second view for the small block the 128-row instruction cannot reach).
//   One (channel, k-tile) is one contiguous Mpad*256-byte span that the X-stage fetches with one plain
//   bulk copy, no tensor map.  Spectra t >= n_t are written as zeros.
// EXACT_FP32:  per subband  [C][M][n_t] float2.
// ---------------------------------------------------------------------------------------------

// One X-stage job = one set of rows of a (subband, channel) k-tile loaded to shared memory plus up
// to kMaxMmaGroups accumulator groups computed from it (see xstage_tc.cu).
struct XMmaGroup {
    int a_row;      // first row of the A operand, relative to the first loaded row (m rows used)
    int b_row;      // first row of the B operand, relative to the first loaded row
    int n;          // number of B rows = accumulator columns (multiple of 16, <= 256)
    int tmem_col;   // first TMEM column of the Re accumulator; Im follows at tmem_col + n
    int out_row;    // global input index of A row 0
    int out_col;    // global input index of B row 0
    int m;          // instruction M: 128, or 64 (accumulator row r then sits in TMEM lane 32 (r / 16) + r % 16)
    int row_min;    // rows (global input index) below this are another group's job and are not stored
    int kind;       // 0: four single-plane products into Re | Im accumulators (2 n columns);
                    // 1: one both-plane product [Zr; Zi] [Zr; Zi]^T of the rows a_row.. (n = 2 x rows per plane,
                    //    n columns), combined into Re / Im by the epilogue
};
struct XJob {
    int ld_row[2];     // two row ranges of the [Mpad][64] block copied to smem back to back
    int ld_nrows[2];   // (second may be empty)
    int n_groups;
    int tmem_cols;     // power of two >= 32 to allocate
    XMmaGroup g[kMaxMmaGroups];
};

// Events bracketing the four kernels of one chunk: e[0] | phase table | e[1] | F-stage | e[2] | history | e[3] | X-stage | e[4]
struct StageEvents {
    cudaEvent_t e[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
};

}  // namespace cobalt

struct cobalt_plan_s {
    int S = 0, B = 0, C = 0, T = 0, bits = 0, mode = COBALT_MODE_TENSOR_FP16;   // bits: what the fused kernel reads (16 or 8)
    int bits_in = 0;                   // what the caller passes (16, 8 or 4); 4 is expanded to 8 by the ingest pre-pass
    int layout = COBALT_LAYOUT_PLANAR; // order of the caller's samples (cobalt_set_input_layout)
    int dumps = 1;                     // D, cobalt_set_dumps
    long long N_in = 0;                // stream stride of the caller's samples (cobalt_set_coarse_delays), >= N
    int *d_coarse = nullptr;           // [S] first sample of each station's block, or nullptr (all zero)
    float2 *d_poff = nullptr;          // [2S] exp(-i phase0) per stream, or nullptr (cobalt_set_phase_offsets)
    void *d_ingest = nullptr;          // planar copy of one chunk for pol-minor / 4-bit input
    int x_splits = 1;                  // X-stage: k-range of a (dump, subband, channel) split over this many jobs
    float2 *d_xpart = nullptr;         // partial visibilities of the split jobs of one chunk
    long long N = 0, n_t = 0, N_u = 0, n_bl = 0;
    int M = 0, Mpad = 0, n_kt = 0;
    int chunk = 1;
    int chunk_user = 0;                // what cobalt_set_chunk_subbands asked for (0 = never called: the default rule); kept by cobalt_set_mode
    int host_chunk = 1;                // subbands per group of cobalt_process_host (<= chunk)
    int device = 0, sm_count = 0;
    double f_s = 195312.5;
    std::vector<double> f_sb;
    bool f_sb_user = false;            // cobalt_set_subband_frequencies was called: cobalt_set_sample_rate keeps the ladder
    bool scratch_ok = false;           // alloc_scratch completed; cobalt_process* refuse to run otherwise
    double *d_f_sb = nullptr;          // [B]
    float *d_weights = nullptr;        // [16][C], tap k (0 = newest block), branch ph
    std::vector<float> h_weights;
    void *d_hist[2] = {nullptr, nullptr};   // raw integer samples [B][S][2][15 C][2]; ping-pong
    int hist_cur = 0;
    float2 *d_phase = nullptr;         // [B][S][C]  b[j] exp(-2 pi i frac(f tau)), built once per call; applied by the X-stage
    float *d_dstep = nullptr;          // [B][S][C] phase step per spectrum in cycles (cobalt_process_interp)
    float zscale = 1.f;                // power-of-two scale s of the fp16 intermediate (reading R1): 2^-e,
                                       // e = ceil(log2(amp_max / 32768)) in TENSOR mode, 1 in EXACT mode
    float amp_max = 0.f;               // worst-case |F| for full-scale input: sum|g| * sqrt(2) * 2^(bits-1)
    void *d_z = nullptr;               // intermediate of one chunk (layout per mode)
    CUtensorMap zmap;                  // TENSOR mode: d_z as (spectrum-in-k-tile, chunk subband * C + channel, plane, row m, k-tile)
    size_t z_subband_bytes = 0;
    std::vector<cobalt::XJob> jobs;    // X-stage jobs of one (subband, channel)
    cobalt::XJob *d_jobs = nullptr;
    size_t x_smem_bytes = 0;
    int x_stages = 0;
    bool x_staged = false;             // X-stage epilogue through a shared-memory image of the channel's output block
    size_t x_out_off = 0;
    size_t x_rot_bytes = 0;            // one of the two per-job rotation tables of the X-stage epilogue
    size_t scratch_bytes = 0;
    // host-buffer path
    cudaStream_t hs[3] = {nullptr, nullptr, nullptr};
    void *d_in[2] = {nullptr, nullptr};
    void *d_out[2] = {nullptr, nullptr};
    double *d_delays_h = nullptr;
    double *d_delays_end_h = nullptr;
    unsigned char *d_valid_h = nullptr;    // [B][S][n_kt] flags of a cobalt_process_host_ex call
    unsigned int *d_counts_h = nullptr;    // [B][D][n_bl] weights of a cobalt_process_host_ex call
    float *d_bandpass_h = nullptr;
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_cmp[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
    // timing
    bool timing = false;
    std::vector<cobalt::StageEvents> events;
    int n_chunks_timed = 0;
    int launches = 0;
    mutable std::string err;
};

namespace cobalt {

inline size_t sample_bytes(int bits) { return bits == 16 ? 4 : 2; }   // one complex sample
// the history carry overwrites the buffer it was read from (no host-side state changes from call to call: a single
// captured call can be replayed); only blocks shorter than the history itself alternate between the two buffers
inline bool history_in_place(const cobalt_plan_s *p) { return p->N_u >= (long long)(kTaps - 1) * p->C; }

// The per-call inputs beyond the plan (cobalt_io_t) as the launch helpers see them for one chunk.
struct FCall {
    const double *delays_end = nullptr;    // device [S] or nullptr (static delay)
    const unsigned char *valid = nullptr;  // device [B][S][n_kt] or nullptr
    const int *coarse = nullptr;           // device [S] or nullptr: first sample of each station's block
    long long n_in = 0;                    // stream stride of the samples the fused kernel reads
};

// What the X-stage applies to the raw correlations of one chunk: V_ik <- V_ik w_i conj(w_k) / s^2 with
// w_m = phase[(b0 + subband) S + m / 2][channel] * poff[m] (steps a5, a6 and reading A22 moved behind the integration: the
// same product, one multiplication per visibility instead of one per sample), s = the fp16 operand scale.
struct XCall {
    const float2 *phase = nullptr;     // plan's d_phase [B][S][C], or nullptr: no rotation (cobalt_debug_correlate)
    const float2 *poff = nullptr;      // [2S] or nullptr
    int b0 = 0;                        // first subband of the chunk
    float inv_s2 = 1.f;
};

// One chunk of a cobalt_beamform call as the launch helper sees it (beamform.cu).
struct BfCall {
    const double *beam_delays = nullptr;   // device [n_beams][S] seconds (coherent products)
    const float *bandpass = nullptr;       // device [C]
    void *out = nullptr;                   // first subband of the chunk in the caller's output
    int n_beams = 0, product = 0, n_stokes = 1, t_int = 1;
};

// fstage.cu ---------------------------------------------------------------------------------
cudaError_t launch_phase_table(const cobalt_plan_s *p, cudaStream_t st, const double *d_delays,
                               const float *d_bandpass, int b0, int nb, const double *d_delays_end);
// samples_b0 points at the first subband of the chunk [b0, b0 + nb)
cudaError_t launch_fstage(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb, const FCall &call);
cudaError_t launch_history_update(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int b0, int nb, const FCall &call);
cudaError_t launch_unpack(cudaStream_t st, int bits, const void *d_in, long long n, float *d_out);
// caller's order / width -> planar int16 / int8 [nb][2S][N] in d_out, coarse offsets applied (layout.cu)
cudaError_t launch_ingest(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int nb, void *d_out);
cudaError_t launch_valid_counts(const cobalt_plan_s *p, cudaStream_t st, const unsigned char *d_valid, int b0, int nb, unsigned int *d_counts);
// layout.cu ---------------------------------------------------------------------------------
// z of one subband -> [C][2S][n_t] complex64, rotated like the X-stage would (xc) so that the tap shows steps a1-a7
cudaError_t launch_z_to_float(const cobalt_plan_s *p, cudaStream_t st, const void *d_zsub, float2 *d_out, const XCall &xc);
cudaError_t launch_float_to_z(const cobalt_plan_s *p, cudaStream_t st, const float2 *d_in, void *d_zsub);
// xstage_simt.cu ----------------------------------------------------------------------------
// d_vis points at subband b0 of dump 0; dump d is dump_stride float2 further
cudaError_t launch_xstage_simt(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int nb, float2 *d_vis, size_t dump_stride, const XCall &xc);
// xstage_tc.cu ------------------------------------------------------------------------------
void build_xjobs(cobalt_plan_s *p);
cudaError_t launch_xstage_tc(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int nb, float2 *d_vis, size_t dump_stride, const XCall &xc);

// beamform.cu -------------------------------------------------------------------------------
// p->d_phase must hold the pure station phases of the call (launch_phase_table with d_bandpass == nullptr)
cudaError_t launch_beamform(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int b0, int nb, const BfCall &bc);
bool bf_tc_shape(const cobalt_plan_s *p, int n_beams, int &bpb, int &stages, size_t &w_bytes, size_t &stage_bytes, size_t &smem);

}  // namespace cobalt
