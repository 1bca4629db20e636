/*
 * cobalt.h -- C ABI of the B200-native Cobalt correlator hot path.
 *
 * The main thing built is the correlator pipeline of "Cobalt: A GPU-based correlator and
 * beamformer for LOFAR" (arXiv:1801.04834), sec 7.5 ("P:L360"):
 *
 *   "The correlator pipeline first channelizes subbands in a polyphase filter using FIR
 *    filters and FFT kernels.  We carry FIR filter history samples across to the next block.
 *    The pipeline then applies fine delay compensation and bandpass correction. [...] the
 *    delay and bandpass kernel transposes data on write-back [...].  The last kernel computes
 *    the correlations of all pairs of antenna fields and averages in time to approximately 1 s."
 *
 * plus the fixed->floating conversion of P:L89 (sec 3.2) and the precision rule of P:L368
 * (phase angles in double precision, everything else single precision).  The paper prints
 * no formulas; the exact arithmetic is the reading listed in DESIGN.md ("Readings A1..A32",
 * taken from SURVEY.md sec 8(c)), summarised at cobalt_process() below.  On top of it sit the
 * rows of SURVEY.md sec 8(f): time-varying delays, phase offsets, dumps, lost-data flags, coarse
 * delays, pol-minor and 4-bit input (cobalt_process_ex and the setters), the beamformer of
 * P:L362-366 at the plan's channel count (cobalt_beamform), and one plan-less entry point for
 * callers that must not allocate (cobalt_correlate_noalloc).
 *
 * Conventions
 *   - Every function returns a cobalt_status (0 = OK, negative = error) and never throws,
 *     aborts or prints.  cobalt_strerror() names a code; cobalt_last_error() gives detail.
 *   - "device" pointers are CUDA device pointers valid on the plan's device; "host" pointers
 *     are ordinary (for cobalt_process_host: preferably pinned) host memory.
 *   - The caller owns every buffer it passes and the stream.  The plan owns the FIR weights,
 *     FIR history, phase table and the intermediate (channelised) scratch.
 *   - cobalt_process() only ENQUEUES work on `cuda_stream` and returns; buffers must stay
 *     alive and unmodified until the stream reaches the end of the call.
 *   - All sizes are validated; nothing is read or written outside the documented extents.
 *   - One plan = one stream = one host thread at a time: cobalt_process*, cobalt_beamform and the
 *     setters update plan state (launch counters, event lists, which history buffer is current)
 *     without locking, and the plan's scratch is shared by every call on it.  Use one plan per
 *     concurrent stream; different plans are independent.
 *   - There is no CPU fallback: without a CUDA device of compute capability 10.x every
 *     entry point that needs the device returns COBALT_ERR_UNSUPPORTED_DEVICE / COBALT_ERR_CUDA.
 *
 * Symbols (S stations, B subbands, C channels, T = 16 taps, N samples per pol per subband
 * per call, n_t = floor(N/C) spectra, N_u = n_t*C consumed samples, n_bl = S(S+1)/2).
 */
#ifndef COBALT_B200_H
#define COBALT_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cobalt_plan_s cobalt_plan_t;   /* opaque */

typedef enum {
    COBALT_OK = 0,
    COBALT_ERR_BAD_ARG = -1,             /* argument out of range / NULL pointer          */
    COBALT_ERR_NO_MEMORY = -2,           /* host or device allocation failed              */
    COBALT_ERR_CUDA = -3,                /* a CUDA runtime call failed (see last_error)   */
    COBALT_ERR_UNSUPPORTED_DEVICE = -4   /* no device, or device is not sm_100 class      */
} cobalt_status;

typedef enum {
    /* X-stage on tcgen05 tensor cores, fp16 operands, fp32 accumulation in TMEM.
     * Tolerance vs the float64 oracle: ||dV||_F / ||V||_F <= 2e-3 per (subband, channel).
     * The fp16 operands carry a power-of-two scale fixed by input_bits and the FIR gain so that full-scale
     * input cannot overflow (undone exactly in the X-stage epilogue). */
    COBALT_MODE_TENSOR_FP16 = 0,
    /* Everything in fp32 (SIMT FMA correlator).  Tolerance: max |dV| / sqrt(V_ii V_kk) <= 1e-4. */
    COBALT_MODE_EXACT_FP32 = 1
} cobalt_mode;

typedef struct {
    int stations, subbands, channels, taps, input_bits, mode;
    long long samples_per_integration;   /* N                                              */
    long long n_spectra;                 /* n_t = floor(N / C)   (reading A11)             */
    long long n_consumed;                /* N_u = n_t * C                                   */
    long long n_baselines;               /* n_bl = S (S+1) / 2, autocorrelations included  */
    long long input_bytes;               /* B*S*2*N*2*(bits/8): extent read from `samples` */
    long long output_bytes;              /* D*B*C*n_bl*4*8: extent written to `visibilities` */
    long long scratch_bytes;             /* device memory owned by the plan                */
    int chunk_subbands;                  /* subbands processed per internal launch group   */
    int sm_count;
    double sample_rate_hz;
    int dumps;                           /* D, cobalt_set_dumps                               */
    int n_tiles;                         /* ceil(n_t / 64): extent of `valid` per station   */
    long long samples_allocated;         /* stream stride of `samples` (cobalt_set_coarse_delays) */
} cobalt_info_t;

/* ---------------------------------------------------------------------------------------
 * cobalt_plan: validate the observation constants, allocate all device state on the current
 * CUDA device, build the FIR weights.  ("Most kernel parameters are fixed throughout
 * an observation"; the paper's run-time compilation becomes template specialisation on
 * (channels, input_bits).)
 *   stations  >= 1 (dual polarisation each), subbands >= 1,
 *   channels  in {16, 64, 256}, taps == 16, input_bits in {16, 8, 4}
 *             (4: one byte per complex sample, re in the low nibble, im in the high nibble, two's complement
 *              -8 .. 7, reading A27 / P:L121; expanded to int8 by a pre-pass, see cobalt_set_input_layout),
 *   samples_per_integration >= channels.
 * The prototype filter is the Hann-windowed sinc of reading A1 (== scipy.signal.firwin(16 C,
 * 1/C, window="hann")), evaluated in double and rounded once to fp32.  History starts as zeros
 * (reading A3).  Default subband centre frequencies f_sb[s] = 100 MHz + (12 + s) * f_s, default
 * f_s = 195312.5 Hz (reading A6); default mode COBALT_MODE_TENSOR_FP16.
 * On failure *out = NULL. */
int cobalt_plan(cobalt_plan_t **out, int stations, int subbands, int channels, int taps,
                long long samples_per_integration, int input_bits);

/* ---------------------------------------------------------------------------------------
 * cobalt_process: one integration period of the whole hot path, enqueued on `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *
 *   d_samples      device, [B][S][2 pol][N][2 (re,im)] int16 (input_bits 16) or int8 (8), or
 *                  [B][S][2 pol][N] bytes holding one 4-bit complex sample each (input_bits 4, A27),
 *                  time contiguous per polarisation (reading A13; cobalt_set_input_layout selects
 *                  LOFAR's pol-minor wire order instead); read only.
 *   d_delays       device, [S] double, seconds; one value per station, both pols (A7).
 *   d_bandpass     device, [C] float, real weight multiplying the voltages (A8).
 *   d_visibilities device, [B][C][n_bl][2][2] complex64 (float re, float im); fully
 *                  overwritten.  Baseline (i <= k) at index k(k+1)/2 + i, then
 *                  [pol of i][pol of k] (A9).  Must be 16-byte aligned in COBALT_MODE_TENSOR_FP16
 *                  (COBALT_ERR_BAD_ARG otherwise); d_samples needs the alignment of one complex
 *                  sample (4 / 2 bytes); 16-byte aligned streams take the bulk-copy path.
 *
 * Per subband s and stream (station a, pol p), with x = the integer samples as floats
 * (bit-exact two's complement value, A12) preceded by the carried history:
 *   y[t][ph] = sum_{k<16} g[(15-k) C + ph] x[(t-k) C + ph]                      (A2)
 *   D[t][c]  = sum_ph y[t][ph] exp(-2 pi i ph c / C),  F[t][j] = D[t][(j + C/2) mod C]  (A4, A5)
 *   f[s][j]  = f_sb[s] + (j - C/2) f_s / C                                       (A6)
 *   z[t][j]  = F[t][j] b[j] exp(-2 pi i frac(f[s][j] tau_a))   (frac in fp64)
 *   V[s][j][bl(i,k)][p][q] = sum_t z_{i,p}[t][j] conj(z_{k,q}[t][j])              (A9, A10)
 * and the last 15 C consumed samples of every stream become the new history (stateful!).
 * The factor w_a[j] = b[j] exp(-2 pi i frac(f[s][j] tau_a)) is constant over the call, so the library correlates F and
 * multiplies each visibility by w_i conj(w_k) (the same product; w from the fp64 phase table, the multiplication in fp32).
 * The call only enqueues kernels on `cuda_stream` (no synchronisation, no allocation) and changes no host-side state, so a
 * single call can be captured in a CUDA graph and replayed block after block (the history is carried in place).  Exception:
 * blocks shorter than the history (N_u < 15 C) alternate between two history buffers; capture those in pairs.
 * Only the first N_u = floor(N/C) C samples of each stream are consumed (A11). */
int cobalt_process(cobalt_plan_t *plan, void *cuda_stream, const void *d_samples,
                   const double *d_delays, const float *d_bandpass, void *d_visibilities);

/* Same computation with HOST buffers (same layouts).  The library streams subband chunks
 * host->device, computes, and streams visibilities device->host on internal streams, double
 * buffered, and returns after everything has completed (synchronous).  Pinned host memory is
 * needed for the copies to overlap; pageable memory works but serialises. */
int cobalt_process_host(cobalt_plan_t *plan, const void *h_samples, const double *h_delays,
                        const float *h_bandpass, void *h_visibilities);
/* cobalt_process_host with the optional members of cobalt_io_t (declared below, at cobalt_process_ex): every pointer
 * of `h_io` is a HOST pointer with the layout of its device counterpart -- samples, delays, bandpass, visibilities
 * ([D][B][C][n_bl][2][2] with D = cobalt_set_dumps) required; delays_end [S], valid [B][S][n_tiles] and valid_counts
 * [B][D][n_bl] optional (NULL = absent).  In the paper the lost-data flags arrive from the host side together with the
 * samples and the blocks are streamed through pinned buffers: this is that path.  The small
 * arrays are copied whole ahead of the first group, the samples and visibilities group by group, double buffered, on
 * three internal streams; valid_counts comes back after the last group.  Synchronous like cobalt_process_host, same
 * history carry; results are bit-identical to cobalt_process_ex on device copies of the same buffers. */
struct cobalt_io_s;
int cobalt_process_host_ex(cobalt_plan_t *plan, const struct cobalt_io_s *h_io);

/* cobalt_process with a delay that varies over the block ("we compute the
 * channel-dependent phase angles [from the residual delay at the start and the end of the block] in double
 * precision ... interpolated linearly ... sin/cos and complex multiplication in single precision").  Reading A21
 * (DESIGN.md): spectrum t (0 <= t < n_t) of station a is rotated with
 *     tau_a(t) = delays_begin[a] + (delays_end[a] - delays_begin[a]) * t / n_t,
 * z = F * b[j] * exp(-2 pi i f[s][j] tau_a(t)).  The phase at t = 0 and the phase step per spectrum
 * f (tau_e - tau_b) / n_t are computed in fp64; the per-spectrum factor in fp32, accurate while
 * |f (tau_e - tau_b)| stays below about 100 cycles per block.  d_delays_end: device [S] doubles; everything else as
 * cobalt_process (same buffers, asynchrony, history carry, errors).  delays_end == delays_begin gives
 * cobalt_process to rounding. */
int cobalt_process_interp(cobalt_plan_t *plan, void *cuda_stream, const void *d_samples,
                          const double *d_delays_begin, const double *d_delays_end, const float *d_bandpass,
                          void *d_visibilities);


/* ---------------------------------------------------------------------------------------
 * cobalt_process_ex: cobalt_process with every optional input and output of SURVEY.md sec 8(f) rows 1-2 in one
 * argument block (cobalt_process / cobalt_process_interp are this call with the optional members NULL).
 * All pointers are DEVICE pointers; same asynchrony, history carry and errors as cobalt_process.
 *   samples, delays, bandpass, visibilities   as cobalt_process (delays = the delay at the first spectrum);
 *   delays_end     NULL, or [S] double: the delay runs linearly to this value over the block (cobalt_process_interp, A21);
 *   valid          NULL (nothing lost), or [B][S][n_tiles] bytes, n_tiles = ceil(n_t / 64): 0 marks the 64 spectra
 *                  [64 v, 64 v + 64) of a station (both polarisations) as lost ("lost data ... encoded in the
 *                  metadata", reading A24): their channelised samples count as zero in the correlation; the FIR still
 *                  runs over whatever the input holds;
 *   valid_counts   NULL, or [B][D][n_bl] unsigned: the number of spectra of dump d in which both stations of the
 *                  baseline are valid -- the weight that goes with the visibility (n_t per dump when valid == NULL);
 *   visibilities   [D][B][C][n_bl][2][2] complex64 with D = cobalt_set_dumps (default 1: the layout of cobalt_process).
 */
typedef struct cobalt_io_s {
    const void *samples;
    const double *delays;
    const double *delays_end;
    const float *bandpass;
    const unsigned char *valid;
    void *visibilities;
    unsigned int *valid_counts;
} cobalt_io_t;
int cobalt_process_ex(cobalt_plan_t *plan, void *cuda_stream, const cobalt_io_t *io);

/* ---------------------------------------------------------------------------------------
 * cobalt_beamform: the beamformer pipeline of SURVEY.md sec 8(f) row 4 for one block, at the
 * plan's channel count ("Cobalt performs delay compensation, bandpass correction and beamforming at 256 channels per
 * subband"); enqueued on `cuda_stream` like cobalt_process, with the same channelisation (steps a1-a4), delay
 * compensation, bandpass, phase offsets, coarse delays, input layouts and valid-sample flags, and the same history
 * carry (stateful; a plan serves either the correlator or the beamformer stream of an observation).  Sharing the
 * correlator's 16-tap channeliser is a reading (A28): in the paper the beamformer "cannot share initial steps
 * with the correlator" and runs a 256-channel PPF of its own; what this call adds is the beam-forming step.
 * Not built (A32): the transform to the requested output resolution with its transposes, and beam
 * delays that vary over the block (beam_delays is one value per (beam, station) and call).
 * With z[a][p][t][j] the delay-compensated, bandpass-corrected channelised sample of station a, polarisation p
 * (cobalt_process, line "z[t][j] = ..."):
 *   coherent beam b (reading A28; "adjusts the beam direction with a phase shift and sums over antenna fields",
 *   P:L368 "The beamforming kernel operates in a similar way": the phase angle in fp64):
 *       Y[b][p][j][t] = sum_a exp(-2 pi i frac(f[s][j] tau_{b,a})) z[a][p][t][j]
 *   Stokes parameters of a dual-polarisation sample (X, Y) (reading A29):
 *       I = |X|^2 + |Y|^2,  Q = |X|^2 - |Y|^2,  U = 2 Re(X conj(Y)),  V = 2 Im(X conj(Y))
 *   time integration (reading A30; Stokes only, "complex voltages cannot be time averaged"): output sample u is the sum
 *       of the t_int spectra [u t_int, (u+1) t_int); n_out = floor(n_t / t_int), the tail is not consumed
 *   incoherent beam (reading A31; "first computes Stokes parameters and then sums over antenna fields"):
 *       S_k[j][t] = sum_a stokes_k(z[a][X][t][j], z[a][Y][t][j]).
 * No division by the number of stations or samples.  The paper's final step, "transforms to the requested output
 * resolution" (an inverse and a second FFT), is not part of this call.
 *   samples, delays, delays_end, bandpass, valid   device, as in cobalt_io_t (delays_end and valid may be NULL)
 *   beam_delays  device [n_beams][S] double, seconds: tau_{b,a}, the delay of station a for beam b relative to the phase
 *                centre, with the sign sense of `delays`; ignored for COBALT_BF_INCOHERENT_STOKES
 *   n_beams      >= 1 (coherent products)
 *   product      COBALT_BF_COHERENT_VOLTAGES   out = [B][n_beams][2 pol][C][n_t] complex64
 *                COBALT_BF_COHERENT_STOKES     out = [B][n_beams][n_stokes][C][n_out] float
 *                COBALT_BF_INCOHERENT_STOKES   out = [B][n_stokes][C][n_out] float
 *   n_stokes     1 (I) or 4 (I, Q, U, V); t_int a power of two in [1, 128] (both ignored for voltages)
 *   out          device, 8-byte aligned, fully overwritten.
 * COBALT_MODE_TENSOR_FP16: the coherent sum runs on tcgen05 from the fp16 intermediate (fp16 weights, fp32 accumulation);
 * tolerance vs the float64 oracle ||dY||_F / ||Y||_F <= 2e-3 per (subband, channel) (same for the Stokes outputs);
 * needs 2 S <= 208 (COBALT_ERR_BAD_ARG otherwise).  COBALT_MODE_EXACT_FP32: fp32 FMAs, 1e-4 of the same norm.
 * For t_int > 32 the tensor path adds two or four partial sums per output sample with atomics (t_int = 128: the order of
 * four fp32 additions is not fixed). */
#define COBALT_BF_COHERENT_VOLTAGES 0
#define COBALT_BF_COHERENT_STOKES 1
#define COBALT_BF_INCOHERENT_STOKES 2
typedef struct {
    const void *samples;
    const double *delays;
    const double *delays_end;
    const float *bandpass;
    const unsigned char *valid;
    const double *beam_delays;
    int n_beams, product, n_stokes, t_int;
    void *out;
} cobalt_bf_io_t;
int cobalt_beamform(cobalt_plan_t *plan, void *cuda_stream, const cobalt_bf_io_t *io);
/* Extent in bytes that cobalt_beamform writes to `out` for these settings (0 on bad arguments). */
long long cobalt_beamform_output_bytes(const cobalt_plan_t *plan, int n_beams, int product, int n_stokes, int t_int);

/* Frees all plan state.  cobalt_destroy(NULL) is a no-op returning COBALT_OK.  The caller must
 * have synchronised every stream that still runs work of this plan. */
int cobalt_destroy(cobalt_plan_t *plan);

/* --------------------------------------------------------------------------- settings */
/* Subband centre (sky) frequencies in Hz, host array [B] (A6).  Takes effect next call. */
int cobalt_set_subband_frequencies(cobalt_plan_t *plan, const double *h_hz);
/* Subband sample rate f_s in Hz (A6: the channel spacing is f_s / C).  While cobalt_set_subband_frequencies has not
 * been called the default ladder f_sb[s] = 100 MHz + (12 + s) f_s is rebuilt with the new rate; a ladder the caller
 * has set is kept as it is.  Takes effect next call. */
int cobalt_set_sample_rate(cobalt_plan_t *plan, double hz);
/* Reading A22 ("bandpass and clock corrections"): a constant phase per (station, polarisation) with the
 * sign sense of the delay term, z <- z exp(-i phase0[a][p]).  h_phase0: host [S][2] doubles, radians, or NULL = none.
 * Applied in fp32 together with the delay rotation: to the visibilities in the X-stage epilogue (V_ik *= w_i conj(w_k)) and
 * to the beam weights of cobalt_beamform.  Takes effect next call. */
int cobalt_set_phase_offsets(cobalt_plan_t *plan, const double *h_phase0);
/* Reading A25 ("coarse delay compensation ... by shifting"): station a's block of N samples starts at sample
 * h_offsets[a] of its input stream, which is samples_allocated >= N + max offset samples long (the stream stride of
 * d_samples becomes samples_allocated).  Applied by the F-stage's loads (free when the offset is a multiple of 16 bytes;
 * other offsets take a slower element-wise load path).  The FIR history is the last 15 C samples the previous call
 * consumed of the shifted stream.  h_offsets: host [S] ints >= 0, or NULL = none (and samples_allocated = N). */
int cobalt_set_coarse_delays(cobalt_plan_t *plan, const int *h_offsets, long long samples_allocated);
/* Reading A23: D dumps per block.  Dump boundaries fall on multiples of 64 spectra: D must divide
 * n_tiles = ceil(n_t / 64); dump d integrates the spectra [d L, min((d + 1) L, n_t)), L = 64 n_tiles / D.  The
 * visibility buffer becomes [D][B][C][n_bl][2][2]. */
int cobalt_set_dumps(cobalt_plan_t *plan, int dumps_per_block);
/* Reading A26: order of d_samples.  COBALT_LAYOUT_PLANAR (default) = [B][S][2 pol][N][2]; COBALT_LAYOUT_POL_MINOR =
 * LOFAR's wire order [B][S][N][2 pol][2] (time-major, polarisation-minor).  Pol-minor input (and 4-bit input in either
 * order) goes through a re-ordering pre-pass into plan-owned scratch (one extra read and write of the input). */
#define COBALT_LAYOUT_PLANAR 0
#define COBALT_LAYOUT_POL_MINOR 1
int cobalt_set_input_layout(cobalt_plan_t *plan, int layout);
/* Switch COBALT_MODE_*; reallocates the intermediate scratch, keeps the history and a launch-group size set with
 * cobalt_set_chunk_subbands (otherwise the default group size of the new mode applies). */
int cobalt_set_mode(cobalt_plan_t *plan, int mode);
/* Subbands per internal launch group (>= 1, clipped to B).  Reallocates scratch.  Default: as many as fit in 8 GiB of
 * intermediate (at most a quarter of the free device memory), split evenly over the call; cobalt_process_host moves
 * and computes in groups of about 1 GiB. */
int cobalt_set_chunk_subbands(cobalt_plan_t *plan, int chunk);
/* Zero the FIR history (as after cobalt_plan).  Enqueued on the legacy default stream and
 * synchronised before returning. */
int cobalt_reset(cobalt_plan_t *plan);
int cobalt_info(const cobalt_plan_t *plan, cobalt_info_t *info);
const char *cobalt_strerror(int status);
/* Text of the most recent failure on this plan (valid until the next call on it). */
const char *cobalt_last_error(const cobalt_plan_t *plan);

/* --------------------------------------------------------------------------- measurement */
/* When enabled, cobalt_process() brackets each stage of each chunk with CUDA events on the
 * caller's stream.  cobalt_get_timing() synchronises those events and returns, for the most
 * recent cobalt_process() call, the summed device time in ms of the F-stage kernels (phase
 * table + unpack/FIR/FFT/rotate/transpose + history update) and of the X-stage kernels, and
 * the number of kernels the call launched.  Any output pointer may be NULL. */
int cobalt_set_timing(cobalt_plan_t *plan, int enabled);
int cobalt_get_timing(cobalt_plan_t *plan, double *f_stage_ms, double *x_stage_ms, int *kernel_launches);
/* The same, per kernel: ms4[0..3] = summed device time over the call's chunks of the phase-table kernel,
 * the fused F-stage kernel (unpack+FIR+FFT+rotate+bandpass+transpose), the history-carry kernel and
 * the X-stage kernel; the roofline figures of bench.py divide by ms4[1] and ms4[3]. */
int cobalt_get_kernel_timing(cobalt_plan_t *plan, double *ms4, int *kernel_launches);

/* --------------------------------------------------------------------------- debug taps */
/* (used by the parity tests to pin individual steps; not needed in production)           */
/* FIR weights exactly as the kernels use them, host [16][C] float, weight of tap k (k = 0 is
 * the newest block) and branch ph at [k*C + ph] == fp32(g[(15-k) C + ph]). */
int cobalt_debug_fir_weights(const cobalt_plan_t *plan, float *h_weights);
/* Step a1 alone: n integer components (int16 or int8 per input_bits) -> n floats, device; input_bits 4: n BYTES ->
 * 2 n floats. */
int cobalt_debug_unpack(void *cuda_stream, int input_bits, const void *d_in, long long n, float *d_out);
/* Steps a1-a7 for ONE subband `sb` of d_samples (full [B][..] array as in cobalt_process):
 * d_z receives z as [C][2S][n_t] complex64 (input index = 2*station + pol).  Reads the history
 * of that subband but does NOT advance it.  In TENSOR_FP16 mode the values are the fp16
 * operands that the X-stage consumes, converted back to fp32 and multiplied by the rotation w_a[j] the X-stage applies. */
int cobalt_debug_channelised(cobalt_plan_t *plan, void *cuda_stream, const void *d_samples,
                             const double *d_delays, const float *d_bandpass, int sb, void *d_z);
/* Step a8-a9 alone for one subband: d_z [C][2S][n_t] complex64 (caller supplied) ->
 * d_vis [C][n_bl][2][2] complex64, through the X-stage of the current mode. */
int cobalt_debug_correlate(cobalt_plan_t *plan, void *cuda_stream, const void *d_z, void *d_vis);

/* --------------------------------------------------------------------------- no-allocation entry point */
/* cobalt_correlate_noalloc: steps a8-a9 ("computes the correlations of all pairs of antenna fields and averages
 * in time") of ONE subband without a plan and without a single device or pinned-host allocation, for callers that must
 * not allocate: a real-time pipeline that took all its buffers from pools before the observation started
 * cannot afford cudaMalloc / cudaFree in mid-run -- both synchronise the whole device, so every stream stalls and a
 * late block of antenna data is dropped -- and on a GPU whose memory is budgeted to the last buffer they may
 * fail; the same goes for code running inside a host application that owns all device memory through its own pool.
 * Every other entry point needs a cobalt_plan, and cobalt_plan allocates.
 *
 * The arithmetic is that of COBALT_MODE_EXACT_FP32 (fp32 FMAs; tolerance vs the float64 oracle 1e-4 of
 * sqrt(V_ii V_kk)), organised like the split X-stage: the time range is cut into at most COBALT_NOALLOC_MAX_SLICES
 * slices whose partial visibilities are added in slice order, so the result is deterministic (it differs from
 * cobalt_debug_correlate only by the order of the fp32 additions).  The partial visibilities live in a fixed
 * COBALT_NOALLOC_SCRATCH_BYTES array inside the library's device image instead of in allocated memory.  Consequences:
 *   - every GPU on which the library's module is loaded holds those 16 MiB until the process exits;
 *   - sizes are limited: channels * n_bl <= COBALT_NOALLOC_MAX_CHANNEL_BASELINES (n_bl = S (S + 1) / 2; e.g. S <= 63
 *     at 64 channels, S <= 31 at 256).  Anything larger returns COBALT_ERR_BAD_ARG with the numbers in h_err and
 *     launches nothing;
 *   - the FIRST call on a device looks up where the array lives on that device (cudaGetSymbolAddress, under a host
 *     mutex) and remembers it; make that first call during start-up, with the device current, before any stream
 *     capture is begun on it.  Later calls on that device only launch two kernels on `cuda_stream`;
 *   - all calls on a device share the array.  It needs no clearing (each call overwrites every slot it later reads),
 *     and calls on the same stream are safe.  Calls that can overlap on the GPU -- different streams, or several host
 *     threads each with a stream -- race on it and produce wrong output; the caller must serialise them.
 *
 *   cuda_stream  cudaStream_t as void* (NULL = legacy default stream); the call only enqueues, it does not synchronise
 *   d_z          device, [C][2 S][n_t] complex64, input index 2 * station + pol (the layout of cobalt_debug_correlate);
 *                read only, 8-byte aligned
 *   stations     S >= 1;  channels C in {16, 64, 256};  n_spectra n_t in [1, 2^30]
 *   d_vis        device, [C][n_bl][2][2] complex64, baseline (i <= k) at k (k + 1) / 2 + i (reading A9); fully
 *                overwritten, 8-byte aligned.  Caller-owned like d_z; both must stay alive until the stream gets there
 *   h_err        host, NULL or a buffer of h_err_len bytes that receives a 0-terminated description of a failure
 *                (there is no plan whose cobalt_last_error could hold it); emptied on success
 * Returns COBALT_OK, COBALT_ERR_BAD_ARG (NULL / misaligned pointer, size out of range or beyond the scratch),
 * COBALT_ERR_UNSUPPORTED_DEVICE (no CUDA device, or not sm_100 class; no CPU fallback) or COBALT_ERR_CUDA.
 * Arguments are checked before the device is touched. */
#define COBALT_NOALLOC_SCRATCH_BYTES 16777216
#define COBALT_NOALLOC_MAX_SLICES 4
#define COBALT_NOALLOC_MAX_CHANNEL_BASELINES 131072   /* SCRATCH_BYTES / (MAX_SLICES * 32 bytes per [2][2] complex64) */
int cobalt_correlate_noalloc(void *cuda_stream, const void *d_z, int stations, int channels, long long n_spectra,
                             void *d_vis, char *h_err, int h_err_len);

#ifdef __cplusplus
}
#endif
#endif /* COBALT_B200_H */
