// Host side of the C ABI (include/cobalt.h): plan construction, the per-call launch sequence
//   [phase table (fp64)] -> [unpack+FIR+FFT+rotate+bandpass+transpose] -> [history carry] -> [correlate]
// per chunk of subbands (P:L360 step order; "a small number of buffers that the CUDA kernels
// alternate between"), the host-buffer streaming variant, settings and the debug taps.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "cobalt_internal.h"

using namespace cobalt;

namespace {

thread_local std::string g_err;   // failures before a plan exists

int fail(const cobalt_plan_s *p, int code, const std::string &msg) {
    if (p) p->err = msg;
    g_err = msg;
    return code;
}

#define CK(p, call)                                                                                        \
    do {                                                                                                   \
        cudaError_t e__ = (call);                                                                          \
        if (e__ != cudaSuccess)                                                                            \
            return fail(p, e__ == cudaErrorMemoryAllocation ? COBALT_ERR_NO_MEMORY : COBALT_ERR_CUDA,      \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                              \
    } while (0)

// Reading A1: Hann-windowed sinc, unit DC gain, double precision, rounded once to fp32.
// weights[k][ph] = g[(15 - k) C + ph]  (reading A2: tap k = 0 multiplies the newest block).
void build_weights(int C, std::vector<float> &w, double &sum_abs) {
    const int L = kTaps * C;
    const double pi = 3.141592653589793238462643383279502884;
    std::vector<double> g(L);
    double sum = 0.0;
    for (int n = 0; n < L; ++n) {
        const double u = ((double)n - 0.5 * (double)(L - 1)) / (double)C;
        const double sinc = u == 0.0 ? 1.0 : std::sin(pi * u) / (pi * u);
        const double hann = 0.5 - 0.5 * std::cos(2.0 * pi * (double)n / (double)(L - 1));
        g[n] = sinc * hann;
        sum += g[n];
    }
    w.resize(L);
    for (int k = 0; k < kTaps; ++k)
        for (int ph = 0; ph < C; ++ph) w[k * C + ph] = (float)(g[(kTaps - 1 - k) * C + ph] / sum);
    sum_abs = 0.0;
    for (float v : w) sum_abs += std::fabs((double)v);
}

// bytes of one complex sample as the CALLER passes it (4-bit: one byte)
size_t caller_sample_bytes(const cobalt_plan_s *p) { return p->bits_in == 16 ? 4 : p->bits_in == 8 ? 2 : 1; }
// one subband of the caller's samples (stream stride N_in) / of one dump of the visibilities
size_t subband_input_bytes(const cobalt_plan_s *p) { return (size_t)p->M * (size_t)p->N_in * caller_sample_bytes(p); }
size_t subband_output_bytes(const cobalt_plan_s *p) { return (size_t)p->C * (size_t)p->n_bl * 4 * sizeof(float2); }
// the fused kernel cannot read the caller's samples directly: pol-minor order or 4-bit samples go through launch_ingest
bool needs_ingest(const cobalt_plan_s *p) { return p->layout != COBALT_LAYOUT_PLANAR || p->bits_in == 4; }

void free_scratch(cobalt_plan_s *p) {
    cudaFree(p->d_ingest);
    cudaFree(p->d_xpart);
    p->d_ingest = nullptr;
    p->d_xpart = nullptr;
    cudaFree(p->d_z);
    cudaFree(p->d_dstep);
    p->d_dstep = nullptr;
    cudaFree(p->d_phase);
    p->d_z = nullptr;
    p->d_phase = nullptr;
    for (int i = 0; i < 2; ++i) {
        cudaFree(p->d_in[i]);
        cudaFree(p->d_out[i]);
        p->d_in[i] = p->d_out[i] = nullptr;
    }
    cudaFree(p->d_valid_h);
    cudaFree(p->d_counts_h);
    p->d_valid_h = nullptr;
    p->d_counts_h = nullptr;
}

// Tensor map of the fp16 intermediate of one chunk for the F-stage's tensor stores (fstage.cu, store issuer).
// Dimensions, innermost first: spectrum within the k-tile (64 fp16 = one 128-byte row), chunk subband * C + channel,
// u = 2 * (row group m / 8) + plane (1024-byte atoms, cobalt_internal.h), row within the group m % 8, k-tile; the box is
// half a row of every (stream of the CTA, plane, channel) -- the CTA's streams share one row group.
int build_zmap(cobalt_plan_s *p) {
    std::memset(&p->zmap, 0, sizeof(p->zmap));
    if (p->mode != COBALT_MODE_TENSOR_FP16) return COBALT_OK;
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CK(p, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(p, COBALT_ERR_CUDA, "cuTensorMapEncodeTiled is not available");
    const cuuint64_t row = 128, atom = 8 * row, kt = (cuuint64_t)p->Mpad * 2 * row, chan = (cuuint64_t)p->n_kt * kt;
    const cuuint64_t dims[5] = {(cuuint64_t)kKTile, (cuuint64_t)p->chunk * p->C, (cuuint64_t)(p->Mpad / 8) * 2, 8, (cuuint64_t)p->n_kt};
    const cuuint64_t strides[4] = {chan, atom, row, kt};   // bytes, dimensions 1..4
    const cuuint32_t box[5] = {(cuuint32_t)kStoreTile, (cuuint32_t)p->C, 2, (cuuint32_t)kStoreBoxStreams(p->C), 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = reinterpret_cast<encode_fn>(fn)(&p->zmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 5, p->d_z, dims, strides, box, estr,
                                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
                                                       CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(p, COBALT_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r));
    return COBALT_OK;
}

// (Re)allocate the per-chunk scratch for the current mode / chunk size.
int alloc_scratch(cobalt_plan_s *p, int chunk_request) {
    p->scratch_ok = false;      // until everything below has succeeded the plan refuses to process
    free_scratch(p);
    if (p->mode == COBALT_MODE_TENSOR_FP16) p->z_subband_bytes = (size_t)p->C * p->n_kt * 2 * p->Mpad * 128;
    else p->z_subband_bytes = (size_t)p->C * p->M * (size_t)p->n_t * sizeof(float2);
    int chunk = chunk_request;
    if (chunk <= 0) {
        // Default: up to 8 GiB of intermediate per launch group, at most a quarter of the free device memory.  Long
        // launches keep the tail of the F-stage (CTAs of equal length on 148 SMs: 8 subbands of config 3 are 8.3 waves)
        // and the kernel switches small: config 3 runs 5 % faster with 61 subbands per group than with 8.
        size_t free_b = 0, total_b = 0;
        size_t budget = (size_t)8 << 30;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b / 4 < budget) budget = free_b / 4;
        chunk = (int)(budget / p->z_subband_bytes);
        if (chunk < 1) chunk = 1;
        // equal groups: B = 244 with room for 64 becomes 4 x 61, not 3 x 64 + 52
        if (chunk < p->B) chunk = (p->B + (p->B + chunk - 1) / chunk - 1) / ((p->B + chunk - 1) / chunk);
    }
    if (chunk > p->B) chunk = p->B;
    p->chunk = chunk;
    // the host-buffer path pipelines H2D / compute / D2H group by group: keep its groups at about 1 GiB of intermediate
    p->host_chunk = (int)(((size_t)1 << 30) / p->z_subband_bytes);
    if (p->host_chunk < 1) p->host_chunk = 1;
    if (p->host_chunk > chunk) p->host_chunk = chunk;
    CK(p, cudaMalloc(&p->d_z, (size_t)chunk * p->z_subband_bytes));
    CK(p, cudaMemset(p->d_z, 0, (size_t)chunk * p->z_subband_bytes));   // zero rows 2S..Mpad stay zero forever
    CK(p, cudaMalloc(&p->d_phase, (size_t)p->B * p->S * p->C * sizeof(float2)));
    CK(p, cudaMalloc(&p->d_dstep, (size_t)p->B * p->S * p->C * sizeof(float)));
    {   // Reading R1: power-of-two scale of the fp16 intermediate so that full-scale input cannot overflow it
        // (|F s| <= amp_max s <= 32768); undone exactly (1/s^2) by the X-stage.  The bandpass no longer enters: it is
        // applied to the visibilities in fp32.
        int e = 0;
        if (p->mode == COBALT_MODE_TENSOR_FP16) e = (int)std::ceil(std::log2((double)p->amp_max / 32768.0));
        p->zscale = std::ldexp(1.f, -e);
    }
    size_t extra = 0;
    if (needs_ingest(p)) {
        extra += (size_t)chunk * p->M * p->N * sample_bytes(p->bits);
        CK(p, cudaMalloc(&p->d_ingest, (size_t)chunk * p->M * p->N * sample_bytes(p->bits)));
    }
    // X-stage in tensor mode: with fewer (dump, subband, channel) problems than two per SM each one's time range is split
    // over up to 8 jobs whose partial blocks are added up afterwards (xstage_tc.cu)
    p->x_splits = 1;
    if (p->mode == COBALT_MODE_TENSOR_FP16) {
        const long long probs = (long long)chunk * p->C * p->dumps * (long long)p->jobs.size();
        if (probs < 2LL * p->sm_count) {
            long long sp = (2LL * p->sm_count + probs - 1) / probs;
            if (sp > 8) sp = 8;
            if (sp > p->n_kt / p->dumps) sp = p->n_kt / p->dumps;
            p->x_splits = sp < 1 ? 1 : (int)sp;
        }
        if (p->x_splits > 1) {
            const size_t bytes = (size_t)chunk * p->C * p->dumps * p->x_splits * p->n_bl * 4 * sizeof(float2);
            extra += bytes;
            CK(p, cudaMalloc(&p->d_xpart, bytes));
        }
    }
    CK(p, cudaDeviceSynchronize());
    {
        const int rc = build_zmap(p);
        if (rc != COBALT_OK) return rc;
    }
    const size_t hist = (size_t)p->B * p->M * (kTaps - 1) * p->C * sample_bytes(p->bits);
    p->scratch_bytes = (size_t)chunk * p->z_subband_bytes + (size_t)p->B * p->S * p->C * (sizeof(float2) + sizeof(float)) + 2 * hist +
                       (size_t)kTaps * p->C * sizeof(float) + (size_t)p->B * sizeof(double) + extra;
    p->scratch_ok = true;
    return COBALT_OK;
}

// Steps a1-a7 + a10 of one chunk of subbands [b0, b0 + nb), shared by the correlator and the beamformer: the fp64 phase table
// of the whole call (with the first chunk; `table_bandpass` = nullptr builds pure station phases, which is what the beamformer
// wants -- afterwards p->d_phase belongs to the caller of this function until its chunk loop ends), the ingest pre-pass where
// the input needs one, the fused F-stage kernel into p->d_z, and the history carry.  Records ev->e[0..3]; adds the launches
// beyond the usual three (phase table, F-stage, history) to *extra.
int enqueue_fstage(cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, const double *delays, const float *table_bandpass,
                   const double *delays_end, const unsigned char *valid, int b0, int nb, StageEvents *ev, int *extra) {
    if (ev) CK(p, cudaEventRecord(ev->e[0], st));
    if (b0 == 0) CK(p, launch_phase_table(p, st, delays, table_bandpass, 0, p->B, delays_end));   // every subband's table in one launch
    if (ev) CK(p, cudaEventRecord(ev->e[1], st));
    FCall call;
    call.delays_end = delays_end;
    call.valid = valid;
    const void *fsamples = samples_b0;
    if (needs_ingest(p)) {     // pol-minor order / 4-bit samples: re-ordered, widened, coarse offsets applied
        CK(p, launch_ingest(p, st, samples_b0, nb, p->d_ingest));
        fsamples = p->d_ingest;
        call.coarse = nullptr;
        call.n_in = p->N;
        *extra += 1;
    } else {
        call.coarse = p->d_coarse;
        call.n_in = p->N_in;
    }
    CK(p, launch_fstage(p, st, fsamples, b0, nb, call));
    if (ev) CK(p, cudaEventRecord(ev->e[2], st));
    CK(p, launch_history_update(p, st, fsamples, b0, nb, call));
    if (ev) CK(p, cudaEventRecord(ev->e[3], st));
    return COBALT_OK;
}

// One chunk of subbands [b0, b0 + nb): samples_b0 / vis_b0 point at subband b0 (of dump 0); io holds the per-call pointers.
// dump_stride: float2 between consecutive dumps at vis_b0 (the caller's [D][B][...] array, or a group-sized staging buffer).
int enqueue_chunk(cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, const cobalt_io_t &io, float2 *vis_b0, size_t dump_stride, int b0,
                  int nb, StageEvents *ev) {
    int extra = 0;
    {
        const int rc = enqueue_fstage(p, st, samples_b0, io.delays, io.bandpass, io.delays_end, io.valid, b0, nb, ev, &extra);
        if (rc != COBALT_OK) return rc;
    }
    XCall xc;
    xc.phase = p->d_phase;
    xc.poff = p->d_poff;
    xc.b0 = b0;
    xc.inv_s2 = 1.f / (p->zscale * p->zscale);
    if (p->mode == COBALT_MODE_TENSOR_FP16) {
        CK(p, launch_xstage_tc(p, st, p->d_z, nb, vis_b0, dump_stride, xc));
        if (p->x_splits > 1) extra += 1;
    } else {
        CK(p, launch_xstage_simt(p, st, p->d_z, nb, vis_b0, dump_stride, xc));
    }
    if (io.valid_counts) {
        CK(p, launch_valid_counts(p, st, io.valid, b0, nb, io.valid_counts));
        extra += 1;
    }
    if (ev) CK(p, cudaEventRecord(ev->e[4], st));
    p->launches += (b0 == 0 ? 4 : 3) + extra;
    return COBALT_OK;
}

int ensure_events(cobalt_plan_s *p, int n) {
    while ((int)p->events.size() < n) {
        StageEvents e;
        for (auto &ev : e.e) CK(p, cudaEventCreate(&ev));
        p->events.push_back(e);
    }
    return COBALT_OK;
}

}  // namespace

extern "C" {

const char *cobalt_strerror(int status) {
    switch (status) {
        case COBALT_OK: return "ok";
        case COBALT_ERR_BAD_ARG: return "bad argument";
        case COBALT_ERR_NO_MEMORY: return "out of memory";
        case COBALT_ERR_CUDA: return "CUDA error";
        case COBALT_ERR_UNSUPPORTED_DEVICE: return "no CUDA device of compute capability 10.x (sm_100)";
    }
    return "unknown status";
}

const char *cobalt_last_error(const cobalt_plan_t *plan) { return plan ? plan->err.c_str() : g_err.c_str(); }

int cobalt_plan(cobalt_plan_t **out, int stations, int subbands, int channels, int taps,
                long long samples_per_integration, int input_bits) {
    if (!out) return fail(nullptr, COBALT_ERR_BAD_ARG, "out is NULL");
    *out = nullptr;
    if (stations < 1 || stations > 16384) return fail(nullptr, COBALT_ERR_BAD_ARG, "stations must be in [1, 16384]");
    if (subbands < 1) return fail(nullptr, COBALT_ERR_BAD_ARG, "subbands must be >= 1");
    if (channels != 16 && channels != 64 && channels != 256)
        return fail(nullptr, COBALT_ERR_BAD_ARG, "channels must be 16, 64 or 256");
    if (taps != kTaps) return fail(nullptr, COBALT_ERR_BAD_ARG, "taps must be 16");
    if (input_bits != 16 && input_bits != 8 && input_bits != 4) return fail(nullptr, COBALT_ERR_BAD_ARG, "input_bits must be 16, 8 or 4");
    if (samples_per_integration < channels)
        return fail(nullptr, COBALT_ERR_BAD_ARG, "samples_per_integration must be >= channels");
    if (samples_per_integration / channels > (1ll << 30))
        return fail(nullptr, COBALT_ERR_BAD_ARG, "samples_per_integration too large");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, COBALT_ERR_UNSUPPORTED_DEVICE, "no CUDA device");
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return fail(nullptr, COBALT_ERR_CUDA, "cudaGetDeviceProperties failed");
    if (prop.major != 10)
        return fail(nullptr, COBALT_ERR_UNSUPPORTED_DEVICE,
                    std::string("device is sm_") + std::to_string(prop.major * 10 + prop.minor) + ", need sm_100");

    cobalt_plan_s *p = new (std::nothrow) cobalt_plan_s();
    if (!p) return fail(nullptr, COBALT_ERR_NO_MEMORY, "host allocation failed");
    p->S = stations;
    p->B = subbands;
    p->C = channels;
    p->T = taps;
    p->bits_in = input_bits;
    p->bits = input_bits == 16 ? 16 : 8;      // 4-bit samples are expanded to int8 by the ingest pre-pass
    p->N = samples_per_integration;
    p->N_in = p->N;
    p->n_t = p->N / p->C;
    p->N_u = p->n_t * p->C;
    p->n_bl = (long long)stations * (stations + 1) / 2;
    p->M = 2 * stations;
    p->Mpad = (p->M + 15) / 16 * 16;
    p->n_kt = (int)((p->n_t + kKTile - 1) / kKTile);
    p->device = dev;
    p->sm_count = prop.multiProcessorCount;
    p->f_sb.resize(subbands);
    for (int s = 0; s < subbands; ++s) p->f_sb[s] = 100.0e6 + (12 + s) * p->f_s;   // reading A6
    double sum_abs_g = 0.0;
    build_weights(p->C, p->h_weights, sum_abs_g);
    // worst-case modulus of a channelised sample for full-scale input: sum|g| sqrt(2) 2^(bits-1)
    p->amp_max = (float)(sum_abs_g * 1.4142135623730951 * (input_bits == 16 ? 32768.0 : input_bits == 8 ? 128.0 : 8.0));
    build_xjobs(p);

    int rc = COBALT_OK;
    auto guard = [&](cudaError_t e, const char *what) {
        if (e != cudaSuccess && rc == COBALT_OK)
            rc = fail(p, e == cudaErrorMemoryAllocation ? COBALT_ERR_NO_MEMORY : COBALT_ERR_CUDA,
                      std::string(what) + ": " + cudaGetErrorString(e));
    };
    const size_t hist = (size_t)p->B * p->M * (kTaps - 1) * p->C * sample_bytes(p->bits);
    guard(cudaMalloc(&p->d_weights, p->h_weights.size() * sizeof(float)), "cudaMalloc weights");
    guard(cudaMalloc(&p->d_f_sb, (size_t)p->B * sizeof(double)), "cudaMalloc f_sb");
    guard(cudaMalloc(&p->d_hist[0], hist), "cudaMalloc history");
    guard(cudaMalloc(&p->d_hist[1], hist), "cudaMalloc history");
    guard(cudaMalloc(&p->d_jobs, p->jobs.size() * sizeof(XJob)), "cudaMalloc jobs");
    if (rc == COBALT_OK) {
        guard(cudaMemcpy(p->d_weights, p->h_weights.data(), p->h_weights.size() * sizeof(float), cudaMemcpyHostToDevice), "weights H2D");
        guard(cudaMemcpy(p->d_f_sb, p->f_sb.data(), (size_t)p->B * sizeof(double), cudaMemcpyHostToDevice), "f_sb H2D");
        guard(cudaMemcpy(p->d_jobs, p->jobs.data(), p->jobs.size() * sizeof(XJob), cudaMemcpyHostToDevice), "jobs H2D");
        guard(cudaMemset(p->d_hist[0], 0, hist), "memset history");   // reading A3
        guard(cudaMemset(p->d_hist[1], 0, hist), "memset history");
    }
    if (rc == COBALT_OK) rc = alloc_scratch(p, 0);
    if (rc != COBALT_OK) {
        g_err = p->err;
        cobalt_destroy(p);
        return rc;
    }
    *out = p;
    return COBALT_OK;
}

int cobalt_destroy(cobalt_plan_t *p) {
    if (!p) return COBALT_OK;
    free_scratch(p);
    cudaFree(p->d_weights);
    cudaFree(p->d_f_sb);
    cudaFree(p->d_hist[0]);
    cudaFree(p->d_hist[1]);
    cudaFree(p->d_jobs);
    cudaFree(p->d_coarse);
    cudaFree(p->d_poff);
    cudaFree(p->d_delays_h);
    cudaFree(p->d_delays_end_h);
    cudaFree(p->d_bandpass_h);
    for (auto &e : p->events)
        for (auto &ev : e.e) cudaEventDestroy(ev);
    for (int i = 0; i < 3; ++i)
        if (p->hs[i]) cudaStreamDestroy(p->hs[i]);
    for (int i = 0; i < 2; ++i) {
        if (p->ev_in[i]) cudaEventDestroy(p->ev_in[i]);
        if (p->ev_cmp[i]) cudaEventDestroy(p->ev_cmp[i]);
        if (p->ev_out[i]) cudaEventDestroy(p->ev_out[i]);
    }
    delete p;
    return COBALT_OK;
}

int cobalt_process_ex(cobalt_plan_t *p, void *cuda_stream, const cobalt_io_t *io) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    if (!io || !io->samples || !io->delays || !io->bandpass || !io->visibilities) return fail(p, COBALT_ERR_BAD_ARG, "NULL buffer");
    if (!p->scratch_ok) return fail(p, COBALT_ERR_NO_MEMORY, "the plan has no scratch (an earlier cobalt_set_mode / cobalt_set_chunk_subbands failed)");
    if ((reinterpret_cast<uintptr_t>(io->samples) & (caller_sample_bytes(p) - 1)) != 0)
        return fail(p, COBALT_ERR_BAD_ARG, "d_samples must be aligned to one complex sample");
    if (p->mode == COBALT_MODE_TENSOR_FP16 && (reinterpret_cast<uintptr_t>(io->visibilities) & 15u) != 0)
        return fail(p, COBALT_ERR_BAD_ARG, "d_visibilities must be 16-byte aligned in COBALT_MODE_TENSOR_FP16");
    // the fp32 correlator puts (subband of the group, dump) in gridDim.z: refuse before anything is enqueued (a launch failure
    // in a later group would leave the in-place FIR history of the earlier groups advanced)
    if (p->mode == COBALT_MODE_EXACT_FP32 && (long long)p->chunk * p->dumps > kMaxGridYZ)
        return fail(p, COBALT_ERR_BAD_ARG, "COBALT_MODE_EXACT_FP32: chunk_subbands * dumps = " + std::to_string((long long)p->chunk * p->dumps) +
                                               " exceeds 65535; lower cobalt_set_chunk_subbands or cobalt_set_dumps");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int n_chunks = (p->B + p->chunk - 1) / p->chunk;
    if (p->timing) {
        int rc = ensure_events(p, n_chunks);
        if (rc != COBALT_OK) return rc;
    }
    p->launches = 0;
    p->n_chunks_timed = 0;
    for (int ci = 0; ci < n_chunks; ++ci) {
        const int b0 = ci * p->chunk;
        const int nb = (p->B - b0) < p->chunk ? (p->B - b0) : p->chunk;
        const unsigned char *sm = static_cast<const unsigned char *>(io->samples) + (size_t)b0 * subband_input_bytes(p);
        float2 *vis = reinterpret_cast<float2 *>(static_cast<unsigned char *>(io->visibilities) + (size_t)b0 * subband_output_bytes(p));
        int rc = enqueue_chunk(p, st, sm, *io, vis, (size_t)p->B * p->C * p->n_bl * 4, b0, nb, p->timing ? &p->events[ci] : nullptr);
        if (rc != COBALT_OK) return rc;
    }
    if (p->timing) p->n_chunks_timed = n_chunks;
    if (!history_in_place(p)) p->hist_cur ^= 1;   // short blocks: the history kernels of this call wrote the other buffer (stream ordered)
    return COBALT_OK;
}

int cobalt_process(cobalt_plan_t *p, void *cuda_stream, const void *d_samples, const double *d_delays,
                   const float *d_bandpass, void *d_visibilities) {
    cobalt_io_t io{};
    io.samples = d_samples;
    io.delays = d_delays;
    io.bandpass = d_bandpass;
    io.visibilities = d_visibilities;
    return cobalt_process_ex(p, cuda_stream, &io);
}

int cobalt_process_interp(cobalt_plan_t *p, void *cuda_stream, const void *d_samples, const double *d_delays_begin,
                          const double *d_delays_end, const float *d_bandpass, void *d_visibilities) {
    if (p && !d_delays_end) return fail(p, COBALT_ERR_BAD_ARG, "NULL buffer");
    cobalt_io_t io{};
    io.samples = d_samples;
    io.delays = d_delays_begin;
    io.delays_end = d_delays_end;
    io.bandpass = d_bandpass;
    io.visibilities = d_visibilities;
    return cobalt_process_ex(p, cuda_stream, &io);
}

long long cobalt_beamform_output_bytes(const cobalt_plan_t *p, int n_beams, int product, int n_stokes, int t_int) {
    if (!p) return 0;
    const bool stokes = product != COBALT_BF_COHERENT_VOLTAGES;
    if (product < COBALT_BF_COHERENT_VOLTAGES || product > COBALT_BF_INCOHERENT_STOKES) return 0;
    if (product != COBALT_BF_INCOHERENT_STOKES && (n_beams < 1 || n_beams > 4096)) return 0;
    if (stokes && ((n_stokes != 1 && n_stokes != 4) || t_int < 1 || t_int > 128 || (t_int & (t_int - 1)) != 0)) return 0;
    const long long beams = product == COBALT_BF_INCOHERENT_STOKES ? 1 : n_beams;
    if (!stokes) return (long long)p->B * beams * 2 * p->C * p->n_t * (long long)sizeof(float2);
    return (long long)p->B * beams * n_stokes * p->C * (p->n_t / t_int) * (long long)sizeof(float);
}

int cobalt_beamform(cobalt_plan_t *p, void *cuda_stream, const cobalt_bf_io_t *io) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    if (!io || !io->samples || !io->delays || !io->bandpass || !io->out) return fail(p, COBALT_ERR_BAD_ARG, "NULL buffer");
    if (!p->scratch_ok) return fail(p, COBALT_ERR_NO_MEMORY, "the plan has no scratch (an earlier cobalt_set_mode / cobalt_set_chunk_subbands failed)");
    const int t_int = io->product == COBALT_BF_COHERENT_VOLTAGES ? 1 : io->t_int;
    const int n_stokes = io->product == COBALT_BF_COHERENT_VOLTAGES ? 1 : io->n_stokes;
    const long long total = cobalt_beamform_output_bytes(p, io->n_beams, io->product, n_stokes, t_int);
    if (total <= 0) return fail(p, COBALT_ERR_BAD_ARG, "bad beamformer settings (product, n_beams, n_stokes in {1, 4}, t_int a power of two <= 128 with floor(n_t / t_int) >= 1)");
    if (io->product != COBALT_BF_INCOHERENT_STOKES && !io->beam_delays) return fail(p, COBALT_ERR_BAD_ARG, "NULL buffer");
    if ((reinterpret_cast<uintptr_t>(io->out) & 7u) != 0) return fail(p, COBALT_ERR_BAD_ARG, "out must be 8-byte aligned");
    if ((reinterpret_cast<uintptr_t>(io->samples) & (caller_sample_bytes(p) - 1)) != 0)
        return fail(p, COBALT_ERR_BAD_ARG, "d_samples must be aligned to one complex sample");
    const bool tensor = p->mode == COBALT_MODE_TENSOR_FP16;
    // the SIMT beamformer kernels (incoherent Stokes in both modes, everything in EXACT mode) put ceil(n_t / 128) in gridDim.y
    if ((!tensor || io->product == COBALT_BF_INCOHERENT_STOKES) && (p->n_t + kBfTBlock - 1) / kBfTBlock > kMaxGridYZ)
        return fail(p, COBALT_ERR_BAD_ARG, "n_t = " + std::to_string(p->n_t) + " spectra per block exceed the " + std::to_string((long long)kMaxGridYZ * kBfTBlock) +
                                               " this beamformer product handles in this mode; use shorter blocks");
    if (tensor && io->product != COBALT_BF_INCOHERENT_STOKES) {
        int bpb, stages;
        size_t wb, sb, sm;
        if (!bf_tc_shape(p, io->n_beams, bpb, stages, wb, sb, sm))
            return fail(p, COBALT_ERR_BAD_ARG, "too many stations for the tensor-core beamformer (2 S <= 208); use COBALT_MODE_EXACT_FP32");
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t out_sb = (size_t)(total / p->B);
    // the tensor path adds the partial sums of windows longer than a warp with atomics: start from zero
    if (tensor && io->product == COBALT_BF_COHERENT_STOKES && t_int > 32) CK(p, cudaMemsetAsync(io->out, 0, (size_t)total, st));
    const int n_chunks = (p->B + p->chunk - 1) / p->chunk;
    if (p->timing) {
        int rc = ensure_events(p, n_chunks);
        if (rc != COBALT_OK) return rc;
    }
    p->launches = 0;
    p->n_chunks_timed = 0;
    for (int ci = 0; ci < n_chunks; ++ci) {
        const int b0 = ci * p->chunk;
        const int nb = (p->B - b0) < p->chunk ? (p->B - b0) : p->chunk;
        const unsigned char *sm = static_cast<const unsigned char *>(io->samples) + (size_t)b0 * subband_input_bytes(p);
        StageEvents *ev = p->timing ? &p->events[ci] : nullptr;
        // pure station phases (no bandpass: the beamformer scales its outputs by b[j] in fp32)
        int extra = 0;
        {
            const int rc = enqueue_fstage(p, st, sm, io->delays, nullptr, io->delays_end, io->valid, b0, nb, ev, &extra);
            if (rc != COBALT_OK) return rc;
        }
        BfCall bc;
        bc.beam_delays = io->beam_delays;
        bc.bandpass = io->bandpass;
        bc.out = static_cast<unsigned char *>(io->out) + (size_t)b0 * out_sb;
        bc.n_beams = io->n_beams;
        bc.product = io->product;
        bc.n_stokes = n_stokes;
        bc.t_int = t_int;
        CK(p, launch_beamform(p, st, p->d_z, b0, nb, bc));
        if (ev) CK(p, cudaEventRecord(ev->e[4], st));
        p->launches += (b0 == 0 ? 4 : 3) + extra;
    }
    if (p->timing) p->n_chunks_timed = n_chunks;
    if (!history_in_place(p)) p->hist_cur ^= 1;
    return COBALT_OK;
}

int cobalt_process_host_ex(cobalt_plan_t *p, const cobalt_io_t *h) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    if (!h || !h->samples || !h->delays || !h->bandpass || !h->visibilities) return fail(p, COBALT_ERR_BAD_ARG, "NULL buffer");
    if (!p->scratch_ok) return fail(p, COBALT_ERR_NO_MEMORY, "the plan has no scratch (an earlier cobalt_set_mode / cobalt_set_chunk_subbands failed)");
    if (p->mode == COBALT_MODE_EXACT_FP32 && (long long)p->host_chunk * p->dumps > kMaxGridYZ)
        return fail(p, COBALT_ERR_BAD_ARG, "COBALT_MODE_EXACT_FP32: subbands per group * dumps exceeds 65535; lower cobalt_set_chunk_subbands or cobalt_set_dumps");
    const size_t in_b = subband_input_bytes(p), out_b = subband_output_bytes(p);
    const int D = p->dumps;
    const size_t valid_b = (size_t)p->B * p->S * p->n_kt, counts_b = (size_t)p->B * D * p->n_bl * sizeof(unsigned int);
    if (!p->hs[0]) {
        for (int i = 0; i < 3; ++i) CK(p, cudaStreamCreateWithFlags(&p->hs[i], cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(p, cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming));
            CK(p, cudaEventCreateWithFlags(&p->ev_cmp[i], cudaEventDisableTiming));
            CK(p, cudaEventCreateWithFlags(&p->ev_out[i], cudaEventDisableTiming));
        }
        CK(p, cudaMalloc(&p->d_delays_h, (size_t)p->S * sizeof(double)));
        CK(p, cudaMalloc(&p->d_delays_end_h, (size_t)p->S * sizeof(double)));
        CK(p, cudaMalloc(&p->d_bandpass_h, (size_t)p->C * sizeof(float)));
    }
    if (!p->d_in[0]) {        // (re)allocated after every change of mode / group size / dumps / layout (free_scratch)
        for (int i = 0; i < 2; ++i) {
            CK(p, cudaMalloc(&p->d_in[i], (size_t)p->host_chunk * in_b));
            CK(p, cudaMalloc(&p->d_out[i], (size_t)p->host_chunk * out_b * D));     // [D][group][C][n_bl][2][2]
        }
    }
    if (h->valid && !p->d_valid_h) CK(p, cudaMalloc(&p->d_valid_h, valid_b));
    if (h->valid_counts && !p->d_counts_h) CK(p, cudaMalloc(&p->d_counts_h, counts_b));
    cudaStream_t s_in = p->hs[0], s_cmp = p->hs[1], s_out = p->hs[2];
    // On any failure below the copies already enqueued still touch the caller's host buffers: drain the three
    // streams before returning the error.
    auto drain = [&](int rc) {
        cudaStreamSynchronize(s_in);
        cudaStreamSynchronize(s_cmp);
        cudaStreamSynchronize(s_out);
        return rc;
    };
#define CKH(call)                                                                                             \
    do {                                                                                                      \
        cudaError_t e__ = (call);                                                                             \
        if (e__ != cudaSuccess)                                                                               \
            return drain(fail(p, COBALT_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)));      \
    } while (0)
    // the small per-call arrays travel whole, ahead of the first group, on the compute stream
    CKH(cudaMemcpyAsync(p->d_delays_h, h->delays, (size_t)p->S * sizeof(double), cudaMemcpyHostToDevice, s_cmp));
    CKH(cudaMemcpyAsync(p->d_bandpass_h, h->bandpass, (size_t)p->C * sizeof(float), cudaMemcpyHostToDevice, s_cmp));
    if (h->delays_end) CKH(cudaMemcpyAsync(p->d_delays_end_h, h->delays_end, (size_t)p->S * sizeof(double), cudaMemcpyHostToDevice, s_cmp));
    if (h->valid) CKH(cudaMemcpyAsync(p->d_valid_h, h->valid, valid_b, cudaMemcpyHostToDevice, s_cmp));
    cobalt_io_t io{};
    io.delays = p->d_delays_h;
    io.bandpass = p->d_bandpass_h;
    io.delays_end = h->delays_end ? p->d_delays_end_h : nullptr;
    io.valid = h->valid ? p->d_valid_h : nullptr;
    io.valid_counts = h->valid_counts ? p->d_counts_h : nullptr;
    const size_t group_stride = (size_t)p->host_chunk * p->C * p->n_bl * 4;     // float2 between dumps in d_out[buf]
    const int n_chunks = (p->B + p->host_chunk - 1) / p->host_chunk;
    p->launches = 0;
    p->n_chunks_timed = 0;
    for (int ci = 0; ci < n_chunks; ++ci) {
        const int buf = ci & 1;
        const int b0 = ci * p->host_chunk;
        const int nb = (p->B - b0) < p->host_chunk ? (p->B - b0) : p->host_chunk;
        if (ci >= 2) CKH(cudaStreamWaitEvent(s_in, p->ev_cmp[buf], 0));     // d_in[buf] consumed
        CKH(cudaMemcpyAsync(p->d_in[buf], static_cast<const unsigned char *>(h->samples) + (size_t)b0 * in_b,
                            (size_t)nb * in_b, cudaMemcpyHostToDevice, s_in));
        CKH(cudaEventRecord(p->ev_in[buf], s_in));
        CKH(cudaStreamWaitEvent(s_cmp, p->ev_in[buf], 0));
        if (ci >= 2) CKH(cudaStreamWaitEvent(s_cmp, p->ev_out[buf], 0));    // d_out[buf] drained
        int rc = enqueue_chunk(p, s_cmp, p->d_in[buf], io, static_cast<float2 *>(p->d_out[buf]), group_stride, b0, nb, nullptr);
        if (rc != COBALT_OK) return drain(rc);
        CKH(cudaEventRecord(p->ev_cmp[buf], s_cmp));
        CKH(cudaStreamWaitEvent(s_out, p->ev_cmp[buf], 0));
        for (int d = 0; d < D; ++d)      // dump d of the group -> subbands [b0, b0 + nb) of dump d of the caller's [D][B][...] array
            CKH(cudaMemcpyAsync(static_cast<unsigned char *>(h->visibilities) + ((size_t)d * p->B + b0) * out_b,
                                static_cast<const unsigned char *>(p->d_out[buf]) + (size_t)d * group_stride * sizeof(float2),
                                (size_t)nb * out_b, cudaMemcpyDeviceToHost, s_out));
        CKH(cudaEventRecord(p->ev_out[buf], s_out));
    }
    if (h->valid_counts) CKH(cudaMemcpyAsync(h->valid_counts, p->d_counts_h, counts_b, cudaMemcpyDeviceToHost, s_cmp));
    if (!history_in_place(p)) p->hist_cur ^= 1;
    CKH(cudaStreamSynchronize(s_in));
    CKH(cudaStreamSynchronize(s_cmp));
    CKH(cudaStreamSynchronize(s_out));
#undef CKH
    return COBALT_OK;
}

int cobalt_process_host(cobalt_plan_t *p, const void *h_samples, const double *h_delays, const float *h_bandpass,
                        void *h_visibilities) {
    cobalt_io_t h{};
    h.samples = h_samples;
    h.delays = h_delays;
    h.bandpass = h_bandpass;
    h.visibilities = h_visibilities;
    return cobalt_process_host_ex(p, &h);
}

int cobalt_set_subband_frequencies(cobalt_plan_t *p, const double *h_hz) {
    if (!p || !h_hz) return fail(p, COBALT_ERR_BAD_ARG, "NULL argument");
    for (int s = 0; s < p->B; ++s)
        if (!(h_hz[s] == h_hz[s]) || std::fabs(h_hz[s]) > 1e12) return fail(p, COBALT_ERR_BAD_ARG, "frequency not finite");
    CK(p, cudaDeviceSynchronize());
    p->f_sb.assign(h_hz, h_hz + p->B);
    p->f_sb_user = true;
    CK(p, cudaMemcpy(p->d_f_sb, p->f_sb.data(), (size_t)p->B * sizeof(double), cudaMemcpyHostToDevice));
    return COBALT_OK;
}

int cobalt_set_sample_rate(cobalt_plan_t *p, double hz) {
    if (!p || !(hz > 0.0) || hz > 1e12) return fail(p, COBALT_ERR_BAD_ARG, "sample rate must be positive and finite");
    p->f_s = hz;
    if (!p->f_sb_user) {   // the default ladder is defined in terms of f_s (reading A6): it follows the new rate
        CK(p, cudaDeviceSynchronize());
        for (int s = 0; s < p->B; ++s) p->f_sb[s] = 100.0e6 + (12 + s) * p->f_s;
        CK(p, cudaMemcpy(p->d_f_sb, p->f_sb.data(), (size_t)p->B * sizeof(double), cudaMemcpyHostToDevice));
    }
    return COBALT_OK;
}

int cobalt_set_phase_offsets(cobalt_plan_t *p, const double *h_phase0) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    CK(p, cudaDeviceSynchronize());
    if (!h_phase0) {
        cudaFree(p->d_poff);
        p->d_poff = nullptr;
        return COBALT_OK;
    }
    std::vector<float2> w((size_t)p->M);
    for (int m = 0; m < p->M; ++m) {
        if (!(h_phase0[m] == h_phase0[m]) || std::fabs(h_phase0[m]) > 1e9) return fail(p, COBALT_ERR_BAD_ARG, "phase offset not finite");
        w[m] = make_float2((float)std::cos(h_phase0[m]), (float)-std::sin(h_phase0[m]));   // exp(-i phase0), reading A22
    }
    if (!p->d_poff) CK(p, cudaMalloc(&p->d_poff, (size_t)p->M * sizeof(float2)));
    CK(p, cudaMemcpy(p->d_poff, w.data(), (size_t)p->M * sizeof(float2), cudaMemcpyHostToDevice));
    return COBALT_OK;
}

int cobalt_set_coarse_delays(cobalt_plan_t *p, const int *h_offsets, long long samples_allocated) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    CK(p, cudaDeviceSynchronize());
    if (!h_offsets) {
        cudaFree(p->d_coarse);
        p->d_coarse = nullptr;
        p->N_in = p->N;
        return COBALT_OK;
    }
    if (samples_allocated < p->N) return fail(p, COBALT_ERR_BAD_ARG, "samples_allocated must be >= samples_per_integration");
    for (int a = 0; a < p->S; ++a)
        if (h_offsets[a] < 0 || (long long)h_offsets[a] + p->N > samples_allocated)
            return fail(p, COBALT_ERR_BAD_ARG, "coarse delay outside [0, samples_allocated - samples_per_integration]");
    if (!p->d_coarse) CK(p, cudaMalloc(&p->d_coarse, (size_t)p->S * sizeof(int)));
    CK(p, cudaMemcpy(p->d_coarse, h_offsets, (size_t)p->S * sizeof(int), cudaMemcpyHostToDevice));
    p->N_in = samples_allocated;
    cudaFree(p->d_in[0]);     // the host-path staging buffers are sized by the stream stride
    cudaFree(p->d_in[1]);
    p->d_in[0] = p->d_in[1] = nullptr;
    return COBALT_OK;
}

int cobalt_set_dumps(cobalt_plan_t *p, int dumps) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    if (dumps < 1 || p->n_kt % dumps != 0) return fail(p, COBALT_ERR_BAD_ARG, "dumps_per_block must divide ceil(n_t / 64)");
    if (dumps == p->dumps) return COBALT_OK;
    CK(p, cudaDeviceSynchronize());
    p->dumps = dumps;
    return alloc_scratch(p, p->chunk);
}

int cobalt_set_input_layout(cobalt_plan_t *p, int layout) {
    if (!p || (layout != COBALT_LAYOUT_PLANAR && layout != COBALT_LAYOUT_POL_MINOR)) return fail(p, COBALT_ERR_BAD_ARG, "unknown layout");
    if (layout == p->layout) return COBALT_OK;
    CK(p, cudaDeviceSynchronize());
    p->layout = layout;
    return alloc_scratch(p, p->chunk);
}

int cobalt_set_mode(cobalt_plan_t *p, int mode) {
    if (!p || (mode != COBALT_MODE_TENSOR_FP16 && mode != COBALT_MODE_EXACT_FP32)) return fail(p, COBALT_ERR_BAD_ARG, "unknown mode");
    if (mode == p->mode) return COBALT_OK;
    CK(p, cudaDeviceSynchronize());
    p->mode = mode;
    return alloc_scratch(p, p->chunk_user);   // a group size the caller chose survives the switch; otherwise the default rule of the new mode
}

int cobalt_set_chunk_subbands(cobalt_plan_t *p, int chunk) {
    if (!p || chunk < 1) return fail(p, COBALT_ERR_BAD_ARG, "chunk must be >= 1");
    CK(p, cudaDeviceSynchronize());
    p->chunk_user = chunk;
    return alloc_scratch(p, chunk);
}

int cobalt_reset(cobalt_plan_t *p) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    CK(p, cudaDeviceSynchronize());
    const size_t hist = (size_t)p->B * p->M * (kTaps - 1) * p->C * sample_bytes(p->bits);
    CK(p, cudaMemset(p->d_hist[0], 0, hist));
    CK(p, cudaMemset(p->d_hist[1], 0, hist));
    CK(p, cudaDeviceSynchronize());
    return COBALT_OK;
}

int cobalt_info(const cobalt_plan_t *p, cobalt_info_t *info) {
    if (!p || !info) return fail(p, COBALT_ERR_BAD_ARG, "NULL argument");
    info->stations = p->S;
    info->subbands = p->B;
    info->channels = p->C;
    info->taps = p->T;
    info->input_bits = p->bits_in;
    info->mode = p->mode;
    info->samples_per_integration = p->N;
    info->n_spectra = p->n_t;
    info->n_consumed = p->N_u;
    info->n_baselines = p->n_bl;
    info->input_bytes = (long long)((size_t)p->B * subband_input_bytes(p));
    info->output_bytes = (long long)((size_t)p->dumps * p->B * subband_output_bytes(p));
    info->scratch_bytes = (long long)p->scratch_bytes;
    info->chunk_subbands = p->chunk;
    info->sm_count = p->sm_count;
    info->sample_rate_hz = p->f_s;
    info->dumps = p->dumps;
    info->n_tiles = p->n_kt;
    info->samples_allocated = p->N_in;
    return COBALT_OK;
}

int cobalt_set_timing(cobalt_plan_t *p, int enabled) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    p->timing = enabled != 0;
    p->n_chunks_timed = 0;
    return COBALT_OK;
}

int cobalt_get_kernel_timing(cobalt_plan_t *p, double *ms4, int *launches) {
    if (!p) return fail(nullptr, COBALT_ERR_BAD_ARG, "plan is NULL");
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int i = 0; i < p->n_chunks_timed; ++i) {
        CK(p, cudaEventSynchronize(p->events[i].e[4]));
        for (int k = 0; k < 4; ++k) {
            float t = 0.f;
            CK(p, cudaEventElapsedTime(&t, p->events[i].e[k], p->events[i].e[k + 1]));
            acc[k] += t;
        }
    }
    if (ms4)
        for (int k = 0; k < 4; ++k) ms4[k] = acc[k];
    if (launches) *launches = p->launches;
    return COBALT_OK;
}

int cobalt_get_timing(cobalt_plan_t *p, double *f_ms, double *x_ms, int *launches) {
    double ms[4];
    int rc = cobalt_get_kernel_timing(p, ms, launches);
    if (rc != COBALT_OK) return rc;
    if (f_ms) *f_ms = ms[0] + ms[1] + ms[2];
    if (x_ms) *x_ms = ms[3];
    return COBALT_OK;
}

int cobalt_debug_fir_weights(const cobalt_plan_t *p, float *h_weights) {
    if (!p || !h_weights) return fail(p, COBALT_ERR_BAD_ARG, "NULL argument");
    std::memcpy(h_weights, p->h_weights.data(), p->h_weights.size() * sizeof(float));
    return COBALT_OK;
}

int cobalt_debug_unpack(void *cuda_stream, int input_bits, const void *d_in, long long n, float *d_out) {
    if ((input_bits != 16 && input_bits != 8 && input_bits != 4) || n < 0 || (n > 0 && (!d_in || !d_out)))
        return fail(nullptr, COBALT_ERR_BAD_ARG, "bad unpack arguments");
    CK(nullptr, launch_unpack(static_cast<cudaStream_t>(cuda_stream), input_bits, d_in, n, d_out));
    return COBALT_OK;
}

int cobalt_debug_channelised(cobalt_plan_t *p, void *cuda_stream, const void *d_samples, const double *d_delays,
                             const float *d_bandpass, int sb, void *d_z) {
    if (!p || !d_samples || !d_delays || !d_bandpass || !d_z) return fail(p, COBALT_ERR_BAD_ARG, "NULL argument");
    if (sb < 0 || sb >= p->B) return fail(p, COBALT_ERR_BAD_ARG, "subband out of range");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const unsigned char *sm = static_cast<const unsigned char *>(d_samples) + (size_t)sb * subband_input_bytes(p);
    CK(p, launch_phase_table(p, st, d_delays, d_bandpass, sb, 1, nullptr));
    FCall call;
    const void *fsamples = sm;
    if (needs_ingest(p)) {
        CK(p, launch_ingest(p, st, sm, 1, p->d_ingest));
        fsamples = p->d_ingest;
        call.n_in = p->N;
    } else {
        call.coarse = p->d_coarse;
        call.n_in = p->N_in;
    }
    CK(p, launch_fstage(p, st, fsamples, sb, 1, call));
    XCall xc;
    xc.phase = p->d_phase;
    xc.poff = p->d_poff;
    xc.b0 = sb;
    xc.inv_s2 = 1.f / (p->zscale * p->zscale);
    CK(p, launch_z_to_float(p, st, p->d_z, static_cast<float2 *>(d_z), xc));
    return COBALT_OK;
}

int cobalt_debug_correlate(cobalt_plan_t *p, void *cuda_stream, const void *d_z, void *d_vis) {
    if (!p || !d_z || !d_vis) return fail(p, COBALT_ERR_BAD_ARG, "NULL argument");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    CK(p, launch_float_to_z(p, st, static_cast<const float2 *>(d_z), p->d_z));
    const size_t dump_stride = (size_t)p->C * p->n_bl * 4;     // one subband: [D][C][n_bl][2][2]
    const XCall xc;                                            // caller-supplied operands are taken as they are: no rotation, unit scale
    if (p->mode == COBALT_MODE_TENSOR_FP16) CK(p, launch_xstage_tc(p, st, p->d_z, 1, static_cast<float2 *>(d_vis), dump_stride, xc));
    else CK(p, launch_xstage_simt(p, st, p->d_z, 1, static_cast<float2 *>(d_vis), dump_stride, xc));
    return COBALT_OK;
}

}  // extern "C"
