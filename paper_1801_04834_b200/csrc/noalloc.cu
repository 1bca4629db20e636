// cobalt_correlate_noalloc (include/cobalt.h): steps a8-a9 ("computes the correlations of all pairs of
// antenna fields and averages in time") for callers that are not allowed to allocate device memory.
//
// Who that is.  The paper's pipeline takes every buffer from pools that are filled before the observation starts
// and then runs against a real-time deadline: cudaMalloc / cudaFree in the middle of it synchronise the
// whole device (every stream stalls, a block of antenna data is late and is dropped), and on a GPU whose memory
// has been budgeted to the last buffer they can simply fail.  The same holds for a plug-in inside a host application that
// owns all device memory through its own pool and forbids the driver's allocator.  Every other entry point of this
// library needs a cobalt_plan, and cobalt_plan allocates; this one needs no plan.
//
// What it is a variant of.  The X-stage splits the time range of small problems over several jobs that write partial
// visibilities to plan-owned scratch (cobalt_plan_s::d_xpart) and sums them afterwards (xsum_kernel, ingest.cu): too few
// (channel, tile pair) jobs would otherwise leave most of the 148 SMs idle.  Here the same two steps run in fp32 (the
// arithmetic of xstage_simt.cu, the COBALT_MODE_EXACT_FP32 arm) and the partial visibilities live in the file-scope
// array below instead of in cudaMalloc'ed memory.
//
// The array.  16 MiB (COBALT_NOALLOC_SCRATCH_BYTES), part of the library's device image: every GPU on which this
// translation unit's module gets loaded holds its own copy until the process exits, whether the entry point is ever
// called or not.  In HOST code the name g_noalloc_scratch is only a handle for the runtime, not a device address (a
// kernel handed `g_noalloc_scratch` from the host side would fault, or scribble over unrelated host-mapped memory), so
// the host asks cudaGetSymbolAddress for the address -- once per device, with that device current -- and passes the
// result to the kernels.
//
// Sharing.  All calls on a device use the same array.  Nothing in it has to start at zero: the first kernel of a call
// writes every partial-sum slot the second kernel of that call reads, so whatever the previous call left behind is never
// looked at.  Calls on ONE stream are ordered by the stream and are safe.  Calls whose kernels may overlap on the GPU (two
// streams, two host threads with a stream each) race on the array and give wrong visibilities: serialise them.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "cobalt_internal.h"

namespace {

constexpr size_t kScratchBytes = COBALT_NOALLOC_SCRATCH_BYTES;
constexpr int kMaxSlices = COBALT_NOALLOC_MAX_SLICES;
constexpr int kTile = 32, kTk = 16;
static_assert((size_t)COBALT_NOALLOC_MAX_CHANNEL_BASELINES * kMaxSlices * 4 * sizeof(float2) == kScratchBytes,
              "the documented size limit must be exactly what the array holds");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

// part[slice][c][bl][p][q] = sum over the spectra of the slice of z_{2i+p}[t] conj(z_{2k+q}[t]); CTA = one 32 x 32 tile of
// input pairs (upper triangle of tiles) of one (channel, slice); the loop body is the one of xstage_simt_kernel.
__global__ void __launch_bounds__(256) xpart_noalloc_kernel(const float2 *__restrict__ z, float2 *__restrict__ part, int M, long long n_t,
                                                            long long n_bl, long long slice_len) {
    __shared__ float2 As[kTk][kTile + 1];
    __shared__ float2 Bs[kTk][kTile + 1];
    const int pair = blockIdx.x;
    int tj = (int)((sqrtf(8.f * (float)pair + 1.f) - 1.f) * 0.5f);
    while (tj * (tj + 1) / 2 > pair) --tj;
    while ((tj + 1) * (tj + 2) / 2 <= pair) ++tj;
    const int ti = pair - tj * (tj + 1) / 2;
    const int c = blockIdx.y, C = gridDim.y, slice = blockIdx.z;
    const long long t_begin = (long long)slice * slice_len, t_end = min(n_t, t_begin + slice_len);
    const float2 *zc = z + (size_t)c * M * n_t;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;

    float2 acc[2][2];
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < 2; ++v) acc[u][v] = make_float2(0.f, 0.f);

    for (long long t0 = t_begin; t0 < t_end; t0 += kTk) {
#pragma unroll
        for (int e = tid; e < kTile * kTk; e += 256) {
            const int tt = e & (kTk - 1), row = e >> 4;
            const long long t = t0 + tt;
            const int ra = ti * kTile + row, rb = tj * kTile + row;
            As[tt][row] = (ra < M && t < t_end) ? zc[(size_t)ra * n_t + t] : make_float2(0.f, 0.f);
            Bs[tt][row] = (rb < M && t < t_end) ? zc[(size_t)rb * n_t + t] : make_float2(0.f, 0.f);
        }
        __syncthreads();
#pragma unroll
        for (int tt = 0; tt < kTk; ++tt) {
            float2 a[2], b[2];
            a[0] = As[tt][ty * 2];
            a[1] = As[tt][ty * 2 + 1];
            b[0] = Bs[tt][tx * 2];
            b[1] = Bs[tt][tx * 2 + 1];
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    acc[u][v].x = fmaf(a[u].x, b[v].x, fmaf(a[u].y, b[v].y, acc[u][v].x));
                    acc[u][v].y = fmaf(a[u].y, b[v].x, fmaf(-a[u].x, b[v].y, acc[u][v].y));
                }
        }
        __syncthreads();
    }
    // every (c, bl, p, q) of this slice is written by exactly one thread of exactly one CTA (an empty slice writes zeros),
    // which is why the array never needs clearing
    float2 *pc = part + ((size_t)slice * C + c) * n_bl * 4;
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            const int a = ti * kTile + ty * 2 + u, b = tj * kTile + tx * 2 + v;
            const int i = a >> 1, k = b >> 1;
            if (a < M && b < M && i <= k) pc[((size_t)k * (k + 1) / 2 + i) * 4 + (a & 1) * 2 + (b & 1)] = acc[u][v];
        }
}

// vis[e] = part[0][e] + part[1][e] + ... in slice order (a fixed order: the result does not depend on scheduling)
__global__ void xsum_noalloc_kernel(const float2 *__restrict__ part, float2 *__restrict__ vis, int slices, long long n_elem) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n_elem; e += (long long)gridDim.x * blockDim.x) {
        float2 acc = part[e];
        for (int s = 1; s < slices; ++s) {
            const float2 v = part[(size_t)s * n_elem + e];
            acc.x += v.x;
            acc.y += v.y;
        }
        vis[e] = acc;
    }
}

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
float2 *g_scratch_of_device[kMaxDevices] = {};   // device address of g_noalloc_scratch on each device, nullptr = not asked yet

int fail(char *h_err, int h_err_len, int code, const char *fmt, ...) {
    if (h_err && h_err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(h_err, (size_t)h_err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// The set-up step: the array's address on the CURRENT device.  First use on a device asks the runtime (which loads this
// module on the device if it is not there yet -- the moment the 16 MiB are taken); later calls read the cached pointer.
int scratch_on_current_device(float2 **out, char *h_err, int h_err_len) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(h_err, h_err_len, COBALT_ERR_UNSUPPORTED_DEVICE, "no usable CUDA device (cudaGetDevice: %s); there is no CPU fallback",
                    cudaGetErrorString(e));
    }
    if (dev < 0 || dev >= kMaxDevices) return fail(h_err, h_err_len, COBALT_ERR_UNSUPPORTED_DEVICE, "device ordinal %d is outside [0, %d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_of_device[dev]) {
        int major = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return fail(h_err, h_err_len, COBALT_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10)
            return fail(h_err, h_err_len, COBALT_ERR_UNSUPPORTED_DEVICE, "device %d has compute capability %d.x; this library is built for sm_100a only", dev, major);
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            return fail(h_err, h_err_len, COBALT_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_scratch_of_device[dev] = static_cast<float2 *>(ptr);
    }
    *out = g_scratch_of_device[dev];
    return COBALT_OK;
}

}  // namespace

extern "C" int cobalt_correlate_noalloc(void *cuda_stream, const void *d_z, int stations, int channels, long long n_spectra, void *d_vis,
                                        char *h_err, int h_err_len) {
    if (h_err && h_err_len > 0) h_err[0] = '\0';
    // 1. arguments -- before anything touches the device, so that a bad size is reported the same way on every machine
    if (!d_z || !d_vis) return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG, "d_z and d_vis must not be NULL");
    if (stations < 1) return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG, "stations must be >= 1 (got %d)", stations);
    if (channels != 16 && channels != 64 && channels != 256) return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG, "channels must be 16, 64 or 256 (got %d)", channels);
    if (n_spectra < 1 || n_spectra > (1LL << 30)) return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG, "n_spectra must be in [1, 2^30] (got %lld)", n_spectra);
    const long long n_bl = (long long)stations * ((long long)stations + 1) / 2;
    if (stations > 1024 || (long long)channels * n_bl > COBALT_NOALLOC_MAX_CHANNEL_BASELINES)
        return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG,
                    "problem too large for the static scratch: channels * n_baselines = %d * %lld = %lld exceeds "
                    "COBALT_NOALLOC_MAX_CHANNEL_BASELINES = %d (%d MiB hold %d partial sums of 32 bytes per (channel, baseline)); "
                    "use cobalt_plan + cobalt_debug_correlate / cobalt_process, which allocate",
                    channels, n_bl, (long long)channels * n_bl, COBALT_NOALLOC_MAX_CHANNEL_BASELINES, (int)(kScratchBytes >> 20), kMaxSlices);
    if ((reinterpret_cast<uintptr_t>(d_z) & 7u) != 0 || (reinterpret_cast<uintptr_t>(d_vis) & 7u) != 0)
        return fail(h_err, h_err_len, COBALT_ERR_BAD_ARG, "d_z and d_vis must be 8-byte aligned (one complex64)");
    // 2. set-up (first call on this device only): where the array lives on the current device
    float2 *part = nullptr;
    const int rc = scratch_on_current_device(&part, h_err, h_err_len);
    if (rc != COBALT_OK) return rc;
    // 3. two launches on the caller's stream, nothing else: no allocation, no synchronisation, no copy
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int M = 2 * stations;
    const long long tiles64 = (n_spectra + cobalt::kKTile - 1) / cobalt::kKTile;
    const int slices = (int)(tiles64 < kMaxSlices ? tiles64 : kMaxSlices);
    const long long slice_len = (n_spectra + slices - 1) / slices;
    const int ntile = (M + kTile - 1) / kTile;
    const dim3 grid((unsigned)(ntile * (ntile + 1) / 2), (unsigned)channels, (unsigned)slices);
    xpart_noalloc_kernel<<<grid, 256, 0, st>>>(static_cast<const float2 *>(d_z), part, M, n_spectra, n_bl, slice_len);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h_err, h_err_len, COBALT_ERR_CUDA, "xpart_noalloc_kernel launch: %s", cudaGetErrorString(e));
    const long long n_elem = (long long)channels * n_bl * 4;
    const unsigned blocks = (unsigned)((n_elem + 255) / 256);
    xsum_noalloc_kernel<<<blocks, 256, 0, st>>>(part, static_cast<float2 *>(d_vis), slices, n_elem);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h_err, h_err_len, COBALT_ERR_CUDA, "xsum_noalloc_kernel launch: %s", cudaGetErrorString(e));
    return COBALT_OK;
}
