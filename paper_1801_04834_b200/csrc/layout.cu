// Conversions between the plan's internal channelised layout (cobalt_internal.h) and the plain
// [C][2S][n_t] complex64 array of the debug taps cobalt_debug_channelised / cobalt_debug_correlate.
// Test plumbing around step a7 ("transposes data on write-back"); not on the production path.
#include "cobalt_internal.h"

namespace cobalt {

namespace {

__device__ __forceinline__ size_t z16_offset(int c, int kt, int plane, int m, int tt, int n_kt, int Mpad) {
    // byte offset of element (channel c, k-tile kt, plane, row m, spectrum tt of the tile)
    return ((((size_t)c * n_kt + kt) * (Mpad >> 3) + (m >> 3)) * 2 + plane) * 1024 + (size_t)(m & 7) * 128 +
           ((((tt >> 3) ^ (m & 7)) << 4) | ((tt & 7) << 1));
}

// rotation of input m, channel c as the X-stage applies it (xstage_tc.cu): phase[(b S + m / 2) C + c] * poff[m]
__device__ __forceinline__ float2 rot_of(const float2 *phase, const float2 *poff, int b, int S, int C, int m, int c) {
    float2 w = phase[((size_t)b * S + (m >> 1)) * C + c];
    if (poff) {
        const float2 q = poff[m];
        w = make_float2(w.x * q.x - w.y * q.y, w.x * q.y + w.y * q.x);
    }
    return w;
}

__global__ void z16_to_float_kernel(const unsigned char *__restrict__ z, float inv_s, const float2 *__restrict__ phase,
                                    const float2 *__restrict__ poff, int b, int S,
                                    float2 *__restrict__ out, int C, int M, int Mpad, int n_kt, long long n_t) {
    const long long total = (long long)C * M * n_t;   // the operands carry the power-of-two scale s (fstage.cu)
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long t = idx % n_t;
        const int m = (int)((idx / n_t) % M);
        const int c = (int)(idx / (n_t * M));
        const int kt = (int)(t / kKTile), tt = (int)(t % kKTile);
        const __half re = *reinterpret_cast<const __half *>(z + z16_offset(c, kt, 0, m, tt, n_kt, Mpad));
        const __half im = *reinterpret_cast<const __half *>(z + z16_offset(c, kt, 1, m, tt, n_kt, Mpad));
        const float2 v = make_float2(__half2float(re) * inv_s, __half2float(im) * inv_s);
        const float2 w = phase ? rot_of(phase, poff, b, S, C, m, c) : make_float2(1.f, 0.f);
        out[idx] = make_float2(v.x * w.x - v.y * w.y, v.x * w.y + v.y * w.x);
    }
}

__global__ void z32_to_float_kernel(const float2 *__restrict__ z, const float2 *__restrict__ phase, const float2 *__restrict__ poff,
                                    int b, int S, float2 *__restrict__ out, int C, int M, long long n_t) {
    const long long total = (long long)C * M * n_t;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int m = (int)((idx / n_t) % M);
        const int c = (int)(idx / (n_t * M));
        const float2 v = z[idx];
        const float2 w = phase ? rot_of(phase, poff, b, S, C, m, c) : make_float2(1.f, 0.f);
        out[idx] = make_float2(v.x * w.x - v.y * w.y, v.x * w.y + v.y * w.x);
    }
}

// Writes every element of the [C][n_kt][Mpad/8][2][8][64] block, zeros in the padding rows / spectra.
__global__ void float_to_z16_kernel(const float2 *__restrict__ in, unsigned char *__restrict__ z, int C, int M,
                                    int Mpad, int n_kt, long long n_t) {
    const long long total = (long long)C * n_kt * Mpad * kKTile;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int tt = (int)(idx % kKTile);
        const int m = (int)((idx / kKTile) % Mpad);
        const int kt = (int)((idx / ((long long)kKTile * Mpad)) % n_kt);
        const int c = (int)(idx / ((long long)kKTile * Mpad * n_kt));
        const long long t = (long long)kt * kKTile + tt;
        float2 v = make_float2(0.f, 0.f);
        if (m < M && t < n_t) v = in[((size_t)c * M + m) * n_t + t];
        *reinterpret_cast<__half *>(z + z16_offset(c, kt, 0, m, tt, n_kt, Mpad)) = __float2half_rn(v.x);
        *reinterpret_cast<__half *>(z + z16_offset(c, kt, 1, m, tt, n_kt, Mpad)) = __float2half_rn(v.y);
    }
}

inline unsigned grid_for(long long total, int threads) {
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 65535) blocks = 65535;
    if (blocks < 1) blocks = 1;
    return (unsigned)blocks;
}

}  // namespace

cudaError_t launch_z_to_float(const cobalt_plan_s *p, cudaStream_t st, const void *d_zsub, float2 *d_out, const XCall &xc) {
    const long long total = (long long)p->C * p->M * p->n_t;
    if (p->mode == COBALT_MODE_TENSOR_FP16)
        z16_to_float_kernel<<<grid_for(total, 256), 256, 0, st>>>(static_cast<const unsigned char *>(d_zsub), 1.f / p->zscale, xc.phase, xc.poff,
                                                                  xc.b0, p->S, d_out, p->C, p->M, p->Mpad, p->n_kt, p->n_t);
    else
        z32_to_float_kernel<<<grid_for(total, 256), 256, 0, st>>>(static_cast<const float2 *>(d_zsub), xc.phase, xc.poff, xc.b0, p->S, d_out,
                                                                  p->C, p->M, p->n_t);
    return cudaGetLastError();
}

cudaError_t launch_float_to_z(const cobalt_plan_s *p, cudaStream_t st, const float2 *d_in, void *d_zsub) {
    if (p->mode == COBALT_MODE_TENSOR_FP16) {
        const long long total = (long long)p->C * p->n_kt * p->Mpad * kKTile;
        float_to_z16_kernel<<<grid_for(total, 256), 256, 0, st>>>(d_in, static_cast<unsigned char *>(d_zsub), p->C,
                                                                  p->M, p->Mpad, p->n_kt, p->n_t);
        return cudaGetLastError();
    }
    const long long total = (long long)p->C * p->M * p->n_t;
    return cudaMemcpyAsync(d_zsub, d_in, (size_t)total * sizeof(float2), cudaMemcpyDeviceToDevice, st);
}

}  // namespace cobalt
