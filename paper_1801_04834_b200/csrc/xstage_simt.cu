// X-stage, EXACT_FP32 mode: plain fp32 FMA correlator (steps a8-a9, "computes the
// correlations of all pairs of antenna fields and averages in time").  This is the fp32 arm of
// BASELINE.json's tolerance ("max relative error of 1e-4 in fp32"); the production arm is the
// tcgen05 kernel in xstage_tc.cu.
//
// CTA = one 32 x 32 tile of (input a, input b) pairs of one (subband, channel), upper triangle of
// tiles only; 256 threads, each a 2 x 2 block of complex accumulators; time staged through shared
// memory 16 spectra at a time.  V[bl(i,k)][p][q] = sum_t z_{2i+p}[t] conj(z_{2k+q}[t]), i <= k.
#include "cobalt_internal.h"

namespace cobalt {

namespace {

constexpr int kTile = 32, kTk = 16;

__global__ void __launch_bounds__(256) xstage_simt_kernel(const float2 *__restrict__ z, float2 *__restrict__ vis, int C,
                                                         int M, long long n_t, long long n_bl, size_t z_sub_elems, int nb,
                                                         long long dump_len, size_t dump_stride, const float2 *__restrict__ phase,
                                                         const float2 *__restrict__ poff, int b0, float inv_s2) {
    __shared__ float2 As[kTk][kTile + 1];
    __shared__ float2 Bs[kTk][kTile + 1];
    const int pair = blockIdx.x;
    int tj = (int)((sqrtf(8.f * (float)pair + 1.f) - 1.f) * 0.5f);
    while (tj * (tj + 1) / 2 > pair) --tj;
    while ((tj + 1) * (tj + 2) / 2 <= pair) ++tj;
    const int ti = pair - tj * (tj + 1) / 2;
    // blockIdx.z = dump * nb + subband of the chunk; dump d integrates the spectra [d dump_len, min((d + 1) dump_len, n_t))
    const int c = blockIdx.y, d = blockIdx.z / nb, bl = blockIdx.z - d * nb;
    const long long t_begin = (long long)d * dump_len, t_end = min(n_t, t_begin + dump_len);
    const float2 *zc = z + (size_t)bl * z_sub_elems + (size_t)c * M * n_t;
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
    float2 *vc = vis + (size_t)d * dump_stride + ((size_t)bl * C + c) * n_bl * 4;
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            const int a = ti * kTile + ty * 2 + u, b = tj * kTile + tx * 2 + v;
            const int i = a >> 1, k = b >> 1;
            if (a < M && b < M && i <= k) {
                // steps a5, a6 (and reading A22) behind the integration: V_ik <- V_ik w_a conj(w_b), w = rotation * bandpass
                float2 r = make_float2(acc[u][v].x * inv_s2, acc[u][v].y * inv_s2);
                if (phase) {
                    const int S = M >> 1;
                    float2 wa = phase[((size_t)(b0 + bl) * S + i) * C + c], wb = phase[((size_t)(b0 + bl) * S + k) * C + c];
                    if (poff) {
                        const float2 qa = poff[a], qb = poff[b];
                        wa = make_float2(wa.x * qa.x - wa.y * qa.y, wa.x * qa.y + wa.y * qa.x);
                        wb = make_float2(wb.x * qb.x - wb.y * qb.y, wb.x * qb.y + wb.y * qb.x);
                    }
                    const float2 t = make_float2(wa.x * wb.x + wa.y * wb.y, wa.y * wb.x - wa.x * wb.y);   // wa conj(wb)
                    r = make_float2(r.x * t.x - r.y * t.y, r.x * t.y + r.y * t.x);
                }
                vc[((size_t)k * (k + 1) / 2 + i) * 4 + (a & 1) * 2 + (b & 1)] = r;
            }
        }
}

}  // namespace

cudaError_t launch_xstage_simt(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int nb, float2 *d_vis, size_t dump_stride,
                               const XCall &xc) {
    const int ntile = (p->M + kTile - 1) / kTile;
    dim3 grid((unsigned)(ntile * (ntile + 1) / 2), (unsigned)p->C, (unsigned)(nb * p->dumps));
    xstage_simt_kernel<<<grid, 256, 0, st>>>(static_cast<const float2 *>(d_z), d_vis, p->C, p->M, p->n_t, p->n_bl,
                                             p->z_subband_bytes / sizeof(float2), nb, (long long)(p->n_kt / p->dumps) * kKTile, dump_stride,
                                             xc.phase, xc.poff, xc.b0, xc.inv_s2);
    return cudaGetLastError();
}

}  // namespace cobalt
