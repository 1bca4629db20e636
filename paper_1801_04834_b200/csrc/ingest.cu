// Small kernels around the fused F- and X-stage kernels for the rows of SURVEY.md sec 8(f):
//   ingest_kernel       pol-minor wire order (reading A26) and / or 4-bit samples (A27) -> the planar int16 / int8
//                       layout the fused F-stage kernel reads, coarse sample offsets (A25) applied on the way;
//   valid_counts_kernel the weight of every visibility: spectra in which both stations are valid (A24);
//   xsum_kernel         sum of the partial visibilities when the X-stage splits a channel's time range over several jobs.
#include "cobalt_internal.h"
#include "ptx.cuh"

namespace cobalt {

namespace {

inline unsigned grid_for(long long total, int threads) {
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 65535 * 8) blocks = 65535 * 8;
    if (blocks < 1) blocks = 1;
    return (unsigned)blocks;
}

// in:  caller's samples of the chunk, stream stride N_in complex samples;
//      planar [nb][S][2][N_in], or pol-minor [nb][S][N_in][2]; element = 4 B (int16), 2 B (int8) or 1 B (4-bit)
// out: planar [nb][S][2][N], element 4 B (int16) or 2 B (int8; also for 4-bit input)
template <int BITS, bool POLMINOR>
__global__ void ingest_kernel(const unsigned char *__restrict__ in, unsigned char *__restrict__ out, const int *__restrict__ coarse,
                              int S, long long N, long long N_in, long long total) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long n = idx % N;
        const long long stream = idx / N;             // (subband of the chunk * S + station) * 2 + pol
        const int pol = (int)(stream & 1);
        const long long bs = stream >> 1;             // subband * S + station
        const long long src_n = n + (coarse ? coarse[bs % S] : 0);
        const long long e = POLMINOR ? (bs * N_in + src_n) * 2 + pol : (bs * 2 + pol) * N_in + src_n;
        if (BITS == 16) {
            reinterpret_cast<uint32_t *>(out)[idx] = reinterpret_cast<const uint32_t *>(in)[e];
        } else if (BITS == 8) {
            reinterpret_cast<unsigned short *>(out)[idx] = reinterpret_cast<const unsigned short *>(in)[e];
        } else {   // 4-bit: the same unpack_sample the debug tap pins, re-packed as int8 (exact: -8 .. 7)
            const float2 v = unpack_sample<4>(in[e]);
            const int re = (int)v.x, im = (int)v.y;
            reinterpret_cast<unsigned short *>(out)[idx] = (unsigned short)((re & 0xff) | ((im & 0xff) << 8));
        }
    }
}

// counts[b][d][bl(i,k)] = sum over the 64-spectrum tiles v of dump d of valid[b][i][v] * valid[b][k][v] * (spectra in tile v)
__global__ void valid_counts_kernel(const unsigned char *__restrict__ valid, unsigned int *__restrict__ counts, int b0, int nb, int S,
                                    int n_kt, int D, long long n_t, long long n_bl) {
    const long long total = (long long)nb * D * n_bl;
    const int K = n_kt / D;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long bl = idx % n_bl;
        const int d = (int)((idx / n_bl) % D);
        const int b = b0 + (int)(idx / (n_bl * D));
        int k = (int)((sqrtf(8.f * (float)bl + 1.f) - 1.f) * 0.5f);
        while ((long long)k * (k + 1) / 2 > bl) --k;
        while ((long long)(k + 1) * (k + 2) / 2 <= bl) ++k;
        const int i = (int)(bl - (long long)k * (k + 1) / 2);
        unsigned int c = 0;
        for (int v = d * K; v < (d + 1) * K; ++v) {
            const long long len = min((long long)kKTile, n_t - (long long)v * kKTile);
            const bool ok = !valid || (valid[((size_t)b * S + i) * n_kt + v] && valid[((size_t)b * S + k) * n_kt + v]);
            if (ok && len > 0) c += (unsigned int)len;
        }
        counts[((size_t)b * D + d) * n_bl + bl] = c;
    }
}

// out[j][e] = sum_s part[j * splits + s][e]: j = (dump, subband of chunk, channel) in the X-stage's job order, e over one
// channel block of n_elem float4 (= n_bl [2][2] complex / 2)
__global__ void xsum_kernel(const float4 *__restrict__ part, float4 *__restrict__ out, int splits, long long n_elem, long long nbC, int D,
                            size_t dump_stride4) {
    const long long total = (long long)D * nbC * n_elem;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long e = idx % n_elem;
        const long long j = idx / n_elem;             // d * nbC + prob
        const int d = (int)(j / nbC);
        const long long prob = j - (long long)d * nbC;
        float4 acc = part[(j * splits) * n_elem + e];
        for (int s = 1; s < splits; ++s) {
            const float4 v = part[(j * splits + s) * n_elem + e];
            acc.x += v.x;
            acc.y += v.y;
            acc.z += v.z;
            acc.w += v.w;
        }
        out[(size_t)d * dump_stride4 + prob * n_elem + e] = acc;
    }
}

}  // namespace

cudaError_t launch_ingest(const cobalt_plan_s *p, cudaStream_t st, const void *samples_b0, int nb, void *d_out) {
    const long long total = (long long)nb * p->M * p->N;
    const unsigned char *in = static_cast<const unsigned char *>(samples_b0);
    unsigned char *out = static_cast<unsigned char *>(d_out);
    const unsigned g = grid_for(total, 256);
    const bool pm = p->layout == COBALT_LAYOUT_POL_MINOR;
#define COBALT_INGEST(B, PM) ingest_kernel<B, PM><<<g, 256, 0, st>>>(in, out, p->d_coarse, p->S, p->N, p->N_in, total)
    if (p->bits_in == 16) { if (pm) COBALT_INGEST(16, true); else COBALT_INGEST(16, false); }
    else if (p->bits_in == 8) { if (pm) COBALT_INGEST(8, true); else COBALT_INGEST(8, false); }
    else { if (pm) COBALT_INGEST(4, true); else COBALT_INGEST(4, false); }
#undef COBALT_INGEST
    return cudaGetLastError();
}

cudaError_t launch_valid_counts(const cobalt_plan_s *p, cudaStream_t st, const unsigned char *d_valid, int b0, int nb, unsigned int *d_counts) {
    const long long total = (long long)nb * p->dumps * p->n_bl;
    valid_counts_kernel<<<grid_for(total, 256), 256, 0, st>>>(d_valid, d_counts, b0, nb, p->S, p->n_kt, p->dumps, p->n_t, p->n_bl);
    return cudaGetLastError();
}

cudaError_t launch_xsum_n(const cobalt_plan_s *p, cudaStream_t st, int nb, float2 *d_vis, size_t dump_stride, int splits) {
    const long long n_elem = p->n_bl * 2;            // float4 per channel block
    const long long total = (long long)p->dumps * nb * p->C * n_elem;
    xsum_kernel<<<grid_for(total, 256), 256, 0, st>>>(reinterpret_cast<const float4 *>(p->d_xpart), reinterpret_cast<float4 *>(d_vis),
                                                      splits, n_elem, (long long)nb * p->C, p->dumps, dump_stride / 2);
    return cudaGetLastError();
}

}  // namespace cobalt
