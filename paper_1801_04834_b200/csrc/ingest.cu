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

// The common case of ingest_kernel -- pol-minor int16 / int8 with N a multiple of G -- with 16-byte accesses: a thread takes G =
// 4 (int16) or 8 (int8) consecutive time samples of one (subband, station), i.e. 32 contiguous bytes of (pol 0, pol 1) pairs, and
// writes 16 bytes to each polarisation's planar stream.  (The element-wise kernel reads every other 4-byte word per warp and
// reached 3.6 TB/s of the 6.5 TB/s a copy gets.)  A source that is not 16-byte aligned (odd coarse offset, odd N_in, a caller's
// base pointer aligned to a sample only) is read sample by sample; the destination (plan-owned) is always aligned.
template <int BITS>
__global__ void ingest_polminor_vec_kernel(const unsigned char *__restrict__ in, unsigned char *__restrict__ out, const int *__restrict__ coarse,
                                           int S, long long N, long long N_in, long long total_groups) {
    constexpr int SB = BITS == 16 ? 4 : 2;         // bytes per complex sample
    constexpr int G = 16 / SB;                     // time samples per thread
    const long long gpr = N / G;                   // groups per (subband, station)
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total_groups; idx += (long long)gridDim.x * blockDim.x) {
        const long long g = idx % gpr, bs = idx / gpr;
        const long long n0 = g * G + (coarse ? coarse[bs % S] : 0);
        const unsigned char *src = in + ((bs * N_in + n0) * 2) * SB;
        uint32_t w[8];                             // 32 bytes: int16 (p0 t0)(p1 t0)(p0 t1)...; int8 (p0 t0 | p1 t0)(p0 t1 | p1 t1)...
        if ((reinterpret_cast<uintptr_t>(src) & 15u) == 0) {
            const uint4 a = reinterpret_cast<const uint4 *>(src)[0], b = reinterpret_cast<const uint4 *>(src)[1];
            w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
            w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w;
        } else if (SB == 4) {
#pragma unroll
            for (int k = 0; k < 8; ++k) w[k] = reinterpret_cast<const uint32_t *>(src)[k];
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                w[k] = (uint32_t) reinterpret_cast<const unsigned short *>(src)[2 * k] | ((uint32_t) reinterpret_cast<const unsigned short *>(src)[2 * k + 1] << 16);
        }
        uint4 o0, o1;
        if (SB == 4) {
            o0 = make_uint4(w[0], w[2], w[4], w[6]);
            o1 = make_uint4(w[1], w[3], w[5], w[7]);
        } else {                                   // low halves = pol 0, high halves = pol 1
            o0 = make_uint4(__byte_perm(w[0], w[1], 0x5410), __byte_perm(w[2], w[3], 0x5410), __byte_perm(w[4], w[5], 0x5410), __byte_perm(w[6], w[7], 0x5410));
            o1 = make_uint4(__byte_perm(w[0], w[1], 0x7632), __byte_perm(w[2], w[3], 0x7632), __byte_perm(w[4], w[5], 0x7632), __byte_perm(w[6], w[7], 0x7632));
        }
        unsigned char *dst = out + ((bs * 2) * N + g * G) * SB;
        *reinterpret_cast<uint4 *>(dst) = o0;
        *reinterpret_cast<uint4 *>(dst + N * SB) = o1;
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
    if (pm && p->bits_in != 4 && p->N % (p->bits_in == 16 ? 4 : 8) == 0) {      // 16-byte accesses (see the kernel)
        const long long groups = (long long)nb * p->S * (p->N / (p->bits_in == 16 ? 4 : 8));
        const unsigned gv = grid_for(groups, 256);
        if (p->bits_in == 16) ingest_polminor_vec_kernel<16><<<gv, 256, 0, st>>>(in, out, p->d_coarse, p->S, p->N, p->N_in, groups);
        else ingest_polminor_vec_kernel<8><<<gv, 256, 0, st>>>(in, out, p->d_coarse, p->S, p->N, p->N_in, groups);
        return cudaGetLastError();
    }
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
