// X-stage, TENSOR_FP16 mode: the Hermitian contraction V = Z Z^H of one (subband, channel) on the
// 5th-generation tensor cores (steps a8-a9 of SURVEY.md sec 8(a); "computes the correlations
// of all pairs of antenna fields and averages in time"; BASELINE.json north_star (c)).
//
// Z is [2S inputs][n_t spectra] complex, held as two fp16 planes (re, im), K-major, already in the
// 128-byte-swizzled shared-memory image with the planes alternating every 8 rows (cobalt_internal.h),
// so one (channel, k-tile) arrives with one plain bulk copy (cp.async.bulk -> UBLKCP) signalled on an
// mbarrier -- no tensor map, no register staging -- and can be read plane by plane (descriptor
// stride 2048) or as the stacked matrix [Zr; Zi] (stride 1024).
//
//   Re V = Zr Zr^T + Zi Zi^T        Im V = Zi Zr^T - Zr Zi^T
//
// is four tcgen05.mma (kind::f16, fp32 accumulate in TMEM) per 16-spectrum k-step into two
// accumulators; the minus sign is the instruction descriptor's negate-A bit, so no negated plane is
// ever stored.  Only tiles on or above the station diagonal are computed: an XJob (built once per
// plan by build_xjobs) names the rows to load and up to two accumulator groups
//   rows [0,128) x cols [0,Mpad)  (M = 128, four products)  and, for the rows the 128-row instruction
//   cannot reach, ONE product W W^T of the stacked rows W = [Zr; Zi][128, Mpad) per k-step (all four
//   real products at once; the epilogue adds / subtracts its quadrants)            (2S <= 192)
// or, for large arrays, one (128-row block) x (<= 256-column chunk) tile per job.
//
// Warp roles (640 threads, persistent CTAs, one per SM): warp 0 = bulk-copy producer, warp 1 = TMEM
// allocator + single-thread MMA issuer, warps 2-3 idle (they complete the warp group that hands its registers
// to the epilogue), warps 4-19 = epilogue (tcgen05.ld -> rotation w_i conj(w_k) / s^2 -> triangular baseline
// index -> 16-byte stores of (re, im) pairs into a shared-memory image of the channel's output block,
// which leaves with one bulk store; direct global stores when the block does not fit).
#include "cobalt_internal.h"
#include "ptx.cuh"

namespace cobalt {

namespace {

constexpr int kEpiWarps = 16;           // four per TMEM lane quarter, taking every fourth 16-column chunk
constexpr int kEpiSub = kEpiWarps / 4;
// Warp group 0 = producer, MMA issuer and two idle warps: it drops to 32 registers so that the four epilogue warp groups can
// rise to 112 (setmaxnreg moves registers between complete groups of four warps of one CTA).
constexpr int kFirstEpiWarp = 4;
constexpr int kThreads = 32 * (kFirstEpiWarp + kEpiWarps);
constexpr int kBarrierBytes = 4096;       // mbarriers (first 512 bytes) + a copy of the job table
constexpr int kMaxSmemJobs = (kBarrierBytes - 512) / (int)sizeof(XJob);

struct XArgs {
    const unsigned char *z;
    float2 *vis;
    const XJob *jobs;
    // V_ik <- V_ik w_i conj(w_k) / s^2 (XCall, cobalt_internal.h): w_m = phase[((b0 + subband) S + m / 2) C + channel] poff[m]
    const float2 *phase, *poff;
    int b0, S;
    float inv_s2;           // 1 / s^2, s = power-of-two scale of the fp16 intermediate (exact)
    uint32_t rot_off, rot_bytes;   // two per-job tables of w_m (one per job parity) in shared memory, before the stages
    size_t z_subband_bytes;
    long long n_bl;
    int C, M, Mpad, n_kt, jobs_per_channel, total_jobs, stages, stage_bytes;
    uint32_t out_off;       // STAGED: byte offset of the visibility staging block from the 1024-aligned smem base
    // dumps (reading A23) and split time ranges: job id = ((dump * nbC + subband-of-chunk * C + channel) * splits + split) *
    // jobs_per_channel + job-of-channel; it integrates the k-tiles [dump * K + K split / splits, dump * K + K (split + 1) / splits)
    float2 *part;           // splits > 1: partial visibilities, one channel block per (dump, subband, channel, split)
    size_t dump_stride;     // float2 between the dumps of `vis`
    int D, K, splits, nbC;
};

struct XWork {
    int jl, prob, kt0, nkt;
    float2 *out;
};
__device__ __forceinline__ XWork decode_job(const XArgs &a, int jid) {
    XWork w;
    w.jl = jid % a.jobs_per_channel;
    const int slot = jid / a.jobs_per_channel;
    const int sp = slot % a.splits, j = slot / a.splits;
    const int d = j / a.nbC;
    w.prob = j - d * a.nbC;
    const int k0 = (a.K * sp) / a.splits, k1 = (a.K * (sp + 1)) / a.splits;
    w.kt0 = d * a.K + k0;
    w.nkt = k1 - k0;
    w.out = a.splits > 1 ? a.part + (size_t)slot * a.n_bl * 4 : a.vis + (size_t)d * a.dump_stride + (size_t)w.prob * a.n_bl * 4;
    return w;
}

// Two visibilities (same row input, column inputs b and b + 1) times u conj(w_b), u conj(w_{b+1}): u = w_row / s^2, wb = (w_b, w_{b+1}).
__device__ __forceinline__ float4 rotate2(float re0, float im0, float re1, float im1, float2 u, float4 wb) {
    const float t0r = u.x * wb.x + u.y * wb.y, t0i = u.y * wb.x - u.x * wb.y;
    const float t1r = u.x * wb.z + u.y * wb.w, t1i = u.y * wb.z - u.x * wb.w;
    return make_float4(re0 * t0r - im0 * t0i, re0 * t0i + im0 * t0r, re1 * t1r - im1 * t1i, re1 * t1i + im1 * t1r);
}

// STAGED (one job per channel and the channel's [n_bl][2][2] block fits in shared memory): the epilogue writes
// the visibilities into a shared-memory image of the channel's output block and one thread sends it to global
// memory with a single bulk copy (cp.async.bulk, SASS UBLKCP) that drains while the next job's MMAs run; the
// accumulators are handed back as soon as the last TMEM load has landed.
template <bool STAGED>
__global__ void __launch_bounds__(kThreads, 1) xstage_tc_kernel(const XArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // carve: [barriers 1 KB][stages ...][slack]; stage base must be 1024-byte aligned for the swizzle
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base;                       // full[s] at +8 s, empty[s] at +8 (16 + s)
    const uint32_t tmem_full = bar_base + 8 * 32, tmem_empty = bar_base + 8 * 33;
    const uint32_t tmem_slot = bar_base + 8 * 34;              // 4 bytes: TMEM base address
    const uint32_t stage_base = smem_base + kBarrierBytes + 2 * a.rot_bytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int stages = a.stages;

    // the job table is read by every role for every job: keep it in shared memory (global-memory latency would sit
    // on the epilogue's critical path)
    const XJob *jobs = a.jobs;
    if (a.jobs_per_channel <= kMaxSmemJobs) {
        int *dst = reinterpret_cast<int *>(smem_raw + (smem_base - smem_u32(smem_raw)) + 512);
        const int *src = reinterpret_cast<const int *>(a.jobs);
        for (int w = threadIdx.x; w < a.jobs_per_channel * (int)(sizeof(XJob) / 4); w += kThreads) dst[w] = src[w];
        jobs = reinterpret_cast<const XJob *>(dst);
    }
    // every job of one plan allocates the same number of columns (max over jobs)
    int tmem_cols = 32;
    for (int j = 0; j < a.jobs_per_channel; ++j) tmem_cols = max(tmem_cols, a.jobs[j].tmem_cols);

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (16 + s), 1);
        }
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, kEpiWarps);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
        if (elect_one()) {
            int s = 0;
            uint32_t ph = 0;
            const size_t kt_bytes = (size_t)a.Mpad * 256;     // [Mpad / 8][2 planes][8 rows][128 B]
            for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x) {
                const XWork w = decode_job(a, jid);
                const int jl = w.jl;
                const int bl = w.prob / a.C, c = w.prob - bl * a.C;   // prob = subband-of-chunk * C + channel
                const int r0 = jobs[jl].ld_row[0], r1 = jobs[jl].ld_row[1];
                const uint32_t b0 = (uint32_t)jobs[jl].ld_nrows[0] * 256, b1 = (uint32_t)jobs[jl].ld_nrows[1] * 256;
                const unsigned char *src = a.z + (size_t)bl * a.z_subband_bytes + ((size_t)c * a.n_kt + w.kt0) * kt_bytes;
                for (int kt = 0; kt < w.nkt; ++kt, src += kt_bytes) {
                    mbar_wait(bar_base + 8 * (16 + s), ph ^ 1);
                    const uint32_t full = bar_base + 8 * s;
                    const uint32_t dst = stage_base + (uint32_t)s * a.stage_bytes;
                    mbar_arrive_expect_tx(full, b0 + b1);
                    bulk_g2s(dst, src + (size_t)r0 * 256, b0, full);
                    if (b1 > 0) bulk_g2s(dst + b0, src + (size_t)r1 * 256, b1, full);
                    if (++s == stages) {
                        s = 0;
                        ph ^= 1;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
        if (elect_one()) {
            int s = 0;
            uint32_t ph = 0, it = 0;
            // shared-memory descriptor of byte offset 0 of stage 0; rows / stages / k-steps only add to the
            // 14-bit start-address field (units of 16 bytes; shared memory is < 256 KB, so it cannot carry out)
            const uint64_t desc_plane = make_smem_desc(stage_base, 2048);   // one plane: atoms 2048 bytes apart
            const uint64_t desc_both = make_smem_desc(stage_base, 1024);    // [Zr; Zi] stacked 8 rows at a time
            const uint32_t stage_units = (uint32_t)a.stage_bytes >> 4;
            for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x, ++it) {
                const XWork w = decode_job(a, jid);
                const XJob *job = jobs + w.jl;
                const int n_groups = job->n_groups;
                uint32_t g_a[kMaxMmaGroups], g_b[kMaxMmaGroups], g_d[kMaxMmaGroups], g_n[kMaxMmaGroups];
                uint32_t g_pos[kMaxMmaGroups], g_neg[kMaxMmaGroups], g_kind[kMaxMmaGroups];
#pragma unroll
                for (int g = 0; g < kMaxMmaGroups; ++g) {
                    const XMmaGroup &grp = job->g[g < n_groups ? g : 0];
                    g_a[g] = (uint32_t)grp.a_row * 16;             // 256 bytes per row of both planes, >> 4
                    g_b[g] = (uint32_t)grp.b_row * 16;
                    g_kind[g] = (uint32_t)grp.kind;
                    g_n[g] = (uint32_t)grp.n;
                    g_d[g] = tmem_base + (uint32_t)grp.tmem_col;
                    g_pos[g] = make_idesc(grp.m, grp.n, 0);
                    g_neg[g] = make_idesc(grp.m, grp.n, 1);
                }
                mbar_wait_spin(tmem_empty, (it & 1) ^ 1);  // epilogue has drained the accumulators
                tc_fence_after();
                for (int kt = 0; kt < w.nkt; ++kt) {
                    mbar_wait(bar_base + 8 * s, ph);
                    tc_fence_after();
                    const uint64_t so = (uint64_t)((uint32_t)s * stage_units);
#pragma unroll
                    for (int g = 0; g < kMaxMmaGroups; ++g) {
                        if (g < n_groups && g_kind[g] == 1) {
                            const uint64_t aw = desc_both + so + g_a[g], bw = desc_both + so + g_b[g];
#pragma unroll
                            for (int ks = 0; ks < kKTile / 16; ++ks)
                                tc_mma(g_d[g], aw + (uint64_t)(ks * 2), bw + (uint64_t)(ks * 2), g_pos[g], (kt | ks) ? 1u : 0u);
                        } else if (g < n_groups) {
                            const uint64_t ar = desc_plane + so + g_a[g], ai = ar + 64;   // im plane: 1024 bytes in
                            const uint64_t br = desc_plane + so + g_b[g], bi = br + 64;
                            const uint32_t d_re = g_d[g], d_im = d_re + g_n[g];
#pragma unroll
                            for (int ks = 0; ks < kKTile / 16; ++ks) {
                                const uint32_t acc = (kt | ks) ? 1u : 0u;
                                const uint64_t ko = (uint64_t)(ks * 2);         // 32 bytes per k-step, >> 4
                                tc_mma(d_re, ar + ko, br + ko, g_pos[g], acc);    // Re  = Zr Zr^T
                                tc_mma(d_re, ai + ko, bi + ko, g_pos[g], 1u);     // Re += Zi Zi^T
                                tc_mma(d_im, ai + ko, br + ko, g_pos[g], acc);    // Im  = Zi Zr^T
                                tc_mma(d_im, ar + ko, bi + ko, g_neg[g], 1u);     // Im -= Zr Zi^T
                            }
                        }
                    }
                    tc_commit(bar_base + 8 * (16 + s));    // stage free once these MMAs have read it
                    if (++s == stages) {
                        s = 0;
                        ph ^= 1;
                    }
                }
                tc_commit(tmem_full);                      // accumulators complete
            }
        }
    } else if (warp < kFirstEpiWarp) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");      // the two idle warps of warp group 0
    } else {
        // ------------------------------------------------------------------ epilogue
        asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
        // Warps 4..19: warp w reads TMEM lane quarter w % 4 (the only one it may access); the two warps of a quarter
        // take alternate 16-column chunks.  The TMEM load of a warp's next chunk is in flight while it stores the
        // current one.
        const int wq = warp & 3;
        const int sub = (warp - kFirstEpiWarp) >> 2;
        const float inv_s2 = a.inv_s2;                     // undo the power-of-two operand scale (exact)
        unsigned char *smem_al = smem_raw + (smem_base - smem_u32(smem_raw));
        uint32_t it = 0;
        for (int jid = blockIdx.x; jid < a.total_jobs; jid += gridDim.x, ++it) {
            const XWork w = decode_job(a, jid);
            const XJob *job = jobs + w.jl;
            const int n_groups = job->n_groups;
            float4 *vg = reinterpret_cast<float4 *>(w.out);
            float4 *vc = STAGED ? reinterpret_cast<float4 *>(smem_al + a.out_off) : vg;
            // this job's rotation table w_m (steps a5, a6, reading A22 applied behind the integration), loaded while the MMAs run;
            // two tables alternate: a warp is never more than one job ahead of the slowest one (tmem_empty needs all of them)
            float2 *rot = reinterpret_cast<float2 *>(smem_al + a.rot_off + (it & 1) * a.rot_bytes);
            {
                const int bl = w.prob / a.C, c = w.prob - bl * a.C;
                for (int m = threadIdx.x - 32 * kFirstEpiWarp; m < a.Mpad; m += 32 * kEpiWarps) {
                    float2 wv = make_float2(1.f, 0.f);
                    if (a.phase && m < a.M) {
                        wv = a.phase[((size_t)(a.b0 + bl) * a.S + (m >> 1)) * a.C + c];
                        if (a.poff) {
                            const float2 q = a.poff[m];
                            wv = make_float2(wv.x * q.x - wv.y * q.y, wv.x * q.y + wv.y * q.x);
                        }
                    }
                    rot[m] = wv;
                }
                asm volatile("bar.sync 3, %0;" ::"n"(32 * kEpiWarps) : "memory");
            }
            if (STAGED && it > 0) {
                // the previous job's bulk store must have read the staging block before it is overwritten
                if (threadIdx.x == 32 * kFirstEpiWarp) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                asm volatile("bar.sync 1, %0;" ::"n"(32 * kEpiWarps) : "memory");
            }
            mbar_wait(tmem_full, it & 1);
            tc_fence_after();
            for (int g = 0; g < n_groups; ++g) {
                const int gm = job->g[g].m, gn = job->g[g].n, row_min = job->g[g].row_min;
                const int out_col = job->g[g].out_col;
                // M = 128: accumulator row = TMEM lane; M = 64: row r in lane 32 (r / 16) + r % 16
                const int rows_w = gm == 128 ? 32 : 16;
                if (job->g[g].kind == 1) {
                    // Stacked product D = W W^T, W = [Zr; Zi] 8 rows at a time: accumulator row (and column)
                    // a = 16 q + 8 plane + r is input out_row + 8 q + r.  A lane and its partner lane ^ 8 hold the
                    // re-plane and im-plane rows of one input; a 16-column chunk is 8 inputs, re columns then im.
                    //   Re V = D[re][re] + D[im][im]        Im V = D[im][re] - D[re][im]
                    const int arow = wq * rows_w + (lane & (rows_w - 1));
                    const int pl = (arow >> 3) & 1;
                    const int mrow = job->g[g].out_row + ((arow >> 4) << 3) + (arow & 7);
                    const bool row_ok = lane < rows_w && arow < gn && mrow < a.M;
                    const int i = mrow >> 1, p = mrow & 1;
                    const uint32_t t0 = tmem_base + ((uint32_t)(wq * 32) << 16) + job->g[g].tmem_col;
                    if (wq * rows_w < gn) {                             // warp-uniform
                        for (int c = sub; c < (gn >> 4); c += kEpiSub) {
                            uint32_t x[16];
                            tmem_ld16(t0 + c * 16, x);
                            tmem_ld_wait();
                            float val[8];
#pragma unroll
                            for (int r = 0; r < 8; ++r) {
                                const float o = __shfl_xor_sync(0xffffffffu, __uint_as_float(x[8 + r]), 8);
                                val[r] = pl ? __uint_as_float(x[r]) - o : __uint_as_float(x[r]) + o;
                            }
                            // re-plane lanes finish columns 0-3 of the chunk, im-plane lanes columns 4-7
                            float re[4], im[4];
#pragma unroll
                            for (int q = 0; q < 4; ++q) {
                                const float got = __shfl_xor_sync(0xffffffffu, pl ? val[q] : val[4 + q], 8);
                                re[q] = pl ? got : val[q];
                                im[q] = pl ? val[4 + q] : got;
                            }
                            const int b0 = job->g[g].out_col + 8 * c + 4 * pl;      // input index of column q = 0
                            const float2 ur = rot[min(mrow, a.Mpad - 1)];
                            const float2 u = make_float2(ur.x * inv_s2, ur.y * inv_s2);
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int b = b0 + 2 * e, k = b >> 1;
                                if (row_ok && b < a.M && i <= k)
                                    vc[((size_t)k * (k + 1) / 2 + i) * 2 + p] = rotate2(re[2 * e], im[2 * e], re[2 * e + 1], im[2 * e + 1], u,
                                                                                    *reinterpret_cast<const float4 *>(rot + b));
                            }
                        }
                    }
                    continue;
                }
                const int row0 = job->g[g].out_row + wq * rows_w;      // first input index of this warp's lanes
                const int arow = row0 + (lane & (rows_w - 1));
                const bool lane_ok = lane < rows_w && arow >= row_min && arow < a.M;
                const int i = arow >> 1, p = arow & 1;
                if (row0 >= a.M || row0 + rows_w <= row_min) continue;
                const uint32_t t0 = tmem_base + ((uint32_t)(wq * 32) << 16) + job->g[g].tmem_col;
                // chunks of this warp: every kEpiSub-th chunk on or above the diagonal, inside the matrix
                const int c_first = (max(0, (max(row0, row_min) & ~1) - out_col) >> 4) + sub;   // first chunk touching k >= i
                const int c_end = (min(gn, a.M - out_col) + 15) >> 4;
                const int i_max = (min(row0 + rows_w, a.M) - 1) >> 1;           // last station of this warp's rows
                // The warp's chunks as pieces of 8 columns (4 station-pol pairs), double buffered: the TMEM load of the next
                // piece is issued before the current one is rotated and stored, so that the load latency (TMEM reads are the
                // floor of this exposed epilogue) overlaps the arithmetic.  tcgen05.wait::ld waits for every outstanding load,
                // hence exactly one load pair is in flight at each wait.
                const float2 ur = rot[min(arow, a.Mpad - 1)];
                const float2 u = make_float2(ur.x * inv_s2, ur.y * inv_s2);
                const int n_pieces = c_first < c_end ? 2 * ((c_end - c_first + kEpiSub - 1) / kEpiSub) : 0;
                auto piece_col = [&](int pc) { return (c_first + (pc >> 1) * kEpiSub) * 16 + 8 * (pc & 1); };   // column within the group
                auto process = [&](const uint32_t (&re)[8], const uint32_t (&im)[8], int pc) {
                    const int col0 = out_col + piece_col(pc);
                    float4 v[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        v[e] = rotate2(__uint_as_float(re[2 * e]), __uint_as_float(im[2 * e]), __uint_as_float(re[2 * e + 1]),
                                       __uint_as_float(im[2 * e + 1]), u, *reinterpret_cast<const float4 *>(rot + col0 + 2 * e));
                    const int k0 = col0 >> 1;
                    if (k0 >= i_max && col0 + 8 <= a.M) {
                        // whole piece above the diagonal for every row of the warp: baseline index of (i, k0 + e) steps by k
                        if (lane_ok) {
                            int idx = (k0 * (k0 + 1) / 2 + i) * 2 + p;
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                vc[idx] = v[e];
                                idx += 2 * (k0 + e + 1);
                            }
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int b = col0 + 2 * e, k = b >> 1;
                            if (lane_ok && b < a.M && i <= k) vc[((size_t)k * (k + 1) / 2 + i) * 2 + p] = v[e];
                        }
                    }
                };
                uint32_t reA[8], imA[8], reB[8], imB[8];
                if (n_pieces > 0) {
                    tmem_ld8(t0 + piece_col(0), reA);
                    tmem_ld8(t0 + gn + piece_col(0), imA);
                }
                for (int pc = 0; pc < n_pieces; pc += 2) {
                    tmem_ld_wait();
                    tmem_ld8(t0 + piece_col(pc + 1), reB);            // n_pieces is even
                    tmem_ld8(t0 + gn + piece_col(pc + 1), imB);
                    process(reA, imA, pc);
                    tmem_ld_wait();
                    if (pc + 2 < n_pieces) {
                        tmem_ld8(t0 + piece_col(pc + 2), reA);
                        tmem_ld8(t0 + gn + piece_col(pc + 2), imA);
                    }
                    process(reB, imB, pc + 1);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty);        // every TMEM load of this warp has completed (wait::ld)
            if (STAGED) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the bulk copy
                asm volatile("bar.sync 2, %0;" ::"n"(32 * kEpiWarps) : "memory");
                if (threadIdx.x == 32 * kFirstEpiWarp) {
                    bulk_s2g(vg, smem_base + a.out_off, (uint32_t)(a.n_bl * 32));
                    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                }
            }
        }
        if (STAGED && threadIdx.x == 32 * kFirstEpiWarp) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }
int pow2_cols(int c) {
    int p = 32;
    while (p < c) p <<= 1;
    return p;
}

}  // namespace

// Tiling of the upper triangle of one channel's (2S x 2S) product into XJobs (see file header).
void build_xjobs(cobalt_plan_s *p) {
    p->jobs.clear();
    const int Mpad = p->Mpad;
    if (Mpad <= 192) {
        XJob j{};
        j.ld_row[0] = 0;
        j.ld_nrows[0] = Mpad;
        j.ld_row[1] = 0;
        j.ld_nrows[1] = 0;
        j.n_groups = 1;
        j.g[0] = XMmaGroup{0, 0, Mpad, 0, 0, 0, 128, 0, 0};
        int cols = 2 * Mpad;
        if (Mpad > 128) {
            j.n_groups = 2;
            // rows and columns [128, Mpad): one stacked product per k-step (kind 1), 2 (Mpad - 128) rows and columns
            const int nw = 2 * (Mpad - 128);
            j.g[1] = XMmaGroup{128, 128, nw, 2 * Mpad, 128, 128, nw <= 64 ? 64 : 128, 128, 1};
            cols += nw;
        }
        j.tmem_cols = pow2_cols(cols);
        p->jobs.push_back(j);
    } else {
        const int nrb = (Mpad + 127) / 128;
        for (int I = 0; I < nrb; ++I) {
            const int r0 = 128 * I;
            const int na = (Mpad - r0) < 128 ? (Mpad - r0) : 128;
            const int width = Mpad - r0;
            const int nchunks = (width + 255) / 256;
            const int cw = round_up((width + nchunks - 1) / nchunks, 16);
            for (int c0 = r0; c0 < Mpad; c0 += cw) {
                const int n = (Mpad - c0) < cw ? (Mpad - c0) : cw;
                XJob j{};
                j.n_groups = 1;
                if (c0 == r0) {   // diagonal chunk: B rows start at the A rows, load the union once
                    j.ld_row[0] = r0;
                    j.ld_nrows[0] = na > n ? na : n;
                    j.ld_row[1] = 0;
                    j.ld_nrows[1] = 0;
                    j.g[0] = XMmaGroup{0, 0, n, 0, r0, c0, na <= 64 ? 64 : 128, r0, 0};
                } else {
                    j.ld_row[0] = r0;
                    j.ld_nrows[0] = na;
                    j.ld_row[1] = c0;
                    j.ld_nrows[1] = n;
                    j.g[0] = XMmaGroup{0, na, n, 0, r0, c0, na <= 64 ? 64 : 128, r0, 0};
                }
                j.tmem_cols = pow2_cols(2 * n);
                p->jobs.push_back(j);
            }
        }
    }
    int max_rows = 0, slack_rows = 0;
    for (const XJob &j : p->jobs) {
        const int rows = j.ld_nrows[0] + j.ld_nrows[1];
        max_rows = rows > max_rows ? rows : max_rows;
    }
    for (const XJob &j : p->jobs)      // an A operand always reads its instruction's M rows, loaded or not
        for (int g = 0; g < j.n_groups; ++g) {
            const int reach = j.g[g].a_row + (j.g[g].kind == 1 ? j.g[g].m / 2 : j.g[g].m);
            slack_rows = reach - max_rows > slack_rows ? reach - max_rows : slack_rows;
        }
    const size_t stage_bytes = (size_t)max_rows * 256;
    const size_t slack = (size_t)slack_rows * 256;
    // staged epilogue: the whole [n_bl][2][2] block of a channel, if that still leaves three load stages
    size_t out_bytes = ((size_t)p->n_bl * 32 + 127) / 128 * 128;
    const size_t rot_bytes = ((size_t)p->Mpad * sizeof(float2) + 511) / 512 * 512;    // two tables: a multiple of 1024 together
    p->x_rot_bytes = rot_bytes;
    const size_t fixed = 1024 /*alignment*/ + kBarrierBytes + 2 * rot_bytes + slack;
    p->x_staged = p->jobs.size() == 1 && fixed + out_bytes + 3 * stage_bytes <= (size_t)227 * 1024;
    if (!p->x_staged) out_bytes = 0;
    const size_t budget = 227 * 1024 - fixed - out_bytes;
    int stages = (int)(budget / stage_bytes);
    if (stages > 8) stages = 8;
    p->x_stages = stages;
    p->x_out_off = kBarrierBytes + 2 * rot_bytes + (size_t)stages * stage_bytes + slack;
    p->x_smem_bytes = fixed + (size_t)stages * stage_bytes + out_bytes;
}

cudaError_t launch_xsum_n(const cobalt_plan_s *p, cudaStream_t st, int nb, float2 *d_vis, size_t dump_stride, int splits);   // ingest.cu

cudaError_t launch_xstage_tc(const cobalt_plan_s *p, cudaStream_t st, const void *d_z, int nb, float2 *d_vis, size_t dump_stride,
                             const XCall &xc) {
    if (p->x_stages < 2) return cudaErrorInvalidConfiguration;
    XArgs a;
    a.z = static_cast<const unsigned char *>(d_z);
    a.vis = d_vis;
    a.jobs = p->d_jobs;
    a.phase = xc.phase;
    a.poff = xc.poff;
    a.b0 = xc.b0;
    a.S = p->S;
    a.inv_s2 = xc.inv_s2;
    a.rot_off = kBarrierBytes;
    a.rot_bytes = (uint32_t)p->x_rot_bytes;
    a.z_subband_bytes = p->z_subband_bytes;
    a.n_bl = p->n_bl;
    a.C = p->C;
    a.M = p->M;
    a.Mpad = p->Mpad;
    a.n_kt = p->n_kt;
    a.jobs_per_channel = (int)p->jobs.size();
    a.D = p->dumps;
    a.K = p->n_kt / p->dumps;
    a.nbC = nb * p->C;
    // too few (dump, subband, channel) problems to fill the SMs (config 2: 64 channels on 148 SMs): split each one's time
    // range over several jobs, into partial blocks that xsum_kernel adds up
    a.splits = 1;
    if (p->d_xpart) {
        // cost of s splits in k-tile times: waves x (k-tiles per job + ~3.5 for the prologue and the exposed epilogue)
        const long long probs = (long long)a.nbC * a.D * a.jobs_per_channel;
        double best = 1e30;
        for (int sp = 1; sp <= p->x_splits && sp <= a.K; ++sp) {
            const long long waves = (probs * sp + p->sm_count - 1) / p->sm_count;
            const double cost = (double)waves * ((double)((a.K + sp - 1) / sp) + 3.5);
            if (cost < best - 1e-9) {
                best = cost;
                a.splits = sp;
            }
        }
    }
    a.part = p->d_xpart;
    a.dump_stride = dump_stride;
    a.total_jobs = a.nbC * a.D * a.splits * a.jobs_per_channel;
    a.stages = p->x_stages;
    int max_rows = 0;
    for (const XJob &j : p->jobs) max_rows = (j.ld_nrows[0] + j.ld_nrows[1]) > max_rows ? (j.ld_nrows[0] + j.ld_nrows[1]) : max_rows;
    a.stage_bytes = max_rows * 256;
    a.out_off = (uint32_t)p->x_out_off;
    auto kern = p->x_staged ? xstage_tc_kernel<true> : xstage_tc_kernel<false>;   // d_vis is 16-byte aligned (cobalt_process)
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->x_smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = a.total_jobs < p->sm_count ? a.total_jobs : p->sm_count;
    kern<<<grid, kThreads, p->x_smem_bytes, st>>>(a);
    e = cudaGetLastError();
    if (e != cudaSuccess || a.splits == 1) return e;
    return launch_xsum_n(p, st, nb, d_vis, dump_stride, a.splits);
}

}  // namespace cobalt
