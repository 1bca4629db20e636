/*
 * cobalt_oracle.c -- float64 CPU ORACLE for the Cobalt correlator hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_1801_04834_b200/csrc/ and never includes anything from there.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, "P:Lnnn" = line nnn):
 *   P:L89  (sec 3.2)  "Data is converted from fixed to floating point"            -> oracle_unpack_*
 *   P:L360 (sec 7.5)  "channelizes subbands in a polyphase filter using FIR
 *                      filters and FFT kernels. We carry FIR filter history
 *                      samples across to the next block."                          -> oracle_fir, oracle_dft
 *   P:L360, P:L368    "fine delay compensation and bandpass correction"; phase
 *                      angles in double precision, rotate each sample               -> oracle_rotate
 *   P:L368            phase angles from the residual delay at block start and end,
 *                      interpolated linearly (reading A21) -> oracle_rotate_interp
 *   P:L360            "computes the correlations of all pairs of antenna fields
 *                      and averages in time"                                        -> oracle_correlate
 * The paper prints no formulas; every formula below is the reading fixed in
 * SURVEY.md sec 8(c) / DESIGN.md "Readings" (A1..A20) and is written out in the
 * order of that algorithm listing, in plain loops, in double precision: direct
 * FIR convolution, naive O(C^2) DFT, explicit per-baseline multiply-accumulate.
 * No blocking, no fusion, no FFT.  OpenMP only splits an outermost independent
 * index (stream, or channel) across cores; it never changes a summation order.
 *
 * Pins (tests/test_oracle_pins.py): P2 firwin, P3 DC, P4 tone closed form, P5
 * impulse, P6 numpy.fft special case, P7 Hermitian, P8 identical streams, P9
 * delay slope, P10 history carry, P11 brute force (oracle_channel_direct below
 * + a numpy brute force), P12 linearity, P13 statistics, P16 time-varying delay
 * (equal ends = static rotation; closed-form geometric series), P17-P21 (coarse shift,
 * phase offsets, dumps, valid-sample flags and counts, 4-bit unpack), P22-P25 (beamformer: coherent sum,
 * Stokes parameters, time integration, incoherent sum; tests/test_oracle_pins_bf.py).  No function here is
 * "parity unpinned".
 *
 * Layouts (all row-major, last index fastest):
 *   samples  [S][2][N][2]      int16 or int8, (re,im) interleaved, one subband
 *   hist     [S][2][(T-1)*C][2] double, the (T-1)*C samples preceding samples[..][0]
 *   g        [T*C]             double prototype filter
 *   F, z     [S][2][n_t][C][2] double (channel index j ascending in frequency)
 *   vis      [C][n_bl][2][2][2] double, n_bl = S(S+1)/2, baseline (i<=k) at k(k+1)/2+i,
 *                               then [pol of i][pol of k][re,im]
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

/* Number of threads the OpenMP loops will use (1 without OpenMP). */
int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ step 1 */
/* fixed -> floating point.  Two's complement value, no scaling, no
 * flagging of extreme values (reading A12). */
void oracle_unpack_i16(const int16_t *in, long long n, double *out) {
    for (long long i = 0; i < n; ++i) out[i] = (double)in[i];
}
void oracle_unpack_i8(const int8_t *in, long long n, double *out) {
    for (long long i = 0; i < n; ++i) out[i] = (double)in[i];
}

/* ------------------------------------------------------------------ step 2 */
/* Reading A1 (BASELINE.json configs: "16-tap FIR (Hann-windowed sinc)"):
 * g[n] = sinc((n-(L-1)/2)/C) * (0.5 - 0.5 cos(2 pi n/(L-1))), L = T*C, then
 * divided by sum(g) so that the DC gain is 1. */
void oracle_fir_prototype(int C, int T, double *g) {
    const int L = T * C;
    double sum = 0.0;
    for (int n = 0; n < L; ++n) {
        double u = ((double)n - 0.5 * (double)(L - 1)) / (double)C;
        double sinc = (u == 0.0) ? 1.0 : sin(ORACLE_PI * u) / (ORACLE_PI * u);
        double hann = 0.5 - 0.5 * cos(2.0 * ORACLE_PI * (double)n / (double)(L - 1));
        g[n] = sinc * hann;
        sum += g[n];
    }
    for (int n = 0; n < L; ++n) g[n] /= sum;
}

/* ------------------------------------------------------------------ step 3 */
/* P:L360 / P:L150 "many FIR filters feeding into an FFT".  One stream.
 * xh = history followed by the block: xh[(T-1)*C + n] = x[n].
 * y[t][ph] = sum_{k=0}^{T-1} g[(T-1-k)*C + ph] * x[(t-k)*C + ph]   (reading A2:
 * k = 0 is the newest block and takes the LAST C prototype taps). */
void oracle_fir(int C, int T, const double *g, const double *xh /*[(T-1)*C + n_t*C][2]*/,
                long long n_t, double *y /*[n_t][C][2]*/) {
    const long long off = (long long)(T - 1) * C;
    for (long long t = 0; t < n_t; ++t) {
        for (int ph = 0; ph < C; ++ph) {
            double re = 0.0, im = 0.0;
            for (int k = 0; k < T; ++k) {
                double w = g[(T - 1 - k) * C + ph];
                long long idx = off + (t - k) * C + ph;
                re += w * xh[2 * idx];
                im += w * xh[2 * idx + 1];
            }
            y[2 * (t * C + ph)] = re;
            y[2 * (t * C + ph) + 1] = im;
        }
    }
}

/* ------------------------------------------------------------- steps 4 + 5 */
/* P:L340 (the paper calls cuFFT): forward, negative exponent, unnormalised
 * (reading A4), written as the naive O(C^2) sum.
 * D[t][c] = sum_ph y[t][ph] exp(-2 pi i ((ph*c) mod C)/C);
 * F[t][j] = D[t][(j + C/2) mod C]   (reading A5: ascending frequency). */
void oracle_dft(int C, const double *y /*[n_t][C][2]*/, long long n_t, double *F /*[n_t][C][2]*/) {
    double *cs = (double *)malloc(sizeof(double) * 2 * (size_t)C);
    for (int m = 0; m < C; ++m) {
        cs[2 * m] = cos(-2.0 * ORACLE_PI * (double)m / (double)C);
        cs[2 * m + 1] = sin(-2.0 * ORACLE_PI * (double)m / (double)C);
    }
    for (long long t = 0; t < n_t; ++t) {
        for (int j = 0; j < C; ++j) {
            int c = (j + C / 2) % C;
            double re = 0.0, im = 0.0;
            for (int ph = 0; ph < C; ++ph) {
                int m = (int)(((long long)ph * c) % C);
                double yr = y[2 * (t * C + ph)], yi = y[2 * (t * C + ph) + 1];
                re += yr * cs[2 * m] - yi * cs[2 * m + 1];
                im += yr * cs[2 * m + 1] + yi * cs[2 * m];
            }
            F[2 * (t * C + j)] = re;
            F[2 * (t * C + j) + 1] = im;
        }
    }
    free(cs);
}

/* ------------------------------------------------------------- steps 6 + 7 */
/* Reading A6: f[j] = f_sb + (j - C/2) f_s/C.  P:L368 + BASELINE.json north_star:
 * z = F * b[j] * exp(-2 pi i frac(f[j] tau)), everything in double here. */
double oracle_channel_frequency(int C, double f_sb, double f_s, int j) {
    return f_sb + ((double)j - 0.5 * (double)C) * f_s / (double)C;
}
void oracle_rotate(int C, double f_sb, double f_s, double tau, const double *bandpass /*[C]*/,
                   long long n_t, double *F /*[n_t][C][2] in/out*/) {
    for (int j = 0; j < C; ++j) {
        double cyc = oracle_channel_frequency(C, f_sb, f_s, j) * tau;
        double frac = cyc - floor(cyc);
        double wr = bandpass[j] * cos(-2.0 * ORACLE_PI * frac);
        double wi = bandpass[j] * sin(-2.0 * ORACLE_PI * frac);
        for (long long t = 0; t < n_t; ++t) {
            double a = F[2 * (t * C + j)], b = F[2 * (t * C + j) + 1];
            F[2 * (t * C + j)] = a * wr - b * wi;
            F[2 * (t * C + j) + 1] = a * wi + b * wr;
        }
    }
}

/* "the phase angles [are computed] from the residual delay at the start and
 * the end of the block ... in double precision [and] interpolated linearly over the block".  Reading A21
 * (DESIGN.md): spectrum t of an n_t-spectrum block is rotated with the delay
 *   tau(t) = tau_b + (tau_e - tau_b) t / n_t,          t = 0 .. n_t - 1,
 * i.e. z[t][j] = F[t][j] b[j] exp(-2 pi i frac(f[j] tau(t))); tau_e = tau_b is oracle_rotate. */
void oracle_rotate_interp(int C, double f_sb, double f_s, double tau_b, double tau_e, const double *bandpass /*[C]*/,
                          long long n_t, double *F /*[n_t][C][2] in/out*/) {
    for (int j = 0; j < C; ++j) {
        const double f = oracle_channel_frequency(C, f_sb, f_s, j);
        for (long long t = 0; t < n_t; ++t) {
            double tau = tau_b + (tau_e - tau_b) * ((double)t / (double)n_t);
            double cyc = f * tau;
            double frac = cyc - floor(cyc);
            double wr = bandpass[j] * cos(-2.0 * ORACLE_PI * frac);
            double wi = bandpass[j] * sin(-2.0 * ORACLE_PI * frac);
            double a = F[2 * (t * C + j)], b = F[2 * (t * C + j) + 1];
            F[2 * (t * C + j)] = a * wr - b * wi;
            F[2 * (t * C + j) + 1] = a * wi + b * wr;
        }
    }
}

/* ------------------------------------------------------------------ step 8 */
/* P:L360.  V[j][bl(i,k)][p][q] = sum_t z[i][p][t][j] conj(z[k][q][t][j]), i <= k
 * (readings A9, A10: plain sum, no division, autos keep all four products). */
void oracle_correlate(int S, int C, long long n_t, const double *z /*[S][2][n_t][C][2]*/,
                      double *vis /*[C][n_bl][2][2][2]*/) {
    const long long n_bl = (long long)S * (S + 1) / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < C; ++j) {
        for (int k = 0; k < S; ++k) {
            for (int i = 0; i <= k; ++i) {
                long long bl = (long long)k * (k + 1) / 2 + i;
                for (int p = 0; p < 2; ++p) {
                    for (int q = 0; q < 2; ++q) {
                        const double *zi = z + 2 * ((((long long)i * 2 + p) * n_t) * C);
                        const double *zk = z + 2 * ((((long long)k * 2 + q) * n_t) * C);
                        double re = 0.0, im = 0.0;
                        for (long long t = 0; t < n_t; ++t) {
                            double ar = zi[2 * (t * C + j)], ai = zi[2 * (t * C + j) + 1];
                            double br = zk[2 * (t * C + j)], bi = zk[2 * (t * C + j) + 1];
                            re += ar * br + ai * bi;
                            im += ai * br - ar * bi;
                        }
                        double *o = vis + 2 * ((((long long)j * n_bl + bl) * 2 + p) * 2 + q);
                        o[0] = re;
                        o[1] = im;
                    }
                }
            }
        }
    }
}

/* --------------------------------------------------- the F-stage, per stream */
/* Steps 1-7 and 9 for every stream of one subband, from double-precision
 * samples (x may come from oracle_unpack_* or, for pins that must avoid
 * quantisation, directly from the test).  hist is read, then replaced by the
 * last (T-1)*C consumed samples (step 9, "carry FIR filter history").
 * delays may be NULL (no rotation, no bandpass: z = F). */
int oracle_fstage_interp_f64(int S, int C, int T, long long N, const double *x /*[S][2][N][2]*/,
                             const double *g /*[T*C]*/, double *hist /*[S][2][(T-1)*C][2]*/,
                             const double *delays /*[S] or NULL*/, const double *delays_end /*[S] or NULL*/,
                             const double *bandpass /*[C]*/, double f_sb, double f_s, double *z /*[S][2][n_t][C][2]*/);
int oracle_fstage_f64(int S, int C, int T, long long N, const double *x /*[S][2][N][2]*/,
                      const double *g /*[T*C]*/, double *hist /*[S][2][(T-1)*C][2]*/,
                      const double *delays /*[S] or NULL*/, const double *bandpass /*[C]*/,
                      double f_sb, double f_s, double *z /*[S][2][n_t][C][2]*/) {
    return oracle_fstage_interp_f64(S, C, T, N, x, g, hist, delays, NULL, bandpass, f_sb, f_s, z);
}
/* delays_end != NULL: time-varying delay of reading A21 (oracle_rotate_interp). */
int oracle_fstage_interp_f64(int S, int C, int T, long long N, const double *x /*[S][2][N][2]*/,
                             const double *g /*[T*C]*/, double *hist /*[S][2][(T-1)*C][2]*/,
                             const double *delays /*[S] or NULL*/, const double *delays_end /*[S] or NULL*/,
                             const double *bandpass /*[C]*/, double f_sb, double f_s, double *z /*[S][2][n_t][C][2]*/) {
    const long long n_t = N / C;          /* reading A11: trailing N - n_t*C samples unused */
    const long long nu = n_t * C;
    const long long nh = (long long)(T - 1) * C;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int sp = 0; sp < 2 * S; ++sp) {
        double *xh = (double *)malloc(sizeof(double) * 2 * (size_t)(nh + nu));
        double *y = (double *)malloc(sizeof(double) * 2 * (size_t)(nu > 0 ? nu : 1));
        if (!xh || !y) {
#pragma omp atomic write
            fail = 1;
            free(xh);
            free(y);
            continue;
        }
        double *h = hist + 2 * (long long)sp * nh;
        memcpy(xh, h, sizeof(double) * 2 * (size_t)nh);
        memcpy(xh + 2 * nh, x + 2 * (long long)sp * N, sizeof(double) * 2 * (size_t)nu);
        double *zz = z + 2 * (long long)sp * nu;
        oracle_fir(C, T, g, xh, n_t, y);
        oracle_dft(C, y, n_t, zz);
        if (delays && delays_end) oracle_rotate_interp(C, f_sb, f_s, delays[sp / 2], delays_end[sp / 2], bandpass, n_t, zz);
        else if (delays) oracle_rotate(C, f_sb, f_s, delays[sp / 2], bandpass, n_t, zz);
        memcpy(h, xh + 2 * nu, sizeof(double) * 2 * (size_t)nh);   /* last nh of hist||block */
        free(xh);
        free(y);
    }
    return fail;
}

/* ---------------------------------------------------------- whole subband */
/* One subband through steps 1-9 from integer samples.  bits = 16 or 8.
 * z_out may be NULL; otherwise receives z [S][2][n_t][C][2].
 * Returns 0, or 1 on allocation failure / bad bits. */
int oracle_process_subband_interp(int S, int C, int T, long long N, int bits, const void *samples,
                                  double *hist, const double *delays, const double *delays_end, const double *bandpass,
                                  double f_sb, double f_s, double *vis, double *z_out);
int oracle_process_subband(int S, int C, int T, long long N, int bits, const void *samples,
                           double *hist, const double *delays, const double *bandpass,
                           double f_sb, double f_s, double *vis, double *z_out) {
    return oracle_process_subband_interp(S, C, T, N, bits, samples, hist, delays, NULL, bandpass, f_sb, f_s, vis, z_out);
}
/* delays_end != NULL: time-varying delay of reading A21. */
int oracle_process_subband_interp(int S, int C, int T, long long N, int bits, const void *samples,
                                  double *hist, const double *delays, const double *delays_end, const double *bandpass,
                                  double f_sb, double f_s, double *vis, double *z_out) {
    const long long n_t = N / C;
    const long long n_in = (long long)S * 2 * N * 2;
    if (bits != 16 && bits != 8) return 1;
    double *x = (double *)malloc(sizeof(double) * (size_t)n_in);
    double *g = (double *)malloc(sizeof(double) * (size_t)T * C);
    double *z = z_out ? z_out : (double *)malloc(sizeof(double) * 2 * (size_t)S * 2 * n_t * C);
    if (!x || !g || !z) {
        free(x);
        free(g);
        if (!z_out) free(z);
        return 1;
    }
    if (bits == 16) oracle_unpack_i16((const int16_t *)samples, n_in, x);
    else oracle_unpack_i8((const int8_t *)samples, n_in, x);
    oracle_fir_prototype(C, T, g);
    int rc = oracle_fstage_interp_f64(S, C, T, N, x, g, hist, delays, delays_end, bandpass, f_sb, f_s, z);
    if (!rc) oracle_correlate(S, C, n_t, z, vis);
    free(x);
    free(g);
    if (!z_out) free(z);
    return rc;
}


/* =====================================================================================================
 * SURVEY.md sec 8(f) rows 1-3 (the rows marked "next"): clock / phase offsets, sub-second dumps, valid-sample
 * weights, 4-bit samples.  Each is the plain definition of the reading named beside it.
 * ===================================================================================================== */

/* Reading A27 ("4-bit ... mode"): one byte per complex sample, re in the low nibble, im in the high
 * nibble, both 4-bit two's complement (-8 .. 7), no scaling. */
void oracle_unpack_i4(const uint8_t *in, long long n_samples, double *out /*[n_samples][2]*/) {
    for (long long i = 0; i < n_samples; ++i) {
        int lo = in[i] & 15, hi = (in[i] >> 4) & 15;
        out[2 * i] = (double)(lo >= 8 ? lo - 16 : lo);
        out[2 * i + 1] = (double)(hi >= 8 ? hi - 16 : hi);
    }
}

/* Reading A22 ("bandpass and clock corrections"): a constant phase per (station, polarisation),
 * phase0 in radians, with the sign sense of the delay term:  z <- z exp(-i phase0[a][p]). */
void oracle_phase_offsets(int S, int C, long long n_t, const double *phase0 /*[S][2]*/, double *z /*[S][2][n_t][C][2]*/) {
    for (int sp = 0; sp < 2 * S; ++sp) {
        const double wr = cos(phase0[sp]), wi = -sin(phase0[sp]);
        double *zz = z + 2 * (long long)sp * n_t * C;
        for (long long i = 0; i < n_t * C; ++i) {
            double a = zz[2 * i], b = zz[2 * i + 1];
            zz[2 * i] = a * wr - b * wi;
            zz[2 * i + 1] = a * wi + b * wr;
        }
    }
}

/* Reading A24 (P:L298 lost data is "encoded in the metadata"; P:L282-288 block granularity): valid[a][v] = 0 marks
 * the spectra [v tile, (v+1) tile) of station a (both polarisations) as lost.  Their channelised samples count as
 * zero in the correlation (the FIR still runs over whatever the input buffer holds: masking happens after it). */
void oracle_flag_tiles(int S, int C, long long n_t, int tile, const unsigned char *valid /*[S][ceil(n_t/tile)]*/,
                       double *z /*[S][2][n_t][C][2]*/) {
    const long long n_vt = (n_t + tile - 1) / tile;
    for (int a = 0; a < S; ++a)
        for (int p = 0; p < 2; ++p)
            for (long long t = 0; t < n_t; ++t)
                if (!valid[a * n_vt + t / tile]) {
                    double *zz = z + 2 * ((((long long)a * 2 + p) * n_t + t) * C);
                    for (int j = 0; j < 2 * C; ++j) zz[j] = 0.0;
                }
}

/* ... and the weight that goes with a visibility: the number of spectra of dump d in which BOTH stations of the
 * baseline are valid.  counts [D][n_bl].  Dumps as in oracle_correlate_dumps. */
void oracle_valid_counts(int S, long long n_t, int D, int tile, const unsigned char *valid, long long *counts) {
    const long long n_vt = (n_t + tile - 1) / tile;
    const long long n_bl = (long long)S * (S + 1) / 2;
    const long long dump_len = ((n_vt / D) * tile);
    for (int d = 0; d < D; ++d)
        for (int k = 0; k < S; ++k)
            for (int i = 0; i <= k; ++i) {
                long long c = 0;
                for (long long t = d * dump_len; t < n_t && t < (d + 1) * dump_len; ++t)
                    if (valid[i * n_vt + t / tile] && valid[k * n_vt + t / tile]) ++c;
                counts[d * n_bl + (long long)k * (k + 1) / 2 + i] = c;
            }
}

/* Reading A23 (P:L103 integration time down to a fraction of a second): D dumps per block.  Dump
 * boundaries fall on multiples of `tile` spectra (the correlator's time tile, 64): with n_vt = ceil(n_t / tile)
 * tiles, D must divide n_vt and dump d integrates the spectra [d L, min((d+1) L, n_t)), L = (n_vt / D) tile; the
 * last dump is shorter when n_t is not a multiple of the tile.  vis [D][C][n_bl][2][2][2]; D = 1 is oracle_correlate.
 * Returns 1 when D does not divide n_vt. */
int oracle_correlate_dumps(int S, int C, long long n_t, int D, int tile, const double *z /*[S][2][n_t][C][2]*/,
                           double *vis /*[D][C][n_bl][2][2][2]*/) {
    const long long n_vt = (n_t + tile - 1) / tile;
    const long long n_bl = (long long)S * (S + 1) / 2;
    if (D < 1 || n_vt % D) return 1;
    const long long L = (n_vt / D) * tile;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < C; ++j)
        for (int d = 0; d < D; ++d)
            for (int k = 0; k < S; ++k)
                for (int i = 0; i <= k; ++i)
                    for (int p = 0; p < 2; ++p)
                        for (int q = 0; q < 2; ++q) {
                            const double *zi = z + 2 * ((((long long)i * 2 + p) * n_t) * C);
                            const double *zk = z + 2 * ((((long long)k * 2 + q) * n_t) * C);
                            double re = 0.0, im = 0.0;
                            for (long long t = d * L; t < n_t && t < (d + 1) * L; ++t) {
                                double ar = zi[2 * (t * C + j)], ai = zi[2 * (t * C + j) + 1];
                                double br = zk[2 * (t * C + j)], bi = zk[2 * (t * C + j) + 1];
                                re += ar * br + ai * bi;
                                im += ai * br - ar * bi;
                            }
                            long long bl = (long long)k * (k + 1) / 2 + i;
                            double *o = vis + 2 * (((((long long)d * C + j) * n_bl + bl) * 2 + p) * 2 + q);
                            o[0] = re;
                            o[1] = im;
                        }
    return 0;
}

/* =====================================================================================================
 * the beamformer pipeline, at the channel resolution of the
 * plan ("Cobalt performs delay compensation, bandpass correction and beamforming at 256 channels per subband").
 * Input of every function below is z, the delay-compensated, bandpass-corrected channelised data of steps 1-7
 * (a reading, A28: the paper's beamformer "cannot share initial steps with the correlator", and
 * channelises on its own).  Readings A28-A31 of DESIGN.md.  The final
 * transformation "to the requested output resolution" (inverse FFT / second FFT) is not part of this row.
 * ===================================================================================================== */

/* Reading A28 ("Coherent beamforming first adjusts the beam direction with a phase shift and sums over
 * antenna fields"; "The beamforming kernel operates in a similar way [to delay compensation] to form beams
 * with an offset from the center": the phase angle of (beam, station, channel) in double precision):
 *   Y[b][p][j][t] = sum_a exp(-2 pi i frac(f[j] taub[b][a])) z[a][p][t][j]
 * taub[b][a] = the delay of station a for beam b relative to the phase centre, seconds, with the sign sense of the
 * station delay of step 7 (a positive value delays station a's signal); f[j] = the channel's sky frequency (A6).
 * No normalisation by the number of stations (like A10: a scalar the caller can apply). */
void oracle_beamform_coherent(int S, int C, long long n_t, int n_beams, const double *beam_delays /*[n_beams][S]*/,
                              double f_sb, double f_s, const double *z /*[S][2][n_t][C][2]*/,
                              double *y /*[n_beams][2][C][n_t][2]*/) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < n_beams; ++b)
        for (int p = 0; p < 2; ++p)
            for (int j = 0; j < C; ++j) {
                const double f = oracle_channel_frequency(C, f_sb, f_s, j);
                for (long long t = 0; t < n_t; ++t) {
                    double re = 0.0, im = 0.0;
                    for (int a = 0; a < S; ++a) {
                        double cyc = f * beam_delays[(long long)b * S + a];
                        double frac = cyc - floor(cyc);
                        double wr = cos(-2.0 * ORACLE_PI * frac), wi = sin(-2.0 * ORACLE_PI * frac);
                        const double *zz = z + 2 * ((((long long)a * 2 + p) * n_t + t) * C + j);
                        re += wr * zz[0] - wi * zz[1];
                        im += wr * zz[1] + wi * zz[0];
                    }
                    double *o = y + 2 * ((((long long)b * 2 + p) * C + j) * n_t + t);
                    o[0] = re;
                    o[1] = im;
                }
            }
}

/* Reading A29 ("Stokes I only or Stokes IQUV"): the Stokes parameters of one dual-polarisation complex
 * sample (X, Y), linear feeds:
 *   I = |X|^2 + |Y|^2,  Q = |X|^2 - |Y|^2,  U = 2 Re(X conj(Y)),  V = 2 Im(X conj(Y)).
 * n_stokes = 1 (I only) or 4.  out [n_stokes][n]. */
void oracle_stokes(long long n, const double *x /*[n][2]*/, const double *y /*[n][2]*/, int n_stokes, double *out) {
    for (long long i = 0; i < n; ++i) {
        double xr = x[2 * i], xi = x[2 * i + 1], yr = y[2 * i], yi = y[2 * i + 1];
        double px = xr * xr + xi * xi, py = yr * yr + yi * yi;
        out[i] = px + py;
        if (n_stokes == 4) {
            out[n + i] = px - py;
            out[2 * n + i] = 2.0 * (xr * yr + xi * yi);
            out[3 * n + i] = 2.0 * (xi * yr - xr * yi);
        }
    }
}

/* Reading A30 ("Time resolution can be traded against frequency resolution"; "complex voltages cannot
 * be time averaged", so Stokes only): output sample u of a row is the plain sum of the t_int input samples
 * [u t_int, (u+1) t_int); n_out = floor(n_t / t_int), trailing samples are not consumed (as in A11).
 * in [rows][n_t] -> out [rows][n_out]. */
void oracle_integrate(long long rows, long long n_t, int t_int, const double *in, double *out) {
    const long long n_out = n_t / t_int;
    for (long long r = 0; r < rows; ++r)
        for (long long u = 0; u < n_out; ++u) {
            double s = 0.0;
            for (int k = 0; k < t_int; ++k) s += in[r * n_t + u * t_int + k];
            out[r * n_out + u] = s;
        }
}

/* P:L362 "coherent beamforming ... sums over antenna fields, then optionally computes Stokes parameters":
 * A28 -> A29 per (beam, channel, spectrum) -> A30.  out [n_beams][n_stokes][C][n_out].  Returns 1 on allocation failure. */
int oracle_coherent_stokes(int S, int C, long long n_t, int n_beams, const double *beam_delays, double f_sb, double f_s,
                           const double *z, int n_stokes, int t_int, double *out) {
    const long long n_out = n_t / t_int, n = (long long)C * n_t;
    double *y = (double *)malloc(sizeof(double) * 2 * (size_t)n_beams * 2 * (size_t)n);
    double *st = (double *)malloc(sizeof(double) * (size_t)n_stokes * (size_t)n);
    if (!y || !st) {
        free(y);
        free(st);
        return 1;
    }
    oracle_beamform_coherent(S, C, n_t, n_beams, beam_delays, f_sb, f_s, z, y);
    for (int b = 0; b < n_beams; ++b) {
        oracle_stokes(n, y + 2 * ((long long)b * 2) * n, y + 2 * ((long long)b * 2 + 1) * n, n_stokes, st);   /* [k][C][n_t] */
        oracle_integrate((long long)n_stokes * C, n_t, t_int, st, out + (long long)b * n_stokes * C * n_out);
    }
    free(y);
    free(st);
    return 0;
}

/* Reading A31 ("incoherent beamforming first computes Stokes parameters and then sums over antenna fields"):
 *   S_k[j][t] = sum_a stokes_k(z[a][X][t][j], z[a][Y][t][j]),  then A30.  out [n_stokes][C][n_out]. */
int oracle_incoherent_stokes(int S, int C, long long n_t, const double *z /*[S][2][n_t][C][2]*/, int n_stokes, int t_int,
                             double *out) {
    const long long n_out = n_t / t_int, n = (long long)C * n_t;
    double *xs = (double *)malloc(sizeof(double) * 2 * (size_t)n);     /* one station, [C][n_t] per polarisation */
    double *ys = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    double *st = (double *)malloc(sizeof(double) * (size_t)n_stokes * (size_t)n);
    double *acc = (double *)calloc((size_t)n_stokes * (size_t)n, sizeof(double));
    if (!xs || !ys || !st || !acc) {
        free(xs);
        free(ys);
        free(st);
        free(acc);
        return 1;
    }
    for (int a = 0; a < S; ++a) {
        for (int j = 0; j < C; ++j)
            for (long long t = 0; t < n_t; ++t) {
                const double *zx = z + 2 * ((((long long)a * 2 + 0) * n_t + t) * C + j);
                const double *zy = z + 2 * ((((long long)a * 2 + 1) * n_t + t) * C + j);
                xs[2 * (j * n_t + t)] = zx[0];
                xs[2 * (j * n_t + t) + 1] = zx[1];
                ys[2 * (j * n_t + t)] = zy[0];
                ys[2 * (j * n_t + t) + 1] = zy[1];
            }
        oracle_stokes(n, xs, ys, n_stokes, st);
        for (long long i = 0; i < (long long)n_stokes * n; ++i) acc[i] += st[i];
    }
    oracle_integrate((long long)n_stokes * C, n_t, t_int, acc, out);
    free(xs);
    free(ys);
    free(st);
    free(acc);
    return 0;
}

/* ------------------------------------------------- pin P11: single-sum form */
/* An independent route to one channel, with a different loop structure from
 * steps 3-5: window the last T*C samples with g in natural order and take one
 * DFT bin of the whole window,
 *   D[t][c] = sum_{n=0}^{TC-1} g[n] x[(t-(T-1))C + n] exp(-2 pi i c n / C),
 * with the exponential evaluated per term by cos/sin of the reduced argument.
 * Produces z for channel j (ascending-frequency index) of every input, then the
 * visibilities of that channel by direct double loops.  Used for sampled checks
 * at full size (one (subband, channel) at a time) and as the brute-force pin.
 * x is double [S][2][N][2]; hist as above (not updated). */
int oracle_channel_direct(int S, int C, int T, long long N, const double *x, const double *hist,
                          const double *g, const double *delays, const double *bandpass,
                          double f_sb, double f_s, int j,
                          double *zc /*[2S][n_t][2]*/, double *vis_c /*[n_bl][2][2][2]*/) {
    const long long n_t = N / C;
    const long long nh = (long long)(T - 1) * C;
    const int L = T * C;
    const int c = (j + C / 2) % C;
    double *er = (double *)malloc(sizeof(double) * (size_t)L);
    double *ei = (double *)malloc(sizeof(double) * (size_t)L);
    if (!er || !ei) {
        free(er);
        free(ei);
        return 1;
    }
    for (int n = 0; n < L; ++n) {
        long long m = ((long long)c * n) % C;            /* reduce before the trig call */
        er[n] = g[n] * cos(2.0 * ORACLE_PI * (double)m / (double)C);
        ei[n] = -g[n] * sin(2.0 * ORACLE_PI * (double)m / (double)C);
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int sp = 0; sp < 2 * S; ++sp) {
        const double *xs = x + 2 * (long long)sp * N;
        const double *hs = hist + 2 * (long long)sp * nh;
        double wr = 1.0, wi = 0.0;
        if (delays) {
            double cyc = (f_sb + ((double)j - 0.5 * (double)C) * f_s / (double)C) * delays[sp / 2];
            double frac = cyc - floor(cyc);
            wr = bandpass[j] * cos(2.0 * ORACLE_PI * frac);
            wi = -bandpass[j] * sin(2.0 * ORACLE_PI * frac);
        }
        for (long long t = 0; t < n_t; ++t) {
            double re = 0.0, im = 0.0;
            long long base = (t - (T - 1)) * C;          /* index of window start in the block */
            for (int n = 0; n < L; ++n) {
                long long idx = base + n;
                double xr, xi;
                if (idx < 0) {
                    xr = hs[2 * (nh + idx)];
                    xi = hs[2 * (nh + idx) + 1];
                } else {
                    xr = xs[2 * idx];
                    xi = xs[2 * idx + 1];
                }
                re += xr * er[n] - xi * ei[n];
                im += xr * ei[n] + xi * er[n];
            }
            zc[2 * (sp * n_t + t)] = re * wr - im * wi;
            zc[2 * (sp * n_t + t) + 1] = re * wi + im * wr;
        }
    }
    if (vis_c) {
        for (int k = 0; k < S; ++k)
            for (int i = 0; i <= k; ++i)
                for (int p = 0; p < 2; ++p)
                    for (int q = 0; q < 2; ++q) {
                        const double *a = zc + 2 * ((long long)(2 * i + p) * n_t);
                        const double *b = zc + 2 * ((long long)(2 * k + q) * n_t);
                        double re = 0.0, im = 0.0;
                        for (long long t = 0; t < n_t; ++t) {
                            re += a[2 * t] * b[2 * t] + a[2 * t + 1] * b[2 * t + 1];
                            im += a[2 * t + 1] * b[2 * t] - a[2 * t] * b[2 * t + 1];
                        }
                        long long bl = (long long)k * (k + 1) / 2 + i;
                        double *o = vis_c + 2 * ((bl * 2 + p) * 2 + q);
                        o[0] = re;
                        o[1] = im;
                    }
    }
    free(er);
    free(ei);
    return 0;
}
