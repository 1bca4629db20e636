"""Pins for the float64 oracle (pins P2..P13).

Nothing here re-types an oracle formula or re-calls its routine as the expectation:
each expectation is a closed form, an invariant, a scipy/numpy library routine on a
special case, or an independent numpy brute force with a different loop structure.
CPU only (`-m "not gpu"`).
"""
import numpy as np
import pytest
import scipy.signal

T = 16
F_S = 195312.5


def crandn(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ------------------------------------------------------------------ P2: filter
@pytest.mark.parametrize("C", [16, 64, 256])
def test_p2_prototype_is_firwin_hann(oracle, C):
    g = oracle.fir_prototype(C, T)
    ref = scipy.signal.firwin(T * C, 1.0 / C, window="hann")   # library routine, reading A1
    assert g.shape == (T * C,)
    np.testing.assert_allclose(g, ref, rtol=0, atol=1e-15)
    np.testing.assert_allclose(g, g[::-1], rtol=0, atol=1e-16)  # symmetric (to rounding)
    assert abs(g.sum() - 1.0) < 1e-14                           # unit DC gain
    # constants quoted in SURVEY.md sec 8(c) P2
    assert abs(np.sum(g * g) * C - 0.9486) < 2e-4
    assert abs(np.sum(np.abs(g)) - 1.680) < 2e-3


# ------------------------------------------------------------------ P3: DC
@pytest.mark.parametrize("C", [16, 64])
def test_p3_dc_goes_to_centre_channel(oracle, C):
    A = 3.0 - 2.0j
    n_t = 40
    x = np.full((1, 2, n_t * C), A, dtype=np.complex128)
    z = oracle.fstage(x, C)[0, 0]                               # [n_t][C]
    steady = z[T - 1:]
    np.testing.assert_allclose(steady[:, C // 2], A, rtol=0, atol=1e-12)
    others = np.delete(steady, C // 2, axis=1)
    assert np.max(np.abs(others)) <= 9.6e-5 * abs(A)            # max_k |G(k/C)| = 9.5e-5


# ------------------------------------------------------------------ P4: tone closed form
@pytest.mark.parametrize("C,nu_ch", [(16, 5 - 8), (16, 2.37), (64, -17.25), (256, 100.5)])
def test_p4_tone_closed_form(oracle, C, nu_ch):
    """x[n] = A exp(2 pi i nu n), nu = nu_ch/C cycles/sample (nu_ch = offset from the subband
    centre in channel widths).  For t >= T-1:
    D[t][c] = A exp(2 pi i nu (t-(T-1)) C) sum_n g[n] exp(2 pi i (nu - c/C) n), F[t][j] = D[t][(j+C/2)%C]."""
    A = 200.0 * np.exp(0.3j)
    nu = nu_ch / C
    n_t = 24
    n = np.arange(n_t * C)
    x = (A * np.exp(2j * np.pi * nu * n)).reshape(1, 1, -1).repeat(2, axis=1)
    z = oracle.fstage(x, C)[0, 1]
    g = scipy.signal.firwin(T * C, 1.0 / C, window="hann")      # independent of the oracle's g
    nn = np.arange(T * C)
    c = (np.arange(C) + C // 2) % C
    G = np.array([np.sum(g * np.exp(2j * np.pi * (nu - cc / C) * nn)) for cc in c])
    for t in (T - 1, T, n_t - 1):
        expect = A * np.exp(2j * np.pi * nu * (t - (T - 1)) * C) * G
        np.testing.assert_allclose(z[t], expect, rtol=0, atol=1e-10 * abs(A))
    # "all power in the expected channel, leakage bounded by the FIR response"
    if float(nu_ch).is_integer():
        j0 = int(nu_ch) + C // 2
        p = np.abs(z[T]) ** 2
        assert np.argmax(p) == j0
        assert abs(np.sqrt(p[j0]) - abs(A)) < 1e-9 * abs(A)
        assert np.sqrt(np.delete(p, j0).max()) < 1e-4 * abs(A)
    if nu_ch == 100.5:   # half-way between channels: |G| = 0.5 in both neighbours
        j0 = int(np.floor(nu_ch)) + C // 2
        np.testing.assert_allclose(np.abs(z[T, j0:j0 + 2]) / abs(A), [0.5, 0.5], atol=2e-3)


# ------------------------------------------------------------------ P5: impulse
def test_p5_impulse_response_is_prototype_branch(oracle):
    C, n_t, t0, ph0 = 16, 40, 7, 11
    x = np.zeros(n_t * C + (T - 1) * C, dtype=np.complex128)   # history (zeros) then block
    x[(T - 1) * C + t0 * C + ph0] = 1.0 + 0.0j
    g = oracle.fir_prototype(C, T)
    y = oracle.fir(x, g, C)
    gref = scipy.signal.firwin(T * C, 1.0 / C, window="hann")
    expect = np.zeros((n_t, C), dtype=np.complex128)
    for d in range(T):
        expect[t0 + d, ph0] = gref[(T - 1 - d) * C + ph0]       # reading A2 (newest block <- last taps)
    np.testing.assert_allclose(y, expect, rtol=0, atol=1e-15)
    assert np.count_nonzero(y) == T


# ------------------------------------------------------------------ P6: numpy.fft special case
@pytest.mark.parametrize("C", [16, 64, 256])
def test_p6_rectangular_prototype_equals_numpy_fft(oracle, C):
    rng = np.random.default_rng(6)
    n_t = 5
    x = crandn(rng, 2, 2, n_t * C)
    g = np.zeros(T * C)
    g[(T - 1) * C:] = 1.0            # one tap on the newest block: y[t][ph] = x[tC+ph]
    z = oracle.fstage(x, C, g=g)
    ref = np.fft.fftshift(np.fft.fft(x.reshape(2, 2, n_t, C), axis=-1), axes=-1)
    np.testing.assert_allclose(z, ref, rtol=0, atol=1e-11)


def test_dft_matches_numpy_fft_on_random_rows(oracle):
    rng = np.random.default_rng(61)
    for C in (16, 64, 256):
        y = crandn(rng, 3, C)
        np.testing.assert_allclose(oracle.dft(y), np.fft.fftshift(np.fft.fft(y, axis=1), axes=1), atol=1e-11)


# ------------------------------------------------------------------ P7: Hermitian / autos
def full_matrix(oracle, vis, S):
    """[n_bl][2][2] triangular store -> [S,2,S,2] using only stored entries (i <= k)."""
    M = np.full((S, 2, S, 2), np.nan + 0j)
    for k in range(S):
        for i in range(k + 1):
            M[i, :, k, :] = vis[oracle.baseline_index(i, k)]
    return M


def test_p7_hermitian_and_autos(oracle):
    rng = np.random.default_rng(7)
    S, C, n_t = 5, 16, 33
    z = crandn(rng, S, 2, n_t, C)
    vis = oracle.correlate(z)                                   # [C][n_bl][2][2]
    assert vis.shape == (C, S * (S + 1) // 2, 2, 2)
    # definition, by numpy einsum over the FULL S x S matrix (library contraction)
    full = np.einsum("iptj,kqtj->jipkq", z, z.conj())
    for j in (0, 7, 15):
        M = full_matrix(oracle, vis[j], S)
        for k in range(S):
            for i in range(k + 1):
                np.testing.assert_allclose(M[i, :, k, :], full[j, i, :, k, :], rtol=1e-12, atol=1e-12)
                # V_ki = conj(V_ik)^T from the full definition
                np.testing.assert_allclose(full[j, k, :, i, :], M[i, :, k, :].conj().T, rtol=1e-12, atol=1e-12)
            a = M[k, :, k, :]
            assert abs(a[0, 0].imag) < 1e-12 and abs(a[1, 1].imag) < 1e-12
            assert a[0, 0].real >= 0 and a[1, 1].real >= 0
            np.testing.assert_allclose(a[1, 0], np.conj(a[0, 1]), rtol=1e-13)


def test_baseline_order_counts(oracle):
    for S, n in ((4, 10), (48, 1176), (77, 3003), (288, 41616)):     # BASELINE.json configs
        assert oracle.n_baselines(S) == n
    seen = sorted(oracle.baseline_index(i, k) for k in range(6) for i in range(k + 1))
    assert seen == list(range(21))


# ------------------------------------------------------------------ P8: identical streams
def test_p8_identical_streams_cross_equals_auto(oracle):
    rng = np.random.default_rng(8)
    S, C, N = 3, 16, 16 * 50
    one = crandn(rng, 1, 2, N)
    x = np.repeat(one, S, axis=0)
    vis = oracle.correlate(oracle.fstage(x, C))
    for j in range(C):
        for k in range(S):
            for i in range(k + 1):
                np.testing.assert_array_equal(vis[j, oracle.baseline_index(i, k)], vis[j, 0])


# ------------------------------------------------------------------ P9: delay -> phase slope
def delayed(s, d):
    """s(n - d) for real d by an FFT phase ramp (circular)."""
    k = np.fft.fftfreq(s.size)
    return np.fft.ifft(np.fft.fft(s) * np.exp(-2j * np.pi * k * d))


def test_p9_delay_is_phase_slope_and_is_compensated(oracle):
    rng = np.random.default_rng(9)
    C, n_t, d = 64, 1200, 9.77
    N = n_t * C
    s = crandn(rng, N)
    x = np.zeros((2, 2, N), dtype=np.complex128)
    x[0, :] = s
    x[1, :] = delayed(s, d)
    # (a) no compensation: arg V01[j] = +2 pi d (j - C/2)/C
    vis = oracle.correlate(oracle.fstage(x, C, delays=np.zeros(2), bandpass=np.ones(C), f_sb=0.0))
    v01 = vis[:, oracle.baseline_index(0, 1), 0, 0]
    ph = np.unwrap(np.angle(v01))
    jj = np.arange(C)
    slope = np.polyfit(jj[4:-4], ph[4:-4], 1)[0]
    assert abs(slope - 2 * np.pi * d / C) < 2e-3
    # (b) baseband (f_sb = 0): advance station 1 by tau = -d/f_s -> flat phase
    vis = oracle.correlate(oracle.fstage(x, C, delays=np.array([0.0, -d / F_S]), bandpass=np.ones(C), f_sb=0.0))
    v01 = vis[:, oracle.baseline_index(0, 1), 0, 0]
    assert np.max(np.abs(np.angle(v01[2:-2]))) < 0.03
    v00 = vis[:, oracle.baseline_index(0, 0), 0, 0].real
    v11 = vis[:, oracle.baseline_index(1, 1), 0, 0].real
    assert np.median(np.abs(v01) / np.sqrt(v00 * v11)) > 0.9        # coherent (no coarse shift: a few % lost)
    # (c) equivalent: delay station 0 by +d/f_s instead
    vis = oracle.correlate(oracle.fstage(x, C, delays=np.array([d / F_S, 0.0]), bandpass=np.ones(C), f_sb=0.0))
    assert np.max(np.abs(np.angle(vis[2:-2, oracle.baseline_index(0, 1), 0, 0]))) < 0.03
    # (d) sky-frequency ladder: the generator applies the fringe term, the same tau flattens it
    f_sb = oracle.default_subband_frequency(3)
    x[1, :] = delayed(s, d) * np.exp(-2j * np.pi * f_sb * d / F_S)
    vis = oracle.correlate(oracle.fstage(x, C, delays=np.array([0.0, -d / F_S]), bandpass=np.ones(C), f_sb=f_sb))
    assert np.max(np.abs(np.angle(vis[2:-2, oracle.baseline_index(0, 1), 0, 0]))) < 0.03


def test_rotation_sign_and_frequency_ladder(oracle):
    """exp(-2 pi i f tau): a positive tau on a single channel turns the phase clockwise by
    2 pi frac(f tau); f[j] = f_sb + (j - C/2) f_s / C."""
    C = 16
    F = np.ones((1, C), dtype=np.complex128)
    tau, f_sb = 1.0e-7, 150.0e6
    z = oracle.rotate(F, tau, np.ones(C), f_sb)[0]
    f = f_sb + (np.arange(C) - C // 2) * F_S / C
    expect = np.exp(-2j * np.pi * np.modf(f * tau)[0])
    np.testing.assert_allclose(z, expect, atol=1e-9)
    # large delay: frac() must be taken in double precision (H4): compare with exact rational arithmetic
    from fractions import Fraction
    tau = 50e-6
    z = oracle.rotate(F, tau, np.ones(C), f_sb)[0]
    for j in (0, 9):
        cyc = (Fraction(f_sb) + Fraction(j - C // 2) * Fraction(F_S) / C) * Fraction(tau)
        fr = float(cyc - (cyc.numerator // cyc.denominator))
        assert abs(np.angle(z[j] * np.exp(2j * np.pi * fr))) < 1e-8


# ------------------------------------------------------------------ P10: history carry
def test_p10_two_calls_equal_one_call(oracle):
    rng = np.random.default_rng(10)
    S, C = 2, 16
    N1, N2 = 16 * 23, 16 * 9          # second block shorter than the history (15*16 = 240 > 144)
    x = crandn(rng, S, 2, N1 + N2)
    whole = oracle.fstage(x, C)
    h = oracle.new_history(S, C)
    a = oracle.fstage(x[:, :, :N1], C, hist=h)
    b = oracle.fstage(x[:, :, N1:], C, hist=h)
    np.testing.assert_allclose(np.concatenate([a, b], axis=2), whole, rtol=0, atol=1e-13)
    np.testing.assert_array_equal(h, x[:, :, -15 * C:])


def test_a11_trailing_samples_are_ignored(oracle):
    rng = np.random.default_rng(11)
    C = 16
    x = crandn(rng, 1, 2, C * 20 + 7)
    h1, h2 = oracle.new_history(1, C), oracle.new_history(1, C)
    a = oracle.fstage(x, C, hist=h1)
    b = oracle.fstage(x[:, :, :C * 20], C, hist=h2)
    assert a.shape == (1, 2, 20, C)
    np.testing.assert_array_equal(a, b)
    np.testing.assert_array_equal(h1, h2)


# ------------------------------------------------------------------ P11: brute force
def numpy_brute_force(x, hist, g, C, delays, bandpass, f_sb):
    """Different loop structure from the oracle: whole-window single sum per (t, j),
    exponent built with np.exp on the un-reduced argument, visibilities by np.vdot."""
    S, _, N = x.shape
    n_t = N // C
    L = T * C
    xx = np.concatenate([hist, x], axis=2)
    z = np.zeros((S, 2, n_t, C), dtype=np.complex128)
    n = np.arange(L)
    for j in range(C):
        c = (j + C // 2) % C
        e = g * np.exp(-2j * np.pi * c * n / C)
        f = f_sb + (j - C / 2) * F_S / C
        for a in range(S):
            w = bandpass[j] * np.exp(-2j * np.pi * ((f * delays[a]) % 1.0))
            for p in range(2):
                for t in range(n_t):
                    z[a, p, t, j] = w * np.sum(e * xx[a, p, t * C:t * C + L])
    vis = np.zeros((C, S * (S + 1) // 2, 2, 2), dtype=np.complex128)
    for j in range(C):
        for k in range(S):
            for i in range(k + 1):
                for p in range(2):
                    for q in range(2):
                        vis[j, k * (k + 1) // 2 + i, p, q] = np.vdot(z[k, q, :, j], z[i, p, :, j])
    return z, vis


def test_p11_brute_force_two_stations(oracle):
    rng = np.random.default_rng(11)
    S, C, n_t = 2, 16, 21
    samples = rng.integers(-300, 300, size=(S, 2, n_t * C + 5, 2)).astype(np.int16)
    hist = crandn(rng, S, 2, (T - 1) * C) * 50
    delays = np.array([1.3e-6, -0.7e-6])
    bandpass = 1.0 + 0.1 * rng.uniform(-1, 1, C)
    f_sb = oracle.default_subband_frequency(5)
    vis, z = oracle.process_subband(samples, C, delays, bandpass, f_sb, hist=hist.copy(), return_z=True)
    x = samples[..., 0].astype(np.float64) + 1j * samples[..., 1]
    gref = scipy.signal.firwin(T * C, 1.0 / C, window="hann")
    zb, vb = numpy_brute_force(x[:, :, :n_t * C], hist, gref, C, delays, bandpass, f_sb)
    scale = np.abs(vb).max()
    np.testing.assert_allclose(z, zb, rtol=0, atol=1e-9 * np.abs(zb).max())
    np.testing.assert_allclose(vis, vb, rtol=0, atol=1e-12 * scale)
    # the oracle's own second route (single-sum C routine) agrees too
    for j in (0, 5, 15):
        zc, vc = oracle.channel_direct(samples, C, j, hist=hist, delays=delays, bandpass=bandpass, f_sb=f_sb)
        np.testing.assert_allclose(zc.reshape(S, 2, n_t), zb[:, :, :, j], rtol=0, atol=1e-9 * np.abs(zb).max())
        np.testing.assert_allclose(vc, vb[j], rtol=0, atol=1e-12 * scale)


def test_unpack_is_the_integer_value(oracle):
    a16 = np.arange(-32768, 32768, dtype=np.int32).astype(np.int16)
    np.testing.assert_array_equal(oracle.unpack(a16), np.arange(-32768, 32768, dtype=np.float64))
    a8 = np.arange(-128, 128, dtype=np.int32).astype(np.int8)
    np.testing.assert_array_equal(oracle.unpack(a8), np.arange(-128, 128, dtype=np.float64))


# ------------------------------------------------------------------ P12: linearity / bandpass
def test_p12_bandpass_and_input_scaling(oracle):
    rng = np.random.default_rng(12)
    S, C, n_t = 2, 16, 30
    samples = rng.integers(-100, 100, size=(S, 2, n_t * C, 2)).astype(np.int16)
    delays = np.array([0.0, 2e-7])
    b = np.ones(C)
    v1 = oracle.process_subband(samples, C, delays, b, 1.2e8)
    b2 = b.copy()
    b2[3] = 1.5
    v2 = oracle.process_subband(samples, C, delays, b2, 1.2e8)
    np.testing.assert_allclose(v2[3], 2.25 * v1[3], rtol=1e-13)
    np.testing.assert_array_equal(np.delete(v2, 3, axis=0), np.delete(v1, 3, axis=0))
    v4 = oracle.process_subband((2 * samples).astype(np.int16), C, delays, b, 1.2e8)
    np.testing.assert_allclose(v4, 4.0 * v1, rtol=1e-13)


# ------------------------------------------------------------------ P13: statistics
def test_p13_noise_power_and_correlation_coefficient(oracle):
    rng = np.random.default_rng(13)
    S, C, n_t, sigma = 3, 16, 6000, 100.0
    N = n_t * C
    common = crandn(rng, 1, 2, N)
    x = sigma * (np.sqrt(0.9) * crandn(rng, S, 2, N) + np.sqrt(0.1) * common)   # reading A15: 10 % of power
    b = 1.0 + 0.1 * rng.uniform(-1, 1, C)
    vis = oracle.correlate(oracle.fstage(x, C, delays=np.zeros(S), bandpass=b, f_sb=1e8))
    g = scipy.signal.firwin(T * C, 1.0 / C, window="hann")
    expect = n_t * 2 * sigma ** 2 * np.sum(g * g) * b ** 2
    for k in range(S):
        auto = vis[:, oracle.baseline_index(k, k), 0, 0].real
        np.testing.assert_allclose(auto, expect, rtol=6.0 / np.sqrt(n_t))
    for (i, k) in ((0, 1), (0, 2), (1, 2)):
        v = vis[:, oracle.baseline_index(i, k)]
        aii = vis[:, oracle.baseline_index(i, i)]
        akk = vis[:, oracle.baseline_index(k, k)]
        rho = np.abs(v[:, 1, 1]) / np.sqrt(aii[:, 1, 1].real * akk[:, 1, 1].real)
        assert np.all(np.abs(rho - 0.1) < 4.0 / np.sqrt(n_t))
        rho_xy = np.abs(v[:, 0, 1]) / np.sqrt(aii[:, 0, 0].real * akk[:, 1, 1].real)
        assert np.all(rho_xy < 4.5 / np.sqrt(n_t))                   # independent pols: only noise


# ------------------------------------------------------------------ frozen tiny case (tests/golden/)
def test_golden_tiny_case_is_reproduced(oracle):
    """The oracle still gives the values frozen by tests/golden/make_golden.py (which calls only the oracle)."""
    import os
    import sys

    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    sys.path.insert(0, here)
    import make_golden as mg

    x = np.loadtxt(os.path.join(here, "tiny_fx_input.txt"), dtype=np.int64).astype(np.int16).reshape(mg.S, 2, mg.N, 2)
    assert np.array_equal(x, mg.inputs())
    exp = np.loadtxt(os.path.join(here, "tiny_fx_expected.txt")).view(np.complex128).reshape(mg.C, 3, 2, 2)
    vis = oracle.process_subband(x, mg.C, mg.DELAYS, mg.BANDPASS, oracle.default_subband_frequency(0))
    assert np.max(np.abs(vis - exp)) <= 1e-9 * np.max(np.abs(exp))


# ------------------------------------------------------------------ P16: time-varying delay (reading A21)
def test_p16_equal_begin_and_end_delays_are_the_static_rotation(oracle):
    rng = np.random.default_rng(16)
    C, S, n_t = 16, 3, 37
    x = rng.integers(-300, 300, size=(S, 2, n_t * C + 5, 2)).astype(np.int16)
    tau = rng.uniform(0, 2e-6, S)
    b = 1.0 + 0.1 * rng.uniform(-1, 1, C)
    f = 1.2e8
    v0 = oracle.process_subband(x, C, tau, b, f)
    v1 = oracle.process_subband(x, C, tau, b, f, delays_end=tau.copy())
    assert np.array_equal(v0, v1)


@pytest.mark.parametrize("drift_cycles", [0.15, -3.7])
def test_p16_linear_delay_drift_is_a_geometric_series(oracle, drift_cycles):
    """Warmed-up DC input puts F[t][C/2] = A in every spectrum, so with station 1 drifting from tau_b to tau_e the
    cross-correlation of the centre channel is a geometric series with a closed form:
      V01 = |A|^2 sum_t exp(+2 pi i f_c (tau_b + (tau_e - tau_b) t / n_t)) = |A|^2 e^{2 pi i f_c tau_b} (1 - r^n_t) / (1 - r),
    r = exp(2 pi i f_c (tau_e - tau_b) / n_t).  Fixes the interpolation end points (t = 0 is tau_b, t = n_t would be
    tau_e), the sign and that the phase is linear in t."""
    C, n_t = 16, 200
    A = 2.0 - 1.5j
    f_c = 1.0e8                                                 # channel C/2 sits at f_sb
    tau_b = 0.3 / f_c
    tau_e = tau_b + drift_cycles / f_c
    x = np.full((2, 2, n_t * C), A, dtype=np.complex128)
    hist = np.full((2, 2, (T - 1) * C), A, dtype=np.complex128)  # filter already warmed up
    z = oracle.fstage(x, C, hist=hist, delays=np.array([0.0, tau_b]), bandpass=np.ones(C), f_sb=f_c,
                      delays_end=np.array([0.0, tau_e]))
    np.testing.assert_allclose(z[0, 0, :, C // 2], A, rtol=0, atol=1e-12)          # station 0: not rotated
    v = oracle.correlate(z)                                     # [C][n_bl][2][2]
    r = np.exp(2j * np.pi * drift_cycles / n_t)
    want = abs(A) ** 2 * np.exp(2j * np.pi * 0.3) * (1 - r ** n_t) / (1 - r)
    got = v[C // 2, oracle.baseline_index(0, 1), 0, 0]
    assert abs(got - want) <= 1e-9 * abs(A) ** 2 * n_t
    # autocorrelation of the drifting station is unaffected (a pure phase)
    assert abs(v[C // 2, oracle.baseline_index(1, 1), 0, 0] - abs(A) ** 2 * n_t) <= 1e-9 * abs(A) ** 2 * n_t


@pytest.mark.parametrize("m", [-5, 3])
def test_p16_drift_at_an_off_centre_channel_uses_that_channels_frequency(oracle, m):
    """Same closed form as above at channel j = C/2 + m: a warmed-up tone at the exact centre of channel j
    (x[n] = A exp(2 pi i m n / C), periodic in C) gives F[t][j] = A in every spectrum, and the drift of station 1 turns
    with THAT channel's sky frequency f_j = f_sb + m f_s / C (reading A6), not with f_sb: the per-channel term of the
    interpolated phase ("channel-dependent phase angles")."""
    C, n_t = 16, 160
    A = 1.25 + 0.5j
    f_sb, f_s = 1.0e8, oracle.F_S
    j = C // 2 + m
    f_j = f_sb + m * f_s / C
    tau_b = 1.0e-6
    tau_e = tau_b + (12 * n_t + 0.1) / f_sb                     # 12 cycles per spectrum at f_sb (+ 0.1 over the block);
                                                                # f_j adds or removes about a cycle over the block
    n = np.arange(-(T - 1) * C, n_t * C)
    tone = A * np.exp(2j * np.pi * m * (n % C) / C)
    hist = np.broadcast_to(tone[:(T - 1) * C], (2, 2, (T - 1) * C)).copy()
    x = np.broadcast_to(tone[(T - 1) * C:], (2, 2, n_t * C)).copy()
    z = oracle.fstage(x, C, hist=hist, delays=np.array([0.0, tau_b]), bandpass=np.ones(C), f_sb=f_sb,
                      delays_end=np.array([0.0, tau_e]))
    np.testing.assert_allclose(z[0, 0, :, j], A, rtol=0, atol=1e-11)
    v = oracle.correlate(z)
    step = f_j * (tau_e - tau_b) / n_t                          # cycles per spectrum
    r = np.exp(2j * np.pi * step)
    want = abs(A) ** 2 * np.exp(2j * np.pi * f_j * tau_b) * (1 - r ** n_t) / (1 - r)
    got = v[j, oracle.baseline_index(0, 1), 0, 0]
    assert abs(got - want) <= 1e-7 * abs(A) ** 2 * n_t
    # and it is NOT the series of the subband centre frequency
    r0 = np.exp(2j * np.pi * f_sb * (tau_e - tau_b) / n_t)
    wrong = abs(A) ** 2 * np.exp(2j * np.pi * f_sb * tau_b) * (1 - r0 ** n_t) / (1 - r0)
    assert abs(got - wrong) > 1e-2 * abs(A) ** 2 * n_t
