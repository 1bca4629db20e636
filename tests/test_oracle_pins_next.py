"""CPU pins of the oracle functions behind SURVEY.md sec 8(f) rows 1-3 (readings A22-A27):
phase offsets, sub-second dumps, valid-sample flags and counts, coarse integer-sample delay, pol-minor order, 4-bit
samples.  Every pin is a closed form, an invariant or a brute force that does not re-use the routine it checks."""
import numpy as np
import pytest

T = 16
F_S = 195312.5


def crandn(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ------------------------------------------------------------------ P18: phase offsets (A22)
def test_p18_phase_offset_turns_exactly_the_products_of_that_input(oracle):
    """z_{1,X} <- z_{1,X} e^{-i phi}:  V01^{XX} = z0X conj(z1X) turns by +phi, V01^{YX} too, V01^{XY} and V01^{YY} do
    not change; the autocorrelation XX of station 1 does not change, its XY turns by -phi and YX by +phi."""
    rng = np.random.default_rng(18)
    S, C, n_t, phi = 3, 16, 40, 0.7345
    z = crandn(rng, S, 2, n_t, C)
    ph = np.zeros((S, 2))
    ph[1, 0] = phi
    v0 = oracle.correlate(z)
    v1 = oracle.correlate(oracle.phase_offsets(z, ph))
    b01, b11, b12, b00, b02 = (oracle.baseline_index(0, 1), oracle.baseline_index(1, 1), oracle.baseline_index(1, 2),
                               oracle.baseline_index(0, 0), oracle.baseline_index(0, 2))
    e = np.exp(1j * phi)
    np.testing.assert_allclose(v1[:, b01, 0, 0], v0[:, b01, 0, 0] * e, rtol=1e-12)
    np.testing.assert_allclose(v1[:, b01, 1, 0], v0[:, b01, 1, 0] * e, rtol=1e-12)
    np.testing.assert_array_equal(v1[:, b01, :, 1], v0[:, b01, :, 1])
    np.testing.assert_allclose(v1[:, b11, 0, 0], v0[:, b11, 0, 0], rtol=1e-12)
    np.testing.assert_allclose(v1[:, b11, 0, 1], v0[:, b11, 0, 1] / e, rtol=1e-12)
    np.testing.assert_allclose(v1[:, b11, 1, 0], v0[:, b11, 1, 0] * e, rtol=1e-12)
    np.testing.assert_allclose(v1[:, b12, 0, :], v0[:, b12, 0, :] / e, rtol=1e-12)      # station 1 is the first of (1, 2)
    np.testing.assert_array_equal(v1[:, b00], v0[:, b00])
    np.testing.assert_array_equal(v1[:, b02], v0[:, b02])


def test_p18_phase_offset_is_a_delay_at_one_frequency(oracle):
    """Same sign sense as the delay term: an offset of 2 pi f tau on both pols of a station equals delaying it by tau in a
    channel of frequency f (here the subband centre)."""
    C, n_t = 16, 8
    F = np.ones((n_t, C), dtype=np.complex128)
    f, tau = 1.0e8, 1.2345e-9
    a = oracle.rotate(F, tau, np.ones(C), f)[:, C // 2]
    z = np.ones((1, 2, n_t, C), dtype=np.complex128)
    b = oracle.phase_offsets(z, np.full((1, 2), 2 * np.pi * f * tau))[0, 0, :, C // 2]
    np.testing.assert_allclose(a, b, atol=1e-7)


# ------------------------------------------------------------------ P19: dumps (A23)
@pytest.mark.parametrize("n_t,D", [(256, 2), (256, 4), (200, 2), (130, 3)])
def test_p19_dumps_partition_the_block(oracle, n_t, D):
    """Dump d integrates the spectra [d L, min((d+1) L, n_t)), L = (ceil(n_t/64)/D) 64: the dumps add up to the one-dump
    result (to rounding: the sum is split), each equals an independent einsum over its own range, and D = 1 is
    oracle_correlate bit for bit."""
    rng = np.random.default_rng(19)
    S, C = 3, 4
    z = crandn(rng, S, 2, n_t, C)
    one = oracle.correlate(z)
    np.testing.assert_array_equal(oracle.correlate_dumps(z, 1)[0], one)
    vd = oracle.correlate_dumps(z, D)
    np.testing.assert_allclose(vd.sum(axis=0), one, rtol=1e-12, atol=1e-12)
    L = (-(-n_t // 64) // D) * 64
    for d in range(D):
        zz = z[:, :, d * L:min((d + 1) * L, n_t), :]
        full = np.einsum("iptj,kqtj->jikpq", zz, zz.conj())
        for k in range(S):
            for i in range(k + 1):
                np.testing.assert_allclose(vd[d][:, oracle.baseline_index(i, k)], full[:, i, k], rtol=1e-12, atol=1e-12)


def test_p19_dumps_must_divide_the_tile_count(oracle):
    z = np.zeros((1, 2, 200, 4), dtype=np.complex128)            # ceil(200 / 64) = 4 tiles
    with pytest.raises(ValueError):
        oracle.correlate_dumps(z, 3)


# ------------------------------------------------------------------ P20: valid-sample flags and counts (A24)
def test_p20_flagged_tiles_count_as_zero_and_counts_are_the_weights(oracle):
    """Warmed-up DC input makes F[t][C/2] = A in every spectrum of every station, so V_ik[C/2] = |A|^2 x (number of
    spectra in which both stations are valid) = |A|^2 counts: ties the flags, the dumps and the counts together."""
    S, C, n_t, D = 3, 16, 300, 5                                    # 5 tiles of 64 (last one 44 spectra)
    A = 1.5 - 0.5j
    x = np.full((S, 2, n_t * C), A, dtype=np.complex128)
    hist = np.full((S, 2, (T - 1) * C), A, dtype=np.complex128)
    z = oracle.fstage(x, C, hist=hist)
    valid = np.ones((S, 5), dtype=np.uint8)
    valid[0, 1] = 0
    valid[1, 1] = valid[1, 4] = 0
    valid[2, :] = 0
    zf = oracle.flag_tiles(z, valid)
    assert np.all(zf[2] == 0) and np.all(zf[0, :, 64:128] == 0) and np.array_equal(zf[0, :, :64], z[0, :, :64])
    v = oracle.correlate_dumps(zf, D)[:, C // 2, :, 0, 0]            # [D][n_bl]
    counts = oracle.valid_counts(S, n_t, valid, D)
    want = np.zeros((D, oracle.n_baselines(S)), dtype=np.int64)
    tile_len = [64, 64, 64, 64, 44]
    for d in range(D):
        for k in range(S):
            for i in range(k + 1):
                want[d, oracle.baseline_index(i, k)] = tile_len[d] * int(valid[i, d]) * int(valid[k, d])
    np.testing.assert_array_equal(counts, want)
    np.testing.assert_allclose(v, abs(A) ** 2 * counts, rtol=1e-11, atol=1e-11)
    # one dump over the block: the counts add up
    np.testing.assert_array_equal(oracle.valid_counts(S, n_t, valid, 1)[0], want.sum(axis=0))


def test_p20_all_valid_changes_nothing(oracle):
    rng = np.random.default_rng(20)
    z = crandn(rng, 2, 2, 100, 4)
    np.testing.assert_array_equal(oracle.flag_tiles(z, np.ones((2, 2), dtype=np.uint8)), z)


# ------------------------------------------------------------------ P17: coarse integer-sample delay (A25)
def _delayed(s, d):
    k = np.fft.fftfreq(s.size)
    return np.fft.ifft(np.fft.fft(s) * np.exp(-2j * np.pi * k * d))


def test_p17_coarse_shift_plus_residual_phase_restores_coherence(oracle):
    """Pin P9 leaves a few per cent of coherence on the table when a 9.77-sample delay is compensated by phase alone.
    Taking the integer part out by starting the late station's block 9 (here: 10, the nearest) samples later and the
    remainder by phase brings the coherence back above 0.99 and flattens the phase."""
    rng = np.random.default_rng(17)
    C, n_t, d = 64, 1200, 9.77
    N, margin = n_t * C, 16
    s = crandn(rng, N + margin)
    x = np.zeros((2, 2, N + margin, 2))
    for a, sig in enumerate((s, _delayed(s, d))):
        x[a, :, :, 0] = sig.real
        x[a, :, :, 1] = sig.imag
    bl01, b00, b11 = oracle.baseline_index(0, 1), oracle.baseline_index(0, 0), oracle.baseline_index(1, 1)

    def coherence(offsets, tau1):
        xs = oracle.coarse_shift(x, offsets, N)
        xc = xs[..., 0] + 1j * xs[..., 1]
        v = oracle.correlate(oracle.fstage(xc, C, delays=np.array([0.0, tau1]), bandpass=np.ones(C), f_sb=0.0))
        coh = np.abs(v[4:-4, bl01, 0, 0]) / np.sqrt(v[4:-4, b00, 0, 0].real * v[4:-4, b11, 0, 0].real)
        return float(np.median(coh)), float(np.max(np.abs(np.angle(v[4:-4, bl01, 0, 0]))))

    c_phase_only, _ = coherence([0, 0], -d / F_S)
    c_both, ph = coherence([0, 10], -(d - 10) / F_S)
    assert c_phase_only < 0.98                                     # P9: a few per cent lost
    assert c_both > 0.99 and ph < 0.02


def test_p17_coarse_shift_is_plain_indexing(oracle):
    x = np.arange(3 * 2 * 20 * 2).reshape(3, 2, 20, 2)
    y = oracle.coarse_shift(x, [0, 3, 8], 12)
    for a, o in enumerate([0, 3, 8]):
        for p in range(2):
            for n in range(12):
                assert np.array_equal(y[a, p, n], x[a, p, n + o])


# ------------------------------------------------------------------ A26 pol-minor order, A27 4-bit samples
def test_pol_minor_reorder_is_plain_indexing(oracle):
    x = np.arange(2 * 7 * 2 * 2).reshape(2, 7, 2, 2)               # [S][N][pol][re/im]
    y = oracle.pol_minor_to_planar(x)
    assert y.shape == (2, 2, 7, 2)
    for a in range(2):
        for n in range(7):
            for p in range(2):
                assert np.array_equal(y[a, p, n], x[a, n, p])


def test_p21_unpack_4bit_every_byte(oracle):
    b = np.arange(256, dtype=np.uint8)
    got = oracle.unpack4(b)
    for v in range(256):
        re, im = v & 15, v >> 4
        assert got[v, 0] == (re - 16 if re & 8 else re) and got[v, 1] == (im - 16 if im & 8 else im)
    assert got.min() == -8 and got.max() == 7


def test_process_subband_ext_reduces_to_process_subband(oracle):
    rng = np.random.default_rng(22)
    S, C, n_t = 2, 16, 70
    x = rng.integers(-300, 300, size=(S, 2, n_t * C + 3, 2)).astype(np.int16)
    tau = rng.uniform(0, 2e-6, S)
    b = 1.0 + 0.1 * rng.uniform(-1, 1, C)
    v0 = oracle.process_subband(x, C, tau, b, 1.2e8)
    v1 = oracle.process_subband_ext(x, C, tau, b, 1.2e8, phase0=np.zeros((S, 2)), valid=np.ones((S, 2), dtype=np.uint8))
    np.testing.assert_array_equal(v1[0], v0)
