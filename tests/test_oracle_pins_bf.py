"""CPU pins of the oracle functions behind SURVEY.md sec 8(f) row 4, the beamformer (readings A28-A31,
DESIGN.md sec 2): coherent sum, Stokes parameters, time integration, incoherent sum.  Every pin is a closed form, an
invariant or a brute force that does not re-use the routine it checks."""
import numpy as np
import pytest

F_S = 195312.5


def crandn(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def chan_freq(C, f_sb, j):
    return f_sb + (j - C / 2) * F_S / C


# ------------------------------------------------------------------ P22: coherent sum (A28)
def test_p22_one_station_zero_delay_is_the_identity(oracle):
    rng = np.random.default_rng(22)
    C, n_t = 16, 10
    z = crandn(rng, 1, 2, n_t, C)
    y = oracle.beamform_coherent(z, np.zeros((3, 1)), 150e6)
    for b in range(3):
        np.testing.assert_array_equal(y[b], np.transpose(z[0], (0, 2, 1)))        # [2][C][n_t], bit for bit


def test_p22_uniform_linear_array_gives_the_dirichlet_kernel(oracle):
    """Stations on a line see a plane wave: z_a = A e^{+2 pi i f a delta} (station a receives the wavefront a delta EARLIER,
    i.e. its signal is the reference advanced by a delta).  A beam that delays station a by a theta gives
       Y = A sum_a e^{2 pi i f a (delta - theta)} = A e^{i pi (S-1) x} sin(pi S x) / sin(pi x),  x = f (delta - theta),
    and |Y| = S A exactly when the beam points at the source (theta = delta): pins the sign of the exponent, the use of the
    channel's own sky frequency and the sum over stations."""
    S, C, n_t, f_sb = 12, 16, 3, 120.0e6
    A = 2.0 - 1.5j
    delta = 3.1e-9
    thetas = np.array([delta, 0.0, 2.0e-9, -1.0e-9, 3.6e-9])
    a = np.arange(S)
    f = chan_freq(C, f_sb, np.arange(C))
    z = np.empty((S, 2, n_t, C), dtype=np.complex128)
    z[:] = (A * np.exp(2j * np.pi * f[None, :] * a[:, None] * delta))[:, None, None, :]
    z[:, 1] *= 0.5                                                                  # pol Y: half the amplitude
    y = oracle.beamform_coherent(z, thetas[:, None] * a[None, :], f_sb)
    for b, th in enumerate(thetas):
        x = f * (delta - th)
        with np.errstate(invalid="ignore", divide="ignore"):
            dk = np.where(np.abs(np.sin(np.pi * x)) < 1e-300, float(S), np.sin(np.pi * S * x) / np.sin(np.pi * x))
        want = A * np.exp(1j * np.pi * (S - 1) * x) * dk
        for t in range(n_t):
            np.testing.assert_allclose(y[b, 0, :, t], want, rtol=0, atol=1e-6 * abs(A) * S)
            np.testing.assert_allclose(y[b, 1, :, t], 0.5 * want, rtol=0, atol=1e-6 * abs(A) * S)
    np.testing.assert_allclose(np.abs(y[0, 0]), S * abs(A), rtol=1e-9)            # on source: full coherent gain
    assert np.all(np.abs(y[1:, 0]) < S * abs(A) * 0.999)                            # off source: less


def test_p22_brute_force_einsum(oracle):
    rng = np.random.default_rng(221)
    S, C, n_t, nb, f_sb = 5, 16, 7, 4, 133.3e6
    z = crandn(rng, S, 2, n_t, C)
    bd = rng.uniform(-30e-9, 30e-9, (nb, S))
    f = chan_freq(C, f_sb, np.arange(C))
    w = np.exp(-2j * np.pi * ((bd[:, :, None] * f[None, None, :]) % 1.0))          # [b][a][j]
    want = np.einsum("baj,aptj->bpjt", w, z)
    np.testing.assert_allclose(oracle.beamform_coherent(z, bd, f_sb), want, rtol=0, atol=1e-9)


def test_p22_beam_delay_equals_station_delay(oracle):
    """A beam delay tau_{b,a} acts exactly like adding tau_{b,a} to the station delay of step 7 (same sign sense)."""
    rng = np.random.default_rng(222)
    S, C, N = 3, 16, 16 * 40
    x = crandn(rng, S, 2, N) * 50
    tau = rng.uniform(0, 1e-6, S)
    extra = rng.uniform(-5e-8, 5e-8, S)
    f_sb = oracle.default_subband_frequency(3)
    z0 = oracle.fstage(x, C, delays=tau, f_sb=f_sb)
    z1 = oracle.fstage(x, C, delays=tau + extra, f_sb=f_sb)
    y0 = oracle.beamform_coherent(z0, extra[None, :], f_sb)
    y1 = oracle.beamform_coherent(z1, np.zeros((1, S)), f_sb)
    np.testing.assert_allclose(y0, y1, rtol=0, atol=1e-6 * np.abs(y1).max())


# ------------------------------------------------------------------ P23: Stokes parameters (A29)
@pytest.mark.parametrize("x,y,want", [
    (1 + 2j, 0, (5, 5, 0, 0)),                 # X only: Q = +I
    (0, 3 - 1j, (10, -10, 0, 0)),              # Y only: Q = -I
    (2 + 1j, 2 + 1j, (10, 0, 10, 0)),          # X = Y (+45 deg linear): U = +I
    (2 + 1j, -(2 + 1j), (10, 0, -10, 0)),      # X = -Y: U = -I
    (1 + 1j, 1j * (1 + 1j), (4, 0, 0, -4)),    # Y = iX: X conj(Y) = -i |X|^2, V = -I
    (1 + 1j, -1j * (1 + 1j), (4, 0, 0, 4)),    # Y = -iX: V = +I
])
def test_p23_stokes_of_pure_states(oracle, x, y, want):
    got = oracle.stokes(np.array([x], dtype=np.complex128), np.array([y], dtype=np.complex128), 4)[:, 0]
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-14)


def test_p23_stokes_identities(oracle):
    rng = np.random.default_rng(23)
    x, y = crandn(rng, 4, 50), crandn(rng, 4, 50)
    s = oracle.stokes(x, y, 4)
    np.testing.assert_allclose(s[0] ** 2, s[1] ** 2 + s[2] ** 2 + s[3] ** 2, rtol=1e-12)     # fully polarised sample
    np.testing.assert_allclose(s[0], np.abs(x) ** 2 + np.abs(y) ** 2, rtol=1e-14)
    np.testing.assert_allclose(s[2] + 1j * s[3], 2 * x * np.conj(y), rtol=1e-13, atol=1e-13)
    np.testing.assert_array_equal(oracle.stokes(x, y, 1)[0], s[0])                            # I only = the I of IQUV
    # a common phase does not change any Stokes parameter; swapping X and Y flips Q and V, keeps I and U
    np.testing.assert_allclose(oracle.stokes(x * np.exp(0.3j), y * np.exp(0.3j), 4), s, rtol=1e-12, atol=1e-12)
    sw = oracle.stokes(y, x, 4)
    np.testing.assert_allclose(sw, s * np.array([1, -1, 1, -1])[:, None, None], rtol=1e-12, atol=1e-12)


# ------------------------------------------------------------------ P24: time integration (A30)
def test_p24_integration(oracle):
    rng = np.random.default_rng(24)
    a = rng.standard_normal((3, 5, 70))
    np.testing.assert_array_equal(oracle.integrate(a, 1), a)                                    # t_int = 1: identity
    for t_int in (2, 4, 16, 64):
        n_out = 70 // t_int
        want = a[..., :n_out * t_int].reshape(3, 5, n_out, t_int).sum(-1)                      # tail dropped
        got = oracle.integrate(a, t_int)
        assert got.shape == (3, 5, n_out)
        np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)
    ones = np.ones((2, 64))
    np.testing.assert_array_equal(oracle.integrate(ones, 16), np.full((2, 4), 16.0))             # a sum, not a mean


# ------------------------------------------------------------------ P25: coherent vs incoherent Stokes (A28-A31)
def test_p25_coherent_and_incoherent_gain(oracle):
    """S identical stations, beam on the phase centre: coherent Stokes = S^2 x one station, incoherent = S x one station
    ("Coherently formed beams are more sensitive")."""
    rng = np.random.default_rng(25)
    S, C, n_t = 6, 16, 32
    one = crandn(rng, 1, 2, n_t, C)
    z = np.repeat(one, S, axis=0)
    single = oracle.integrate(oracle.stokes(np.transpose(one[0, 0]), np.transpose(one[0, 1]), 4), 8)   # [4][C][n_out]
    coh = oracle.coherent_stokes(z, np.zeros((1, S)), 140e6, 4, 8)
    inc = oracle.incoherent_stokes(z, 4, 8)
    np.testing.assert_allclose(coh[0], S * S * single, rtol=1e-12, atol=1e-9)
    np.testing.assert_allclose(inc, S * single, rtol=1e-12, atol=1e-9)


def test_p25_compositions_against_numpy(oracle):
    rng = np.random.default_rng(251)
    S, C, n_t, nb, f_sb, t_int = 4, 16, 37, 3, 127.7e6, 4
    z = crandn(rng, S, 2, n_t, C)
    bd = rng.uniform(-20e-9, 20e-9, (nb, S))
    f = chan_freq(C, f_sb, np.arange(C))
    w = np.exp(-2j * np.pi * bd[:, :, None] * f[None, None, :])
    y = np.einsum("baj,aptj->bpjt", w, z)
    n_out = n_t // t_int

    def integ(a):
        return a[..., :n_out * t_int].reshape(a.shape[:-1] + (n_out, t_int)).sum(-1)

    X, Y = y[:, 0], y[:, 1]
    want = np.stack([np.abs(X) ** 2 + np.abs(Y) ** 2, np.abs(X) ** 2 - np.abs(Y) ** 2, 2 * (X * np.conj(Y)).real,
                     2 * (X * np.conj(Y)).imag], axis=1)                                        # [b][4][C][n_t]
    got = oracle.coherent_stokes(z, bd, f_sb, 4, t_int)
    np.testing.assert_allclose(got, integ(want), rtol=0, atol=1e-9 * np.abs(want).max())
    np.testing.assert_allclose(oracle.coherent_stokes(z, bd, f_sb, 1, t_int)[:, 0], integ(want)[:, 0], rtol=0, atol=1e-9 * np.abs(want).max())
    zx, zy = np.transpose(z[:, 0], (0, 2, 1)), np.transpose(z[:, 1], (0, 2, 1))                 # [S][C][n_t]
    winc = np.stack([np.abs(zx) ** 2 + np.abs(zy) ** 2, np.abs(zx) ** 2 - np.abs(zy) ** 2, 2 * (zx * np.conj(zy)).real,
                     2 * (zx * np.conj(zy)).imag], axis=0).sum(1)                               # [4][C][n_t]
    np.testing.assert_allclose(oracle.incoherent_stokes(z, 4, t_int), integ(winc), rtol=0, atol=1e-9 * np.abs(winc).max())
    # the incoherent beam does not depend on any station phase
    ph = np.exp(1j * rng.uniform(0, 6.28, (S, 1, 1, 1)))
    np.testing.assert_allclose(oracle.incoherent_stokes(z * ph, 4, t_int), oracle.incoherent_stokes(z, 4, t_int), rtol=1e-11, atol=1e-11)


def test_p25_point_source_beam_pattern_from_integer_samples(oracle):
    """End to end from quantised station samples: a common noise source delayed per station by its geometric delay;
    the beam whose delays cancel the geometric delays collects (nearly) S^2 x the single-station source power, a beam far
    off collects about S x (incoherent level): coherent / incoherent Stokes I ratio ~ S on source."""
    rng = np.random.default_rng(252)
    S, C, n_t = 8, 16, 256
    N = C * n_t
    f_sb = oracle.default_subband_frequency(0)
    src = crandn(rng, N + 64) * 300.0
    geo = rng.uniform(0, 4.0e-6, S)                      # < 1 sample each (5.12 us): fractional delays
    freqs = np.fft.fftfreq(N + 64, d=1.0 / F_S)
    x = np.empty((S, 2, N), dtype=np.complex128)
    for a in range(S):
        d = np.fft.ifft(np.fft.fft(src) * np.exp(-2j * np.pi * (freqs + f_sb) * geo[a]))[32:32 + N]   # delayed + fringe term
        x[a, 0] = d
        x[a, 1] = 0.5 * d
    samples = np.stack([np.rint(x.real), np.rint(x.imag)], axis=-1).astype(np.int16)
    z = oracle.channelise_subband(samples, C, np.zeros(S), np.ones(C), f_sb)
    on = -geo[None, :]
    off = on + rng.uniform(-3e-8, 3e-8, (1, S))          # several cycles of phase error at 100 MHz
    coh = oracle.coherent_stokes(z, np.concatenate([on, off]), f_sb, 1, 64)[:, 0, 2:C - 2, 1:]    # inner channels, warmed up
    inc = oracle.incoherent_stokes(z, 1, 64)[0, 2:C - 2, 1:]
    ratio_on = coh[0].sum() / inc.sum()
    ratio_off = coh[1].sum() / inc.sum()
    assert 0.97 * S < ratio_on <= S * 1.0001
    assert ratio_off < 0.5 * S
