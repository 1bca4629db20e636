"""ctypes front-end of the float64 CPU oracle (``oracle/cobalt_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_1801_04834_b200`` and the CUDA path imports nothing from here.

Every function is argument marshalling around one C routine; the arithmetic and its
citations (PAPER.md lines, SURVEY.md sec 8(c) readings) live in the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cobalt_oracle.c")
_LIB = os.path.join(_HERE, "libcobalt_oracle.so")

F_S = 195312.5  # Hz, subband sample rate (BASELINE.json north_star; "195 kHz")
TAPS = 16


def default_subband_frequency(s: int) -> float:
    """Reading A6: default sky-frequency ladder f_sb[s] = 100 MHz + (12 + s) f_s."""
    return 100.0e6 + (12 + s) * F_S


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP) into oracle/libcobalt_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True, text=True)
    return _LIB


_lib = None
_D = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_fir_prototype.argtypes = [ctypes.c_int, ctypes.c_int, _D]
        lib.oracle_fir.argtypes = [ctypes.c_int, ctypes.c_int, _D, _D, ctypes.c_longlong, _D]
        lib.oracle_dft.argtypes = [ctypes.c_int, _D, ctypes.c_longlong, _D]
        lib.oracle_rotate.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                      _D, ctypes.c_longlong, _D]
        lib.oracle_correlate.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, _D]
        lib.oracle_unpack_i16.argtypes = [ctypes.c_void_p, ctypes.c_longlong, _D]
        lib.oracle_unpack_i8.argtypes = [ctypes.c_void_p, ctypes.c_longlong, _D]
        lib.oracle_fstage_f64.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, _D, _D,
                                          _D, _D, ctypes.c_double, ctypes.c_double, _D]
        lib.oracle_fstage_f64.restype = ctypes.c_int
        lib.oracle_process_subband.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_longlong,
                                               ctypes.c_int, ctypes.c_void_p, _D, _D, _D, ctypes.c_double,
                                               ctypes.c_double, _D, _D]
        lib.oracle_process_subband.restype = ctypes.c_int
        lib.oracle_fstage_interp_f64.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, _D, _D,
                                                 _D, _D, _D, ctypes.c_double, ctypes.c_double, _D]
        lib.oracle_fstage_interp_f64.restype = ctypes.c_int
        lib.oracle_process_subband_interp.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_longlong,
                                                      ctypes.c_int, ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_double,
                                                      ctypes.c_double, _D, _D]
        lib.oracle_process_subband_interp.restype = ctypes.c_int
        lib.oracle_channel_direct.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, _D,
                                              _D, _D, _D, ctypes.c_double, ctypes.c_double, ctypes.c_int, _D, _D]
        lib.oracle_channel_direct.restype = ctypes.c_int
        lib.oracle_unpack_i4.argtypes = [ctypes.c_void_p, ctypes.c_longlong, _D]
        lib.oracle_phase_offsets.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, _D]
        lib.oracle_flag_tiles.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p, _D]
        lib.oracle_valid_counts.argtypes = [ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        lib.oracle_correlate_dumps.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_int, _D, _D]
        lib.oracle_correlate_dumps.restype = ctypes.c_int
        lib.oracle_beamform_coherent.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int, _D,
                                                 ctypes.c_double, ctypes.c_double, _D, _D]
        lib.oracle_stokes.argtypes = [ctypes.c_longlong, _D, _D, ctypes.c_int, _D]
        lib.oracle_integrate.argtypes = [ctypes.c_longlong, ctypes.c_longlong, ctypes.c_int, _D, _D]
        lib.oracle_coherent_stokes.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int, _D, ctypes.c_double,
                                               ctypes.c_double, _D, ctypes.c_int, ctypes.c_int, _D]
        lib.oracle_coherent_stokes.restype = ctypes.c_int
        lib.oracle_incoherent_stokes.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _D, ctypes.c_int, ctypes.c_int, _D]
        lib.oracle_incoherent_stokes.restype = ctypes.c_int
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_D)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _c2r(a):
    """complex128 array -> float64 view with a trailing (re, im) axis."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64).reshape(a.shape + (2,))


def _r2c(a):
    return a.view(np.complex128).reshape(a.shape[:-1])


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def n_baselines(S: int) -> int:
    return S * (S + 1) // 2


def baseline_index(i: int, k: int) -> int:
    """Reading A9: baseline (i <= k) is stored at k(k+1)/2 + i."""
    assert 0 <= i <= k
    return k * (k + 1) // 2 + i


def fir_prototype(C: int, T: int = TAPS) -> np.ndarray:
    g = np.empty(T * C, dtype=np.float64)
    _load().oracle_fir_prototype(C, T, _p(g))
    return g


def unpack(samples: np.ndarray) -> np.ndarray:
    """int16 / int8 array -> float64, same shape (step 1)."""
    s = np.ascontiguousarray(samples)
    out = np.empty(s.shape, dtype=np.float64)
    fn = {np.dtype(np.int16): _load().oracle_unpack_i16, np.dtype(np.int8): _load().oracle_unpack_i8}[s.dtype]
    fn(s.ctypes.data, s.size, _p(out))
    return out


def fir(xh: np.ndarray, g: np.ndarray, C: int, T: int = TAPS) -> np.ndarray:
    """xh: complex [(T-1)*C + n_t*C] (history then block) -> y complex [n_t][C] (step 3)."""
    xr = _c2r(xh)
    n_t = (xr.shape[0] - (T - 1) * C) // C
    assert xr.shape[0] == (T - 1) * C + n_t * C
    y = np.empty((n_t, C, 2), dtype=np.float64)
    _load().oracle_fir(C, T, _p(_f64(g, (T * C,))), _p(xr), n_t, _p(y))
    return _r2c(y)


def dft(y: np.ndarray) -> np.ndarray:
    """y complex [n_t][C] -> F complex [n_t][C], channel j ascending in frequency (steps 4-5)."""
    yr = _c2r(y)
    n_t, C = yr.shape[0], yr.shape[1]
    F = np.empty((n_t, C, 2), dtype=np.float64)
    _load().oracle_dft(C, _p(yr), n_t, _p(F))
    return _r2c(F)


def rotate(F: np.ndarray, tau: float, bandpass: np.ndarray, f_sb: float, f_s: float = F_S) -> np.ndarray:
    """F complex [n_t][C] -> z = F b[j] exp(-2 pi i frac(f[j] tau)) (steps 6-7)."""
    Fr = _c2r(F).copy()
    n_t, C = Fr.shape[0], Fr.shape[1]
    _load().oracle_rotate(C, f_sb, f_s, tau, _p(_f64(bandpass, (C,))), n_t, _p(Fr))
    return _r2c(Fr)


def correlate(z: np.ndarray) -> np.ndarray:
    """z complex [S][2][n_t][C] -> vis complex [C][n_bl][2][2] (step 8)."""
    zr = _c2r(z)
    S, two, n_t, C = zr.shape[:4]
    assert two == 2
    vis = np.empty((C, n_baselines(S), 2, 2, 2), dtype=np.float64)
    _load().oracle_correlate(S, C, n_t, _p(zr), _p(vis))
    return _r2c(vis)


def new_history(S: int, C: int, T: int = TAPS) -> np.ndarray:
    """Zero history (reading A3), complex [S][2][(T-1)*C]."""
    return np.zeros((S, 2, (T - 1) * C), dtype=np.complex128)


def fstage(x: np.ndarray, C: int, hist: np.ndarray | None = None, delays=None, bandpass=None,
           f_sb: float = 0.0, f_s: float = F_S, g: np.ndarray | None = None, T: int = TAPS, delays_end=None) -> np.ndarray:
    """Float entry of the F-stage (steps 2-7, 9): x complex [S][2][N] -> z complex [S][2][n_t][C].

    ``hist`` (complex [S][2][(T-1)*C]) is updated in place when given.  ``g`` overrides the
    prototype filter (pin P6 needs a rectangular one)."""
    xr = _c2r(x)
    S, two, N = xr.shape[:3]
    assert two == 2
    if g is None:
        g = fir_prototype(C, T)
    if hist is None:
        hist = new_history(S, C, T)
    assert hist.dtype == np.complex128 and hist.flags.c_contiguous and hist.shape == (S, 2, (T - 1) * C)
    hr = hist.view(np.float64)
    n_t = N // C
    z = np.empty((S, 2, n_t, C, 2), dtype=np.float64)
    d = None if delays is None else _f64(delays, (S,))
    b = _f64(np.ones(C) if bandpass is None else bandpass, (C,))
    de = None if delays_end is None else _f64(delays_end, (S,))
    rc = _load().oracle_fstage_interp_f64(S, C, T, N, _p(xr), _p(_f64(g, (T * C,))), _p(hr), _p(d), _p(de), _p(b), f_sb, f_s, _p(z))
    if rc:
        raise MemoryError("oracle_fstage_interp_f64")
    return _r2c(z)


def process_subband(samples: np.ndarray, C: int, delays, bandpass, f_sb: float, hist: np.ndarray | None = None,
                    f_s: float = F_S, T: int = TAPS, return_z: bool = False, delays_end=None):
    """One subband, steps 1-9.  samples int16/int8 [S][2][N][2] -> vis complex [C][n_bl][2][2].
    ``delays_end`` given: the delay of spectrum t is delays + (delays_end - delays) t / n_t (reading A21)."""
    s = np.ascontiguousarray(samples)
    S, two, N, ri = s.shape
    assert two == 2 and ri == 2 and s.dtype in (np.int16, np.int8)
    bits = 16 if s.dtype == np.int16 else 8
    if hist is None:
        hist = new_history(S, C, T)
    assert hist.dtype == np.complex128 and hist.flags.c_contiguous and hist.shape == (S, 2, (T - 1) * C)
    n_t = N // C
    vis = np.empty((C, n_baselines(S), 2, 2, 2), dtype=np.float64)
    z = np.empty((S, 2, n_t, C, 2), dtype=np.float64) if return_z else None
    de = None if delays_end is None else _f64(delays_end, (S,))
    rc = _load().oracle_process_subband_interp(S, C, T, N, bits, s.ctypes.data, _p(hist.view(np.float64)),
                                               _p(_f64(delays, (S,))), _p(de), _p(_f64(bandpass, (C,))), f_sb, f_s, _p(vis), _p(z))
    if rc:
        raise MemoryError("oracle_process_subband")
    return (_r2c(vis), _r2c(z)) if return_z else _r2c(vis)


def process(samples: np.ndarray, C: int, delays, bandpass, f_sb=None, hist: np.ndarray | None = None,
            f_s: float = F_S, T: int = TAPS) -> np.ndarray:
    """All subbands: samples [B][S][2][N][2] -> vis complex [B][C][n_bl][2][2].

    ``hist`` complex [B][S][2][(T-1)*C], updated in place when given."""
    B = samples.shape[0]
    out = []
    for sb in range(B):
        f = default_subband_frequency(sb) if f_sb is None else float(f_sb[sb])
        h = None if hist is None else hist[sb]
        out.append(process_subband(samples[sb], C, delays, bandpass, f, h, f_s, T))
    return np.stack(out)


def channel_direct(x: np.ndarray, C: int, j: int, hist: np.ndarray | None = None, delays=None, bandpass=None,
                   f_sb: float = 0.0, f_s: float = F_S, g: np.ndarray | None = None, T: int = TAPS):
    """Pin P11 / sampled full-size checks: channel j by the single-sum form.

    x complex (or integer [S][2][N][2]) -> (z_c complex [2S][n_t], vis_c complex [n_bl][2][2])."""
    if np.issubdtype(np.asarray(x).dtype, np.integer):
        xr = unpack(x)
    else:
        xr = _c2r(x)
    S, two, N = xr.shape[:3]
    if g is None:
        g = fir_prototype(C, T)
    if hist is None:
        hist = new_history(S, C, T)
    n_t = N // C
    zc = np.empty((2 * S, n_t, 2), dtype=np.float64)
    vc = np.empty((n_baselines(S), 2, 2, 2), dtype=np.float64)
    d = None if delays is None else _f64(delays, (S,))
    b = _f64(np.ones(C) if bandpass is None else bandpass, (C,))
    rc = _load().oracle_channel_direct(S, C, T, N, _p(np.ascontiguousarray(xr)), _p(_c2r(hist)),
                                       _p(_f64(g, (T * C,))), _p(d), _p(b), f_sb, f_s, j, _p(zc), _p(vc))
    if rc:
        raise MemoryError("oracle_channel_direct")
    return _r2c(zc), _r2c(vc)


# ------------------------------------------------------------------ SURVEY.md sec 8(f) rows 1-3
TILE = 64  # spectra per valid-sample tile and per dump granule (the correlator's time tile, readings A23 / A24)


def unpack4(packed: np.ndarray) -> np.ndarray:
    """uint8 [...] (re low nibble, im high nibble, 4-bit two's complement) -> float64 [..., 2] (reading A27)."""
    s = np.ascontiguousarray(packed, dtype=np.uint8)
    out = np.empty(s.shape + (2,), dtype=np.float64)
    _load().oracle_unpack_i4(s.ctypes.data, s.size, _p(out))
    return out


def coarse_shift(samples: np.ndarray, offsets, N: int) -> np.ndarray:
    """Reading A25 ("coarse delay compensation ... by shifting"): station a's block of N samples starts at sample
    offsets[a] of its (longer) input stream.  samples [S][2][N_in][2] -> [S][2][N][2]; pure indexing."""
    S = samples.shape[0]
    out = np.empty((S, 2, N, 2), dtype=samples.dtype)
    for a in range(S):
        o = int(offsets[a])
        assert 0 <= o and o + N <= samples.shape[2]
        out[a] = samples[a, :, o:o + N, :]
    return out


def pol_minor_to_planar(x: np.ndarray) -> np.ndarray:
    """Reading A26: LOFAR wire order [S][N][2 pol][2] (time-major, polarisation-minor) -> [S][2][N][2]; pure indexing."""
    return np.ascontiguousarray(np.swapaxes(x, 1, 2))


def phase_offsets(z: np.ndarray, phase0) -> np.ndarray:
    """z complex [S][2][n_t][C] -> z exp(-i phase0[a][p]) (reading A22)."""
    zr = _c2r(z).copy()
    S, _, n_t, C = zr.shape[:4]
    _load().oracle_phase_offsets(S, C, n_t, _p(_f64(phase0, (S, 2))), _p(zr))
    return _r2c(zr)


def flag_tiles(z: np.ndarray, valid) -> np.ndarray:
    """z complex [S][2][n_t][C], valid uint8 [S][ceil(n_t / 64)] -> z with the lost tiles zeroed (reading A24)."""
    zr = _c2r(z).copy()
    S, _, n_t, C = zr.shape[:4]
    v = np.ascontiguousarray(valid, dtype=np.uint8)
    assert v.shape == (S, (n_t + TILE - 1) // TILE)
    _load().oracle_flag_tiles(S, C, n_t, TILE, v.ctypes.data, _p(zr))
    return _r2c(zr)


def valid_counts(S: int, n_t: int, valid, dumps: int = 1) -> np.ndarray:
    """-> int64 [dumps][n_bl]: spectra of each dump in which both stations of the baseline are valid."""
    v = np.ascontiguousarray(valid, dtype=np.uint8)
    out = np.empty((dumps, n_baselines(S)), dtype=np.int64)
    _load().oracle_valid_counts(S, n_t, dumps, TILE, v.ctypes.data, out.ctypes.data)
    return out


def correlate_dumps(z: np.ndarray, dumps: int) -> np.ndarray:
    """z complex [S][2][n_t][C] -> vis complex [dumps][C][n_bl][2][2] (reading A23)."""
    zr = _c2r(z)
    S, two, n_t, C = zr.shape[:4]
    vis = np.empty((dumps, C, n_baselines(S), 2, 2, 2), dtype=np.float64)
    if _load().oracle_correlate_dumps(S, C, n_t, dumps, TILE, _p(zr), _p(vis)):
        raise ValueError("dumps must divide ceil(n_t / 64)")
    return _r2c(vis)


def process_subband_ext(samples: np.ndarray, C: int, delays, bandpass, f_sb: float, hist: np.ndarray | None = None,
                        f_s: float = F_S, T: int = TAPS, delays_end=None, phase0=None, valid=None, dumps: int = 1):
    """process_subband with the rows of SURVEY.md sec 8(f): per-(station, pol) phase offsets (A22), valid-sample
    flags (A24) and several dumps per block (A23).  samples int16/int8 [S][2][N][2] (or uint8 [S][2][N] 4-bit packed,
    A27) -> vis complex [dumps][C][n_bl][2][2]."""
    s = np.ascontiguousarray(samples)
    if s.dtype == np.uint8:
        x = _r2c(unpack4(s))
    else:
        x = _r2c(unpack(s))
    S = x.shape[0]
    z = fstage(x, C, hist=hist, delays=delays, bandpass=bandpass, f_sb=f_sb, f_s=f_s, T=T, delays_end=delays_end)
    if phase0 is not None:
        z = phase_offsets(z, phase0)
    if valid is not None:
        z = flag_tiles(z, valid)
    return correlate_dumps(z, dumps)


# ------------------------------------------------------------------ beamformer
def beamform_coherent(z: np.ndarray, beam_delays, f_sb: float, f_s: float = F_S) -> np.ndarray:
    """z complex [S][2][n_t][C], beam_delays [n_beams][S] seconds -> Y complex [n_beams][2][C][n_t] (reading A28)."""
    zr = _c2r(z)
    S, _, n_t, C = zr.shape[:4]
    bd = _f64(beam_delays)
    assert bd.ndim == 2 and bd.shape[1] == S
    y = np.empty((bd.shape[0], 2, C, n_t, 2), dtype=np.float64)
    _load().oracle_beamform_coherent(S, C, n_t, bd.shape[0], _p(bd), f_sb, f_s, _p(zr), _p(y))
    return _r2c(y)


def stokes(x: np.ndarray, y: np.ndarray, n_stokes: int = 4) -> np.ndarray:
    """x, y complex [...] -> float64 [n_stokes][...]: I, Q, U, V of the dual-polarisation sample (reading A29)."""
    assert n_stokes in (1, 4) and x.shape == y.shape
    xr, yr = _c2r(x), _c2r(y)
    out = np.empty((n_stokes,) + x.shape, dtype=np.float64)
    _load().oracle_stokes(x.size, _p(xr), _p(yr), n_stokes, _p(out))
    return out


def integrate(a: np.ndarray, t_int: int) -> np.ndarray:
    """float64 [..., n_t] -> [..., n_t // t_int]: sums of t_int consecutive samples, tail dropped (reading A30)."""
    a = _f64(a)
    n_t = a.shape[-1]
    out = np.empty(a.shape[:-1] + (n_t // t_int,), dtype=np.float64)
    _load().oracle_integrate(a.size // n_t if n_t else 0, n_t, t_int, _p(a), _p(out))
    return out


def coherent_stokes(z: np.ndarray, beam_delays, f_sb: float, n_stokes: int, t_int: int, f_s: float = F_S) -> np.ndarray:
    """z complex [S][2][n_t][C] -> float64 [n_beams][n_stokes][C][n_t // t_int] (A28 -> A29 -> A30)."""
    zr = _c2r(z)
    S, _, n_t, C = zr.shape[:4]
    bd = _f64(beam_delays)
    out = np.empty((bd.shape[0], n_stokes, C, n_t // t_int), dtype=np.float64)
    if _load().oracle_coherent_stokes(S, C, n_t, bd.shape[0], _p(bd), f_sb, f_s, _p(zr), n_stokes, t_int, _p(out)):
        raise MemoryError("oracle_coherent_stokes")
    return out


def incoherent_stokes(z: np.ndarray, n_stokes: int, t_int: int) -> np.ndarray:
    """z complex [S][2][n_t][C] -> float64 [n_stokes][C][n_t // t_int] (reading A31)."""
    zr = _c2r(z)
    S, _, n_t, C = zr.shape[:4]
    out = np.empty((n_stokes, C, n_t // t_int), dtype=np.float64)
    if _load().oracle_incoherent_stokes(S, C, n_t, _p(zr), n_stokes, t_int, _p(out)):
        raise MemoryError("oracle_incoherent_stokes")
    return out


def channelise_subband(samples: np.ndarray, C: int, delays, bandpass, f_sb: float, hist: np.ndarray | None = None,
                       f_s: float = F_S, T: int = TAPS, delays_end=None, phase0=None, valid=None) -> np.ndarray:
    """Steps 1-7 (+ A22 offsets, A24 flags) of one subband: integer samples [S][2][N][2] -> z complex [S][2][n_t][C]:
    the input of the beamformer functions above (reading A28: the beamformer of this build is fed by the correlator's
    channeliser; the paper's has one of its own)."""
    s = np.ascontiguousarray(samples)
    x = _r2c(unpack4(s)) if s.dtype == np.uint8 else _r2c(unpack(s))
    z = fstage(x, C, hist=hist, delays=delays, bandpass=bandpass, f_sb=f_sb, f_s=f_s, T=T, delays_end=delays_end)
    if phase0 is not None:
        z = phase_offsets(z, phase0)
    if valid is not None:
        z = flag_tiles(z, valid)
    return z
