"""Thin ctypes binding of libcobalt_b200.so (include/cobalt.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels under ``csrc/``; PyTorch supplies device
memory and streams.  There is no CPU fallback: ``load()`` raises when the shared library is
missing, and every entry point returns an error status without a B200-class device.

The functions ``cobalt_plan / cobalt_process / cobalt_process_host / cobalt_destroy / ...`` take
the same arguments as the C ABI (tensors or numpy arrays are turned into raw pointers);
``Correlator`` is a small convenience wrapper around them.
"""
from __future__ import annotations

import ctypes
import os

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libcobalt_b200.so")

COBALT_OK = 0
COBALT_ERR_BAD_ARG = -1
COBALT_ERR_NO_MEMORY = -2
COBALT_ERR_CUDA = -3
COBALT_ERR_UNSUPPORTED_DEVICE = -4
COBALT_MODE_TENSOR_FP16 = 0
COBALT_MODE_EXACT_FP32 = 1
COBALT_LAYOUT_PLANAR = 0
COBALT_LAYOUT_POL_MINOR = 1
COBALT_BF_COHERENT_VOLTAGES = 0
COBALT_BF_COHERENT_STOKES = 1
COBALT_BF_INCOHERENT_STOKES = 2
COBALT_NOALLOC_SCRATCH_BYTES = 16777216
COBALT_NOALLOC_MAX_SLICES = 4
COBALT_NOALLOC_MAX_CHANNEL_BASELINES = 131072

F_S = 195312.5

# every symbol include/cobalt.h declares (tests check the library exports exactly these)
ABI_SYMBOLS = (
    "cobalt_plan", "cobalt_process", "cobalt_process_interp", "cobalt_process_ex", "cobalt_process_host", "cobalt_destroy",
    "cobalt_set_subband_frequencies", "cobalt_set_sample_rate", "cobalt_set_mode",
    "cobalt_set_phase_offsets", "cobalt_set_coarse_delays", "cobalt_set_dumps", "cobalt_set_input_layout",
    "cobalt_set_chunk_subbands", "cobalt_reset", "cobalt_info", "cobalt_strerror", "cobalt_last_error",
    "cobalt_set_timing", "cobalt_get_timing", "cobalt_get_kernel_timing",
    "cobalt_debug_fir_weights", "cobalt_debug_unpack", "cobalt_debug_channelised", "cobalt_debug_correlate",
    "cobalt_beamform", "cobalt_beamform_output_bytes",
    "cobalt_correlate_noalloc", "cobalt_process_host_ex",
)


class CobaltError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = status
        super().__init__(f"cobalt status {status} ({_strerror(status)}){': ' + detail if detail else ''}")


class cobalt_info_t(ctypes.Structure):
    _fields_ = [
        ("stations", ctypes.c_int), ("subbands", ctypes.c_int), ("channels", ctypes.c_int), ("taps", ctypes.c_int),
        ("input_bits", ctypes.c_int), ("mode", ctypes.c_int),
        ("samples_per_integration", ctypes.c_longlong), ("n_spectra", ctypes.c_longlong),
        ("n_consumed", ctypes.c_longlong), ("n_baselines", ctypes.c_longlong),
        ("input_bytes", ctypes.c_longlong), ("output_bytes", ctypes.c_longlong), ("scratch_bytes", ctypes.c_longlong),
        ("chunk_subbands", ctypes.c_int), ("sm_count", ctypes.c_int), ("sample_rate_hz", ctypes.c_double),
        ("dumps", ctypes.c_int), ("n_tiles", ctypes.c_int), ("samples_allocated", ctypes.c_longlong),
    ]


class cobalt_io_t(ctypes.Structure):
    _fields_ = [
        ("samples", ctypes.c_void_p), ("delays", ctypes.c_void_p), ("delays_end", ctypes.c_void_p),
        ("bandpass", ctypes.c_void_p), ("valid", ctypes.c_void_p), ("visibilities", ctypes.c_void_p),
        ("valid_counts", ctypes.c_void_p),
    ]


class cobalt_bf_io_t(ctypes.Structure):
    _fields_ = [
        ("samples", ctypes.c_void_p), ("delays", ctypes.c_void_p), ("delays_end", ctypes.c_void_p),
        ("bandpass", ctypes.c_void_p), ("valid", ctypes.c_void_p), ("beam_delays", ctypes.c_void_p),
        ("n_beams", ctypes.c_int), ("product", ctypes.c_int), ("n_stokes", ctypes.c_int), ("t_int", ctypes.c_int),
        ("out", ctypes.c_void_p),
    ]


_lib = None
_vp = ctypes.c_void_p


def load(path: str | None = None):
    """dlopen the CUDA library.  Raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = ctypes.CDLL(path)
    lib.cobalt_plan.argtypes = [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                ctypes.c_longlong, ctypes.c_int]
    lib.cobalt_process.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
    lib.cobalt_process_interp.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.cobalt_process_ex.argtypes = [_vp, _vp, ctypes.POINTER(cobalt_io_t)]
    lib.cobalt_process_host.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.cobalt_process_host_ex.argtypes = [_vp, ctypes.POINTER(cobalt_io_t)]
    lib.cobalt_set_phase_offsets.argtypes = [_vp, _vp]
    lib.cobalt_set_coarse_delays.argtypes = [_vp, _vp, ctypes.c_longlong]
    lib.cobalt_set_dumps.argtypes = [_vp, ctypes.c_int]
    lib.cobalt_set_input_layout.argtypes = [_vp, ctypes.c_int]
    lib.cobalt_destroy.argtypes = [_vp]
    lib.cobalt_set_subband_frequencies.argtypes = [_vp, _vp]
    lib.cobalt_set_sample_rate.argtypes = [_vp, ctypes.c_double]
    lib.cobalt_set_mode.argtypes = [_vp, ctypes.c_int]
    lib.cobalt_set_chunk_subbands.argtypes = [_vp, ctypes.c_int]
    lib.cobalt_reset.argtypes = [_vp]
    lib.cobalt_info.argtypes = [_vp, ctypes.POINTER(cobalt_info_t)]
    lib.cobalt_strerror.argtypes = [ctypes.c_int]
    lib.cobalt_strerror.restype = ctypes.c_char_p
    lib.cobalt_last_error.argtypes = [_vp]
    lib.cobalt_last_error.restype = ctypes.c_char_p
    lib.cobalt_set_timing.argtypes = [_vp, ctypes.c_int]
    lib.cobalt_get_timing.argtypes = [_vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                      ctypes.POINTER(ctypes.c_int)]
    lib.cobalt_get_kernel_timing.argtypes = [_vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)]
    lib.cobalt_debug_fir_weights.argtypes = [_vp, _vp]
    lib.cobalt_debug_unpack.argtypes = [_vp, ctypes.c_int, _vp, ctypes.c_longlong, _vp]
    lib.cobalt_debug_channelised.argtypes = [_vp, _vp, _vp, _vp, _vp, ctypes.c_int, _vp]
    lib.cobalt_debug_correlate.argtypes = [_vp, _vp, _vp, _vp]
    lib.cobalt_beamform.argtypes = [_vp, _vp, ctypes.POINTER(cobalt_bf_io_t)]
    lib.cobalt_beamform_output_bytes.argtypes = [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib.cobalt_beamform_output_bytes.restype = ctypes.c_longlong
    lib.cobalt_correlate_noalloc.argtypes = [_vp, _vp, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, _vp, ctypes.c_char_p, ctypes.c_int]
    for name in ABI_SYMBOLS:
        fn = getattr(lib, name)
        if name not in ("cobalt_strerror", "cobalt_last_error", "cobalt_beamform_output_bytes"):
            fn.restype = ctypes.c_int
    _lib = lib
    return lib


def _strerror(status: int) -> str:
    try:
        return load().cobalt_strerror(status).decode()
    except Exception:  # library missing: still give a readable message
        return "?"


def _ptr(x):
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream_ptr(stream):
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(status: int, plan=None):
    if status != COBALT_OK:
        detail = load().cobalt_last_error(plan).decode() if _lib is not None else ""
        raise CobaltError(status, detail)


# ------------------------------------------------------------------ C ABI, same names
def cobalt_plan(stations, subbands, channels, taps, samples_per_integration, input_bits):
    h = _vp()
    _check(load().cobalt_plan(ctypes.byref(h), stations, subbands, channels, taps, samples_per_integration, input_bits))
    return h


def cobalt_process(plan, stream, d_samples, d_delays, d_bandpass, d_visibilities):
    _check(load().cobalt_process(plan, _stream_ptr(stream), _ptr(d_samples), _ptr(d_delays), _ptr(d_bandpass),
                                 _ptr(d_visibilities)), plan)


def cobalt_process_interp(plan, stream, d_samples, d_delays_begin, d_delays_end, d_bandpass, d_visibilities):
    _check(load().cobalt_process_interp(plan, _stream_ptr(stream), _ptr(d_samples), _ptr(d_delays_begin), _ptr(d_delays_end),
                                        _ptr(d_bandpass), _ptr(d_visibilities)), plan)


def cobalt_process_ex(plan, stream, d_samples, d_delays, d_bandpass, d_visibilities, d_delays_end=None, d_valid=None,
                      d_valid_counts=None):
    io = cobalt_io_t(_ptr(d_samples), _ptr(d_delays), _ptr(d_delays_end), _ptr(d_bandpass), _ptr(d_valid), _ptr(d_visibilities),
                     _ptr(d_valid_counts))
    _check(load().cobalt_process_ex(plan, _stream_ptr(stream), ctypes.byref(io)), plan)


def cobalt_process_host(plan, h_samples, h_delays, h_bandpass, h_visibilities):
    _check(load().cobalt_process_host(plan, _ptr(h_samples), _ptr(h_delays), _ptr(h_bandpass), _ptr(h_visibilities)), plan)


def cobalt_process_host_ex(plan, h_samples, h_delays, h_bandpass, h_visibilities, h_delays_end=None, h_valid=None, h_valid_counts=None):
    io = cobalt_io_t(_ptr(h_samples), _ptr(h_delays), _ptr(h_delays_end), _ptr(h_bandpass), _ptr(h_valid), _ptr(h_visibilities),
                     _ptr(h_valid_counts))
    _check(load().cobalt_process_host_ex(plan, ctypes.byref(io)), plan)


def cobalt_beamform(plan, stream, d_samples, d_delays, d_bandpass, d_beam_delays, n_beams, product, n_stokes, t_int, d_out,
                    d_delays_end=None, d_valid=None):
    io = cobalt_bf_io_t(_ptr(d_samples), _ptr(d_delays), _ptr(d_delays_end), _ptr(d_bandpass), _ptr(d_valid), _ptr(d_beam_delays),
                        int(n_beams), int(product), int(n_stokes), int(t_int), _ptr(d_out))
    _check(load().cobalt_beamform(plan, _stream_ptr(stream), ctypes.byref(io)), plan)


def cobalt_correlate_noalloc(stream, d_z, stations, channels, n_spectra, d_vis):
    """Steps a8-a9 of one subband for callers that must not allocate device memory (a running real-time pipeline, a host
    application with its own memory pool): no plan, fp32, partial sums in a fixed 16 MiB array inside the library.
    d_z [C][2S][n_t] complex64 -> d_vis [C][n_bl][2][2] complex64, both device memory of the caller;
    channels * n_bl <= COBALT_NOALLOC_MAX_CHANNEL_BASELINES.  Calls that overlap on the GPU race on that array."""
    err = ctypes.create_string_buffer(512)
    status = load().cobalt_correlate_noalloc(_stream_ptr(stream), _ptr(d_z), int(stations), int(channels), int(n_spectra),
                                             _ptr(d_vis), err, len(err))
    if status != COBALT_OK:
        raise CobaltError(status, err.value.decode())


def cobalt_destroy(plan):
    _check(load().cobalt_destroy(plan))


def cobalt_info(plan) -> cobalt_info_t:
    info = cobalt_info_t()
    _check(load().cobalt_info(plan, ctypes.byref(info)), plan)
    return info


class Correlator:
    """Owns one cobalt_plan.  Tensors are torch CUDA tensors (device memory + streams only)."""

    def __init__(self, stations, subbands, channels, samples_per_integration, input_bits=16, taps=16, mode=None):
        self._h = cobalt_plan(stations, subbands, channels, taps, samples_per_integration, input_bits)
        if mode is not None:
            self.set_mode(mode)
        self.info = cobalt_info(self._h)

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None:
            import torch

            torch.cuda.synchronize()
            cobalt_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- settings
    def set_mode(self, mode):
        _check(load().cobalt_set_mode(self._h, mode), self._h)
        self.info = cobalt_info(self._h)

    def set_chunk_subbands(self, chunk):
        _check(load().cobalt_set_chunk_subbands(self._h, chunk), self._h)
        self.info = cobalt_info(self._h)

    def set_subband_frequencies(self, hz):
        import numpy as np

        a = np.ascontiguousarray(hz, dtype=np.float64)
        assert a.shape == (self.info.subbands,)
        _check(load().cobalt_set_subband_frequencies(self._h, a.ctypes.data), self._h)

    def set_sample_rate(self, hz):
        _check(load().cobalt_set_sample_rate(self._h, float(hz)), self._h)

    def set_phase_offsets(self, phase0):
        """phase0: [S][2] radians (host), or None to clear (reading A22)."""
        import numpy as np

        if phase0 is None:
            _check(load().cobalt_set_phase_offsets(self._h, None), self._h)
            return
        a = np.ascontiguousarray(phase0, dtype=np.float64)
        assert a.shape == (self.info.stations, 2)
        _check(load().cobalt_set_phase_offsets(self._h, a.ctypes.data), self._h)

    def set_coarse_delays(self, offsets, samples_allocated=0):
        """offsets: [S] first sample of each station's block (host ints), or None to clear (reading A25)."""
        import numpy as np

        if offsets is None:
            _check(load().cobalt_set_coarse_delays(self._h, None, 0), self._h)
        else:
            a = np.ascontiguousarray(offsets, dtype=np.int32)
            assert a.shape == (self.info.stations,)
            _check(load().cobalt_set_coarse_delays(self._h, a.ctypes.data, int(samples_allocated)), self._h)
        self.info = cobalt_info(self._h)

    def set_dumps(self, dumps):
        _check(load().cobalt_set_dumps(self._h, int(dumps)), self._h)
        self.info = cobalt_info(self._h)

    def set_input_layout(self, layout):
        _check(load().cobalt_set_input_layout(self._h, int(layout)), self._h)
        self.info = cobalt_info(self._h)

    def reset(self):
        _check(load().cobalt_reset(self._h), self._h)

    def set_timing(self, enabled=True):
        _check(load().cobalt_set_timing(self._h, int(enabled)), self._h)

    def get_timing(self):
        f, x, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_int()
        _check(load().cobalt_get_timing(self._h, ctypes.byref(f), ctypes.byref(x), ctypes.byref(n)), self._h)
        return f.value, x.value, n.value

    def get_kernel_timing(self):
        """(phase-table ms, F-stage ms, history ms, X-stage ms, kernel launches) of the last process() call."""
        ms, n = (ctypes.c_double * 4)(), ctypes.c_int()
        _check(load().cobalt_get_kernel_timing(self._h, ms, ctypes.byref(n)), self._h)
        return ms[0], ms[1], ms[2], ms[3], n.value

    # -- the hot path
    def vis_shape(self):
        i = self.info
        one = (i.subbands, i.channels, i.n_baselines, 2, 2)
        return one if i.dumps == 1 else (i.dumps,) + one

    def samples_shape(self, layout=COBALT_LAYOUT_PLANAR):
        """Shape of the sample tensor the plan expects (4-bit: uint8, one byte per complex sample, no trailing axis)."""
        i = self.info
        n = i.samples_allocated
        s = (i.subbands, i.stations, 2, n) if layout == COBALT_LAYOUT_PLANAR else (i.subbands, i.stations, n, 2)
        return s if i.input_bits == 4 else s + (2,)

    def process(self, samples, delays, bandpass, out=None, stream=None, delays_end=None, valid=None, valid_counts=None,
                layout=COBALT_LAYOUT_PLANAR):
        """samples int16/int8 [B][S][2][N][2], delays float64 [S], bandpass float32 [C] (CUDA tensors)
        -> complex64 [B][C][n_bl][2][2].  Enqueues on ``stream`` (default: torch's current stream).
        ``delays_end`` (float64 [S]) selects cobalt_process_interp: the delay runs linearly from ``delays`` at the first
        spectrum to ``delays_end`` at the end of the block."""
        import torch

        i = self.info
        want = {16: torch.int16, 8: torch.int8, 4: torch.uint8}[i.input_bits]
        assert samples.is_cuda and samples.is_contiguous() and samples.dtype == want
        assert tuple(samples.shape) == self.samples_shape(layout), (tuple(samples.shape), self.samples_shape(layout))
        assert delays.is_cuda and delays.dtype == torch.float64 and delays.is_contiguous() and delays.numel() == i.stations
        assert bandpass.is_cuda and bandpass.dtype == torch.float32 and bandpass.is_contiguous() and bandpass.numel() == i.channels
        if out is None:
            out = torch.empty(self.vis_shape(), dtype=torch.complex64, device=samples.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.complex64 and tuple(out.shape) == self.vis_shape()
        if valid is not None:
            assert valid.is_cuda and valid.dtype == torch.uint8 and valid.is_contiguous()
            assert tuple(valid.shape) == (i.subbands, i.stations, i.n_tiles)
        if valid_counts is not None:
            assert valid_counts.is_cuda and valid_counts.dtype == torch.int32 and valid_counts.is_contiguous()
            assert tuple(valid_counts.shape) == (i.subbands, i.dumps, i.n_baselines)
        if delays_end is not None:
            assert delays_end.is_cuda and delays_end.dtype == torch.float64 and delays_end.is_contiguous() and delays_end.numel() == i.stations
        if valid is None and valid_counts is None and i.dumps == 1:
            if delays_end is None:
                cobalt_process(self._h, stream, samples, delays, bandpass, out)
            else:
                cobalt_process_interp(self._h, stream, samples, delays, delays_end, bandpass, out)
        else:
            cobalt_process_ex(self._h, stream, samples, delays, bandpass, out, delays_end, valid, valid_counts)
        return out

    def beamform_shape(self, product, n_beams=1, n_stokes=1, t_int=1):
        """Shape and dtype name of the output of ``beamform`` (reading A32)."""
        i = self.info
        if product == COBALT_BF_COHERENT_VOLTAGES:
            return (i.subbands, n_beams, 2, i.channels, i.n_spectra), "complex64"
        n_out = i.n_spectra // t_int
        if product == COBALT_BF_COHERENT_STOKES:
            return (i.subbands, n_beams, n_stokes, i.channels, n_out), "float32"
        return (i.subbands, n_stokes, i.channels, n_out), "float32"

    def beamform(self, samples, delays, bandpass, product, beam_delays=None, n_stokes=1, t_int=1, out=None, stream=None,
                 delays_end=None, valid=None, layout=COBALT_LAYOUT_PLANAR):
        """cobalt_beamform: samples, delays, bandpass as in ``process``; beam_delays float64
        [n_beams][S] (CUDA) for the coherent products.  Returns the output tensor (see ``beamform_shape``)."""
        import torch

        i = self.info
        want = {16: torch.int16, 8: torch.int8, 4: torch.uint8}[i.input_bits]
        assert samples.is_cuda and samples.is_contiguous() and samples.dtype == want
        assert tuple(samples.shape) == self.samples_shape(layout), (tuple(samples.shape), self.samples_shape(layout))
        assert delays.is_cuda and delays.dtype == torch.float64 and delays.is_contiguous() and delays.numel() == i.stations
        assert bandpass.is_cuda and bandpass.dtype == torch.float32 and bandpass.is_contiguous() and bandpass.numel() == i.channels
        n_beams = 1
        if product != COBALT_BF_INCOHERENT_STOKES:
            assert beam_delays.is_cuda and beam_delays.dtype == torch.float64 and beam_delays.is_contiguous()
            assert beam_delays.dim() == 2 and beam_delays.shape[1] == i.stations
            n_beams = beam_delays.shape[0]
        shape, dt = self.beamform_shape(product, n_beams, n_stokes, t_int)
        if out is None:
            out = torch.empty(shape, dtype=getattr(torch, dt), device=samples.device)
        assert out.is_cuda and out.is_contiguous() and tuple(out.shape) == shape and out.dtype == getattr(torch, dt)
        nbytes = load().cobalt_beamform_output_bytes(self._h, n_beams, product, n_stokes, t_int)
        assert nbytes == out.numel() * out.element_size(), (nbytes, out.numel() * out.element_size())
        cobalt_beamform(self._h, stream, samples, delays, bandpass, beam_delays, n_beams, product, n_stokes, t_int, out,
                        delays_end, valid)
        return out

    def process_host(self, samples, delays, bandpass, out, delays_end=None, valid=None, valid_counts=None):
        """Host buffers (numpy arrays or pinned CPU tensors), same layouts; synchronous.  The optional arrays select
        cobalt_process_host_ex (also used when the plan writes several dumps per block)."""
        i = self.info
        sizes = [(samples, i.input_bytes), (delays, 8 * i.stations), (bandpass, 4 * i.channels), (out, i.output_bytes)]
        if delays_end is not None:
            sizes.append((delays_end, 8 * i.stations))
        if valid is not None:
            sizes.append((valid, i.subbands * i.stations * i.n_tiles))
        if valid_counts is not None:
            sizes.append((valid_counts, 4 * i.subbands * i.dumps * i.n_baselines))
        for a, nbytes in sizes:
            n = a.numel() * a.element_size() if hasattr(a, "numel") else a.nbytes
            assert n == nbytes, (n, nbytes)
        if delays_end is None and valid is None and valid_counts is None:
            cobalt_process_host(self._h, samples, delays, bandpass, out)
        else:
            cobalt_process_host_ex(self._h, samples, delays, bandpass, out, delays_end, valid, valid_counts)
        return out

    # -- debug taps
    def fir_weights(self):
        import numpy as np

        w = np.empty((16, self.info.channels), dtype=np.float32)
        _check(load().cobalt_debug_fir_weights(self._h, w.ctypes.data), self._h)
        return w

    def channelised(self, samples, delays, bandpass, sb=0, stream=None):
        import torch

        i = self.info
        z = torch.empty((i.channels, 2 * i.stations, i.n_spectra), dtype=torch.complex64, device=samples.device)
        _check(load().cobalt_debug_channelised(self._h, _stream_ptr(stream), samples.data_ptr(), delays.data_ptr(),
                                               bandpass.data_ptr(), sb, z.data_ptr()), self._h)
        return z

    def correlate(self, z, stream=None):
        import torch

        i = self.info
        assert z.is_cuda and z.is_contiguous() and z.dtype == torch.complex64
        assert tuple(z.shape) == (i.channels, 2 * i.stations, i.n_spectra)
        shape = (i.channels, i.n_baselines, 2, 2)
        vis = torch.empty(shape if i.dumps == 1 else (i.dumps,) + shape, dtype=torch.complex64, device=z.device)
        _check(load().cobalt_debug_correlate(self._h, _stream_ptr(stream), z.data_ptr(), vis.data_ptr()), self._h)
        return vis


def unpack(x, stream=None):
    """Step a1 alone: int16/int8 CUDA tensor -> float32 CUDA tensor of the same shape; uint8 (4-bit packed complex
    samples, reading A27) -> float32 [..., 2]."""
    import torch

    assert x.is_cuda and x.is_contiguous() and x.dtype in (torch.int16, torch.int8, torch.uint8)
    out = torch.empty(x.shape + (2,) if x.dtype == torch.uint8 else x.shape, dtype=torch.float32, device=x.device)
    bits = 16 if x.dtype == torch.int16 else 8 if x.dtype == torch.int8 else 4
    _check(load().cobalt_debug_unpack(_stream_ptr(stream), bits, x.data_ptr(), x.numel(), out.data_ptr()))
    return out
