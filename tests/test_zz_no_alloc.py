"""cobalt_correlate_noalloc: the one entry point of the library that allocates nothing.

Some users of a correlator library cannot allocate device memory when they call it: the paper's pipeline takes all its
buffers from pools filled before the observation starts and then runs against a real-time deadline, where a
cudaMalloc / cudaFree would synchronise the whole device and cost a block of antenna data, or simply fail on a
GPU whose memory is already handed out; a plug-in inside an application with its own device-memory pool is in the same
position.  For them the library keeps a fixed 16 MiB array in its device image and runs the split X-stage (partial
visibilities per time slice, then their sum) out of it.  These tests check that entry point against the path everybody
else uses (cobalt_plan + cobalt_debug_correlate in COBALT_MODE_EXACT_FP32, which allocates its scratch), at the fp32
tolerance of the other parity tests, on calls that follow each other directly on one stream -- the shared array keeps
whatever the previous call wrote, so a second call with another shape is the case that would expose a dependence on it.

The file is named test_zz_* so that pytest collects it after every other test file: with `-x` a failure here must not
hide the parity tests.  It has to pass alone in a fresh process (its first call then does the per-device set-up) and after
the rest of the suite (the library is already loaded and other kernels have run).
"""
import ctypes

import numpy as np
import pytest

from parity_util import TOL_FP32, err_fp32


def _z(torch, C, S, n_t, seed):
    """Seeded complex64 [C][2S][n_t] with station-to-station correlation (a common signal plus noise), on the GPU."""
    g = torch.Generator(device="cpu").manual_seed(seed)
    common = torch.randn(C, 1, n_t, 2, generator=g)
    noise = torch.randn(C, 2 * S, n_t, 2, generator=g)
    gain = torch.rand(1, 2 * S, 1, 1, generator=g) + 0.5
    z = torch.view_as_complex(((0.7 * common + noise) * gain * 100.0).contiguous())
    return z.to(torch.complex64).cuda().contiguous()


def _existing_path(cobalt, torch, z, S, C, n_t):
    """The allocating path: a plan in EXACT_FP32 mode and its correlate tap (single pass over the time range)."""
    with cobalt.Correlator(S, 1, C, C * n_t, 16, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        assert cor.info.n_spectra == n_t
        v = cor.correlate(z)
        torch.cuda.synchronize()
        return v.cpu().numpy()


@pytest.mark.gpu
def test_noalloc_matches_the_allocating_path_on_consecutive_calls(cobalt):
    import torch

    n_bl = lambda S: S * (S + 1) // 2
    # (S, C, n_t): 4 slices with a ragged tail and several 32-row tiles; then a much smaller problem with 2 slices that
    # re-uses the front of the array the first call filled; then 1 slice; then the largest size the array admits at C = 256
    shapes = [(48, 64, 300), (5, 16, 70), (3, 16, 9), (31, 256, 130)]
    inputs = [_z(torch, C, S, n_t, 1000 + i) for i, (S, C, n_t) in enumerate(shapes)]
    outs = [torch.full((C, n_bl(S), 2, 2), float("nan"), dtype=torch.complex64, device="cuda") for (S, C, n_t) in shapes]
    # all calls back to back on the current stream, nothing in between: no synchronisation, no allocation by the library
    for (S, C, n_t), z, v in zip(shapes, inputs, outs):
        cobalt.cobalt_correlate_noalloc(None, z, S, C, n_t, v)
    # and the first problem once more into a fresh buffer: what the calls in between left in the array must not matter
    again = torch.full_like(outs[0], float("nan"))
    cobalt.cobalt_correlate_noalloc(None, inputs[0], *shapes[0], again)
    torch.cuda.synchronize()
    for (S, C, n_t), z, v in zip(shapes, inputs, outs):
        got = v.cpu().numpy()
        assert np.isfinite(got.view(np.float32)).all(), (S, C, n_t)         # every element was written
        want = _existing_path(cobalt, torch, z, S, C, n_t)
        err = err_fp32(got, want)
        assert err <= TOL_FP32, (S, C, n_t, err)
    assert np.array_equal(again.cpu().numpy().view(np.float32), outs[0].cpu().numpy().view(np.float32))


@pytest.mark.gpu
def test_noalloc_matches_the_oracle(cobalt, oracle):
    """The same entry point against the float64 oracle's correlate (P7-pinned), at the EXACT_FP32 tolerance."""
    import torch

    S, C, n_t = 6, 16, 200
    z = _z(torch, C, S, n_t, 77)
    v = torch.empty((C, S * (S + 1) // 2, 2, 2), dtype=torch.complex64, device="cuda")
    cobalt.cobalt_correlate_noalloc(None, z, S, C, n_t, v)
    torch.cuda.synchronize()
    zc = z.cpu().numpy().astype(np.complex128)                                          # [C][2 S][n_t]
    want = oracle.correlate(np.ascontiguousarray(zc.reshape(C, S, 2, n_t).transpose(1, 2, 3, 0)))   # the oracle takes [S][2][n_t][C]
    assert err_fp32(v.cpu().numpy(), want) <= TOL_FP32


def test_noalloc_rejects_sizes_beyond_the_array(cobalt):
    """Runs without a GPU: sizes are checked before the device is touched, and the message carries the numbers."""
    lib = cobalt.load()
    err = ctypes.create_string_buffer(512)
    assert cobalt.COBALT_NOALLOC_MAX_CHANNEL_BASELINES * cobalt.COBALT_NOALLOC_MAX_SLICES * 32 == cobalt.COBALT_NOALLOC_SCRATCH_BYTES
    for S, C in ((64, 64), (32, 256), (512, 16)):
        assert C * S * (S + 1) // 2 > cobalt.COBALT_NOALLOC_MAX_CHANNEL_BASELINES
        rc = lib.cobalt_correlate_noalloc(None, 256, S, C, 100, 256, err, len(err))
        assert rc == cobalt.COBALT_ERR_BAD_ARG
        assert b"too large" in err.value and str(C * S * (S + 1) // 2).encode() in err.value
    for args in ((None, 0, 4, 16, 100, 256), (None, 256, 4, 16, 100, 0), (None, 256, 0, 16, 100, 256), (None, 256, 4, 32, 100, 256),
                 (None, 256, 4, 16, 0, 256), (None, 260, 4, 16, 100, 256), (None, 256, 4, 16, 100, 260)):
        assert lib.cobalt_correlate_noalloc(*args, err, len(err)) == cobalt.COBALT_ERR_BAD_ARG, args
        assert err.value
    assert lib.cobalt_correlate_noalloc(None, 0, 4, 16, 100, 256, None, 0) == cobalt.COBALT_ERR_BAD_ARG   # no buffer: still no crash
    with pytest.raises(cobalt.CobaltError) as e:
        cobalt.cobalt_correlate_noalloc(0, 256, 64, 64, 100, 256)
    assert e.value.status == cobalt.COBALT_ERR_BAD_ARG and "COBALT_NOALLOC_MAX_CHANNEL_BASELINES" in str(e.value)
