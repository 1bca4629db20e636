"""GPU parity for SURVEY.md sec 8(f) row 4, the beamformer (readings A28-A32): cobalt_beamform through the C
ABI against the float64 oracle on the same seeded integers, element by element, in both modes: coherent complex voltages,
coherent Stokes I / IQUV with time integration, incoherent Stokes; with bandpass, delays, phase offsets, lost tiles,
several subbands per launch group and across two calls (history carry)."""
import numpy as np
import pytest

from parity_util import TOL_FP32, TOL_TENSOR

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run through gpurun)")
    return torch.device("cuda:0")


def _mode(cobalt, tensor):
    return cobalt.COBALT_MODE_TENSOR_FP16 if tensor else cobalt.COBALT_MODE_EXACT_FP32


def _err(got, want, chan_axis):
    """max over (subband, channel) of ||d||_F / ||want||_F; `got`, `want` [B][...] with the channel at chan_axis."""
    axes = tuple(i for i in range(1, want.ndim) if i != chan_axis)
    num = np.sqrt((np.abs(got - want) ** 2).sum(axis=axes))
    den = np.sqrt((np.abs(want) ** 2).sum(axis=axes))
    assert np.all(den > 0)
    return float((num / den).max())


def _check(got, want, chan_axis, tensor, what):
    assert got.shape == want.shape, (got.shape, want.shape)
    assert np.all(np.isfinite(got)), what
    e = _err(got, want, chan_axis)
    tol = TOL_TENSOR if tensor else TOL_FP32
    assert e <= tol, f"{what}: error {e:.3e} > {tol}"


def _data(rng, B, S, N, bits):
    lim = 2000 if bits == 16 else 100
    x = rng.integers(-lim, lim + 1, size=(B, S, 2, N, 2))
    c = rng.integers(-lim // 2, lim // 2 + 1, size=(B, 1, 1, N, 2))      # a common signal: the beams are not pure noise
    return np.clip(x // 2 + c, -lim, lim).astype(np.int16 if bits == 16 else np.int8)


def _oracle_z(oracle, x, C, delays, bp, hist=None, phase0=None, valid=None):
    B = x.shape[0]
    return [oracle.channelise_subband(x[b], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(b),
                                      hist=None if hist is None else hist[b], phase0=phase0,
                                      valid=None if valid is None else valid[b]) for b in range(B)]


@pytest.mark.parametrize("C,bits,S,n_t,n_beams", [
    (16, 16, 3, 130, 5),        # one row group, one beam block, ragged last 128-spectrum block
    (64, 16, 5, 200, 70),       # two beam blocks (64 per block at this size), two k-tiles in the last block
    (256, 8, 4, 70, 3),         # one-and-a-bit k-tiles
    (64, 16, 48, 330, 17),      # the paper's beamformer array (48 core stations): 12 k-steps, odd number of k-tiles
    (16, 16, 77, 128, 9),       # full array: 20 k-steps, narrower beam blocks
])
@pytest.mark.parametrize("tensor", [False, True])
def test_coherent_voltages_match_oracle(cobalt, oracle, dev, C, bits, S, n_t, n_beams, tensor):
    rng = np.random.default_rng(2800 + C + S)
    B, N = 2, n_t * C + 3
    x = _data(rng, B, S, N, bits)
    delays = rng.uniform(-20e-6, 20e-6, S)
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    bd = rng.uniform(-40e-9, 40e-9, (n_beams, S))
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        got = cor.beamform(torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev),
                           cobalt.COBALT_BF_COHERENT_VOLTAGES, beam_delays=torch.from_numpy(bd).to(dev))
        torch.cuda.synchronize()
        got = got.cpu().numpy()
    z = _oracle_z(oracle, x, C, delays, bp)
    want = np.stack([oracle.beamform_coherent(z[b], bd, oracle.default_subband_frequency(b)) for b in range(B)])
    _check(got, want, 3, tensor, "coherent voltages")


@pytest.mark.parametrize("C,S,n_t,n_beams,n_stokes,t_int", [
    (16, 3, 130, 5, 4, 1), (16, 3, 130, 5, 1, 4), (64, 6, 260, 9, 4, 16), (64, 6, 260, 9, 1, 32),
    (16, 4, 400, 3, 4, 64), (16, 4, 400, 3, 4, 128), (256, 48, 70, 6, 4, 2), (64, 5, 200, 70, 1, 8),
])
@pytest.mark.parametrize("tensor", [False, True])
def test_coherent_stokes_match_oracle(cobalt, oracle, dev, C, S, n_t, n_beams, n_stokes, t_int, tensor):
    rng = np.random.default_rng(2900 + C + S + t_int)
    B, N, bits = 2, n_t * C, 16
    x = _data(rng, B, S, N, bits)
    delays = rng.uniform(-20e-6, 20e-6, S)
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    bd = rng.uniform(-40e-9, 40e-9, (n_beams, S))
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        got = cor.beamform(torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev),
                           cobalt.COBALT_BF_COHERENT_STOKES, beam_delays=torch.from_numpy(bd).to(dev), n_stokes=n_stokes, t_int=t_int)
        torch.cuda.synchronize()
        got = got.cpu().numpy()
    z = _oracle_z(oracle, x, C, delays, bp)
    want = np.stack([oracle.coherent_stokes(z[b], bd, oracle.default_subband_frequency(b), n_stokes, t_int) for b in range(B)])
    assert want.shape[-1] == n_t // t_int
    _check(got, want, 3, tensor, f"coherent Stokes, n_stokes {n_stokes}, t_int {t_int}")


@pytest.mark.parametrize("C,bits,S,n_t,n_stokes,t_int", [(16, 16, 3, 130, 4, 1), (64, 8, 7, 260, 4, 16), (256, 16, 48, 70, 1, 64),
                                                         (64, 16, 77, 300, 4, 128)])
@pytest.mark.parametrize("tensor", [False, True])
def test_incoherent_stokes_match_oracle(cobalt, oracle, dev, C, bits, S, n_t, n_stokes, t_int, tensor):
    rng = np.random.default_rng(3000 + C + S)
    B, N = 2, n_t * C + 1
    x = _data(rng, B, S, N, bits)
    delays = rng.uniform(-20e-6, 20e-6, S)
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))                     # the relative X-Y phase of a station turns its U and V
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_phase_offsets(ph0)
        got = cor.beamform(torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev),
                           cobalt.COBALT_BF_INCOHERENT_STOKES, n_stokes=n_stokes, t_int=t_int)
        torch.cuda.synchronize()
        got = got.cpu().numpy()
    z = _oracle_z(oracle, x, C, delays, bp, phase0=ph0)
    want = np.stack([oracle.incoherent_stokes(z[b], n_stokes, t_int) for b in range(B)])
    _check(got, want, 2, tensor, "incoherent Stokes")


@pytest.mark.parametrize("tensor", [False, True])
def test_every_input_option_and_two_calls(cobalt, oracle, dev, tensor):
    """Phase offsets, lost tiles, one subband per launch group, and a second call that continues from the first call's FIR
    history: in this build the beamformer is fed by the correlator's steps a1-a7 (reading A28; the paper's beamformer has a
    channeliser of its own)."""
    rng = np.random.default_rng(3100)
    B, S, C, n_t, bits, n_beams = 3, 6, 64, 192, 16, 7
    N = n_t * C
    delays = rng.uniform(-20e-6, 20e-6, S)
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    bd = rng.uniform(-40e-9, 40e-9, (n_beams, S))
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))
    hist = [oracle.new_history(S, C) for _ in range(B)]
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_chunk_subbands(1)
        cor.set_phase_offsets(ph0)
        for call in range(2):
            x = _data(rng, B, S, N, bits)
            valid = (rng.uniform(size=(B, S, cor.info.n_tiles)) > 0.3).astype(np.uint8)
            args = (torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev))
            got = cor.beamform(*args, cobalt.COBALT_BF_COHERENT_STOKES, beam_delays=torch.from_numpy(bd).to(dev), n_stokes=4,
                               t_int=8, valid=torch.from_numpy(valid).to(dev))
            torch.cuda.synchronize()
            got = got.cpu().numpy()
            z = _oracle_z(oracle, x, C, delays, bp, hist=hist, phase0=ph0, valid=valid)
            want = np.stack([oracle.coherent_stokes(z[b], bd, oracle.default_subband_frequency(b), 4, 8) for b in range(B)])
            _check(got, want, 3, tensor, f"call {call}")


def test_point_source_coherent_gain_on_gpu(cobalt, oracle, dev):
    """GPU version of pin P25: a common source with per-station geometric delays; the beam that cancels them collects ~S x
    the incoherent power, a beam several cycles off collects far less."""
    rng = np.random.default_rng(3200)
    S, C, n_t = 8, 16, 256
    N, F_S = C * n_t, 195312.5
    f_sb = oracle.default_subband_frequency(0)
    src = (rng.standard_normal(N + 64) + 1j * rng.standard_normal(N + 64)) * 300.0
    geo = rng.uniform(0, 4.0e-6, S)
    freqs = np.fft.fftfreq(N + 64, d=1.0 / F_S)
    x = np.empty((1, S, 2, N, 2), dtype=np.int16)
    for a in range(S):
        d = np.fft.ifft(np.fft.fft(src) * np.exp(-2j * np.pi * (freqs + f_sb) * geo[a]))[32:32 + N]
        x[0, a, 0, :, 0], x[0, a, 0, :, 1] = np.rint(d.real), np.rint(d.imag)
        x[0, a, 1] = x[0, a, 0] // 2
    bd = np.stack([-geo, -geo + rng.uniform(-3e-8, 3e-8, S)])
    with cobalt.Correlator(S, 1, C, N, 16) as cor:
        args = (torch.from_numpy(x).to(dev), torch.zeros(S, dtype=torch.float64, device=dev), torch.ones(C, dtype=torch.float32, device=dev))
        coh = cor.beamform(*args, cobalt.COBALT_BF_COHERENT_STOKES, beam_delays=torch.from_numpy(bd).to(dev), n_stokes=1, t_int=64).cpu().numpy()
        cor.reset()
        inc = cor.beamform(*args, cobalt.COBALT_BF_INCOHERENT_STOKES, n_stokes=1, t_int=64).cpu().numpy()
    coh, inc = coh[0, :, 0, 2:C - 2, 1:], inc[0, 0, 2:C - 2, 1:]
    assert 0.97 * S < coh[0].sum() / inc.sum() <= S * 1.001
    assert coh[1].sum() / inc.sum() < 0.5 * S


def test_beamform_rejects_bad_settings(cobalt, dev):
    S, C, N = 3, 16, 16 * 64
    with cobalt.Correlator(S, 1, C, N, 16) as cor:
        x = torch.zeros(cor.samples_shape(), dtype=torch.int16, device=dev)
        d = torch.zeros(S, dtype=torch.float64, device=dev)
        b = torch.ones(C, dtype=torch.float32, device=dev)
        bd = torch.zeros((2, S), dtype=torch.float64, device=dev)
        out = torch.empty(1 << 16, dtype=torch.float32, device=dev)
        for kw in (dict(product=cobalt.COBALT_BF_COHERENT_STOKES, n_stokes=2, t_int=4), dict(product=cobalt.COBALT_BF_COHERENT_STOKES, n_stokes=4, t_int=3),
                   dict(product=cobalt.COBALT_BF_COHERENT_STOKES, n_stokes=4, t_int=256), dict(product=7, n_stokes=1, t_int=1),
                   dict(product=cobalt.COBALT_BF_INCOHERENT_STOKES, n_stokes=1, t_int=128)):      # n_t = 64 < t_int: no output sample
            with pytest.raises(cobalt.CobaltError) as ei:
                cobalt.cobalt_beamform(cor._h, None, x, d, b, bd, 2, kw["product"], kw["n_stokes"], kw["t_int"], out)
            assert ei.value.status == cobalt.COBALT_ERR_BAD_ARG
        with pytest.raises(cobalt.CobaltError):                                                       # coherent product without beam delays
            cobalt.cobalt_beamform(cor._h, None, x, d, b, None, 2, cobalt.COBALT_BF_COHERENT_VOLTAGES, 1, 1, out)
    with cobalt.Correlator(120, 1, C, N, 16) as cor:                                                  # 2 S = 240 > 208 in tensor mode
        x = torch.zeros(cor.samples_shape(), dtype=torch.int16, device=dev)
        d = torch.zeros(120, dtype=torch.float64, device=dev)
        bd = torch.zeros((2, 120), dtype=torch.float64, device=dev)
        out = torch.empty(1 << 16, dtype=torch.float32, device=dev)
        with pytest.raises(cobalt.CobaltError) as ei:
            cobalt.cobalt_beamform(cor._h, None, x, d, torch.ones(C, dtype=torch.float32, device=dev), bd, 2, cobalt.COBALT_BF_COHERENT_VOLTAGES, 1, 1, out)
        assert ei.value.status == cobalt.COBALT_ERR_BAD_ARG


def test_beamformer_workload_shape_sampled(cobalt, oracle, dev):
    """The shape bench.py --beamform times (48 stations, 256 channels, 195312 samples, 127 beams, Stokes I at t_int = 16; three
    subbands here, one launch group), checked on 32 sampled (subband, channel) pairs that the oracle computes one by one through its
    single-sum channeliser (oracle.channel_direct) and its beamformer functions applied to that one channel."""
    from paper_1801_04834_b200 import synth

    cfg = synth.scaled(synth.CONFIGS[6], B=3)
    n_beams, t_int = 127, 16
    data = synth.generate(cfg, device=dev)
    bd = synth.beam_delays(cfg, n_beams, dev)
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits) as cor:
        got = cor.beamform(data["samples"], data["delays"], data["bandpass"], cobalt.COBALT_BF_COHERENT_STOKES, beam_delays=bd,
                           n_stokes=1, t_int=t_int)
        cor.reset()
        gv = cor.beamform(data["samples"], data["delays"], data["bandpass"], cobalt.COBALT_BF_COHERENT_VOLTAGES, beam_delays=bd)
        torch.cuda.synchronize()
        got, gv = got.cpu().numpy(), gv.cpu().numpy()
    delays, bp, bdh = data["delays"].cpu().numpy(), data["bandpass"].cpu().numpy().astype(np.float64), bd.cpu().numpy()
    rng = np.random.default_rng(3300)
    pairs = [(0, 0), (2, cfg.C - 1), (1, cfg.C // 2)] + [(int(rng.integers(cfg.B)), int(rng.integers(cfg.C))) for _ in range(29)]
    pairs.sort()                                                    # one subband of host memory at a time
    for sb, j in pairs:
        x = data["samples"][sb].cpu().numpy()
        f_sb = oracle.default_subband_frequency(sb)
        zc, _ = oracle.channel_direct(x, cfg.C, j, delays=delays, bandpass=bp, f_sb=f_sb)             # [2S][n_t]
        z1 = np.ascontiguousarray(zc.reshape(cfg.S, 2, cfg.n_t, 1))                                  # one channel as a C = 1 array
        f_j = f_sb + (j - cfg.C / 2) * oracle.F_S / cfg.C
        # oracle_channel_frequency(C = 1, f, f_s, 0) = f - f_s / 2: pass the channel's frequency through that formula
        y = oracle.beamform_coherent(z1, bdh, f_j + 0.5 * oracle.F_S)[:, :, 0, :]                   # [n_beams][2][n_t]
        st = oracle.coherent_stokes(z1, bdh, f_j + 0.5 * oracle.F_S, 1, t_int)[:, 0, 0, :]         # [n_beams][n_out]
        ev = np.sqrt((np.abs(gv[sb, :, :, j, :] - y) ** 2).sum() / (np.abs(y) ** 2).sum())
        es = np.sqrt(((got[sb, :, 0, j, :] - st) ** 2).sum() / (st ** 2).sum())
        assert ev <= TOL_TENSOR and es <= TOL_TENSOR, f"subband {sb}, channel {j}: voltages {ev:.3e}, Stokes I {es:.3e}"
