"""GPU parity for product paths that take a different branch than the cases of the other files (round-2 review):

  * the F-stage with SEVERAL time segments per stream (launch_f cuts a stream when a launch has few stream groups and
    >= 8 k-tiles) under the time-varying delay (A21) and the coarse delay (A25): the per-CTA step table taken from a
    segment's first spectrum, the non-persistent launch, and the warm-up rows of a later segment that come from the
    shifted stream instead of the history; every case over two calls (history carry), whole subbands against
    `oracle.process_subband_ext`, both modes;
  * cobalt_beamform with delays_end, coarse delays, pol-minor and 4-bit input, lost tiles and several launch groups
    (include/cobalt.h promises all of them; the beamformer channelises like the correlator, reading A28);
  * the rotation as the PRODUCT applies it (w_i conj(w_k) in the X-stage epilogue, reading R4) pinned through
    cobalt_process: a DC input with tau = 50 us against the exact rational phase (the angle in double precision);
  * EXACT_FP32 mode at the per-subband sizes of configs 4 and 5.
"""
from fractions import Fraction

import numpy as np
import pytest

from parity_util import TOL_FP32, TOL_TENSOR, err_fp32, err_frobenius

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run through gpurun)")
    return torch.device("cuda:0")


def _mode(cobalt, tensor):
    return cobalt.COBALT_MODE_TENSOR_FP16 if tensor else cobalt.COBALT_MODE_EXACT_FP32


def _check(vg, vo, tensor, what):
    assert np.all(np.isfinite(vg)), what
    e = err_frobenius(vg, vo) if tensor else err_fp32(vg, vo)
    tol = TOL_TENSOR if tensor else TOL_FP32
    assert e <= tol, f"{what}: error {e:.3e} > {tol}"


def _data(rng, B, S, N, bits):
    lim = 2000 if bits == 16 else 100
    x = rng.integers(-lim, lim + 1, size=(B, S, 2, N, 2))
    c = rng.integers(-lim // 2, lim // 2 + 1, size=(B, 1, 1, N, 2))      # a common signal: cross terms are not pure noise
    return np.clip(x // 2 + c, -lim, lim).astype(np.int16 if bits == 16 else np.int8)


# ------------------------------------------------------------------ several time segments per stream
@pytest.mark.parametrize("C,bits,S,B,n_t", [
    (64, 16, 4, 2, 64 * 9 + 20),      # 10 k-tiles: 3 segments of 4, 4, 2 tiles, the last one ragged
    (256, 16, 3, 1, 64 * 12 + 1),     # 13 k-tiles, one stream per CTA pass (C = 256 takes both polarisations back to back)
    (256, 8, 2, 2, 64 * 8),           # exactly 8 k-tiles: two full segments
    (16, 8, 5, 1, 64 * 16 + 63),      # 17 k-tiles, C = 16
])
@pytest.mark.parametrize("tensor", [False, True])
def test_interp_and_coarse_delays_with_several_time_segments(cobalt, oracle, dev, C, bits, S, B, n_t, tensor):
    rng = np.random.default_rng(4100 + C + bits + S)
    N, margin = n_t * C + 2, 40
    offsets = np.array([0, 8, 5, 23, 16][:S], dtype=np.int32)            # 16-byte multiples (bulk path) and odd ones
    tau_b = rng.uniform(-20e-6, 20e-6, S)
    tau_e = tau_b + rng.uniform(-1, 1, S) * 2e-8                         # up to ~2 cycles of phase drift over the block
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))
    hist = [None] * B
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        assert cor.info.n_tiles >= 8
        cor.set_coarse_delays(offsets, N + margin)
        cor.set_phase_offsets(ph0)
        for call in range(2):
            x = _data(rng, B, S, N + margin, bits)
            valid = (rng.uniform(size=(B, S, cor.info.n_tiles)) > 0.2).astype(np.uint8)
            vg = cor.process(torch.from_numpy(x).to(dev), torch.from_numpy(tau_b).to(dev), torch.from_numpy(bp).to(dev),
                             delays_end=torch.from_numpy(tau_e).to(dev), valid=torch.from_numpy(valid).to(dev)).cpu().numpy()
            for b in range(B):
                xs = oracle.coarse_shift(x[b], offsets, N)
                if hist[b] is None:
                    hist[b] = oracle.new_history(S, C)
                vo = oracle.process_subband_ext(xs, C, tau_b, bp.astype(np.float64), oracle.default_subband_frequency(b), hist=hist[b],
                                                delays_end=tau_e, phase0=ph0, valid=valid[b])
                _check(vg[b], vo[0], tensor, f"call {call}, subband {b}")


@pytest.mark.parametrize("tensor", [False, True])
def test_interp_and_coarse_delays_at_config2_shape(cobalt, oracle, dev, tensor):
    """48 stations, 1 subband, 64 channels, 3072 spectra (BASELINE.json config 2): launch_f gives 12 segments per stream."""
    from paper_1801_04834_b200 import synth

    cfg = synth.CONFIGS[2]
    rng = np.random.default_rng(4200)
    margin = 32
    data = synth.generate(synth.scaled(cfg, N=cfg.N + margin), device=dev)
    x = data["samples"]
    offsets = rng.integers(0, margin + 1, cfg.S).astype(np.int32)
    offsets[:4] = [0, 8, 16, 3]
    tau_b = data["delays"].cpu().numpy()
    tau_e = tau_b + rng.uniform(-1, 1, cfg.S) * 2e-8
    bp = data["bandpass"].cpu().numpy()
    with cobalt.Correlator(cfg.S, 1, cfg.C, cfg.N, cfg.bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_coarse_delays(offsets, cfg.N + margin)
        vg = cor.process(x, data["delays"], data["bandpass"], delays_end=torch.from_numpy(tau_e).to(dev)).cpu().numpy()
    vo = oracle.process_subband_ext(oracle.coarse_shift(x[0].cpu().numpy(), offsets, cfg.N), cfg.C, tau_b, bp.astype(np.float64),
                                    oracle.default_subband_frequency(0), delays_end=tau_e)
    _check(vg[0], vo[0], tensor, "config 2 shape, interp + coarse")


def test_interp_at_config5_shape(cobalt, oracle, dev):
    """288 receivers, 64 channels, 3072 spectra (config 5): many stream groups AND several segments, tensor mode."""
    from paper_1801_04834_b200 import synth

    cfg = synth.CONFIGS[5]
    rng = np.random.default_rng(4300)
    data = synth.generate(cfg, device=dev)
    tau_b = rng.uniform(-5e-6, 5e-6, cfg.S)
    tau_e = tau_b + rng.uniform(-1, 1, cfg.S) * 2e-8
    bp = data["bandpass"].cpu().numpy()
    with cobalt.Correlator(cfg.S, 1, cfg.C, cfg.N, cfg.bits) as cor:
        vg = cor.process(data["samples"], torch.from_numpy(tau_b).to(dev), data["bandpass"], delays_end=torch.from_numpy(tau_e).to(dev)).cpu().numpy()
    vo = oracle.process_subband_ext(data["samples"][0].cpu().numpy(), cfg.C, tau_b, bp.astype(np.float64), oracle.default_subband_frequency(0),
                                    delays_end=tau_e)
    _check(vg[0], vo[0], True, "config 5 shape, interp")


# ------------------------------------------------------------------ beamformer with every input option of the F-stage
def _bf_err(got, want, chan_axis):
    axes = tuple(i for i in range(want.ndim) if i != chan_axis)
    num = np.sqrt((np.abs(got - want) ** 2).sum(axis=axes))
    den = np.sqrt((np.abs(want) ** 2).sum(axis=axes))
    assert np.all(den > 0)
    return float((num / den).max())


@pytest.mark.parametrize("bits,pol_minor", [(16, True), (8, False), (4, True), (4, False)])
@pytest.mark.parametrize("tensor", [False, True])
def test_beamform_with_delays_end_coarse_delays_and_input_layouts(cobalt, oracle, dev, bits, pol_minor, tensor):
    """3 subbands in launch groups of 2 (ragged last group), time-varying station delay (pure-phase table + the INTERP
    F-stage), coarse offsets, lost tiles, phase offsets, pol-minor and / or 4-bit samples, two calls: coherent Stokes IQUV
    and, on the second call's input, the complex voltages."""
    rng = np.random.default_rng(4400 + bits + pol_minor)
    B, S, C, n_t, n_beams, margin = 3, 5, 64, 64 * 9 + 7, 6, 24
    N = n_t * C
    offsets = np.array([0, 8, 5, 23, 16], dtype=np.int32)
    tau_b = rng.uniform(-20e-6, 20e-6, S)
    tau_e = tau_b + rng.uniform(-1, 1, S) * 2e-8
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    bd = rng.uniform(-40e-9, 40e-9, (n_beams, S))
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))
    lay = cobalt.COBALT_LAYOUT_POL_MINOR if pol_minor else cobalt.COBALT_LAYOUT_PLANAR
    hist = [oracle.new_history(S, C) for _ in range(B)]

    def draw():
        if bits == 4:
            return rng.integers(0, 256, size=(B, S, 2, N + margin)).astype(np.uint8)
        return _data(rng, B, S, N + margin, bits)

    def shift(xb):                                                        # oracle.coarse_shift wants a trailing (re, im) axis
        if bits == 4:
            return np.ascontiguousarray(oracle.coarse_shift(np.repeat(xb[..., None], 2, axis=-1), offsets, N)[..., 0])
        return oracle.coarse_shift(xb, offsets, N)

    def wire(x):                                                          # planar [B][S][2][N(,2)] -> the caller's order
        if not pol_minor:
            return x
        return np.ascontiguousarray(x.transpose(0, 1, 3, 2) if bits == 4 else x.transpose(0, 1, 3, 2, 4))

    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_chunk_subbands(2)
        cor.set_input_layout(lay)
        cor.set_coarse_delays(offsets, N + margin)
        cor.set_phase_offsets(ph0)
        d_b, d_e = torch.from_numpy(tau_b).to(dev), torch.from_numpy(tau_e).to(dev)
        d_bp, d_bd = torch.from_numpy(bp).to(dev), torch.from_numpy(bd).to(dev)
        for call in range(2):
            x = draw()
            valid = (rng.uniform(size=(B, S, cor.info.n_tiles)) > 0.2).astype(np.uint8)
            got = cor.beamform(torch.from_numpy(wire(x)).to(dev), d_b, d_bp, cobalt.COBALT_BF_COHERENT_STOKES, beam_delays=d_bd, n_stokes=4,
                               t_int=8, delays_end=d_e, valid=torch.from_numpy(valid).to(dev), layout=lay)
            torch.cuda.synchronize()
            got = got.cpu().numpy()
            z = [oracle.channelise_subband(shift(x[b]), C, tau_b, bp.astype(np.float64),
                                           oracle.default_subband_frequency(b), hist=hist[b], delays_end=tau_e, phase0=ph0, valid=valid[b])
                 for b in range(B)]
            tol = TOL_TENSOR if tensor else TOL_FP32
            for b in range(B):
                want = oracle.coherent_stokes(z[b], bd, oracle.default_subband_frequency(b), 4, 8)
                e = _bf_err(got[b], want, 2)
                assert e <= tol, f"call {call}, subband {b}: Stokes error {e:.3e} > {tol}"
        # the complex voltages of the second block: put the history back to what it was before that block
        # (cobalt_reset + one call on the first block would do the same; a fresh plan is the shortest way to say it)
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_chunk_subbands(2)
        cor.set_input_layout(lay)
        cor.set_coarse_delays(offsets, N + margin)
        cor.set_phase_offsets(ph0)
        gv = cor.beamform(torch.from_numpy(wire(x)).to(dev), d_b, d_bp, cobalt.COBALT_BF_COHERENT_VOLTAGES, beam_delays=d_bd,
                          delays_end=d_e, valid=torch.from_numpy(valid).to(dev), layout=lay)
        torch.cuda.synchronize()
        gv = gv.cpu().numpy()
    for b in range(B):
        zb = oracle.channelise_subband(shift(x[b]), C, tau_b, bp.astype(np.float64), oracle.default_subband_frequency(b),
                                       hist=oracle.new_history(S, C), delays_end=tau_e, phase0=ph0, valid=valid[b])
        want = oracle.beamform_coherent(zb, bd, oracle.default_subband_frequency(b))
        e = _bf_err(gv[b], want, 2)
        assert e <= (TOL_TENSOR if tensor else TOL_FP32), f"voltages, subband {b}: error {e:.3e}"


# ------------------------------------------------------------------ the rotation as the product applies it
@pytest.mark.parametrize("C", [64, 256])
@pytest.mark.parametrize("tensor", [False, True])
def test_p15_rotation_through_cobalt_process(cobalt, oracle, dev, C, tensor):
    """DC input on every stream -> only the centre channel (f = f_sb exactly) carries power and F is the same for every
    stream, so arg V_ik[C/2] = 2 pi frac(f_sb (tau_k - tau_i)) is all rotation: checked against exact rational arithmetic.
    tau = 50 us at ~100 MHz is ~5000 cycles; fp32 phase arithmetic would be off by ~3e-3 rad."""
    S, n_t = 3, 80
    samples = np.zeros((2, S, 2, n_t * C, 2), dtype=np.int16)
    samples[..., 0] = 1000
    delays = np.array([50e-6, -37.123456e-6, 0.0])
    bandpass = np.ones(C, dtype=np.float32)
    with cobalt.Correlator(S, 2, C, n_t * C, 16, mode=_mode(cobalt, tensor)) as cor:
        vis = cor.process(torch.from_numpy(samples).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bandpass).to(dev)).cpu().numpy()
    for sb in range(2):
        f = Fraction(oracle.default_subband_frequency(sb))
        for i in range(S):
            for k in range(i, S):
                # z_a = F exp(-2 pi i f tau_a)  =>  V_ik = |F|^2 n_t exp(-2 pi i f (tau_i - tau_k))
                cycles = f * (Fraction(float(delays[k])) - Fraction(float(delays[i])))
                want = 2 * np.pi * float(cycles - (cycles.numerator // cycles.denominator))
                for p in range(2):
                    for q in range(2):
                        got = np.angle(vis[sb, C // 2, k * (k + 1) // 2 + i, p, q])
                        d = np.angle(np.exp(1j * (got - want)))
                        assert abs(d) < 1e-5, (sb, i, k, p, q, d)


# ------------------------------------------------------------------ EXACT_FP32 at the sizes of configs 4 and 5
@pytest.mark.parametrize("index", [4, 5])
def test_exact_mode_at_config4_and_config5_shapes(cobalt, oracle, dev, index):
    """One subband of config 4 (77 stations, 64 channels, int8) and config 5 (288 receivers) in EXACT_FP32 mode, on sampled
    channels the oracle computes one by one (oracle.channel_direct), in the 1e-4 metric."""
    from paper_1801_04834_b200 import synth

    cfg = synth.scaled(synth.CONFIGS[index], B=1)
    data = synth.generate(cfg, device=dev)
    with cobalt.Correlator(cfg.S, 1, cfg.C, cfg.N, cfg.bits, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        vis = cor.process(data["samples"], data["delays"], data["bandpass"])
        torch.cuda.synchronize()
    assert bool(torch.isfinite(torch.view_as_real(vis)).all())
    x = data["samples"][0].cpu().numpy()
    delays, bp = data["delays"].cpu().numpy(), data["bandpass"].cpu().numpy().astype(np.float64)
    for j in (0, 17, cfg.C // 2, cfg.C - 1):
        _, vo = oracle.channel_direct(x, cfg.C, j, delays=delays, bandpass=bp, f_sb=oracle.default_subband_frequency(0))
        e = err_fp32(vis[0, j].cpu().numpy(), vo)
        assert e <= TOL_FP32, f"{cfg.name} channel {j}: error {e:.3e} > {TOL_FP32}"


# ------------------------------------------------------------------ plan state and launch limits (round-2 advice)
def test_set_mode_keeps_a_chunk_size_the_caller_chose(cobalt, dev):
    with cobalt.Correlator(3, 6, 16, 16 * 64, 16) as cor:
        default_chunk = cor.info.chunk_subbands
        cor.set_mode(cobalt.COBALT_MODE_EXACT_FP32)
        assert cor.info.chunk_subbands == default_chunk                 # never set: the default rule again
        cor.set_chunk_subbands(2)
        cor.set_mode(cobalt.COBALT_MODE_TENSOR_FP16)
        assert cor.info.chunk_subbands == 2
        cor.set_dumps(1)
        cor.set_mode(cobalt.COBALT_MODE_EXACT_FP32)
        assert cor.info.chunk_subbands == 2


def test_oversized_grids_are_refused_before_anything_is_enqueued(cobalt, dev):
    """Settings whose kernels would need gridDim.y / .z > 65535 used to fail at launch, after earlier launch groups had
    already advanced the in-place FIR history; now they are COBALT_ERR_BAD_ARG up front."""
    dummy = torch.zeros(1 << 20, dtype=torch.uint8, device=dev)          # never read: the call is refused first
    with cobalt.Correlator(1, 1024, 16, 16 * 64 * 64, 16, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        cor.set_chunk_subbands(1024)
        cor.set_dumps(64)                                                # 1024 * 64 = 65536 (subband, dump) pairs in gridDim.z
        with pytest.raises(cobalt.CobaltError) as e:
            cobalt.cobalt_process_ex(cor._h, None, dummy, dummy, dummy, dummy)
        assert e.value.status == cobalt.COBALT_ERR_BAD_ARG and "65535" in str(e.value)
        cor.set_chunk_subbands(512)                                      # two groups of 512: fine
        x = torch.zeros(cor.samples_shape(), dtype=torch.int16, device=dev)
        x[..., 0] = 3
        vis = cor.process(x, torch.zeros(1, dtype=torch.float64, device=dev), torch.ones(16, dtype=torch.float32, device=dev))
        torch.cuda.synchronize()
        assert vis.shape == (64, 1024, 16, 1, 2, 2) and bool(torch.isfinite(torch.view_as_real(vis)).all())
        assert float(vis[:, :, 8, 0, 0, 0].real.min()) > 0               # DC input: power in the centre channel of every dump
    n_t = 65535 * 128 + 1
    with cobalt.Correlator(1, 1, 16, 16 * n_t, 8, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        with pytest.raises(cobalt.CobaltError) as e:
            cobalt.cobalt_beamform(cor._h, None, dummy, dummy, dummy, dummy, 1, cobalt.COBALT_BF_INCOHERENT_STOKES, 1, 1, dummy)
        assert e.value.status == cobalt.COBALT_ERR_BAD_ARG and "spectra" in str(e.value)


# ------------------------------------------------------------------ the host-buffer call with every optional array
@pytest.mark.parametrize("tensor", [False, True])
def test_process_host_ex_is_bit_identical_to_the_device_path(cobalt, dev, tensor):
    """cobalt_process_host_ex (pinned host buffers: dumps, lost-data flags, weights, time-varying delay; groups of 2 + 2 + 1
    subbands) on one plan against cobalt_process_ex with device copies of the same buffers on a second plan, over two
    consecutive blocks (history carry): the same kernels on the same data, so bit for bit.  Then the plain
    cobalt_process_host on plans that write two dumps per block (it used to refuse them)."""
    from paper_1801_04834_b200 import synth

    cfg = synth.scaled(synth.CONFIGS[3], S=6, B=5, C=64, N=64 * 64 * 4)
    D = 2
    rng = np.random.default_rng(4500)
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=_mode(cobalt, tensor)) as on_dev, \
            cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=_mode(cobalt, tensor)) as on_host:
        for cor in (on_dev, on_host):
            cor.set_chunk_subbands(2)
            cor.set_dumps(D)
        i = on_host.info
        for call in range(2):
            data = synth.generate(synth.scaled(cfg, sigma=cfg.sigma * (1 + call)), device="cpu")
            tau_e = data["delays"] + torch.from_numpy(rng.uniform(-1, 1, cfg.S) * 2e-8)
            valid = torch.from_numpy((rng.uniform(size=(cfg.B, cfg.S, i.n_tiles)) > 0.3).astype(np.uint8))
            want_counts = torch.zeros((cfg.B, D, i.n_baselines), dtype=torch.int32, device=dev)
            want = on_dev.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev), delays_end=tau_e.to(dev),
                                  valid=valid.to(dev), valid_counts=want_counts).cpu().numpy()
            out = torch.full(on_host.vis_shape(), float("nan"), dtype=torch.complex64).pin_memory()
            counts = torch.full((cfg.B, D, i.n_baselines), -1, dtype=torch.int32).pin_memory()
            on_host.process_host(data["samples"].pin_memory(), data["delays"], data["bandpass"], out, delays_end=tau_e, valid=valid.pin_memory(),
                                 valid_counts=counts)
            assert out.shape[0] == D and want.shape == tuple(out.shape)
            assert np.array_equal(want.view(np.float32), out.numpy().view(np.float32)), f"block {call}"
            assert np.array_equal(want_counts.cpu().numpy(), counts.numpy()), f"block {call}"
        for cor in (on_dev, on_host):
            cor.reset()
        plain_d = on_dev.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev)).cpu().numpy()
        plain_h = torch.empty(on_host.vis_shape(), dtype=torch.complex64).pin_memory()
        on_host.process_host(data["samples"].pin_memory(), data["delays"], data["bandpass"], plain_h)
        assert np.array_equal(plain_d.view(np.float32), plain_h.numpy().view(np.float32))
