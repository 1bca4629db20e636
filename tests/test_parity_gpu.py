"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the float64 oracle,
element by element on the same seeded integer inputs (SURVEY.md sec 8(c) pins P1, P10, P14, P15 and
reading A17 for the error metrics).  Runs on the B200 box: `pytest -m gpu`.

Tolerances (BASELINE.json north_star): fp32 mode max |dV| / sqrt(V_ii V_kk) <= 1e-4; tensor-core
(fp16 operand) mode ||dV||_F / ||V||_F <= 2e-3 per (subband, channel); integer unpack and the
channel / baseline / polarisation indexing bit-exact.
"""
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


def _synth():
    from paper_1801_04834_b200 import synth

    return synth


def _run_gpu(cobalt, cfg, data, mode, dev, chunk=None, calls=1):
    """Whole path through cobalt_process; returns the list of visibilities of each call."""
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=mode) as cor:
        if chunk is not None:
            cor.set_chunk_subbands(chunk)
        outs = []
        for _ in range(calls):
            vis = cor.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev))
            torch.cuda.synchronize()
            outs.append(vis.cpu().numpy())
    return outs


def _run_oracle(oracle, cfg, data, calls=1, subbands=None):
    sb = range(cfg.B) if subbands is None else subbands
    samples = data["samples"].cpu().numpy()
    hist = {s: oracle.new_history(cfg.S, cfg.C) for s in sb}
    outs = []
    for _ in range(calls):
        v = [oracle.process_subband(samples[s], cfg.C, data["delays"].cpu().numpy(), data["bandpass"].cpu().numpy().astype(np.float64),
                                    oracle.default_subband_frequency(s), hist[s]) for s in sb]
        outs.append(np.stack(v))
    return outs


def _assert_parity(vg, vo, mode_tensor, what):
    assert np.all(np.isfinite(vg)), f"{what}: non-finite GPU output"
    if mode_tensor:
        e = err_frobenius(vg, vo)
        assert e <= TOL_TENSOR, f"{what}: Frobenius error {e:.3e} > {TOL_TENSOR}"
    else:
        e = err_fp32(vg, vo)
        assert e <= TOL_FP32, f"{what}: autocorrelation-normalised error {e:.3e} > {TOL_FP32}"
    return e


# ------------------------------------------------------------------ P1: unpack bit-exact
@pytest.mark.parametrize("bits", [16, 8])
def test_p1_unpack_every_value_bit_exact(cobalt, oracle, dev, bits):
    """cobalt_debug_unpack runs unpack_sample<BITS> of csrc/ptx.cuh on packed complex samples: the very routine (not
    a look-alike) the fused F-stage kernels apply to the words they read from shared memory.  Every value appears
    both as the re (low) and as the im (high) half of a sample; the odd length exercises the single-component tail."""
    if bits == 16:
        x = np.arange(-32768, 32768, dtype=np.int64).astype(np.int16)
    else:
        x = np.arange(-128, 128, dtype=np.int64).astype(np.int8)
    x = np.concatenate([x, x[::-1], x[: 37]])                      # ragged length
    got = cobalt.unpack(torch.from_numpy(x).to(dev)).cpu().numpy()
    want = oracle.unpack(x)
    assert got.dtype == np.float32
    assert np.array_equal(got.astype(np.float64), want)


def test_unpack_empty(cobalt, dev):
    out = cobalt.unpack(torch.empty(0, dtype=torch.int16, device=dev))
    assert out.numel() == 0


# ------------------------------------------------------------------ FIR weights (A1, A2)
@pytest.mark.parametrize("C", [16, 64, 256])
def test_fir_weights_are_the_rounded_prototype(cobalt, oracle, dev, C):
    with cobalt.Correlator(2, 1, C, 4 * C) as cor:
        w = cor.fir_weights()                                      # [k][ph], k = 0 newest block
    g = oracle.fir_prototype(C)
    want = g.reshape(16, C)[::-1].astype(np.float32)               # w[k][ph] = g[(15-k) C + ph]
    assert np.array_equal(w, want)


# ------------------------------------------------------------------ F-stage alone (steps a1-a7)
@pytest.mark.parametrize("C,bits,S,n_t", [(16, 16, 3, 150), (64, 16, 2, 203), (256, 16, 2, 70), (64, 8, 3, 130), (256, 8, 1, 65), (16, 8, 2, 64)])
@pytest.mark.parametrize("mode_tensor", [False, True])
def test_channelised_matches_oracle(cobalt, oracle, dev, C, bits, S, n_t, mode_tensor):
    """z (after rotation, bandpass, channel reorder) for one subband of a 2-subband input, ragged tail
    (N not a multiple of C, n_t not a multiple of the 64-spectrum tile)."""
    rng = np.random.default_rng(1000 + C + bits + S)
    N = n_t * C + 7
    lim = 3000 if bits == 16 else 100
    samples = rng.integers(-lim, lim + 1, size=(2, S, 2, N, 2)).astype(np.int16 if bits == 16 else np.int8)
    delays = rng.uniform(-50e-6, 50e-6, S)
    bandpass = (1.0 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    with cobalt.Correlator(S, 2, C, N, bits, mode=mode) as cor:
        z = cor.channelised(torch.from_numpy(samples).to(dev), torch.from_numpy(delays).to(dev),
                            torch.from_numpy(bandpass).to(dev), sb=1)
        torch.cuda.synchronize()
        z = z.cpu().numpy()                                        # [C][2S][n_t]
    _, zo = oracle.process_subband(samples[1], C, delays, bandpass.astype(np.float64),
                                   oracle.default_subband_frequency(1), return_z=True)
    zo = zo.reshape(2 * S, n_t, C).transpose(2, 0, 1)              # [S][2][n_t][C] -> [C][2S][n_t]
    scale = np.sqrt(np.mean(np.abs(zo) ** 2))
    err = np.max(np.abs(z - zo)) / scale
    # fp32 arithmetic: 16 taps + log2(C) butterfly levels, ~1e-6; fp16 operands: 2^-11 relative rounding
    assert err <= (2e-3 if mode_tensor else 2e-5), err


# ------------------------------------------------------------------ P14: X-stage indexing, bit-exact
@pytest.mark.parametrize("S,n_t", [(1, 5), (3, 64), (8, 100), (48, 130), (64, 66), (70, 66), (77, 70), (81, 129), (88, 64), (96, 70), (100, 64), (130, 65), (288, 40)])
@pytest.mark.parametrize("mode_tensor", [False, True])
def test_p14_correlate_small_integers_bit_exact(cobalt, oracle, dev, S, n_t, mode_tensor):
    """Small integers are exact in fp16 and their sums exact in fp32, so the X-stage must equal integer
    arithmetic bit for bit: pins the conjugation side, baseline order k(k+1)/2 + i and pol order."""
    C = 16
    rng = np.random.default_rng(77 + S)
    zr = rng.integers(-8, 9, size=(C, 2 * S, n_t))
    zi = rng.integers(-8, 9, size=(C, 2 * S, n_t))
    z = (zr + 1j * zi).astype(np.complex64)
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    with cobalt.Correlator(S, 1, C, n_t * C, 16, mode=mode) as cor:
        vis = cor.correlate(torch.from_numpy(z).to(dev))
        torch.cuda.synchronize()
        vis = vis.cpu().numpy()                                    # [C][n_bl][2][2]
    zo = z.astype(np.complex128).reshape(C, S, 2, n_t).transpose(1, 2, 3, 0)   # -> [S][2][n_t][C]
    want = oracle.correlate(np.ascontiguousarray(zo))
    assert np.array_equal(vis.astype(np.complex128), want)


@pytest.mark.parametrize("S,C,n_t", [(77, 256, 768), (77, 64, 1500), (288, 64, 768), (130, 64, 700), (48, 64, 3072)])
def test_p14_bit_exact_through_the_full_size_control_paths(cobalt, oracle, dev, S, C, n_t):
    """P14 at sizes where a CTA runs several jobs one after the other (C * jobs-per-channel > 148 SMs: second and
    later jobs flip the tmem_full / tmem_empty phases and reuse the staged output block), the load ring wraps many
    times (n_t / 64 k-tiles > ring depth) and, for S = 48 with few jobs, the k-range of a channel is split over
    several CTAs.  Integers |v| <= 8: every product and every partial sum is exact in fp32 (< 2^24), so the result
    must equal integer arithmetic bit for bit, element by element."""
    rng = np.random.default_rng(1400 + S + C)
    z = torch.from_numpy(rng.integers(-8, 9, size=(C, 2 * S, n_t, 2)).astype(np.float32))
    zc = torch.view_as_complex(z).contiguous()
    with cobalt.Correlator(S, 1, C, n_t * C, 16, mode=cobalt.COBALT_MODE_TENSOR_FP16) as cor:
        vis = cor.correlate(zc.to(dev))
        torch.cuda.synchronize()
        vis = vis.cpu().numpy()
    zo = zc.numpy().astype(np.complex128).reshape(C, S, 2, n_t).transpose(1, 2, 3, 0)   # -> [S][2][n_t][C]
    want = oracle.correlate(np.ascontiguousarray(zo))
    assert np.array_equal(vis.astype(np.complex128), want)


# ------------------------------------------------------------------ whole path, configs 1 and 2 in full
@pytest.mark.parametrize("mode_tensor", [False, True])
def test_config1_tiny_full_parity(cobalt, oracle, dev, mode_tensor):
    synth = _synth()
    cfg = synth.CONFIGS[1]
    data = synth.generate(cfg, device="cpu")
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    vg = _run_gpu(cobalt, cfg, data, mode, dev, calls=2)
    vo = _run_oracle(oracle, cfg, data, calls=2)
    for call in range(2):                                          # second call: carried history (P10)
        _assert_parity(vg[call], vo[call], mode_tensor, f"config 1 call {call}")
    # the tone of reading A16 sits in channel 5
    p = np.abs(vo[0][0, :, 0, 0, 0])
    assert int(np.argmax(p)) == 5


@pytest.mark.parametrize("mode_tensor", [False, True])
def test_config2_core_like_full_parity(cobalt, oracle, dev, mode_tensor):
    synth = _synth()
    cfg = synth.CONFIGS[2]
    data = synth.generate(cfg, device=dev)
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    vg = _run_gpu(cobalt, cfg, data, mode, dev)
    vo = _run_oracle(oracle, cfg, data)
    _assert_parity(vg[0], vo[0], mode_tensor, "config 2")
    # P13 / A15: 10 % common power => cross-correlation coefficient ~0.1 after delay compensation
    v = vo[0][0]
    auto0 = v[:, 0, 0, 0].real
    auto1 = v[:, 2, 0, 0].real
    rho = np.abs(v[8:-8, 1, 0, 0]) / np.sqrt(auto0[8:-8] * auto1[8:-8])
    assert 0.06 < float(np.median(rho)) < 0.12


# ------------------------------------------------------------------ chunking, history, ragged shapes
@pytest.mark.parametrize("mode_tensor", [False, True])
def test_subband_chunking_and_history_carry(cobalt, oracle, dev, mode_tensor):
    """5 subbands processed 2 per launch group (ragged last chunk), two consecutive calls."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[3], S=5, B=5, C=64, N=64 * 150 + 13)
    data = synth.generate(cfg, device="cpu")
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    vg = _run_gpu(cobalt, cfg, data, mode, dev, chunk=2, calls=2)
    vo = _run_oracle(oracle, cfg, data, calls=2)
    for call in range(2):
        _assert_parity(vg[call], vo[call], mode_tensor, f"chunked call {call}")


def test_short_block_history_older_than_block(cobalt, oracle, dev):
    """N = C (one spectrum per call): the new history is mostly the old one shifted (step a10)."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[1], N=16)
    data = synth.generate(synth.scaled(synth.CONFIGS[1], N=16 * 6), device="cpu")
    full = data["samples"]
    hist = oracle.new_history(cfg.S, cfg.C)
    with cobalt.Correlator(cfg.S, 1, cfg.C, 16, 16, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        for blk in range(6):
            s = full[:, :, :, 16 * blk:16 * (blk + 1), :].contiguous()
            vg = cor.process(s.to(dev), data["delays"].to(dev), data["bandpass"].to(dev)).cpu().numpy()
            vo = oracle.process_subband(s[0].numpy(), cfg.C, data["delays"].numpy(), data["bandpass"].numpy().astype(np.float64),
                                        oracle.default_subband_frequency(0), hist)
            _assert_parity(vg[0], vo, False, f"block {blk}")


@pytest.mark.parametrize("mode_tensor", [False, True])
def test_reset_zeroes_history(cobalt, dev, mode_tensor):
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[1], N=16 * 70)
    data = synth.generate(cfg, device="cpu")
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    with cobalt.Correlator(cfg.S, 1, cfg.C, cfg.N, 16, mode=mode) as cor:
        args = (data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev))
        a = cor.process(*args).cpu().numpy()
        b = cor.process(*args).cpu().numpy()
        cor.reset()
        c = cor.process(*args).cpu().numpy()
    assert np.array_equal(a, c)
    assert not np.array_equal(a, b)


# ------------------------------------------------------------------ extreme integers (A12)
@pytest.mark.parametrize("C,n_t", [(64, 80), (256, 48)])
@pytest.mark.parametrize("bits", [16, 8])
def test_extreme_sample_values(cobalt, oracle, dev, bits, C, n_t):
    """Full-scale input incl. -32768 / -128: no overflow of the fp16 intermediate, parity holds."""
    synth = _synth()
    S = 2
    rng = np.random.default_rng(5)
    lo, hi = (-32768, 32767) if bits == 16 else (-128, 127)
    samples = rng.choice(np.array([lo, hi, 0, -1, 1]), size=(1, S, 2, n_t * C, 2)).astype(np.int16 if bits == 16 else np.int8)
    data = {"samples": torch.from_numpy(samples), "delays": torch.zeros(S, dtype=torch.float64),
            "bandpass": torch.ones(C, dtype=torch.float32)}
    cfg = synth.scaled(synth.CONFIGS[1], S=S, C=C, N=n_t * C, bits=bits)
    for mode_tensor in (False, True):
        mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
        vg = _run_gpu(cobalt, cfg, data, mode, dev)
        vo = _run_oracle(oracle, cfg, data)
        _assert_parity(vg[0], vo[0], mode_tensor, f"extreme values, tensor={mode_tensor}")


# ------------------------------------------------------------------ P15: fp64 phase
def test_p15_large_delay_phase_needs_fp64(cobalt, oracle, dev):
    """tau = 50 us at ~100 MHz is ~5000 cycles: the rotation must agree with float64 to ~1e-6 rad
    (fp32 phase arithmetic would be off by ~3e-3).  Checked through z of a DC input."""
    C, S, n_t = 64, 2, 80
    samples = np.zeros((1, S, 2, n_t * C, 2), dtype=np.int16)
    samples[..., 0] = 1000                                          # DC -> centre channel C/2
    delays = np.array([50e-6, -37.123456e-6])
    bandpass = np.ones(C, dtype=np.float32)
    with cobalt.Correlator(S, 1, C, n_t * C, 16, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        z = cor.channelised(torch.from_numpy(samples).to(dev), torch.from_numpy(delays).to(dev),
                            torch.from_numpy(bandpass).to(dev)).cpu().numpy()
    f = oracle.default_subband_frequency(0)                         # channel C/2 is the subband centre
    for a in range(S):
        want = -2 * np.pi * ((f * delays[a]) % 1.0)
        got = np.angle(z[C // 2, 2 * a, 40])
        d = np.angle(np.exp(1j * (got - want)))
        assert abs(d) < 2e-6, (a, d)


# ------------------------------------------------------------------ host-buffer entry (e2e path)
def test_process_host_matches_device_path(cobalt, dev):
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[3], S=6, B=5, C=64, N=64 * 100)
    data = synth.generate(cfg, device="cpu")
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits) as cor:
        cor.set_chunk_subbands(2)
        a = cor.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev)).cpu().numpy()
        cor.reset()
        out = torch.empty(cor.vis_shape(), dtype=torch.complex64).pin_memory()
        cor.process_host(data["samples"].pin_memory(), data["delays"], data["bandpass"], out)
    assert np.array_equal(a, out.numpy())


# ------------------------------------------------------------------ fp16 operand scale
@pytest.mark.parametrize("C,n_t,t0", [(64, 64, 40), (256, 32, 20)])
def test_fp16_scale_worst_case_amplitude(cobalt, oracle, dev, C, n_t, t0):
    """Sign-matched full-scale input rotated by 45 degrees drives one component of z to
    sum|g| * sqrt(2) * 32767 ~ 7.8e4 > 65504: without the power-of-two operand scale fp16 overflows.  Every channel
    but the centre one is empty here (leakage only), so the per-channel 2e-3 also checks that the F-stage keeps the
    dynamic range of an fp32 filter bank."""
    S = 2
    g = oracle.fir_prototype(C)
    samples = np.zeros((1, S, 2, n_t * C, 2), dtype=np.int16)
    seg = (32767 * np.sign(g)).astype(np.int16)                     # window of spectrum t0, natural order
    samples[0, :, :, (t0 - 15) * C:(t0 + 1) * C, 0] = seg
    samples[0, :, :, (t0 - 15) * C:(t0 + 1) * C, 1] = seg
    f = oracle.default_subband_frequency(0)
    tau = (np.floor(f * 1e-6) + 0.125) / f                          # frac(f tau) = 1/8 at the centre channel
    delays = np.array([tau, 0.0])
    bandpass = np.ones(C, dtype=np.float32)
    _, zo = oracle.process_subband(samples[0], C, delays, bandpass.astype(np.float64), f, return_z=True)
    assert np.max(np.abs(zo[0].real)) > 65504                       # the case really is out of fp16 range
    with cobalt.Correlator(S, 1, C, n_t * C, 16) as cor:
        vg = cor.process(torch.from_numpy(samples).to(dev), torch.from_numpy(delays).to(dev),
                         torch.from_numpy(bandpass).to(dev)).cpu().numpy()
    vo = oracle.process_subband(samples[0], C, delays, bandpass.astype(np.float64), f)
    _assert_parity(vg[0], vo, True, "worst-case amplitude")


@pytest.mark.parametrize("gain", [1e-4, 300.0])
def test_fp16_scale_follows_bandpass_gain(cobalt, oracle, dev, gain):
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[2], S=4, N=64 * 200)
    data = synth.generate(cfg, device="cpu")
    data["bandpass"] = (data["bandpass"] * gain * (1 + 0.2 * torch.rand(cfg.C))).to(torch.float32)
    vg = _run_gpu(cobalt, cfg, data, cobalt.COBALT_MODE_TENSOR_FP16, dev)
    vo = _run_oracle(oracle, cfg, data)
    _assert_parity(vg[0], vo[0], True, f"bandpass gain {gain}")


# ------------------------------------------------------------------ time-varying delay (reading A21)
@pytest.mark.parametrize("C,bits,S,n_t,drift", [(16, 16, 3, 150, 0.15), (64, 16, 2, 203, -2.5), (256, 16, 2, 70, 0.15),
                                                (64, 8, 3, 130, 30.0), (256, 8, 1, 65, -0.4)])
@pytest.mark.parametrize("mode_tensor", [False, True])
def test_time_varying_delay_matches_oracle(cobalt, oracle, dev, C, bits, S, n_t, drift, mode_tensor):
    """cobalt_process_interp: the delay runs linearly from delays to delays_end over the block; drift =
    phase change of the subband centre over the block in cycles (LOFAR rates give ~0.15; 30 stresses the fp32 step)."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[2 if bits == 16 else 4], S=S, B=2, C=C, N=n_t * C + 3, bits=bits)
    data = synth.generate(cfg, device="cpu")
    rng = np.random.default_rng(21)
    tau_b = data["delays"].numpy()
    tau_e = tau_b + drift / oracle.default_subband_frequency(0) * rng.uniform(0.5, 1.0, S)
    bp = data["bandpass"].numpy().astype(np.float64)
    samples = data["samples"].numpy()
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=mode) as cor:
        vg = cor.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev),
                         delays_end=torch.from_numpy(tau_e).to(dev))
        vs = cor.process(data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev))   # second call: history carried
        torch.cuda.synchronize()
        vg = vg.cpu().numpy()
    for b in range(cfg.B):
        vo = oracle.process_subband(samples[b], C, tau_b, bp, oracle.default_subband_frequency(b), delays_end=tau_e)
        _assert_parity(vg[b], vo, mode_tensor, f"time-varying delay, subband {b}")
        if S > 1:
            static = oracle.process_subband(samples[b], C, tau_b, bp, oracle.default_subband_frequency(b))
            assert np.max(np.abs(static - vo)) > 1e-3 * np.max(np.abs(vo))      # the drift really changes the result
    assert np.all(np.isfinite(vs.cpu().numpy()))


def test_time_varying_delay_with_equal_ends_is_the_static_call(cobalt, dev):
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[2], S=4, B=1, C=64, N=64 * 90)
    data = synth.generate(cfg, device="cpu")
    out = []
    for interp in (False, True):
        with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
            d = data["delays"].to(dev)
            v = cor.process(data["samples"].to(dev), d, data["bandpass"].to(dev), delays_end=d.clone() if interp else None)
            torch.cuda.synchronize()
            out.append(v.cpu().numpy())
    scale = np.max(np.abs(out[0]))
    assert np.max(np.abs(out[0] - out[1])) <= 2e-6 * scale


def test_output_pointer_not_16_byte_aligned_is_rejected_in_tensor_mode(cobalt, dev):
    """The tensor-mode X-stage writes 16-byte pieces (and whole channel blocks with one bulk store): an 8-byte
    aligned visibility buffer is a COBALT_ERR_BAD_ARG, not a fault; EXACT mode (8-byte stores) accepts it."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[2], S=5, B=2, C=64, N=64 * 70)
    data = synth.generate(cfg, device="cpu")
    args = (data["samples"].to(dev), data["delays"].to(dev), data["bandpass"].to(dev))
    for mode in (cobalt.COBALT_MODE_TENSOR_FP16, cobalt.COBALT_MODE_EXACT_FP32):
        with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=mode) as cor:
            ref = cor.process(*args)
            cor.reset()
            shape = cor.vis_shape()
            flat = torch.zeros(int(np.prod(shape)) + 1, dtype=torch.complex64, device=dev)
            out = flat[1:].view(shape)
            assert out.data_ptr() % 16 == 8
            if mode == cobalt.COBALT_MODE_TENSOR_FP16:
                with pytest.raises(Exception, match="16-byte"):
                    cor.process(*args, out=out)
            else:
                cor.process(*args, out=out)
                torch.cuda.synchronize()
                assert torch.equal(ref, out) and flat[0] == 0


def test_streaming_under_a_cuda_graph(cobalt, oracle, dev):
    """SURVEY.md sec 8(f) row 2 (streaming): cobalt_process only enqueues kernels on the caller's stream, so two
    consecutive blocks can be captured in a
    CUDA graph and replayed on new data; the history carries across replays exactly as across plain calls."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[2], S=3, B=2, C=64, N=64 * 40)
    blocks = [synth.generate(synth.scaled(cfg, N=cfg.N), device="cpu") for _ in range(1)]
    rng = np.random.default_rng(8)
    data = [torch.from_numpy(rng.integers(-300, 300, size=(cfg.B, cfg.S, 2, cfg.N, 2)).astype(np.int16)) for _ in range(4)]
    delays, bandpass = blocks[0]["delays"], blocks[0]["bandpass"]
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits) as cor:
        x0 = torch.empty_like(data[0], device=dev)
        x1 = torch.empty_like(data[0], device=dev)
        v0 = torch.empty(cor.vis_shape(), dtype=torch.complex64, device=dev)
        v1 = torch.empty_like(v0)
        d, b = delays.to(dev), bandpass.to(dev)
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            cor.process(x0, d, b, out=v0, stream=torch.cuda.current_stream())
            cor.process(x1, d, b, out=v1, stream=torch.cuda.current_stream())
        cor.reset()                                              # capture did not run anything; start from zero history
        got = []
        for r in range(2):
            x0.copy_(data[2 * r]); x1.copy_(data[2 * r + 1])
            g.replay()
            torch.cuda.synchronize()
            got += [v0.cpu().numpy().copy(), v1.cpu().numpy().copy()]
    for sb in range(cfg.B):
        hist = oracle.new_history(cfg.S, cfg.C)
        for k in range(4):
            vo = oracle.process_subband(data[k].numpy()[sb], cfg.C, delays.numpy(), bandpass.numpy().astype(np.float64),
                                        oracle.default_subband_frequency(sb), hist)
            _assert_parity(got[k][sb], vo, True, f"graph replay, block {k}, subband {sb}")


def test_one_captured_call_replays_block_after_block(cobalt, oracle, dev):
    """A single captured cobalt_process replayed on three consecutive blocks: the FIR history is carried in place, no
    host-side state changes between calls."""
    rng = np.random.default_rng(81)
    S, B, C, n_t = 3, 2, 64, 40
    N = C * n_t
    data = [torch.from_numpy(rng.integers(-300, 300, size=(B, S, 2, N, 2)).astype(np.int16)) for _ in range(3)]
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    with cobalt.Correlator(S, B, C, N, 16) as cor:
        x = torch.empty_like(data[0], device=dev)
        v = torch.empty(cor.vis_shape(), dtype=torch.complex64, device=dev)
        d, b = torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev)
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            cor.process(x, d, b, out=v, stream=torch.cuda.current_stream())
        cor.reset()
        got = []
        for r in range(3):
            x.copy_(data[r])
            g.replay()
            torch.cuda.synchronize()
            got.append(v.cpu().numpy().copy())
    for sb in range(B):
        hist = oracle.new_history(S, C)
        for k in range(3):
            vo = oracle.process_subband(data[k].numpy()[sb], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(sb), hist)
            _assert_parity(got[k][sb], vo, True, f"single-call graph replay, block {k}, subband {sb}")


def test_golden_tiny_case_on_gpu(cobalt, dev):
    """The frozen oracle values of tests/golden/ (written by the oracle alone) against both GPU modes."""
    import os
    import sys

    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    sys.path.insert(0, here)
    import make_golden as mg

    x = np.loadtxt(os.path.join(here, "tiny_fx_input.txt"), dtype=np.int64).astype(np.int16).reshape(1, mg.S, 2, mg.N, 2)
    exp = np.loadtxt(os.path.join(here, "tiny_fx_expected.txt")).view(np.complex128).reshape(1, mg.C, 3, 2, 2)
    for mode, tensor in ((cobalt.COBALT_MODE_EXACT_FP32, False), (cobalt.COBALT_MODE_TENSOR_FP16, True)):
        with cobalt.Correlator(mg.S, 1, mg.C, mg.N, 16, mode=mode) as cor:
            vis = cor.process(torch.from_numpy(x).to(dev), torch.from_numpy(mg.DELAYS).to(dev),
                              torch.from_numpy(mg.BANDPASS.astype(np.float32)).to(dev))
            torch.cuda.synchronize()
        _assert_parity(vis.cpu().numpy(), exp, tensor, f"golden tiny case, tensor={tensor}")


# ------------------------------------------------------------------ frequency settings (reading A6)
def _delayed(s, d):
    k = np.fft.fftfreq(s.size)
    return np.fft.ifft(np.fft.fft(s) * np.exp(-2j * np.pi * k * d))


@pytest.mark.parametrize("mode_tensor", [False, True])
def test_p9_baseband_delay_slope_and_compensation_on_gpu(cobalt, oracle, dev, mode_tensor):
    """GPU counterpart of pin P9 through cobalt_set_subband_frequencies: with f_sb = 0 (pure baseband) a station
    delayed by d samples shows arg V01[j] = 2 pi d (j - C/2) / C, and tau_1 = -d / f_s flattens it; the same with a
    non-default sample rate through cobalt_set_sample_rate.  Checked against the closed form AND the oracle."""
    rng = np.random.default_rng(909)
    C, n_t, d, S = 64, 1200, 9.77, 2
    N = n_t * C
    s0 = (rng.standard_normal(N) + 1j * rng.standard_normal(N)) * 2000.0
    x = np.zeros((1, S, 2, N, 2), dtype=np.int16)
    for a, sig in enumerate((s0, _delayed(s0, d))):
        x[0, a, :, :, 0] = np.rint(sig.real)
        x[0, a, :, :, 1] = np.rint(sig.imag)
    bandpass = np.ones(C, dtype=np.float32)
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    bl01 = oracle.baseline_index(0, 1)
    for f_s in (oracle.F_S, 200.0e3):
        with cobalt.Correlator(S, 1, C, N, 16, mode=mode) as cor:
            cor.set_subband_frequencies(np.array([0.0]))
            if f_s != oracle.F_S:
                cor.set_sample_rate(f_s)
            args = (torch.from_numpy(x).to(dev), torch.from_numpy(bandpass).to(dev))
            v_raw = cor.process(args[0], torch.zeros(S, dtype=torch.float64, device=dev), args[1]).cpu().numpy()[0]
            cor.reset()
            tau = np.array([0.0, -d / f_s])
            v_cmp = cor.process(args[0], torch.from_numpy(tau).to(dev), args[1]).cpu().numpy()[0]
        ph = np.unwrap(np.angle(v_raw[:, bl01, 0, 0]))
        slope = np.polyfit(np.arange(C)[4:-4], ph[4:-4], 1)[0]
        assert abs(slope - 2 * np.pi * d / C) < 2e-3, slope
        assert np.max(np.abs(np.angle(v_cmp[2:-2, bl01, 0, 0]))) < 0.03
        vo = oracle.process_subband(x[0], C, tau, bandpass.astype(np.float64), 0.0, f_s=f_s)
        _assert_parity(v_cmp, vo, mode_tensor, f"baseband P9, f_s = {f_s}")


@pytest.mark.parametrize("mode_tensor", [False, True])
def test_shuffled_frequency_ladder_and_sample_rate_match_oracle(cobalt, oracle, dev, mode_tensor):
    """cobalt_set_subband_frequencies with a non-monotonic ladder (incl. a negative and a zero frequency) and
    cobalt_set_sample_rate, several launch groups: every subband is rotated with ITS frequency."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[3], S=4, B=5, C=64, N=64 * 90 + 5)
    data = synth.generate(cfg, device="cpu")
    f_sb = np.array([151.3e6, 0.0, 37.25e6, -12.5e6, 240.0e6])
    f_s = 180.0e3
    delays = np.random.default_rng(3).uniform(-40e-6, 40e-6, cfg.S)
    mode = cobalt.COBALT_MODE_TENSOR_FP16 if mode_tensor else cobalt.COBALT_MODE_EXACT_FP32
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=mode) as cor:
        cor.set_chunk_subbands(2)
        cor.set_subband_frequencies(f_sb)
        cor.set_sample_rate(f_s)                     # a ladder the caller has set is kept
        vg = cor.process(data["samples"].to(dev), torch.from_numpy(delays).to(dev), data["bandpass"].to(dev)).cpu().numpy()
    bp = data["bandpass"].numpy().astype(np.float64)
    for b in range(cfg.B):
        vo = oracle.process_subband(data["samples"].numpy()[b], cfg.C, delays, bp, float(f_sb[b]), f_s=f_s)
        _assert_parity(vg[b], vo, mode_tensor, f"custom ladder, subband {b}")
    # the ladder matters: subband 0 with the default frequency is a different answer
    wrong = oracle.process_subband(data["samples"].numpy()[0], cfg.C, delays, bp, oracle.default_subband_frequency(0), f_s=f_s)
    assert err_frobenius(vg[0], wrong) > 10 * TOL_TENSOR


def test_set_sample_rate_rebuilds_the_default_ladder(cobalt, oracle, dev):
    """include/cobalt.h: while the caller has not set the ladder, f_sb[s] = 100 MHz + (12 + s) f_s follows f_s."""
    synth = _synth()
    cfg = synth.scaled(synth.CONFIGS[3], S=3, B=3, C=16, N=16 * 130)
    data = synth.generate(cfg, device="cpu")
    f_s = 150.0e3
    delays = np.array([0.0, 31.7e-6, -18.2e-6])
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        cor.set_sample_rate(f_s)
        vg = cor.process(data["samples"].to(dev), torch.from_numpy(delays).to(dev), data["bandpass"].to(dev)).cpu().numpy()
    bp = data["bandpass"].numpy().astype(np.float64)
    for b in range(cfg.B):
        vo = oracle.process_subband(data["samples"].numpy()[b], cfg.C, delays, bp, 100.0e6 + (12 + b) * f_s, f_s=f_s)
        _assert_parity(vg[b], vo, False, f"default ladder at f_s = {f_s}, subband {b}")


@pytest.mark.parametrize("S,B,C,n_t", [(77, 2, 256, 762), (40, 3, 64, 3000)])
def test_exact_mode_many_units_per_cta(cobalt, oracle, dev, S, B, C, n_t):
    """Several (stream group, time segment) units per persistent F-stage CTA in EXACT mode, where nothing paces the two FFT
    teams against each other: the FIR -> FFT hand-over uses one named barrier per (y buffer, team), so a team that runs ahead
    cannot take the other team's barrier generation (a shared barrier deadlocked here).  Sampled channels against the oracle."""
    rng = np.random.default_rng(4100 + S)
    N = n_t * C
    x = rng.integers(-500, 500, size=(B, S, 2, N, 2)).astype(np.int16)
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    with cobalt.Correlator(S, B, C, N, 16, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        vis = cor.process(torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev))
        torch.cuda.synchronize()
        vis = vis.cpu().numpy()
    for sb, j in [(0, 1), (B - 1, C // 2), (B - 1, C - 1)]:
        _, vo = oracle.channel_direct(x[sb], C, j, delays=delays, bandpass=bp.astype(np.float64), f_sb=oracle.default_subband_frequency(sb))
        _assert_parity(vis[sb, j][None], vo[None], False, f"exact mode, subband {sb}, channel {j}")
