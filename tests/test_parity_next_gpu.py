"""GPU parity for the rows of SURVEY.md sec 8(f) built in round 2: per-(station, pol) phase offsets (A22), dumps (A23),
valid-sample flags and counts (A24), coarse integer-sample delay (A25), pol-minor wire order (A26), 4-bit samples (A27), and
the X-stage's split time ranges.  Each case runs through the C ABI (cobalt_process_ex and the setters) and is compared
element by element with the float64 oracle on the same seeded integers, in both modes."""
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


def _data(rng, B, S, N, bits, lim=None):
    lim = lim or (2000 if bits == 16 else 100)
    x = rng.integers(-lim, lim + 1, size=(B, S, 2, N, 2)).astype(np.int16 if bits == 16 else np.int8)
    # a common signal so that the cross-correlations are not pure noise
    c = rng.integers(-lim // 2, lim // 2 + 1, size=(B, 1, 1, N, 2))
    x = np.clip(x // 2 + c, -lim, lim).astype(x.dtype)
    return x


# ------------------------------------------------------------------ phase offsets (A22)
@pytest.mark.parametrize("C,bits,S,n_t", [(64, 16, 3, 130), (256, 16, 3, 70), (256, 8, 2, 65), (16, 8, 2, 100)])
@pytest.mark.parametrize("tensor", [False, True])
def test_phase_offsets_match_oracle(cobalt, oracle, dev, C, bits, S, n_t, tensor):
    """C = 256 also exercises the one-stream-per-CTA launch (the two polarisations no longer share a rotation table)."""
    rng = np.random.default_rng(220 + C + bits)
    B, N = 2, n_t * C + 5
    x = _data(rng, B, S, N, bits)
    delays = rng.uniform(-20e-6, 20e-6, S)
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        args = (torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev))
        plain = cor.process(*args).cpu().numpy()
        cor.reset()
        cor.set_phase_offsets(ph0)
        vg = cor.process(*args).cpu().numpy()
        cor.reset()
        cor.set_phase_offsets(None)
        again = cor.process(*args).cpu().numpy()
    assert np.array_equal(plain, again)                               # clearing the offsets restores the plain path
    for b in range(B):
        vo = oracle.process_subband_ext(x[b], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(b), phase0=ph0)[0]
        _check(vg[b], vo, tensor, f"phase offsets, subband {b}")
    # closed form (pin P18 on the GPU): baseline (0, 1) XX turns by phase0[1][X] - phase0[0][X]
    bl = oracle.baseline_index(0, 1)
    turn = np.exp(1j * (ph0[1, 0] - ph0[0, 0]))
    big = np.abs(plain[0, :, bl, 0, 0]) > 0.2 * np.abs(plain[0, :, bl, 0, 0]).max()
    np.testing.assert_allclose(vg[0, big, bl, 0, 0], plain[0, big, bl, 0, 0] * turn, rtol=5e-3 if tensor else 1e-4)


# ------------------------------------------------------------------ dumps (A23), flags and counts (A24)
@pytest.mark.parametrize("C,bits,S,n_t,D", [(64, 16, 5, 256, 4), (16, 16, 3, 200, 2), (256, 8, 2, 130, 3), (64, 8, 4, 640, 5)])
@pytest.mark.parametrize("tensor", [False, True])
def test_dumps_flags_and_counts_match_oracle(cobalt, oracle, dev, C, bits, S, n_t, D, tensor):
    rng = np.random.default_rng(230 + C + D)
    B, N = 3, n_t * C
    x = _data(rng, B, S, N, bits)
    delays = rng.uniform(-5e-6, 5e-6, S)
    bp = np.ones(C, dtype=np.float32)
    n_tiles = -(-n_t // 64)
    valid = (rng.uniform(size=(B, S, n_tiles)) > 0.3).astype(np.uint8)
    valid[0] = 1                                                      # subband 0: nothing lost
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        cor.set_chunk_subbands(2)
        args = (torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev))
        one = cor.process(*args).cpu().numpy()                        # [B][C][n_bl][2][2]
        cor.reset()
        cor.set_dumps(D)
        assert cor.info.dumps == D and cor.info.n_tiles == n_tiles
        counts = torch.zeros((B, D, cor.info.n_baselines), dtype=torch.int32, device=dev)
        vg = cor.process(*args, valid=torch.from_numpy(valid).to(dev), valid_counts=counts).cpu().numpy()   # [D][B][...]
        cor.reset()
        nof = cor.process(*args).cpu().numpy()                        # dumps, no flags
    assert vg.shape == (D, B, C, S * (S + 1) // 2, 2, 2)
    for b in range(B):
        vo = oracle.process_subband_ext(x[b], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(b),
                                        valid=valid[b], dumps=D)
        for d in range(D):
            _check(vg[d, b], vo[d], tensor, f"dump {d}, subband {b}")
        np.testing.assert_array_equal(counts[b].cpu().numpy(), oracle.valid_counts(S, n_t, valid[b], D))
    # nothing lost in subband 0: the flagged call equals the unflagged one bit for bit, and the dumps add up to the block
    assert np.array_equal(vg[:, 0], nof[:, 0])
    scale = np.abs(one[0]).max()
    assert np.max(np.abs(nof[:, 0].sum(axis=0) - one[0])) <= (2e-3 if tensor else 2e-5) * scale


def test_dumps_must_divide_the_tile_count(cobalt, dev):
    with cobalt.Correlator(2, 1, 16, 16 * 200, 16) as cor:            # 4 tiles
        with pytest.raises(Exception, match="divide"):
            cor.set_dumps(3)
        cor.set_dumps(4)


# ------------------------------------------------------------------ coarse integer-sample delay (A25)
@pytest.mark.parametrize("C,bits,n_t", [(64, 16, 150), (256, 8, 66), (16, 16, 130)])
@pytest.mark.parametrize("tensor", [False, True])
def test_coarse_delays_match_oracle_over_two_calls(cobalt, oracle, dev, C, bits, n_t, tensor):
    """Offsets that are and are not multiples of 16 bytes (bulk-copy and element-wise load paths); the second call
    carries the history of the shifted streams."""
    rng = np.random.default_rng(250 + C)
    B, S, N, margin = 2, 4, n_t * C + 3, 24
    offsets = np.array([0, 8, 5, 23], dtype=np.int32)
    xs = [_data(rng, B, S, N + margin, bits) for _ in range(2)]
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    with cobalt.Correlator(S, B, C, N, bits, mode=_mode(cobalt, tensor)) as cor:
        with pytest.raises(Exception):
            cor.set_coarse_delays(offsets, N + 10)                    # 23 + N > allocated
        cor.set_coarse_delays(offsets, N + margin)
        assert cor.info.samples_allocated == N + margin
        got = [cor.process(torch.from_numpy(x).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev)).cpu().numpy()
               for x in xs]
    for b in range(B):
        hist = oracle.new_history(S, C)
        for call, x in enumerate(xs):
            vo = oracle.process_subband(oracle.coarse_shift(x[b], offsets, N), C, delays, bp.astype(np.float64),
                                        oracle.default_subband_frequency(b), hist)
            _check(got[call][b], vo, tensor, f"coarse delays, call {call}, subband {b}")


# ------------------------------------------------------------------ pol-minor order (A26) and 4-bit samples (A27)
@pytest.mark.parametrize("tail", [9, 8, 4])      # N a multiple of 8 / of 4 only / odd: the 16-byte and the element-wise re-ordering
@pytest.mark.parametrize("bits", [16, 8])
def test_pol_minor_input_is_bit_identical_to_planar(cobalt, oracle, dev, bits, tail):
    rng = np.random.default_rng(260 + bits)
    B, S, C, N = 2, 3, 64, 64 * 70 + tail
    x = _data(rng, B, S, N, bits)                                     # planar [B][S][2][N][2]
    xm = np.ascontiguousarray(x.transpose(0, 1, 3, 2, 4))             # pol-minor [B][S][N][2][2]
    assert np.array_equal(oracle.pol_minor_to_planar(xm[0]), x[0])
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    d, b_ = torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev)
    with cobalt.Correlator(S, B, C, N, bits) as cor:
        a = cor.process(torch.from_numpy(x).to(dev), d, b_).cpu().numpy()
        cor.reset()
        cor.set_input_layout(cobalt.COBALT_LAYOUT_POL_MINOR)
        m = cor.process(torch.from_numpy(xm).to(dev), d, b_, layout=cobalt.COBALT_LAYOUT_POL_MINOR).cpu().numpy()
        m2 = cor.process(torch.from_numpy(xm).to(dev), d, b_, layout=cobalt.COBALT_LAYOUT_POL_MINOR).cpu().numpy()
    assert np.array_equal(a, m)                                       # a pure re-ordering: bit for bit
    assert not np.array_equal(m, m2)                                  # (the second call carries history)
    vo = oracle.process_subband(x[1], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(1))
    _check(m[1], vo, True, "pol-minor input")


def test_p21_unpack_4bit_every_byte_on_gpu(cobalt, oracle, dev):
    b = np.arange(256, dtype=np.uint8)
    b = np.concatenate([b, b[::-1], b[:5]])
    got = cobalt.unpack(torch.from_numpy(b).to(dev)).cpu().numpy()
    assert np.array_equal(got.astype(np.float64), oracle.unpack4(b))


@pytest.mark.parametrize("layout_minor", [False, True])
@pytest.mark.parametrize("tensor", [False, True])
def test_4bit_samples_match_oracle(cobalt, oracle, dev, layout_minor, tensor):
    rng = np.random.default_rng(270)
    B, S, C, N = 2, 3, 64, 64 * 80 + 6
    x = rng.integers(0, 256, size=(B, S, 2, N)).astype(np.uint8)      # every nibble pattern incl. -8
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    lay = cobalt.COBALT_LAYOUT_POL_MINOR if layout_minor else cobalt.COBALT_LAYOUT_PLANAR
    xin = np.ascontiguousarray(x.transpose(0, 1, 3, 2)) if layout_minor else x
    with cobalt.Correlator(S, B, C, N, 4, mode=_mode(cobalt, tensor)) as cor:
        cor.set_input_layout(lay)
        vg = cor.process(torch.from_numpy(xin).to(dev), torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev),
                         layout=lay).cpu().numpy()
    for b in range(B):
        vo = oracle.process_subband_ext(x[b], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(b))[0]
        _check(vg[b], vo, tensor, f"4-bit, subband {b}")


# ------------------------------------------------------------------ X-stage: split time ranges, all rows together
def test_split_time_ranges_match_oracle_and_unsplit_result(cobalt, oracle, dev):
    """One subband x 64 channels = 64 problems on 148 SMs: the tensor X-stage splits every channel's k-range over several
    CTAs and adds the partial blocks; a plan with many subbands (no split) must agree to rounding."""
    rng = np.random.default_rng(280)
    S, C, n_t = 6, 64, 64 * 12
    N = n_t * C
    x = _data(rng, 1, S, N, 16)
    delays = rng.uniform(-1e-6, 1e-6, S)
    bp = np.ones(C, dtype=np.float32)
    d, b_ = torch.from_numpy(delays).to(dev), torch.from_numpy(bp).to(dev)
    with cobalt.Correlator(S, 1, C, N, 16) as cor:
        v1 = cor.process(torch.from_numpy(x).to(dev), d, b_).cpu().numpy()
    x8 = np.repeat(x, 8, axis=0)
    with cobalt.Correlator(S, 8, C, N, 16) as cor:
        cor.set_subband_frequencies(np.full(8, oracle.default_subband_frequency(0)))
        v8 = cor.process(torch.from_numpy(x8).to(dev), d, b_).cpu().numpy()
    vo = oracle.process_subband(x[0], C, delays, bp.astype(np.float64), oracle.default_subband_frequency(0))
    _check(v1[0], vo, True, "split k-range")
    assert np.max(np.abs(v1[0] - v8[3])) <= 1e-5 * np.abs(vo).max()   # fp32 sums split differently, same operands


@pytest.mark.parametrize("tensor", [False, True])
def test_every_row_at_once(cobalt, oracle, dev, tensor):
    """Time-varying delay + phase offsets + coarse delays + flags + dumps in one cobalt_process_ex call."""
    rng = np.random.default_rng(290)
    B, S, C, n_t, D, margin = 2, 3, 64, 256, 2, 16
    N = n_t * C
    offsets = np.array([4, 0, 11], dtype=np.int32)
    x = _data(rng, B, S, N + margin, 16)
    tau_b = rng.uniform(-2e-6, 2e-6, S)
    tau_e = tau_b + rng.uniform(-1, 1, S) * 0.3 / 1.0e8
    bp = (1 + 0.1 * rng.uniform(-1, 1, C)).astype(np.float32)
    ph0 = rng.uniform(-np.pi, np.pi, (S, 2))
    valid = (rng.uniform(size=(B, S, 4)) > 0.25).astype(np.uint8)
    with cobalt.Correlator(S, B, C, N, 16, mode=_mode(cobalt, tensor)) as cor:
        cor.set_coarse_delays(offsets, N + margin)
        cor.set_phase_offsets(ph0)
        cor.set_dumps(D)
        counts = torch.zeros((B, D, cor.info.n_baselines), dtype=torch.int32, device=dev)
        vg = cor.process(torch.from_numpy(x).to(dev), torch.from_numpy(tau_b).to(dev), torch.from_numpy(bp).to(dev),
                         delays_end=torch.from_numpy(tau_e).to(dev), valid=torch.from_numpy(valid).to(dev),
                         valid_counts=counts).cpu().numpy()
    for b in range(B):
        vo = oracle.process_subband_ext(oracle.coarse_shift(x[b], offsets, N), C, tau_b, bp.astype(np.float64),
                                        oracle.default_subband_frequency(b), delays_end=tau_e, phase0=ph0, valid=valid[b], dumps=D)
        for d in range(D):
            _check(vg[d, b], vo[d], tensor, f"all rows, dump {d}, subband {b}")
        np.testing.assert_array_equal(counts[b].cpu().numpy(), oracle.valid_counts(S, n_t, valid[b], D))
