"""GPU parity at BASELINE.json's FULL sizes (configs 3, 4, 5), in the launch configuration bench.py times
(default chunking, TENSOR_FP16 mode, one cobalt_process over the whole config), checked

  * on the first, the middle and the last WHOLE subband (every channel, every visibility) against
    `oracle.process_subband`, plus >= 32 seeded (subband, channel) spot checks that the oracle computes one by one
    with its single-sum form (`oracle.channel_direct`, SURVEY.md sec 8(c) pin P11 / sec 8(d)); and
  * via properties that hold at any size (finite everywhere, autocorrelations real and positive, XY of an
    autocorrelation = conj(YX), reading A9).

The whole float64 oracle on these configs would take hours; configs 1 and 2 are compared in
full in test_parity_gpu.py.  Tolerance: ||dV||_F / ||V||_F <= 2e-3 per (subband, channel) (BASELINE.json).
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


def _sampled_pairs(cfg, n_random, seed):
    """(subband, channel) pairs: corners and centre, plus seeded random ones."""
    rng = np.random.default_rng(seed)
    sbs = sorted({0, cfg.B // 2, cfg.B - 1})
    pairs = [(sbs[0], 0), (sbs[len(sbs) // 2], cfg.C // 2), (sbs[-1], cfg.C - 1)]
    for _ in range(n_random):
        pairs.append((int(rng.integers(cfg.B)), int(rng.integers(cfg.C))))
    return pairs


def _invariants(vis, S):
    """Properties of reading A9 that hold at any size; vis is a torch complex tensor [B][C][n_bl][2][2] on the GPU."""
    assert bool(torch.isfinite(torch.view_as_real(vis)).all()), "non-finite visibility"
    k = torch.arange(S, device=vis.device)
    diag = vis[:, :, k * (k + 1) // 2 + k]                         # autocorrelations [B][C][S][2][2]
    xx, yy = diag[..., 0, 0], diag[..., 1, 1]
    assert bool((xx.real > 0).all()) and bool((yy.real > 0).all()), "autocorrelation power not positive"
    scale = torch.sqrt(xx.real * yy.real)
    assert float((xx.imag.abs() / xx.real).max()) <= 1e-6 and float((yy.imag.abs() / yy.real).max()) <= 1e-6
    assert float(((diag[..., 0, 1] - diag[..., 1, 0].conj()).abs() / scale).max()) <= 1e-5, "auto XY != conj(YX)"


def _check_sampled(oracle, cfg, data, vis, pairs, mode_tensor=True):
    delays = data["delays"].cpu().numpy()
    bandpass = data["bandpass"].cpu().numpy().astype(np.float64)
    worst = 0.0
    cache = {}
    for sb, j in pairs:
        if sb not in cache:
            cache.clear()                                           # one subband of host memory at a time
            cache[sb] = data["samples"][sb].cpu().numpy()
        _, vo = oracle.channel_direct(cache[sb], cfg.C, j, delays=delays, bandpass=bandpass,
                                      f_sb=oracle.default_subband_frequency(sb))
        vg = vis[sb, j].cpu().numpy()
        e = err_frobenius(vg, vo) if mode_tensor else err_fp32(vg, vo)
        tol = TOL_TENSOR if mode_tensor else TOL_FP32
        assert e <= tol, f"{cfg.name} subband {sb} channel {j}: error {e:.3e} > {tol}"
        worst = max(worst, e)
    return worst


def _check_whole_subbands(oracle, cfg, data, vis, subbands):
    delays = data["delays"].cpu().numpy()
    bandpass = data["bandpass"].cpu().numpy().astype(np.float64)
    worst = 0.0
    for sb in subbands:
        vo = oracle.process_subband(data["samples"][sb].cpu().numpy(), cfg.C, delays, bandpass, oracle.default_subband_frequency(sb))
        e = err_frobenius(vis[sb].cpu().numpy(), vo)
        assert e <= TOL_TENSOR, f"{cfg.name} whole subband {sb}: worst channel error {e:.3e} > {TOL_TENSOR}"
        worst = max(worst, e)
    return worst


def _full_config(cobalt, oracle, dev, index, n_random, subbands=0):
    from paper_1801_04834_b200 import synth

    cfg = synth.CONFIGS[index] if subbands == 0 else synth.scaled(synth.CONFIGS[index], B=subbands)
    data = synth.generate(cfg, device=dev)
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=cobalt.COBALT_MODE_TENSOR_FP16) as cor:
        assert cor.info.n_baselines == cfg.n_bl and cor.info.n_spectra == cfg.n_t
        vis = cor.process(data["samples"], data["delays"], data["bandpass"])
        torch.cuda.synchronize()
    _invariants(vis, cfg.S)
    worst = _check_sampled(oracle, cfg, data, vis, _sampled_pairs(cfg, n_random, 1000 + index))
    worst = max(worst, _check_whole_subbands(oracle, cfg, data, vis, sorted({0, cfg.B // 2, cfg.B - 1})))
    del vis, data
    torch.cuda.empty_cache()
    return worst


def test_config3_full_array_16bit_sampled(cobalt, oracle, dev):
    """77 stations, 244 subbands, 256 channels, 195312 int16 samples: 29.4 GB in, 6.0 GB out."""
    _full_config(cobalt, oracle, dev, 3, n_random=32)


def test_config4_full_array_8bit_sampled(cobalt, oracle, dev):
    """77 stations, 488 subbands, 64 channels, 195312 int8 samples."""
    _full_config(cobalt, oracle, dev, 4, n_random=32)


def test_config5_large_n_whole(cobalt, oracle, dev):
    """288 receivers (41616 baselines), 64 channels: the multi-job tiling of the X-stage at full size; the config
    has one subband, compared in full (plus the spot checks through the other oracle routine)."""
    _full_config(cobalt, oracle, dev, 5, n_random=8)


def test_config3_exact_mode_two_chunks_sampled(cobalt, oracle, dev):
    """EXACT_FP32 mode at config 3's per-subband size, 3 subbands in chunks of 2 (ragged last chunk), 1e-4 metric."""
    from paper_1801_04834_b200 import synth

    cfg = synth.scaled(synth.CONFIGS[3], B=3)
    data = synth.generate(cfg, device=dev)
    with cobalt.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=cobalt.COBALT_MODE_EXACT_FP32) as cor:
        cor.set_chunk_subbands(2)
        vis = cor.process(data["samples"], data["delays"], data["bandpass"])
        torch.cuda.synchronize()
    _invariants(vis, cfg.S)
    _check_sampled(oracle, cfg, data, vis, [(0, 0), (1, 128), (2, 255), (2, 77)], mode_tensor=False)
