"""Seeded synthetic LOFAR-shaped inputs for tests and bench (BASELINE.json configs 1-5).

This module holds NONE of the method's arithmetic (no FIR, no channeliser, no correlator): it only
draws station voltages with the shapes, value distributions and correlation structure of the
paper's workloads (sec 5, Table 5; recipe in DESIGN.md "Input recipe", readings
A14-A16).  It stands in for real LOFAR station data, which is not available.  Both the CUDA path and
the oracle are fed the SAME integer arrays produced here (copied, never regenerated).

Everything is torch so the big configs can be drawn on the GPU; pass device="cpu" for CPU tests.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import torch

F_S = 195312.5
C_LIGHT = 299792458.0
SEED0 = 180104834


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    S: int
    B: int
    C: int
    N: int
    bits: int
    sigma: float
    common_power: float      # fraction of the per-stream power that is the common sky signal (A15)
    max_delay: float         # seconds
    ripple: float            # bandpass ripple amplitude
    kind: str                # "tone" | "sky" | "sources"

    @property
    def n_t(self):
        return self.N // self.C

    @property
    def n_bl(self):
        return self.S * (self.S + 1) // 2

    @property
    def input_bytes(self):
        return self.B * self.S * 2 * self.N * 2 * (self.bits // 8)

    @property
    def output_bytes(self):
        return self.B * self.C * self.n_bl * 4 * 8


CONFIGS = {
    1: Config(1, "tiny-fx", 4, 1, 16, 4096, 16, 100.0, 0.0, 0.0, 0.0, "tone"),
    2: Config(2, "lofar-core-like", 48, 1, 64, 196608, 16, 100.0, 0.10, 2e-6, 0.0, "sky"),
    3: Config(3, "full-array-16bit", 77, 244, 256, 195312, 16, 100.0, 0.10, 50e-6, 0.1, "sky"),
    4: Config(4, "full-array-8bit", 77, 488, 64, 195312, 8, 16.0, 0.10, 50e-6, 0.0, "sky"),
    5: Config(5, "large-n-stress", 288, 1, 64, 196608, 16, 100.0, 0.0, 0.0, 0.0, "sources"),
    # not a BASELINE.json config: the beamformer workload of P:L111 ("127 time domain data streams using all 48 core antenna
    # fields in 16-bit mode at full bandwidth"), at the 256 channels per subband of P:L362; same recipe as config 3
    6: Config(6, "beamformer-core-16bit", 48, 244, 256, 195312, 16, 100.0, 0.10, 2e-6, 0.1, "sky"),
}


def default_subband_frequency(s: int) -> float:
    return 100.0e6 + (12 + s) * F_S


def scaled(cfg: Config, **kw) -> Config:
    """A smaller instance of a config (fewer subbands / samples) with the same recipe."""
    d = dict(cfg.__dict__)
    d.update(kw)
    return Config(**d)


def _crandn(shape, gen, device):
    return torch.complex(torch.randn(shape, generator=gen, device=device, dtype=torch.float32),
                         torch.randn(shape, generator=gen, device=device, dtype=torch.float32))


def _delay(common_f, d_samples, N):
    """common_f: FFT of [..., N]; returns the sequences delayed by d_samples[a] (circular phase ramp)."""
    k = torch.fft.fftfreq(N, device=common_f.device, dtype=torch.float64)
    ph = -2.0 * math.pi * (d_samples.to(torch.float64)[:, None] * k[None, :])
    ramp = torch.polar(torch.ones_like(ph), ph).to(torch.complex64)          # [A][N]
    return torch.fft.ifft(common_f[None, ...] * ramp[:, None, :], dim=-1)     # [A][2][N]


def _quantise(x, cfg: Config):
    lim_lo, lim_hi = (-32768, 32767) if cfg.bits == 16 else (-127, 127)     # A14; config 4: clip to [-127, 127]
    q = torch.view_as_real(x).round().clamp_(lim_lo, lim_hi)
    return q.to(torch.int16 if cfg.bits == 16 else torch.int8)


def geometry(cfg: Config, device="cpu"):
    """Seeded per-config constants: delays handed to the library, bandpass, source geometry."""
    gen = torch.Generator(device="cpu").manual_seed(SEED0 + cfg.index)
    out = {}
    if cfg.kind == "sky":
        tau = torch.rand(cfg.S, generator=gen, dtype=torch.float64) * cfg.max_delay
        out["tau_true"] = tau                       # delay of the sky signal at each station
        out["delays"] = -tau                        # what the library is asked to apply (flattens the phase)
    elif cfg.kind == "sources":
        r = 1500.0 * torch.sqrt(torch.rand(cfg.S, generator=gen, dtype=torch.float64))
        th = 2 * math.pi * torch.rand(cfg.S, generator=gen, dtype=torch.float64)
        x, y = r * torch.cos(th), r * torch.sin(th)
        lm = (torch.rand(3, 2, generator=gen, dtype=torch.float64) * 2 - 1) * 0.3 / math.sqrt(2.0)
        tau_src = (x[None, :] * lm[:, 0:1] + y[None, :] * lm[:, 1:2]) / C_LIGHT      # [3][S]
        out["tau_src"] = tau_src
        out["powers"] = torch.tensor([0.10, 0.05, 0.02], dtype=torch.float64)
        out["delays"] = -tau_src[0]                 # track source 1
    else:
        out["delays"] = torch.zeros(cfg.S, dtype=torch.float64)
    if cfg.ripple > 0:
        out["bandpass"] = (1.0 + cfg.ripple * (torch.rand(cfg.C, generator=gen, dtype=torch.float64) * 2 - 1)).to(torch.float32)
    else:
        out["bandpass"] = torch.ones(cfg.C, dtype=torch.float32)
    return {k: v.to(device) for k, v in out.items()}


def beam_delays(cfg: Config, n_beams: int, device="cpu") -> torch.Tensor:
    """Seeded tied-array beam delays tau[b][a] (seconds), [n_beams][S] float64: beam 0 is the phase centre, the others are
    plane-wave offsets over stations in a 1 km disc, up to ~1 degree off (a few tens of ns)."""
    gen = torch.Generator(device="cpu").manual_seed(SEED0 + 77 * cfg.index + n_beams)
    r = 1000.0 * torch.sqrt(torch.rand(cfg.S, generator=gen, dtype=torch.float64))
    th = 2 * math.pi * torch.rand(cfg.S, generator=gen, dtype=torch.float64)
    x, y = r * torch.cos(th), r * torch.sin(th)
    lm = (torch.rand(n_beams, 2, generator=gen, dtype=torch.float64) * 2 - 1) * 0.017
    lm[0] = 0.0
    return ((x[None, :] * lm[:, 0:1] + y[None, :] * lm[:, 1:2]) / C_LIGHT).contiguous().to(device)


def generate_subband(cfg: Config, sb: int, device="cpu", geo=None) -> torch.Tensor:
    """Samples of one subband, [S][2][N][2] int16/int8, seeded by (config, subband)."""
    geo = geo if geo is not None else geometry(cfg, device)
    gen = torch.Generator(device=device).manual_seed(SEED0 * 1000 + cfg.index * 100000 + sb)
    S, N = cfg.S, cfg.N
    noise = _crandn((S, 2, N), gen, device)
    if cfg.kind == "tone":
        # A16: complex exponential at the centre of output channel 5, amplitude 200, all streams
        n = torch.arange(N, device=device, dtype=torch.float64)
        nu = (5 - cfg.C // 2) / cfg.C
        tone = torch.polar(torch.full_like(n, 200.0), 2 * math.pi * nu * n).to(torch.complex64)
        x = cfg.sigma * noise + tone[None, None, :]
    elif cfg.kind == "sky":
        f_sb = default_subband_frequency(sb)
        common = _crandn((2, N), gen, device)
        tau = geo["tau_true"].to(device)
        sky = _delay(torch.fft.fft(common, dim=-1), tau * F_S, N)
        fringe = torch.polar(torch.ones_like(tau), -2 * math.pi * torch.frac(f_sb * tau)).to(torch.complex64)
        sky = sky * fringe[:, None, None]
        rho = cfg.common_power
        x = cfg.sigma * (math.sqrt(1 - rho) * noise + math.sqrt(rho) * sky)
    else:
        f_sb = default_subband_frequency(sb)
        x = noise.clone()
        for s in range(3):
            common = _crandn((2, N), gen, device)
            tau = geo["tau_src"][s].to(device)
            sky = _delay(torch.fft.fft(common, dim=-1), tau * F_S, N)
            fringe = torch.polar(torch.ones_like(tau), -2 * math.pi * torch.frac(f_sb * tau)).to(torch.complex64)
            x = x + math.sqrt(float(geo["powers"][s])) * sky * fringe[:, None, None]
        x = cfg.sigma * x
    return _quantise(x, cfg)


def generate(cfg: Config, device="cpu", out: torch.Tensor | None = None):
    """All subbands: dict(samples [B][S][2][N][2], delays [S] f64, bandpass [C] f32)."""
    geo = geometry(cfg, device)
    dt = torch.int16 if cfg.bits == 16 else torch.int8
    if out is None:
        out = torch.empty((cfg.B, cfg.S, 2, cfg.N, 2), dtype=dt, device=device)
    for sb in range(cfg.B):
        out[sb].copy_(generate_subband(cfg, sb, device, geo))
    return {"samples": out, "delays": geo["delays"].contiguous(), "bandpass": geo["bandpass"].contiguous()}
