#!/usr/bin/env python
"""bench.py -- one JSON line for the Cobalt correlator hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A step is one pass of the whole hot path (cobalt_process: phase table -> unpack+FIR+FFT+rotate+
bandpass+transpose -> history carry -> correlate, every subband) over one integration period of
synthetic LOFAR-shaped input.  Default workload: BASELINE.json's full-array 16-bit config (77 stations,
244 subbands, 256 channels, 195312 samples), the one the north_star targets are stated on; it fits one
GPU.  `value` = baseline*channel*samples per second of the whole job with inputs resident in HBM;
`e2e` = the same through cobalt_process_host (pinned host buffers, H2D/D2H inside the timed region).
With N > 1 (torchrun) every rank runs the same workload on its own GPU (the path shards by subband
with no exchange step: replicas, weak scaling) and value aggregates over ranks on the max time.

`--impl reference` times the float64 CPU oracle (oracle/, as it stands) on a bounded sample of the
same workload; it is a deliberately slow baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

F_S = 195312.5
METRIC = "baseline-channel-samples/s"
UNIT = "baseline*channel*samples/s"
# SURVEY.md sec 8(d) / DESIGN.md: algorithmic HBM bytes of the F-stage per complex sample per pol
# (raw input + 16-bit complex intermediate) and algorithmic flops of the X-stage per baseline-sample.
F_BYTES_PER_SAMPLE = {16: 4 + 4, 8: 2 + 4}
X_FLOP_PER_BASELINE_SAMPLE = 32


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (1-5)")
    ap.add_argument("--subbands", type=int, default=0, help="override the number of subbands (debugging)")
    ap.add_argument("--mode", default="tensor", choices=["tensor", "exact"])
    ap.add_argument("--interp", action="store_true",
                    help="time cobalt_process_interp (delay running linearly over the block, SURVEY.md sec 8(f) row 1)")
    ap.add_argument("--layout", default="planar", choices=["planar", "pol-minor"],
                    help="order of the samples: pol-minor = LOFAR's wire order, which goes through the ingest pre-pass (one extra read + write of the input)")
    ap.add_argument("--chunk", type=int, default=0, help="subbands per launch group (0 = library default)")
    ap.add_argument("--beamform", default="", choices=["", "stokes-i", "iquv", "voltages", "incoherent"],
                    help="time cobalt_beamform (SURVEY.md sec 8(f) row 4) on the beamformer workload (synth config 6) instead")
    ap.add_argument("--beams", type=int, default=127)
    ap.add_argument("--t-int", type=int, default=16)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args(argv)


# ----------------------------------------------------------------------------- multi-process plumbing
def dist_setup():
    """(rank, world_size, local_rank); initialises torch.distributed when launched by torchrun."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist

        if not dist.is_initialized():
            backend = "nccl" if torch.cuda.is_available() else "gloo"
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def dist_barrier():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max(x: float, device=None) -> float:
    """Max over ranks of a per-rank scalar (the job takes as long as its slowest rank)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Replicas (weak scaling): every rank processed units_per_rank in at most seconds_max."""
    return units_per_rank * world / seconds_max


# ----------------------------------------------------------------------------- clocks during the timed region
class ClockSampler(threading.Thread):
    def __init__(self, index: int, period: float = 0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown",
            nv.nvmlClocksThrottleReasonApplicationsClocksSetting: "applications_clocks_setting",
        }
        while not self._halt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            self._halt.wait(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        s, w = sorted(self.samples), sorted(self.power)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "power_w": w[len(w) // 2] if w else None, "power_w_max": w[-1] if w else None}


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:  # noqa: BLE001
            return local_rank
    return local_rank


# ----------------------------------------------------------------------------- roofline denominators
def measured_peaks():
    """MEASURED_PEAKS.json (driver-written) or the fallback B200_PROFILING.md states."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "tensor_tflops_burst": float(d["bf16_tflops"]),
                "tensor_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    except Exception:  # noqa: BLE001
        return {"hbm_gbs": 6650.0, "tensor_tflops_burst": 1590.0, "tensor_tflops_sustained": 1400.0, "source": "fallback"}


def stored_traffic(key: str):
    """DRAM bytes per launch of a kernel from the committed `ncu --set full` capture named in profiles/traffic.json.
    bench.py cannot run ncu on itself, so the figure is a stored one: it is only reported while the kernel's source
    file still has the sha256 recorded with the capture; otherwise None (and `traffic_source` says why)."""
    import hashlib

    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            ent = json.load(f).get(key)
        if not isinstance(ent, dict):
            return None, "no capture recorded"
        with open(os.path.join(ROOT, ent["file"]), "rb") as f:
            sha = hashlib.sha256(f.read()).hexdigest()
        if sha != ent["sha256"]:
            return None, f"stale: {ent['file']} changed since {ent['source']}"
        return ent["bytes"], ent["source"]
    except Exception as e:  # noqa: BLE001
        return None, f"unavailable: {e!r}"


def workload(args):
    from paper_1801_04834_b200 import synth

    cfg = synth.CONFIGS[6 if (args.beamform and args.config == 3) else args.config]
    if args.subbands > 0:
        cfg = synth.scaled(cfg, B=args.subbands)
    return cfg


def units_per_step(cfg) -> float:
    """baseline * channel * samples of one step: n_bl * B * N_u (N_u = n_t * C consumed samples)."""
    return float(cfg.n_bl) * cfg.B * (cfg.n_t * cfg.C)


# ----------------------------------------------------------------------------- the oracle leg (CPU)
def oracle_sample(cfg, steps: int, warmup: int):
    """Times oracle.process_subband on the first, middle and last subband of the workload (one
    subband when the workload has fewer than three), zero history, the first n_t_sample spectra of each, per step;
    the throughput is the sample's and stands, extrapolated linearly, for the whole config.
    Returns (units/s, seconds per step, description, threads)."""
    import numpy as np

    import oracle
    from paper_1801_04834_b200 import synth

    oracle.build()
    sbs = sorted({0, cfg.B // 2, cfg.B - 1})
    # bound the sample to roughly 10-30 s of CPU work: ~1.2e11 naive flop (DFT 8 C^2 + X 32 n_bl per spectrum-channel)
    flop_per_spectrum = 2 * cfg.S * 8.0 * cfg.C * cfg.C + 32.0 * cfg.n_bl * cfg.C
    n_t_s = int(max(16, min(cfg.n_t, 1.2e11 // (flop_per_spectrum * len(sbs)))))
    sub = synth.scaled(cfg, B=1, N=n_t_s * cfg.C)
    geo = synth.geometry(cfg, "cpu")
    samples = [synth.generate_subband(cfg, sb, "cpu", geo)[:, :, : sub.N, :].contiguous().numpy() for sb in sbs]
    delays = geo["delays"].numpy()
    bandpass = geo["bandpass"].numpy().astype(np.float64)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        for sb, x in zip(sbs, samples):
            oracle.process_subband(x, cfg.C, delays, bandpass, oracle.default_subband_frequency(sb))
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    sec = sum(times) / len(times)
    units = float(cfg.n_bl) * n_t_s * cfg.C * len(sbs)
    desc = (f"oracle.process_subband on subbands {sbs} of {cfg.B}, first {n_t_s} of {cfg.n_t} spectra of each "
            f"({cfg.S} stations, {cfg.C} channels); float64, direct FIR, naive O(C^2) DFT, per-baseline loops; "
            f"throughput of the sample, extrapolated linearly to the whole config")
    return units / sec, sec, desc, oracle.num_threads()


def run_reference(args, rank, world):
    if rank != 0:
        return 0
    cfg = workload(args)
    value, sec, desc, threads = oracle_sample(cfg, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "stations": cfg.S, "subbands": cfg.B, "channels": cfg.C, "samples": cfg.N,
                   "input_bits": cfg.bits, "note": "each step is a bounded sample of the workload (see cpu_baseline.sample)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------- the CUDA leg
def host_budget_bytes(world_local: int) -> int:
    try:
        with open("/proc/meminfo") as f:
            for ln in f:
                if ln.startswith("MemAvailable:"):
                    return int(int(ln.split()[1]) * 1024 * 0.55 / max(1, world_local))
    except Exception:  # noqa: BLE001
        pass
    return 8 << 30


def run_ours(args, rank, world, local):
    import torch

    import paper_1801_04834_b200 as pkg
    from paper_1801_04834_b200 import synth

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl ours needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    pkg.load()
    cfg = workload(args)
    peaks = measured_peaks()
    mode = pkg.COBALT_MODE_TENSOR_FP16 if args.mode == "tensor" else pkg.COBALT_MODE_EXACT_FP32

    # ---- synthetic input, generated on the device subband by subband
    data = synth.generate(cfg, device=dev)
    samples, delays, bandpass = data["samples"], data["delays"], data["bandpass"]
    torch.cuda.synchronize()

    cor = pkg.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=mode)
    if args.chunk > 0:
        cor.set_chunk_subbands(args.chunk)
    layout = pkg.COBALT_LAYOUT_PLANAR
    if args.layout == "pol-minor":
        # the same samples in the wire order [B][S][N][2 pol][2], re-ordered in place subband by subband (untimed)
        minor = samples.view(cfg.B, cfg.S, cfg.N, 2, 2)
        for b in range(cfg.B):
            minor[b].copy_(samples[b].permute(0, 2, 1, 3).contiguous())
        samples = minor
        layout = pkg.COBALT_LAYOUT_POL_MINOR
        cor.set_input_layout(layout)
        torch.cuda.synchronize()
    info = cor.info
    vis = torch.empty(cor.vis_shape(), dtype=torch.complex64, device=dev)
    stream = torch.cuda.current_stream()
    cor.set_timing(True)

    # --interp: a LOFAR-like drift of 0.15 cycles of the first subband's centre frequency over the block
    delays_end = (delays + 0.15 / 1.0e8) if args.interp else None
    for _ in range(args.warmup):
        cor.process(samples, delays, bandpass, out=vis, delays_end=delays_end, layout=layout)
    torch.cuda.synchronize()

    sampler = ClockSampler(physical_gpu_index(local))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    kt = [0.0, 0.0, 0.0, 0.0]
    launches = 0
    dist_barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev[0].record(stream)
    for i in range(args.steps):
        cor.process(samples, delays, bandpass, out=vis, delays_end=delays_end, layout=layout)
        ev[i + 1].record(stream)
        ms = cor.get_kernel_timing()          # waits for this step's events (device time per kernel)
        for k in range(4):
            kt[k] += ms[k]
        launches += ms[4]
    torch.cuda.synchronize()
    dist_barrier()
    clocks = sampler.stop()
    total_ms = ev[0].elapsed_time(ev[-1])
    sec_step = dist_max(total_ms / 1e3 / args.steps, dev)
    # SURVEY.md sec 8(d) asks for the median of the timed calls next to the mean: under the board's power cap the clock
    # wanders from step to step, which the mean hides
    step_ms = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps))
    med_ms = step_ms[len(step_ms) // 2] if len(step_ms) % 2 else 0.5 * (step_ms[len(step_ms) // 2 - 1] + step_ms[len(step_ms) // 2])
    sec_step_median = dist_max(med_ms / 1e3, dev)
    step_ms_min, step_ms_max = step_ms[0], step_ms[-1]
    n_chunks = (cfg.B + info.chunk_subbands - 1) // info.chunk_subbands
    t_phase, t_f, t_hist, t_x = (dist_max(v / 1e3 / args.steps, dev) for v in kt)

    units = units_per_step(cfg)
    value = whole_job_value(units, world, sec_step)
    n_samples = float(cfg.B) * 2 * cfg.S * (cfg.n_t * cfg.C)               # complex samples per pol-stream
    f_bytes = n_samples * F_BYTES_PER_SAMPLE[cfg.bits] if args.mode == "tensor" else n_samples * (cfg.bits // 4 + 8)
    x_flop = units * X_FLOP_PER_BASELINE_SAMPLE
    f_kernel = "fstage_kernel"
    tr_f, tr_f_src = stored_traffic(f_kernel) if (cfg.name == "full-array-16bit" and args.mode == "tensor") else (None, "captured for config 3 only")
    tr_x, tr_x_src = stored_traffic("xstage_tc_kernel") if (cfg.name == "full-array-16bit" and args.mode == "tensor") else (None, "captured for config 3 only")
    roof_f = {"kernel": f_kernel, "bound": "hbm", "achieved": f_bytes / t_f / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
              "frac": f_bytes / t_f / 1e9 / peaks["hbm_gbs"], "traffic": tr_f, "traffic_source": tr_f_src,
              "peak_source": peaks["source"], "ms_per_launch": t_f * 1e3 / n_chunks, "launches_per_step": n_chunks,
              "algorithmic_bytes_per_launch": f_bytes / n_chunks}
    # the F-stage is bound by FP32 dispatch, not by HBM: the same launches against the FP32 peak
    import math
    f_flop = n_samples * (64 + 5 * math.log2(cfg.C) + 8)
    alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
    roof_alu = {"kernel": f_kernel, "bound": "alu", "achieved": f_flop / t_f / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                "frac": f_flop / t_f / 1e12 / alu_peak, "traffic": None,
                "peak_source": "nominal, not measured: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz (DESIGN.md); the run's clock is in `clocks`",
                "algorithmic_flop_per_sample": 64 + 5 * math.log2(cfg.C) + 8}
    if clocks and clocks.get("sm_mhz"):
        # the same figure against the FP32 peak at the clock this run actually held (median of the samples under load)
        roof_alu["frac_at_run_clock"] = roof_alu["achieved"] / (148 * 128 * 2 * clocks["sm_mhz"] * 1e6 / 1e12)
    roof_x = {"kernel": "xstage_tc_kernel" if args.mode == "tensor" else "xstage_simt_kernel", "bound": "tensor",
              "achieved": x_flop / t_x / 1e12, "peak": peaks["tensor_tflops_sustained"], "unit": "TFLOP/s",
              "frac": x_flop / t_x / 1e12 / peaks["tensor_tflops_sustained"],
              "traffic": tr_x, "traffic_source": tr_x_src,
              "peak_source": peaks["source"] + " (sustained bf16; fp16 runs at the same rate)",
              "ms_per_launch": t_x * 1e3 / n_chunks, "launches_per_step": n_chunks,
              "algorithmic_flop_per_launch": x_flop / n_chunks,
              "hbm_gbs": (n_samples * 4 + cfg.output_bytes) / t_x / 1e9}
    dominant, other = (roof_f, roof_x) if t_f >= t_x else (roof_x, roof_f)

    # ---- end to end through the public host-buffer call (pinned host memory, H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e and not args.interp and args.layout == "planar":
        e2e = run_e2e(args, cfg, cor, samples, delays, bandpass, world, dev)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, sec, desc, threads = oracle_sample(cfg, 1, 0)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc, "seconds": sec}

    cor.close()
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": sec_step * 1e3, "ms_per_step_median": sec_step_median * 1e3, "ms_per_step_min": step_ms_min,
            "ms_per_step_max": step_ms_max, "value_at_median": whole_job_value(units, world, sec_step_median), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (fp16 tensor-core operands, fp32 accumulate; fp64 phase angles)" if args.mode == "tensor" else "f32",
            "data": "synthetic",
            "config": {"workload": cfg.name, "stations": cfg.S, "subbands": cfg.B, "channels": cfg.C, "taps": 16,
                       "samples_per_integration": cfg.N, "input_bits": cfg.bits, "baselines": cfg.n_bl, "mode": args.mode, "layout": args.layout,
                       "call": "cobalt_process_interp" if args.interp else "cobalt_process",
                       "chunk_subbands": info.chunk_subbands, "parallelism": "replicas" if world > 1 else "single-gpu",
                       "l2": f"inputs ({cfg.input_bytes / 1e9:.2f} GB per step) exceed the 126 MB L2; no flush needed"},
            "roofline": dominant, "roofline_other": other, "roofline_alu": roof_alu,
            "stage_ms": {"phase_table": t_phase * 1e3, "f_stage": t_f * 1e3, "history": t_hist * 1e3, "x_stage": t_x * 1e3},
            "x_stage": {"baseline_channel_samples_per_s": units / t_x, "visibility_gflops": x_flop / t_x / 1e9},
            "f_stage": {"ppf_input_gbs": cfg.input_bytes / t_f / 1e9, "samples_per_s": n_samples / t_f},
            "real_time_factor": (cfg.n_t * cfg.C / F_S) / sec_step,
            "clocks": clocks, "gpu_launches": int(launches), "e2e": e2e, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    return 0


def oracle_beamform_sample(cfg, beam_delays, product, n_stokes, t_int, pkg):
    """The oracle (as it stands) on a bounded sample of the beamformer workload: the first subband, the first 2 t_int-blocks of
    at least 32 spectra; float64, direct FIR, naive DFT, a cos/sin per (beam, station, channel, spectrum) term."""
    import numpy as np

    import oracle
    from paper_1801_04834_b200 import synth

    oracle.build()
    n_t_s = max(32, 2 * t_int)
    geo = synth.geometry(cfg, "cpu")
    x = synth.generate_subband(cfg, 0, "cpu", geo)[:, :, : n_t_s * cfg.C, :].contiguous().numpy()
    t0 = time.perf_counter()
    z = oracle.channelise_subband(x, cfg.C, geo["delays"].numpy(), geo["bandpass"].numpy().astype(np.float64), oracle.default_subband_frequency(0))
    if product == pkg.COBALT_BF_COHERENT_VOLTAGES:
        oracle.beamform_coherent(z, beam_delays, oracle.default_subband_frequency(0))
    elif product == pkg.COBALT_BF_COHERENT_STOKES:
        oracle.coherent_stokes(z, beam_delays, oracle.default_subband_frequency(0), n_stokes, t_int)
    else:
        oracle.incoherent_stokes(z, n_stokes, t_int)
    sec = time.perf_counter() - t0
    units = float(beam_delays.shape[0]) * n_t_s * cfg.C
    return {"value": units / sec, "unit": "beam*channel*samples/s", "cores": oracle.num_threads(), "kind": "oracle", "seconds": sec,
            "sample": f"oracle channeliser + beamformer on subband 0 of {cfg.B}, first {n_t_s} of {cfg.n_t} spectra ({cfg.S} stations, "
                      f"{cfg.C} channels, {beam_delays.shape[0]} beams); float64, naive DFT, a cos/sin per term; throughput of the sample, "
                      "extrapolated linearly to the whole workload"}


def run_beamform(args, rank, world, local):
    """`--beamform`: one step = one cobalt_beamform over the whole beamformer workload (F-stage + beamformer kernel)."""
    import torch

    import paper_1801_04834_b200 as pkg
    from paper_1801_04834_b200 import synth

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl ours needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    pkg.load()
    cfg = workload(args)
    peaks = measured_peaks()
    product = {"stokes-i": pkg.COBALT_BF_COHERENT_STOKES, "iquv": pkg.COBALT_BF_COHERENT_STOKES,
               "voltages": pkg.COBALT_BF_COHERENT_VOLTAGES, "incoherent": pkg.COBALT_BF_INCOHERENT_STOKES}[args.beamform]
    n_stokes = 4 if args.beamform == "iquv" else 1
    t_int = 1 if args.beamform == "voltages" else args.t_int
    n_beams = 1 if args.beamform == "incoherent" else args.beams
    if args.beamform == "voltages" and args.subbands <= 0:      # complex voltages of 127 beams: 0.4 GB per subband
        cfg = synth.scaled(cfg, B=32)
    data = synth.generate(cfg, device=dev)
    samples, delays, bandpass = data["samples"], data["delays"], data["bandpass"]
    bd = synth.beam_delays(cfg, n_beams, dev)
    cor = pkg.Correlator(cfg.S, cfg.B, cfg.C, cfg.N, cfg.bits, mode=pkg.COBALT_MODE_TENSOR_FP16 if args.mode == "tensor" else pkg.COBALT_MODE_EXACT_FP32)
    if args.chunk > 0:
        cor.set_chunk_subbands(args.chunk)
    info = cor.info
    shape, dt = cor.beamform_shape(product, n_beams, n_stokes, t_int)
    out = torch.empty(shape, dtype=getattr(torch, dt), device=dev)
    stream = torch.cuda.current_stream()
    cor.set_timing(True)
    call = lambda: cor.beamform(samples, delays, bandpass, product, beam_delays=bd, n_stokes=n_stokes, t_int=t_int, out=out)  # noqa: E731
    for _ in range(args.warmup):
        call()
    torch.cuda.synchronize()
    sampler = ClockSampler(physical_gpu_index(local))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    kt = [0.0, 0.0, 0.0, 0.0]
    launches = 0
    dist_barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev[0].record(stream)
    for _ in range(args.steps):
        call()
        ms = cor.get_kernel_timing()
        for k in range(4):
            kt[k] += ms[k]
        launches += ms[4]
    ev[1].record(stream)
    torch.cuda.synchronize()
    dist_barrier()
    clocks = sampler.stop()
    sec_step = dist_max(ev[0].elapsed_time(ev[1]) / 1e3 / args.steps, dev)
    t_phase, t_f, t_hist, t_b = (dist_max(v / 1e3 / args.steps, dev) for v in kt)
    n_chunks = (cfg.B + info.chunk_subbands - 1) // info.chunk_subbands
    n_cs = float(cfg.B) * cfg.n_t * cfg.C                                    # channel-samples per polarisation stream
    units = n_beams * n_cs
    out_bytes = out.numel() * out.element_size()
    z_bytes = n_cs * 2 * cfg.S * 4                                           # fp16 re + im of every input, read once
    f_bytes = n_cs * 2 * cfg.S * F_BYTES_PER_SAMPLE[cfg.bits]
    b_flop = 8.0 * cfg.S * 2 * n_beams * n_cs if product != pkg.COBALT_BF_INCOHERENT_STOKES else 0.0   # complex MAC per (beam, pol, station)
    roof_f = {"kernel": "fstage_kernel", "bound": "hbm", "achieved": f_bytes / t_f / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
              "frac": f_bytes / t_f / 1e9 / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"],
              "ms_per_launch": t_f * 1e3 / n_chunks, "launches_per_step": n_chunks, "algorithmic_bytes_per_launch": f_bytes / n_chunks}
    bname = "incoherent_kernel" if product == pkg.COBALT_BF_INCOHERENT_STOKES else ("bf_tc_kernel" if args.mode == "tensor" else "bf_simt_kernel")
    roof_b = {"kernel": bname, "bound": "hbm", "achieved": (z_bytes + out_bytes) / t_b / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
              "frac": (z_bytes + out_bytes) / t_b / 1e9 / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"],
              "ms_per_launch": t_b * 1e3 / n_chunks, "launches_per_step": n_chunks,
              "algorithmic_bytes_per_launch": (z_bytes + out_bytes) / n_chunks,
              "tensor_tflops": b_flop / t_b / 1e12, "tensor_frac_of_sustained_peak": b_flop / t_b / 1e12 / peaks["tensor_tflops_sustained"],
              "note": "algorithmic flops = 8 per (beam, polarisation, station, channel-sample); the kernel issues twice that (the weight rows are zero on the other polarisation)"}
    dominant, other = (roof_f, roof_b) if t_f >= t_b else (roof_b, roof_f)
    cor.close()
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_beamform_sample(cfg, bd.cpu().numpy(), product, n_stokes, t_int, pkg)
    if rank == 0:
        line = {
            "metric": "beam-channel-samples/s", "value": whole_job_value(units, world, sec_step), "unit": "beam*channel*samples/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_step * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (fp16 tensor-core operands, fp32 accumulate; fp64 phase angles)" if args.mode == "tensor" else "f32",
            "data": "synthetic",
            "config": {"workload": cfg.name, "call": "cobalt_beamform", "product": args.beamform, "stations": cfg.S, "subbands": cfg.B,
                       "channels": cfg.C, "beams": n_beams, "n_stokes": n_stokes, "t_int": t_int, "samples_per_integration": cfg.N,
                       "input_bits": cfg.bits, "mode": args.mode, "chunk_subbands": info.chunk_subbands,
                       "l2": f"inputs ({cfg.input_bytes / 1e9:.2f} GB per step) exceed the 126 MB L2; no flush needed"},
            "roofline": dominant, "roofline_other": other,
            "stage_ms": {"phase_table": t_phase * 1e3, "f_stage": t_f * 1e3, "history": t_hist * 1e3, "beamform": t_b * 1e3},
            "real_time_factor": (cfg.n_t * cfg.C / F_S) / sec_step, "output_bytes": out_bytes,
            "clocks": clocks, "gpu_launches": int(launches), "e2e": None, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    return 0


def run_e2e(args, cfg, cor, samples, delays, bandpass, world, dev):
    import torch

    import paper_1801_04834_b200 as pkg
    from paper_1801_04834_b200 import synth

    in_b, out_b = cfg.input_bytes // cfg.B, cfg.output_bytes // cfg.B
    budget = host_budget_bytes(world)
    b_e2e = int(max(1, min(cfg.B, budget // (in_b + out_b))))
    steps = min(args.steps, 5)
    if b_e2e == cfg.B:
        c2, own = cor, False
        c2.reset()
    else:
        c2, own = pkg.Correlator(cfg.S, b_e2e, cfg.C, cfg.N, cfg.bits, mode=cor.info.mode), True
    c2.set_timing(False)
    h_in = torch.empty((b_e2e,) + tuple(samples.shape[1:]), dtype=samples.dtype, pin_memory=True)
    h_in.copy_(samples[:b_e2e])
    h_out = torch.empty((b_e2e,) + tuple(cor.vis_shape()[1:]), dtype=torch.complex64, pin_memory=True)
    h_del, h_bp = delays.cpu(), bandpass.cpu()
    torch.cuda.synchronize()
    for _ in range(min(args.warmup, 3)):
        c2.process_host(h_in, h_del, h_bp, h_out)
    dist_barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        c2.process_host(h_in, h_del, h_bp, h_out)       # synchronous: returns when the visibilities are in h_out
    torch.cuda.synchronize()
    sec = dist_max((time.perf_counter() - t0) / steps, dev)
    dist_barrier()
    sub = synth.scaled(cfg, B=b_e2e)
    out = {"value": whole_job_value(units_per_step(sub), world, sec), "unit": UNIT,
           "h2d_bytes_per_step": int(h_in.numel() * h_in.element_size() + 8 * cfg.S + 4 * cfg.C),
           "d2h_bytes_per_step": int(h_out.numel() * h_out.element_size()), "ms_per_step": sec * 1e3, "steps": steps,
           "subbands": b_e2e, "api": "cobalt_process_host (pinned host buffers, chunked H2D / compute / D2H overlap)",
           "real_time_factor": (cfg.n_t * cfg.C / F_S) / sec,
           "pcie_gbs": (h_in.numel() * h_in.element_size() + h_out.numel() * h_out.element_size()) / sec / 1e9}
    if own:
        c2.close()
    del h_in, h_out
    return out


def main(argv=None):
    args = parse_args(argv)
    if args.impl == "reference":
        # rank 0 alone runs the oracle; the other ranks exit 0 without work and no process group is formed
        rank = int(os.environ.get("RANK", "0"))
        return run_reference(args, rank, int(os.environ.get("WORLD_SIZE", "1")))
    rank, world, local = dist_setup()
    rc = run_beamform(args, rank, world, local) if args.beamform else run_ours(args, rank, world, local)
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
    return rc


if __name__ == "__main__":
    sys.exit(main())
