"""bench.py's N > 1 path on CPU: world_size-2 gloo (replicas only, the only collectives are the
barrier and the max-reduction of the timing), and the reference arm's rank-0-only rule."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(script_args, world, extra_env=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable] + script_args, cwd=ROOT, env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_world_size_2_gloo_max_over_ranks_and_aggregate():
    outs = _spawn([os.path.join(ROOT, "tests", "dist_worker.py")], 2)
    res = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda r: r["rank"])
    assert [r["rank"] for r in res] == [0, 1] and all(r["world"] == 2 for r in res)
    for r in res:
        assert abs(r["sec_max"] - 0.020) < 1e-12          # the slowest rank's time, on every rank
        assert abs(r["value"] - 2 * 1000.0 / 0.020) < 1e-6  # replicas: units of all ranks / max time


def test_reference_arm_runs_on_rank_0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 without work."""
    outs = _spawn([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--config", "1"], 2)
    lines0 = [ln for ln in outs[0].splitlines() if ln.startswith("{")]
    assert len(lines0) == 1 and outs[1].strip() == ""
    d = json.loads(lines0[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "tiny-fx"


def test_single_process_helpers_without_a_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.dist_max(0.5) == 0.5
    assert bench.whole_job_value(10.0, 4, 2.0) == 20.0
    args = bench.parse_args([])
    assert args.gpus == 1 and args.config == 3 and args.warmup >= 3


def test_beamformer_bench_host_side():
    """bench.py --beamform without a GPU: argument parsing, the workload it selects (synth config 6) and the oracle leg of its
    cpu_baseline on a scaled-down instance."""
    sys.path.insert(0, ROOT)
    import bench
    import paper_1801_04834_b200 as pkg
    from paper_1801_04834_b200 import synth

    args = bench.parse_args(["--beamform", "stokes-i", "--beams", "5", "--t-int", "4"])
    cfg = bench.workload(args)
    assert cfg.name == "beamformer-core-16bit" and (cfg.S, cfg.C) == (48, 256)
    small = synth.scaled(cfg, S=3, B=1, C=16, N=16 * 64)
    bd = synth.beam_delays(small, 5, "cpu").numpy()
    assert bd.shape == (5, 3) and abs(bd[0]).max() == 0.0              # beam 0 is the phase centre
    r = bench.oracle_beamform_sample(small, bd, pkg.COBALT_BF_COHERENT_STOKES, 1, 4, pkg)
    assert r["kind"] == "oracle" and r["value"] > 0 and r["cores"] >= 1
