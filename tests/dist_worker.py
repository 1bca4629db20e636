"""Worker of tests/test_bench_dist.py: one rank of a world_size-2 gloo group exercising bench.py's multi-process
plumbing (rendezvous from the torchrun environment, barrier, max-over-ranks timing, whole-job aggregation)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def main():
    rank, world, local = bench.dist_setup()
    bench.dist_barrier()
    # each rank "measures" a different step time; the job takes as long as its slowest rank
    sec = 0.010 * (rank + 1)
    sec_max = bench.dist_max(sec)
    units = 1000.0
    out = {"rank": rank, "world": world, "local": local, "sec_max": sec_max,
           "value": bench.whole_job_value(units, world, sec_max)}
    bench.dist_barrier()
    import torch.distributed as dist

    dist.destroy_process_group()
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
