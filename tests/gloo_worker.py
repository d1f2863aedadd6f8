"""Worker of tests/test_multiproc.py: one rank of a world_size-2 gloo job on CPU.

Exercises the only cross-rank logic the N > 1 path has ("replicas only"):
per-rank replica seeds, MAX-over-ranks timings, SUM-over-ranks counts, barrier."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist  # noqa: E402

import bench  # noqa: E402
from paper_2106_11286_b200 import workloads  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    cfg = workloads.CONFIGS["c4"]
    seed = bench.replica_seed(cfg, rank)
    # rank r pretends its timed region took 10 + 5 r ms and launched 100 + r kernels
    (ms, ms_sweeps), (launches, attempts) = bench.reduce_over_ranks(
        [10.0 + 5.0 * rank, 8.0 - rank], [100 + rank, 1000 * (rank + 1)], "cpu")
    (dt,), none = bench.reduce_over_ranks([0.5 * (rank + 1)], [], "cpu")
    seeds = [None] * world
    dist.all_gather_object(seeds, seed)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"world": world, "ms": ms, "ms_sweeps": ms_sweeps, "launches": launches,
                          "attempts": attempts, "dt": dt, "none": none, "seeds": seeds}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
