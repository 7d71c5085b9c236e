"""Run by tests/test_bench_multirank.py under torch.distributed.run with 2 CPU ranks (gloo): exercises the host-side
multi-rank logic of bench.py (replicas only: seeds per rank, MAX over ranks, whole-job value).  No GPU, no oracle."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    local_ms = 100.0 + 25.0 * rank                       # rank 1 is the slow one
    dist.barrier()
    ms = bench.max_over_ranks(torch, dist, local_ms, device="cpu")
    out = {"rank": rank, "world": world, "seed": bench.replica_seed(rank), "ms_max": ms,
           "value": bench.aggregate_value(world, 4 * 32 ** 4, 10, ms)}
    gathered = [None] * world
    dist.all_gather_object(gathered, out)
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("RANKS " + json.dumps(gathered), flush=True)


if __name__ == "__main__":
    main()
