"""Worker of tests/test_multirank.py: one rank of a world_size-2 gloo job on CPU.  Exercises the
multi-rank plumbing of bench.py (max-over-ranks timing, whole-job value, rank-0-only reference arm)."""
import json
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    dev = torch.device("cpu")
    ms = [10.0, 14.5][rank]                                   # rank 1 is the slow replica
    mx = bench.max_over_ranks(ms, world, dev)
    val = bench.job_value(1000, 3, world, mx)
    dist.barrier()
    out = {"rank": rank, "world": world, "max_ms": mx, "value": val}
    with open(os.path.join(sys.argv[1], "rank%d.json" % rank), "w") as f:
        json.dump(out, f)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
