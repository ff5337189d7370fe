"""Worker of tests/test_multirank_gloo.py: one rank of a world_size-2 gloo job on CPU.  Exercises
the host logic bench.py's N > 1 path uses (replicas only): the round-robin deal of
sources and the MAX-time / SUM-work reduction.  Writes one JSON file per rank."""
import json
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def main():
    out_dir = sys.argv[1]
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    steps, nsrc = 3, 4
    mine = [bench.source_for(rank, steps, k, nsrc) for k in range(steps)]
    # rank r "takes" (r + 1) seconds and does (10 * (r + 1), 7) units of work
    secs, work = bench.reduce_over_ranks(torch, dist, world, float(rank + 1), [10 * (rank + 1), 7], "cpu")
    dist.barrier()
    with open(os.path.join(out_dir, "rank%d.json" % rank), "w") as f:
        json.dump({"rank": rank, "world": world, "sources": mine, "secs": secs, "work": work}, f)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
