"""Worker of tests/test_replicas_gloo.py: one of two `gloo` ranks exercising bench.py's replica logic on the CPU."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from workloads import make_config  # noqa: E402


def main():
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # every rank builds its own replica: different seeds -> different fields, same shape
    seed = bench.replica_seed(5, rank, world)
    w = make_config(5, n=16, seed=seed)
    digest = float(np.asarray(w.n0[0], np.float64).sum())
    all_digests = [None] * world
    dist.all_gather_object(all_digests, digest)
    # the job's time is the slowest rank's; its value counts every replica's units
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, "cpu")
    value = bench.whole_job_value(16 ** 3 * w.G, 5, world, ms)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"seeds_differ": len(set(all_digests)) == world, "ms": ms, "value": value, "world": world,
                          "seed0": bench.replica_seed(5, 0, 1), "units": 16 ** 3 * w.G}), flush=True)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
