"""Worker for test_bench_dist.py: exercises bench.py's N>1 plumbing (replicas only) under gloo on CPU."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import torch  # noqa: E402

import bench  # noqa: E402

world, rank, local = bench.dist_setup(int(os.environ["WORLD_SIZE"]))
assert world == int(os.environ["WORLD_SIZE"]) and rank == int(os.environ["RANK"])
bench.barrier(world)
# device-time aggregation: the slowest replica defines the step time
m = bench.max_over_ranks(1.5 + rank, world, torch.device("cpu"))
assert m == 1.5 + (world - 1), m
# whole-job value = replicas * iterations / max time
value = world * 20 * 4 / m
bench.barrier(world)
if rank == 0:
    print(f"DIST_OK world={world} max={m} value={value}")
