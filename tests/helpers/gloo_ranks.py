"""Two-rank CPU (gloo) exercise of bench.py's multi-process logic: max-over-ranks and the replica aggregate."""
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import bench  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
mine = [10.0 + rank, 5.0 - rank, 1.0 + 0.5 * rank]
got = bench.max_over_ranks(mine, world, torch.device("cpu"))
assert got == [10.0 + world - 1, 5.0, 1.0 + 0.5 * (world - 1)], got
p = bench.make_problem("C0", rank)
other = bench.make_problem("C0", (rank + 1) % world)
assert p.seed != other.seed and p.state_steps == other.state_steps   # independent replicas, same size
if rank == 0:
    print("RATE", bench.aggregate_rate(p.state_steps, 4, world, got[0]))
dist.barrier()
dist.destroy_process_group()
