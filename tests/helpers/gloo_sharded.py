"""Two-rank CPU (gloo) exercise of the K-sharded step's host logic: shard_problem + gather_partials of the
product, with the oracle standing in for the kernels (per-shard rollouts and partials in fp64)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import oracle as O  # noqa: E402
from paper_2209_12842_b200 import sharded  # noqa: E402
from paper_2209_12842_b200 import workloads as W  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
p = W.config0(K=45, M=16, T=8, near_obstacle=True)
p = p.replace(v=W.random_mean_control(p, 0), lam=50.0, eta=0.2)       # soft weights, both eta branches live
orc = O.Oracle(p)
sp = sharded.shard_problem(p, world, rank)
k0, k1 = sp.k_offset, sp.k_offset + sp.K
assert sp.K_total == p.K and (k0, k1) == sharded.shard_bounds(p.K, world, rank)
r = orc.rollout_costs(k_begin=k0, k_end=k1)                            # the global-k rows of this rank
part = torch.from_numpy(O.shard_partial(r["S_tilde"], r["u"], p.lam))
parts = sharded.gather_partials(part)                                  # the product's collective wrapper
assert parts.shape == (world, 2 + 2 * p.T) and torch.equal(parts[rank], part)
vp = O.combine_partials(parts.numpy(), p.lam, p.u_min, p.u_max)
full = orc.rollout_costs()
ref = orc.weights_update(full["S_tilde"], full["u"])["v_plus"]
err = float(np.abs(vp - ref).max())
assert err < 1e-12, err
gathered = [None] * world
dist.all_gather_object(gathered, vp.tobytes())
assert all(g == gathered[0] for g in gathered)                         # every rank holds the same v+
if rank == 0:
    print("SHARDED_OK", err)
dist.barrier()
dist.destroy_process_group()
