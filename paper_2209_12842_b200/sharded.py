"""K-sharded RA-MPPI step over several GPUs, one process per GPU.

The K control samples are independent until the weights (17) PAPER.md:134, so rank g rolls out the samples
k in shard_bounds(K, world, g) (Philox counters carry the global k, so the draws do not depend on the partition),
reduces them to {beta_g, Z_g, N_g[T,2]} (ra_mppi_step_partial), one all-gather moves the 2+2T doubles of every
rank, and every rank forms the same v+ (ra_mppi_combine_partials).  The exchange is (2+2T)*8 bytes per rank
(816 B at T = 50): latency-bound, so it is a plain NCCL all-gather, not a fused kernel.

Marshalling and the collective only: all arithmetic runs in libra_mppi.so.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_bounds(K: int, world: int, rank: int):
    """Samples [k_begin, k_end) of rank `rank`: contiguous, sizes differ by at most one, larger shards first."""
    if not (0 <= rank < world) or K < world:
        raise ValueError(f"cannot shard K={K} over world={world} (rank {rank}): every rank needs >= 1 sample")
    base, extra = divmod(K, world)
    k_begin = rank * base + min(rank, extra)
    return k_begin, k_begin + base + (1 if rank < extra else 0)


def shard_problem(p, world: int, rank: int):
    """The workloads.Problem of one shard: K = its sample count, k_offset / K_total name its place."""
    k_begin, k_end = shard_bounds(p.K, world, rank)
    return p.replace(K=k_end - k_begin, k_offset=k_begin, K_total=p.K)


def gather_partials(partial: torch.Tensor, group=None) -> torch.Tensor:
    """All-gather one [2+2T] fp64 partial per rank into [world, 2+2T], row r from rank r (any backend)."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        return partial.reshape(1, -1).contiguous()
    out = torch.empty(world * partial.numel(), dtype=partial.dtype, device=partial.device)
    dist.all_gather_into_tensor(out, partial.reshape(-1).contiguous(), group=group)
    return out.view(world, partial.numel())


class ShardedRaMppi:
    """One rank of a K-sharded controller: `RaMppi` on this rank's shard + the exchange step."""

    def __init__(self, problem, device: int = 0, group=None):
        from .controller import RaMppi
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.problem = problem
        self.ctl = RaMppi(shard_problem(problem, self.world, self.rank), device=device)
        self._partial = torch.empty(2 + 2 * problem.T, device=self.ctl.device, dtype=torch.float64)

    def step(self, d_x0: torch.Tensor, d_v: torch.Tensor, iteration: int = 0):
        """In place on every rank: d_v [T,2] <- v+ of the whole K-sample problem."""
        self.ctl.step_partial(d_x0, d_v, iteration, out=self._partial)
        parts = gather_partials(self._partial, self.group)
        return self.ctl.combine_partials(parts, d_v)

    def close(self):
        self.ctl.close()
