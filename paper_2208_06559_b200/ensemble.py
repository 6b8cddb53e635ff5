"""Multi-GPU plumbing for the ensemble: chains never interact (PAPER.md:66, :166,
:301), so ranks own contiguous blocks of GLOBAL chain ids and exchange only the 2 x NOBS ensemble
accumulator.  No arithmetic of the method lives here; works with any torch.distributed backend."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard(rank: int, world: int, chains_per_rank: int) -> int:
    """global id of this rank's local chain 0 (weak scaling: every rank owns chains_per_rank chains)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return rank * chains_per_rank


def reduce_ensemble(ens: torch.Tensor) -> torch.Tensor:
    """sum the [2][NOBS] accumulator (row 0 sums, row 1 sums of squares) over all ranks, in place."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(ens, op=dist.ReduceOp.SUM)
    return ens


def max_over_ranks(value: float, device=None) -> float:
    """device-timed milliseconds -> max over ranks (the slowest rank defines the step time)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([value], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())
    return float(value)


def mean_and_se(ens: torch.Tensor, n_chains_total: int):
    """ensemble mean and standard error of every observable from the reduced accumulator."""
    mean = ens[0] / n_chains_total
    var = torch.clamp(ens[1] / n_chains_total - mean * mean, min=0.0)
    return mean, torch.sqrt(var / n_chains_total)
