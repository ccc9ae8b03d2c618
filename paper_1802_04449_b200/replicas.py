"""Host logic of the N > 1 path: the hydro step does not shard across GPUs in this build ("replicas only",
DESIGN.md section 7) -- every rank evolves its own seeded event with no data-path collective.  The only
cross-rank operations are a barrier and a MAX reduction of the device-timed interval."""
from __future__ import annotations

from . import inputs


def rank_seed(config_index: int, rank: int) -> int:
    """One seeded event per rank (variant = rank)."""
    return inputs.seed_for(config_index, variant=rank)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (nccl: pass the rank's CUDA device; gloo: device None)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(cells_per_rank: int, steps: int, ms_local: float, world: int, device=None):
    """Whole-job throughput: all ranks' cell-updates divided by the slowest rank's time.  Returns (rate, ms)."""
    ms = max_over_ranks(ms_local, device)
    return world * cells_per_rank * steps / (ms * 1e-3), ms
