"""Host-side logic of the N-GPU run: the path does not shard (DESIGN.md "replicas
only"), so rank r dedisperses its own independently seeded beams and the job's
time is the maximum over ranks.  No data-path collective exists; torch.distributed
carries only the barrier and the timing reduction (NCCL on GPUs, gloo in CPU tests)."""
from __future__ import annotations


def beam_indices(rank: int, nbeams_per_rank: int) -> list[int]:
    """Global beam indices (=> generator seeds/streams) owned by a rank: disjoint across ranks."""
    return [rank * nbeams_per_rank + b for b in range(nbeams_per_rank)]


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a per-rank scalar (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: int, world: int, seconds_max_over_ranks: float) -> float:
    """Whole-job aggregate: units all ranks processed / the slowest rank's time."""
    return units_per_rank * world / seconds_max_over_ranks
