"""Host-side logic of the N-GPU run.  Dedispersion itself does not shard (DESIGN.md "replicas
only"): rank r dedisperses its own independently seeded beams and the job's time is the maximum
over ranks; torch.distributed carries the barrier and the timing reduction (NCCL on GPUs, gloo in
CPU tests).  The one step of the paper's pipeline that needs data from every beam is the multibeam
coincidence RFI test (one beam per GPU is the paper's deployment):
each rank counts its own beams above threshold (dedisp_rfi_beam_counts), the uint8 counts are
summed across ranks here (all-reduce over NCCL / NVLink), and every rank thresholds the sum
(dedisp_rfi_mask_from_counts)."""
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


def allreduce_beam_counts(counts, total_beams: int, group=None):
    """SUM all-reduce (in place) of the per-rank uint8 beam counts [nseries, nsamps]: afterwards every rank
    holds the number of beams of the WHOLE receiver above threshold per sample.  ``total_beams`` (all ranks
    together) must fit the uint8 counters.  Identity when not distributed.  Returns ``counts``."""
    import torch
    import torch.distributed as dist
    if total_beams > 255:
        raise ValueError("beam counts are uint8: at most 255 beams in total")
    if counts.dtype != torch.uint8:
        raise TypeError("counts must be a uint8 tensor")
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
    return counts
