"""Host-side plumbing of the multi-GPU path: replicas only.

The standard variant of one image does not shard (a halo exchange per family step would be needed), so
N GPUs run N independent replicas; a batched stack shards by frame.  No collective touches the data path:
torch.distributed is used for the barrier and for the max-over-ranks time only.
"""
from __future__ import annotations


def frame_shard(batch: int, rank: int, world: int) -> tuple[int, int]:
    """(first frame, frame count) of `rank` when `batch` independent frames are split over `world` ranks."""
    if not (0 <= rank < world) or batch < 0:
        raise ValueError("bad rank / world / batch")
    base, extra = divmod(batch, world)
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def shard_workload(y, rank: int, world: int):
    """The part of a workload `rank` projects and how the job scales.

    A stack of independent frames [B,H,W] with B >= world is split by frame (strong scaling: the job is the whole
    stack; no collective, every frame's output stays on its rank).  A single image, or fewer frames than ranks,
    does not shard: every rank runs a replica of the whole workload (weak scaling).
    Returns (y_part, first_frame, n_frames_total_in_job, scaling)."""
    if getattr(y, "ndim", 0) == 3 and y.shape[0] >= world and world > 1:
        first, count = frame_shard(int(y.shape[0]), rank, world)
        return y[first:first + count], first, int(y.shape[0]), "strong"
    frames = int(y.shape[0]) if getattr(y, "ndim", 0) == 3 else 1
    return y, 0, frames * world, "weak"


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Max of a per-rank scalar (device time of the timed region); identity without a process group."""
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Whole-job throughput: units processed by all ranks / max-over-ranks time."""
    return units_per_rank * world / seconds_max
