"""Host-side sharding of the frame-set stream over ranks (one process per GPU).

Frame sets are independent given the rig (one depth map per synchronized frame set), so the path shards
with no data-path collective: every rank gets its own contiguous block of frames and the only communication is the
barrier and the reduction of the timing (max over ranks) and of the unit counts (sum over ranks)."""
from __future__ import annotations


def frames_for_rank(first_frame: int, frames_per_rank: int, rank: int, world: int):
    """Weak scaling: rank r owns frames [first + r*n, first + (r+1)*n)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    start = first_frame + rank * frames_per_rank
    return list(range(start, start + frames_per_rank))


def split_stream(n_frames: int, rank: int, world: int):
    """Strong scaling of a fixed stream: contiguous, balanced to within one frame, covering every frame once."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    base, extra = divmod(n_frames, world)
    start = rank * base + min(rank, extra)
    return list(range(start, start + base + (1 if rank < extra else 0)))


def reduce_timing(ms_values, unit_counts, device=None):
    """(max over ranks of each time, sum over ranks of each count); identity without torch.distributed."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(ms_values), dtype=torch.float64, device=device)
    n = torch.tensor(list(unit_counts), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [float(x) for x in n]
