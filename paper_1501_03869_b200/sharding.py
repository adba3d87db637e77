"""Multi-GPU plumbing of the path: frames are independent in Eq. 7, so the path
shards over frames with NO data-path collective -- every rank owns a table copy and its own frames.
Only the timing is reduced (max over ranks).  Host logic only; no arithmetic of the method."""


def rank_frame_range(rank: int, world: int, frames_per_rank: int):
    """Weak scaling: rank r owns global frames [r*frames_per_rank, (r+1)*frames_per_rank)."""
    if not (0 <= rank < world) or frames_per_rank < 0:
        raise ValueError("bad rank / world / frames_per_rank")
    return rank * frames_per_rank, (rank + 1) * frames_per_rank


def split_frames(nframes: int, world: int):
    """Strong scaling: contiguous, balanced split of nframes frames; returns [(begin, end)] per rank."""
    if nframes < 0 or world < 1:
        raise ValueError("bad nframes / world")
    return [(nframes * r // world, nframes * (r + 1) // world) for r in range(world)]


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Device time of a multi-rank step = max over ranks (torch.distributed all_reduce MAX)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
