"""Replica-level plumbing for N > 1 (the path shards only by frame; no data-path collective).
Host logic only: which frames a rank renders and how per-rank device times become one whole-job number."""
import torch
import torch.distributed as dist


def frames_of_rank(n_frames, rank, world):
    """Contiguous split of a frame sequence over ranks; the first (n_frames % world) ranks get one more."""
    base, extra = divmod(n_frames, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of per-rank numbers (device times in ms) over the default process group."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_fps(ms_per_step_local, world, device="cpu"):
    """Weak scaling: every rank renders one frame per step; job rate = world frames per slowest rank's step time."""
    ms = max_over_ranks([ms_per_step_local], device)[0]
    return world * 1e3 / ms, ms
