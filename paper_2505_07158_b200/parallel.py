"""Multi-GPU plumbing of bench.py: the path shards by frame with no exchange step, so the only
cross-rank operations are the timing barrier and the max-over-ranks reduction.  No cipher arithmetic lives here; the
helpers work on any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests)."""
from __future__ import annotations

from . import synth


def rank_clip_config(cfg: "synth.Config", rank: int, frames: int) -> "synth.Config":
    """Weak scaling: rank r encrypts its own clip of the same shape (seed shifted by 100 r), at least `frames` long."""
    return synth.Config(cfg.name, cfg.w, cfg.h, max(frames, cfg.frames), cfg.seed + 100 * rank, cfg.kind, cfg.sigma,
                        cfg.batch, cfg.n_streams)


def max_over_ranks(values, device="cpu"):
    """Element-wise maximum of a list of floats over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_rate(world: int, frames_per_rank: int, steps: int, seconds: float) -> float:
    """Frames per second of the whole job: every rank processed frames_per_rank * steps frames in `seconds` (max over ranks)."""
    return world * frames_per_rank * steps / seconds
