"""Frame sharding for N > 1 GPUs: host-side index arithmetic only (no FIR / DFT math here).

Every output frame depends only on its own M*P input samples (Eq. (20), then a
per-frame DFT), so ranks split the work with NO data-path collective:
  * independent streams (config 4): whole streams per rank (`shard_streams`);
  * one long stream (config 5): contiguous frame ranges, each rank reading its range plus a
    read-only (M-1)*P-sample halo (`shard_frames`).
The only communication is the max-over-ranks of the elapsed time (`max_over_ranks`).
"""
from __future__ import annotations


def shard_streams(S: int, world: int, rank: int) -> range:
    """Streams [lo, hi) owned by `rank` (sizes differ by at most one)."""
    base, extra = divmod(S, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def shard_frames(n_samples: int, P: int, M: int, world: int, rank: int):
    """Contiguous frame range of one stream for `rank`.

    Returns (f_lo, f_hi, s_lo, s_hi): frames [f_lo, f_hi) of the full output are produced by
    running the PFB on samples [s_lo, s_hi) = blocks [f_lo, f_hi + M - 1).  Empty shard: f_lo == f_hi.
    """
    F = n_samples // P - M + 1
    if F < 1:
        raise ValueError("n_samples too short")
    base, extra = divmod(F, world)
    f_lo = rank * base + min(rank, extra)
    f_hi = f_lo + base + (1 if rank < extra else 0)
    if f_hi == f_lo:
        return f_lo, f_hi, 0, 0
    return f_lo, f_hi, f_lo * P, (f_hi + M - 1) * P


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar over the default process group (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
