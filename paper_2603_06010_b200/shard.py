"""Multi-GPU plumbing: the path shards over the templates (rows of H), nothing else.

Each template's log-likelihood depends only on (d, h_b, handle state), so B rows are split into
contiguous slices, one per rank; every rank builds its own handle (O(N) state, replicated) and
writes its slice of `out`.  There is NO data-path collective (the paper's own
parallelism is a process pool over proposals).  `gather_out` is an
optional convenience for callers that want the whole vector on every rank: one all_gather of
8*B bytes.  No arithmetic of the method lives here.
"""
from __future__ import annotations

from typing import List, Tuple


def row_slice(B: int, rank: int, world: int) -> Tuple[int, int]:
    """[lo, hi) of the rows of H owned by `rank`: contiguous, balanced to within one row,
    the first B % world ranks take the extra row.  Empty slices are legal (B < world)."""
    if B < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad shard request B={B} rank={rank} world={world}")
    q, r = divmod(B, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def all_slices(B: int, world: int) -> List[Tuple[int, int]]:
    return [row_slice(B, r, world) for r in range(world)]


def gather_out(out_local, B: int, group=None):
    """All-gather the per-rank slices of `out` into the full [B] vector (same on every rank).
    `out_local` is this rank's slice (torch tensor, any device the process group supports).
    Slices may differ in length by one row, so they are padded to the longest for the collective."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    sl = all_slices(B, world)
    lo, hi = sl[rank]
    if out_local.numel() != hi - lo:
        raise ValueError(f"rank {rank} holds {out_local.numel()} values, its slice has {hi - lo}")
    longest = max(h - l for l, h in sl)
    pad = torch.zeros(longest, dtype=out_local.dtype, device=out_local.device)
    pad[: hi - lo] = out_local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[: h - l] for p, (l, h) in zip(parts, sl)])


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Timing rule of bench.py: a multi-GPU time is the max over ranks."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
