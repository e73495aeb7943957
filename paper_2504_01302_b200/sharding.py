"""Multi-GPU use of the path: parameter vectors are independent, so a batch is cut into contiguous chunks,
one per rank, with static data replicated and NO data-path collective.  The only exchange a
sampler needs is the all-gather of B log-likelihood floats, done here with torch.distributed (NCCL on GPUs,
gloo in the CPU tests)."""
from __future__ import annotations

import torch


def shard_range(B: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous chunk [lo, hi) of a batch of B vectors for `rank`; sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(B, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def gather_loglike(local: torch.Tensor, B: int, rank: int, world: int, dist=None) -> torch.Tensor:
    """All-gather the per-rank log-likelihood chunks into the full [B] vector (ragged chunks padded by one)."""
    if world == 1:
        return local.clone()
    import torch.distributed as d
    dist = dist or d
    width = -(-B // world)
    buf = torch.full((width,), float("nan"), dtype=local.dtype, device=local.device)
    buf[: local.numel()] = local
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf)
    out = torch.empty(B, dtype=local.dtype, device=local.device)
    for r in range(world):
        lo, hi = shard_range(B, r, world)
        out[lo:hi] = parts[r][: hi - lo]
    return out
