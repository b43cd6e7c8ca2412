"""the N x N oracle pass (A1) sharded by QUERY over the ranks of one node.

The all-pairs pass is N independent queries against the same N points ("parallel
brute-force frontier oracle ... N^2 kernel"): rank r of W takes the contiguous id range
``query_slice(N, r, W)``, runs ``kc_frontier_oracle`` on it against its own copy of the positions,
and the ranks exchange the finished certificate columns (20 B per point) with one all-gather.  The
positions are never exchanged: every rank already holds them (they are the step's input), and the
O(N) rows of the step are cheap enough to run replicated.  Nothing here is arithmetic of the method:
slicing and the exchange only, on any initialised process group (nccl on the GPU box, gloo in the
CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def query_slice(n: int, rank: int, world: int) -> tuple[int, int]:
    """Ids [lo, hi) of rank ``rank``: contiguous, sizes differ by at most one, lower ranks first."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("query_slice: need world >= 1, 0 <= rank < world, n >= 0")
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def slice_width(n: int, world: int) -> int:
    """Columns of the exchange buffer: the widest slice (every rank sends the same amount)."""
    return -(-n // world)


def gather_columns(buf: torch.Tensor, n: int, group=None) -> torch.Tensor:
    """All-gather of certificate columns.  ``buf`` is this rank's (rows, >= n) tensor whose columns
    ``query_slice(n, rank, world)`` are final; on return the columns [0, n) of ``buf`` are final on
    every rank.  One collective: every rank contributes ``slice_width`` columns (the tail of a short
    slice is padding and is dropped on arrival).  Without a process group (one rank) it is a no-op."""
    if not (dist.is_available() and dist.is_initialized()):
        return buf
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    if world == 1:
        return buf
    rows, w = buf.shape[0], slice_width(n, world)
    lo, hi = query_slice(n, rank, world)
    send = torch.zeros((rows, w), dtype=buf.dtype, device=buf.device)
    send[:, : hi - lo] = buf[:, lo:hi]
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send, group=group)
    for r in range(world):
        a, b = query_slice(n, r, world)
        if r != rank:
            buf[:, a:b] = recv[r][:, : b - a]
    return buf
