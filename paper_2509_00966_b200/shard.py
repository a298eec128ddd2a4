"""Domain sharding across ranks: divide-and-conquer domains are independent inside a
time step, so a multi-GPU job gives every rank a contiguous block of domains and
its own handle; there is no collective on the data path.  Host-side index logic only."""
from __future__ import annotations

from typing import Tuple


def domain_block(ndom_total: int, rank: int, world: int) -> Tuple[int, int]:
    """[first, last) global domain indices owned by `rank`: blocks differ in size by at most one."""
    if not (0 <= rank < world) or ndom_total < 0:
        raise ValueError("bad rank/world/ndom")
    base, extra = divmod(ndom_total, world)
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


def weak_scaling_block(ndom_per_rank: int, rank: int) -> Tuple[int, int]:
    """bench.py's weak-scaling layout: every rank owns `ndom_per_rank` domains with global indices
    (= generator seeds) rank*ndom_per_rank .. (rank+1)*ndom_per_rank."""
    return rank * ndom_per_rank, (rank + 1) * ndom_per_rank
