"""Host-side plumbing for N > 1 processes (one per GPU).  The path runs on one GPU by construction (BASELINE.json
north_star): a single lattice is stepped as N independent replicas, a batch of specimens
(BASELINE.json configs[3]) is split into contiguous specimen ranges, one per rank.  There is no data-path collective;
torch.distributed is used only for the barrier and for the max-over-ranks of the device-measured time."""
from __future__ import annotations

from typing import Sequence, Tuple


def shard_units(n_units: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced split of n_units independent units: rank r gets [lo, hi); sizes differ by at most 1 and
    the first (n_units % world) ranks get the larger share."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_over_ranks(values: Sequence[float], op: str = "max", dist=None, device=None):
    """Element-wise max / sum of per-rank float values over all ranks (identity when not distributed)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device or "cpu")
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return [float(v) for v in t.cpu()]
