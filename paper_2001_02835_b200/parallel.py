"""Direction split of the TEK staple over ranks.

The paper's only parallel scheme assigns the four directions mu of the TEK model to four GPUs: every star-product stays inside
one card, and the link series are exchanged once per molecular-dynamics step.  This module is that scheme for the one step of
the path this library owns, the staple: every rank holds all four link series U_mu (replicated), computes S_mu for the
directions it owns with ``nspt_staple_dir`` -- no collective inside a product -- and one all-gather makes all four S_mu (or,
in an NSPT driver, the four updated links: same shape, same call) available on every rank.

One process per GPU, ``torch.distributed`` for the plumbing (NCCL over NVLink on GPUs; the host logic below is backend
agnostic and is tested with gloo on CPU tensors and an injected compute function).  world sizes 1, 2 and 4 are supported:
rank r owns the directions mu with mu % world == r.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence

__all__ = ["owned_directions", "all_gather_series", "staple_direction_split"]


def owned_directions(rank: int, world: int) -> List[int]:
    """Directions of rank `rank`: mu % world == rank (world in {1, 2, 4})."""
    if world not in (1, 2, 4):
        raise ValueError("the four directions split over 1, 2 or 4 ranks")
    if not 0 <= rank < world:
        raise ValueError("rank out of range")
    return [mu for mu in range(4) if mu % world == rank]


def all_gather_series(owned: Sequence, rank: int, world: int, group=None) -> list:
    """All-gather of per-direction series: `owned` holds this rank's series in the order of owned_directions(rank, world);
    returns the four series in direction order on every rank.  4/world tensors of (Ntrunc+1) x N x N complex128 leave each
    rank (207 MB in all at N = 225, N_trunc = 63)."""
    import torch
    import torch.distributed as dist
    mine = owned_directions(rank, world)
    if len(owned) != len(mine):
        raise ValueError("one series per owned direction expected")
    if world == 1:
        return list(owned)
    local = torch.stack(list(owned))                       # (4/world, n, N, N)
    parts = [torch.empty_like(local) for _ in range(world)]
    dist.all_gather(parts, local, group=group)
    out: list = [None] * 4
    for r in range(world):
        for i, mu in enumerate(owned_directions(r, world)):
            out[mu] = parts[r][i]
    return out


def staple_direction_split(U: Sequence, z, rank: Optional[int] = None, world: Optional[int] = None, group=None,
                           compute: Optional[Callable] = None) -> list:
    """[S_0, S_1, S_2, S_3] of eq. 2.3 on every rank, each S_mu computed by the rank that owns direction mu.

    U: the four link series, replicated on every rank.  compute(U, z, mu) -> S_mu defaults to ``nspt_staple_dir`` on the
    current CUDA device; tests inject a CPU implementation."""
    import torch.distributed as dist
    if world is None:
        world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
    if rank is None:
        rank = dist.get_rank(group) if world > 1 else 0
    if compute is None:
        from . import binding as nspt
        compute = nspt.nspt_staple_dir
    owned = [compute(U, z, mu) for mu in owned_directions(rank, world)]
    return all_gather_series(owned, rank, world, group)
