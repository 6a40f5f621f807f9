"""Algorithm 1 of the paper across processes, one process per GPU (reading R28 of DESIGN.md).

Every rank holds the whole data set on its own GPU (the paper reads the preprocessed histories on every node), runs
`pct_reconstruct_regions` for ITS regions only -- hull intersection of all histories, membership, K1 and the DROP solve
on the members, slice selection -- and the kept slices are then collected: one broadcast per region from its owner.
That collection is the only transfer ("eliminating the need of data transfers among the GPUs"; "the final
image will be made of slices 0-9 from the first region and 10-19 of the second"); there is no collective on
the data path.  Only argument marshalling and torch.distributed plumbing live here; every step of Algorithm 1 runs in
libpct.so (csrc/regions.cu).
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence, Tuple

import torch
import torch.distributed as dist


def region_owner(n_regions: int, world_size: int) -> List[int]:
    """Rank that runs region g: contiguous runs of regions per rank, the first `n_regions % world_size` ranks take one
    more (with n_regions == world_size, the paper's case, rank g runs region g)."""
    if n_regions < 1 or world_size < 1:
        raise ValueError("n_regions and world_size must be positive")
    base, extra = divmod(n_regions, world_size)
    owner: List[int] = []
    for r in range(world_size):
        owner += [r] * (base + (1 if r < extra else 0))
    return owner


def my_regions(n_regions: int, rank: int, world_size: int) -> Tuple[int, int]:
    """(first region, number of regions) of `rank`; the count is 0 for ranks beyond the number of regions."""
    owner = region_owner(n_regions, world_size)
    mine = [g for g, r in enumerate(owner) if r == rank]
    return (mine[0], len(mine)) if mine else (0, 0)


def assemble_slices(x_local: torch.Tensor, keep: Sequence[Tuple[int, int]], owner: Sequence[int], slice_elems: int,
                    group=None) -> torch.Tensor:
    """selectSlice() across ranks: slices [keep_lo, keep_hi) of region g are broadcast from owner[g]; on return every rank
    holds the final image in x_local.  Works on any backend (NCCL on the GPUs, gloo on CPU tensors in the tests)."""
    for (lo, hi), src in zip(keep, owner):
        if hi > lo:
            dist.broadcast(x_local[lo * slice_elems: hi * slice_elems], src=src, group=group)
    return x_local


def reconstruct_regions_distributed(ctx, protons: Dict[str, torch.Tensor], u_in_mm: float, u_out_mm: float,
                                    hull: Optional[torch.Tensor], b: torch.Tensor, x0: Optional[torch.Tensor],
                                    ext: int, iters: int, block_size: int, lam: float, n_regions: Optional[int] = None,
                                    group=None):
    """Algorithm 1 with one region (or a run of regions) per rank.  Returns (final image on every rank, members per region
    of the regions this rank ran, -1 elsewhere)."""
    from . import binding
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    n_regions = world if n_regions is None else int(n_regions)
    regions = binding.regions_setup(ctx.geom.nz, n_regions, ext)
    first, count = my_regions(n_regions, rank, world)
    x, members = ctx.reconstruct_regions(protons, u_in_mm, u_out_mm, hull, b, x0, n_regions, ext, iters, block_size, lam,
                                         region_first=first, region_count=count)
    keep = [(r.keep_lo, r.keep_hi) for r in regions]
    assemble_slices(x, keep, region_owner(n_regions, world), ctx.geom.nx * ctx.geom.ny, group)
    return x, members
