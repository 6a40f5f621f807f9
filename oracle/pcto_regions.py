"""CPU oracle of Algorithm 1 of the paper, "multi-GPU based reconstruction".  TEST INFRASTRUCTURE ONLY:
imported by tests/ (and nothing of the product); plain numpy around the oracle's own MLP / DROP routines (pcto.py), one
function per step of the algorithm, in the paper's order and words.  Shares nothing with the CUDA path.

    1: setupImageRegions()  2: identifyProtonsPassingRegions()  3: allocateMemoryForProtonsPerGPU()
    4: iterativelySolvePerGPU()  5: selectSlice()

Readings (R28), where the paper gives an example but no formula:
  * "division of the reconstruction volume into several overlapping regions based on the number of available GPUs"
    (PAPER.md:45): the nz slices are cut into G consecutive parts of equal height (boundaries floor(g nz / G)); a region is
    its part plus `ext` slices of each neighbouring part.  The paper's example fixes this: 20 slices, 2 GPUs -> regions
    0-12 and 7-19, overlap 7-12, final image 0-9 / 10-19, i.e. ext = 3, overlap = 2 ext ("the overlap is set
    at twice the slices for a 96 % coverage", Table I: 94-96 % of the protons span at most 3 slices).
  * "each proton is associated with the image region entered to and exited from": a history belongs to
    region g if the slice of its hull entry voxel OR the slice of its hull exit voxel lies in region g; histories that A1
    rejects (no hull intersection, order, depth, non-finite record) belong to none.
  * "we select the reconstruction that is closest to the non-overlapped slices of its region": slice z of the
    final image comes from the region whose own part contains z.
Parity: pinned by tests/test_oracle_regions.py (the paper's worked example from tests/golden/, partition invariants,
membership by brute force, and the special cases G = 1 and ext >= nz that must reproduce the plain solver).
"""
from __future__ import annotations

from typing import List, Optional, Tuple

import numpy as np

from . import pcto

A1_REJECT = pcto.REJ_MISS | pcto.REJ_ORDER | pcto.REJ_DEPTH | pcto.REJ_NONFINITE


def setup_image_regions(nz: int, n_regions: int, ext: int) -> List[Tuple[int, int, int, int]]:
    """Step 1 -> [(z_lo, z_hi, keep_lo, keep_hi)] per region, half-open slice ranges."""
    if not (1 <= n_regions <= nz) or ext < 0:
        raise ValueError("need 1 <= n_regions <= nz and ext >= 0")
    cuts = [(g * nz) // n_regions for g in range(n_regions + 1)]              # own parts: [cuts[g], cuts[g+1])
    regions = []
    for g in range(n_regions):
        keep_lo, keep_hi = cuts[g], cuts[g + 1]
        z_lo = keep_lo if g == 0 else max(0, keep_lo - ext)                   # widened towards every neighbour
        z_hi = keep_hi if g == n_regions - 1 else min(nz, keep_hi + ext)
        regions.append((z_lo, z_hi, keep_lo, keep_hi))
    return regions


def hull_ends(geom, params, protons, hull, flags: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Hull entry and exit voxel (V_s, V_e of R4) of every history, -1 / -1 where A1 rejects it."""
    m = protons.m
    v_in = np.full(m, -1, dtype=np.int64)
    v_out = np.full(m, -1, dtype=np.int64)
    for i in range(m):
        if flags[i] & A1_REJECT:
            continue
        got = pcto.polyline(geom, params, protons, i, hull)
        if got is not None:
            v_in[i], v_out[i] = got[1], got[2]
    return v_in, v_out


def identify_protons_passing_region(v_in: np.ndarray, v_out: np.ndarray, slice_elems: int, z_lo: int, z_hi: int) -> np.ndarray:
    """Step 2 -> ascending indices of the histories that enter or exit the region."""
    ok = (v_in >= 0) & (v_out >= 0)
    za, zb = v_in // slice_elems, v_out // slice_elems
    inside = ((za >= z_lo) & (za < z_hi)) | ((zb >= z_lo) & (zb < z_hi))
    return np.nonzero(ok & inside)[0]


def reconstruct(geom, params, arrays: dict, u_in_mm: float, u_out_mm: float, hull: Optional[np.ndarray], b: np.ndarray,
                x0: Optional[np.ndarray], n_regions: int, ext: int, iters: int, block_size: int, lam: float):
    """Steps 1-5 -> (final image float32[n], [member indices per region], [image of every region])."""
    n = geom.nx * geom.ny * geom.nz
    slice_elems = geom.nx * geom.ny
    pa = pcto.ProtonArrays(arrays, u_in_mm, u_out_mm)
    all_paths = pcto.Paths(geom, params, pa, hull)
    flags = all_paths.rows()[3]
    v_in, v_out = hull_ends(geom, params, pa, hull, flags)
    start = np.ones(n, dtype=np.float32) if x0 is None else np.asarray(x0, dtype=np.float32).reshape(-1)
    x_final = np.zeros(n, dtype=np.float32)
    members, images = [], []
    for (z_lo, z_hi, keep_lo, keep_hi) in setup_image_regions(geom.nz, n_regions, ext):            # step 1
        idx = identify_protons_passing_region(v_in, v_out, slice_elems, z_lo, z_hi)               # step 2
        sub = {k: np.ascontiguousarray(np.asarray(v)[idx]) for k, v in arrays.items()}            # step 3: the region's own copy
        sub_b = np.ascontiguousarray(np.asarray(b, dtype=np.float32)[idx])
        if idx.size:
            paths = pcto.Paths(geom, params, pcto.ProtonArrays(sub, u_in_mm, u_out_mm), hull)
            x_g = paths.solve(sub_b, start, iters, block_size, lam)                               # step 4: no exchange
        else:
            x_g = start.copy()
        x_final[keep_lo * slice_elems: keep_hi * slice_elems] = x_g[keep_lo * slice_elems: keep_hi * slice_elems]   # step 5
        members.append(idx)
        images.append(x_g)
    return x_final, members, images
