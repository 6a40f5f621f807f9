"""Pins for Algorithm 1 of the paper (R28): the oracle (oracle/pcto_regions.py), the host-only
step 1 of the library (pct_regions_setup: pure arithmetic, no GPU), and the process plumbing
(paper_1802_01070_b200/regions.py) on the gloo backend with world_size 2.

What fixes the oracle here, other than itself: the region table the paper prints (tests/golden/regions_paper_example.txt);
partition invariants that hold for any (nz, G, ext); membership by brute force over all voxel pairs of a small grid; and the
two special cases in which Algorithm 1 must reproduce the plain solver (already pinned against a dense-matrix DROP in
test_oracle_solver.py): one region, and an extension that makes every region the whole volume."""
import os
import socket

import numpy as np
import pytest
import torch

import synth
from helpers import oracle_setup

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def paper_example():
    rows, meta = [], {}
    for line in open(os.path.join(ROOT, "tests", "golden", "regions_paper_example.txt")):
        if line.startswith("# nz") or line.startswith("# n_regions") or line.startswith("# overlap"):
            _, k, v = line.split()
            meta[k] = int(v)
        elif not line.startswith("#") and line.strip():
            rows.append(tuple(int(t) for t in line.split()))
    return meta, rows


@pytest.fixture(scope="module")
def regions_oracle(oracle):
    from oracle import pcto_regions
    return pcto_regions


def test_paper_example(regions_oracle):
    meta, rows = paper_example()
    assert meta == {"nz": 20, "n_regions": 2, "overlap_first": 7, "overlap_last": 12}
    got = regions_oracle.setup_image_regions(meta["nz"], meta["n_regions"], 3)
    # the fixture holds the paper's inclusive slice numbers; the oracle returns half-open ranges
    assert [(g, lo, hi - 1, klo, khi - 1) for g, (lo, hi, klo, khi) in enumerate(got)] == rows
    # overlap of the two regions = slices 7..12 = twice the extension ("the overlap is set at twice the slices")
    assert (got[1][0], got[0][1] - 1) == (meta["overlap_first"], meta["overlap_last"])
    assert got[0][1] - got[1][0] == 2 * 3
    # a plausible mistake (extension on one side only, or kept parts cut at the region edge) does not give the paper's table
    assert regions_oracle.setup_image_regions(20, 2, 2) != got and regions_oracle.setup_image_regions(20, 2, 4) != got


def test_library_step_1_prints_the_papers_table():
    """pct_regions_setup is host arithmetic: callable without a GPU."""
    from paper_1802_01070_b200 import binding
    meta, rows = paper_example()
    got = binding.regions_setup(meta["nz"], meta["n_regions"], 3)
    assert [(g, r.z_lo, r.z_hi - 1, r.keep_lo, r.keep_hi - 1) for g, r in enumerate(got)] == rows
    for bad in ((20, 0, 3), (20, 21, 0), (20, 2, -1), (0, 1, 0)):
        with pytest.raises(binding.PctError):
            binding.regions_setup(*bad)


@pytest.mark.parametrize("nz,G,ext", [(20, 2, 3), (128, 2, 4), (128, 3, 4), (160, 8, 2), (7, 7, 1), (9, 4, 0), (8, 2, 100), (5, 1, 2)])
def test_partition_invariants(regions_oracle, nz, G, ext):
    from paper_1802_01070_b200 import binding
    R = regions_oracle.setup_image_regions(nz, G, ext)
    assert len(R) == G
    kept = np.zeros(nz, dtype=int)
    for g, (lo, hi, klo, khi) in enumerate(R):
        assert 0 <= lo <= klo < khi <= hi <= nz                               # a region holds its own, non-empty part
        kept[klo:khi] += 1
        assert klo - lo == (0 if g == 0 else min(ext, klo))                   # widened by ext towards every neighbour, clipped
        assert hi - khi == (0 if g == G - 1 else min(ext, nz - khi))
        assert abs((khi - klo) - nz / G) < 1.0                                # parts of equal height up to rounding
    assert np.all(kept == 1)                                                  # the kept parts tile [0, nz) exactly once
    assert [(r.z_lo, r.z_hi, r.keep_lo, r.keep_hi) for r in binding.regions_setup(nz, G, ext)] == R


def test_membership_by_brute_force(regions_oracle):
    nx, ny, nz = 3, 2, 6
    sl = nx * ny
    n = sl * nz
    pairs = np.array([(a, b) for a in range(-1, n) for b in range(-1, n)])
    v_in, v_out = pairs[:, 0].copy(), pairs[:, 1].copy()
    rej = (v_in < 0) | (v_out < 0)
    v_in[rej] = -1; v_out[rej] = -1                                           # A1 rejects a history as a whole
    for (lo, hi, _, _) in regions_oracle.setup_image_regions(nz, 3, 1):
        got = set(regions_oracle.identify_protons_passing_region(v_in, v_out, sl, lo, hi).tolist())
        want = set()
        for i, (a, b) in enumerate(zip(v_in, v_out)):
            if a < 0:
                continue
            za, zb = a // sl, b // sl                                          # slice of a linear voxel index (R1)
            if lo <= za < hi or lo <= zb < hi:                                 # "entered to and exited from"
                want.add(i)
        assert got == want and len(got) > 0
    # a history that only passes THROUGH a region (enters below, exits above) is not a member of it: the paper assigns by the
    # entry and exit regions only
    thr = regions_oracle.identify_protons_passing_region(np.array([0]), np.array([n - 1]), sl, 2, 4)
    assert thr.size == 0


# ORACLE_REGIONS_PART_2
