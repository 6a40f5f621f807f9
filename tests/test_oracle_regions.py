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


def tiny_case(oracle, m=3000):
    cfg = synth.scaled(synth.CONFIGS["tiny"], m)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    arrays = {k: v.cpu().numpy() for k, v in pr.items() if k != "wepl"}
    return cfg, g, p, arrays, hull.numpy(), pr["wepl"].numpy(), P


def test_special_cases_reproduce_the_plain_solver(oracle, regions_oracle):
    cfg, g, p, arrays, hull, b, P = tiny_case(oracle)
    n = cfg.nx * cfg.ny * cfg.nz
    x_plain = P.solve(b, np.ones(n, np.float32), 2, cfg.block, cfg.lam)
    flags = P.rows()[3]
    accepted = int(np.count_nonzero((flags & regions_oracle.A1_REJECT) == 0))
    # one region: every accepted history is a member, the image is the plain solver's (rejected rows are empty: same sums)
    x1, mem1, _ = regions_oracle.reconstruct(g, p, arrays, -cfg.u_tracker, cfg.u_tracker, hull, b, None, 1, 0, 2, cfg.block, cfg.lam)
    assert mem1[0].size == accepted and np.all(np.diff(mem1[0]) > 0)
    # blocks are consecutive ranges of the MEMBER list: with the rejected histories dropped the block boundaries move, so the
    # comparison uses one block per sweep (block >= m), where membership cannot change the blocking
    x_plain_1 = P.solve(b, np.ones(n, np.float32), 2, cfg.m, cfg.lam)
    x1b, _, _ = regions_oracle.reconstruct(g, p, arrays, -cfg.u_tracker, cfg.u_tracker, hull, b, None, 1, 0, 2, cfg.m, cfg.lam)
    assert np.abs(x1b - x_plain_1).max() < 1e-5
    # an extension of nz slices makes every region the whole volume: every region's image is the plain solver's
    x3, mem3, imgs = regions_oracle.reconstruct(g, p, arrays, -cfg.u_tracker, cfg.u_tracker, hull, b, None, 3, cfg.nz, 2, cfg.m, cfg.lam)
    assert all(mm.size == accepted for mm in mem3)
    for img in imgs:
        assert np.abs(img - x_plain_1).max() < 1e-5
    assert np.abs(x3 - x_plain_1).max() < 1e-5
    assert np.abs(x_plain - 1.0).max() > 0.05 and np.abs(x1 - 1.0).max() > 0.05          # the solves did something


def test_regions_without_overlap_differ_only_near_the_cuts(oracle, regions_oracle):
    """Table I of the paper: a path hardly moves along z, so a region solved on its own histories reproduces the joint solve away
    from the cut; with ext = 0 the slices next to a cut see histories that the neighbour also updates, and may differ."""
    cfg, g, p, arrays, hull, b, P = tiny_case(oracle, 6000)
    n, sl = cfg.nx * cfg.ny * cfg.nz, cfg.nx * cfg.ny
    x_plain = P.solve(b, np.ones(n, np.float32), 3, cfg.m, cfg.lam).reshape(cfg.nz, -1)
    x2, mem, _ = regions_oracle.reconstruct(g, p, arrays, -cfg.u_tracker, cfg.u_tracker, hull, b, None, 2, 2, 3, cfg.m, cfg.lam)
    x2 = x2.reshape(cfg.nz, -1)
    assert 0 < mem[0].size < 6000 and 0 < mem[1].size < 6000
    assert np.intersect1d(mem[0], mem[1]).size > 0                             # the overlap's histories go to both regions
    # DROP divides a block's update by the per-voxel count of the BLOCK: dropping far-away histories leaves the near slices'
    # sums and counts unchanged, so the first and last slices agree with the joint solve to rounding
    assert np.abs(x2[0] - x_plain[0]).max() < 1e-5 and np.abs(x2[-1] - x_plain[-1]).max() < 1e-5


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _gloo_worker(rank, world, port, n_regions, nz, slice_elems, out_q):
    import torch.distributed as dist
    from paper_1802_01070_b200 import regions
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        owner = regions.region_owner(n_regions, world)
        first, count = regions.my_regions(n_regions, rank, world)
        cuts = [(g * nz) // n_regions for g in range(n_regions + 1)]
        keep = [(cuts[g], cuts[g + 1]) for g in range(n_regions)]
        # every rank fills the kept slices of ITS regions with a value that names (region, slice); the rest stays -1
        x = torch.full((nz * slice_elems,), -1.0)
        for g in range(first, first + count):
            for z in range(*keep[g]):
                x[z * slice_elems:(z + 1) * slice_elems] = 100.0 * g + z
        regions.assemble_slices(x, keep, owner, slice_elems)
        out_q.put((rank, first, count, x.numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_regions", [2, 3])
def test_slice_assembly_across_two_processes(n_regions):
    """selectSlice() across ranks (gloo, world_size 2): afterwards every rank holds every slice from the region that keeps it."""
    import torch.multiprocessing as mp
    from paper_1802_01070_b200 import regions
    nz, slice_elems, world = 8, 6, 2
    assert regions.region_owner(2, 2) == [0, 1] and regions.region_owner(3, 2) == [0, 0, 1] and regions.region_owner(1, 2) == [0]
    assert regions.my_regions(1, 1, 2) == (0, 0)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, world, port, n_regions, nz, slice_elems, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    cuts = [(g * nz) // n_regions for g in range(n_regions + 1)]
    want = np.empty(nz * slice_elems, dtype=np.float32)
    for g in range(n_regions):
        for z in range(cuts[g], cuts[g + 1]):
            want[z * slice_elems:(z + 1) * slice_elems] = 100.0 * g + z
    assert sorted(r for r, _, _, _ in got) == [0, 1]
    assert sum(c for _, _, c, _ in got) == n_regions
    for _, _, _, x in got:
        assert np.array_equal(x, want)
