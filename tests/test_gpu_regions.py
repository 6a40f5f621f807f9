"""Parity of Algorithm 1 of the paper (R28) through the C-ABI binding against the CPU oracle
(oracle/pcto_regions.py): hull entry/exit voxels and region membership bit-exact (integer work), the gathered histories
bit-exact (copies), the reconstructed image within the solver's tolerance (north_star: rel-L2 1e-4, max-abs 1e-3)."""
import numpy as np
import pytest
import torch

import synth
from helpers import oracle_setup

pytestmark = pytest.mark.gpu
REL_L2_TOL, MAX_ABS_TOL = 1e-4, 1e-3


@pytest.fixture(scope="module")
def binding():
    from paper_1802_01070_b200 import binding as b
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    b.load_library()
    return b


@pytest.fixture(scope="module")
def regions_oracle(oracle):
    from oracle import pcto_regions
    return pcto_regions


def case(binding, oracle, name, m, nan_at=None):
    cfg = synth.scaled(synth.CONFIGS[name], m)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    if nan_at is not None:
        pr["t_out"][nan_at] = float("nan")                        # rejected: non-finite record
        pr["t_in"][nan_at + 1] = 1e3; pr["t_out"][nan_at + 1] = 1e3       # rejected: misses the grid
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    arrays = {k: pr[k].cpu().numpy() for k in binding.PROTON_KEYS}
    return cfg, ctx, dev, arrays, hull, pr["wepl"].cuda().contiguous(), pr["wepl"].numpy()


def test_hull_intersect_and_membership_match_oracle(binding, oracle, regions_oracle):
    cfg, ctx, dev, arrays, hull, b_d, b_h = case(binding, oracle, "tiny", 4000, nan_at=5)
    u = cfg.u_tracker
    g, p, pa, P = oracle_setup(oracle, cfg, dict(arrays), hull)
    flags = P.rows()[3]
    vi_o, vo_o = regions_oracle.hull_ends(g, p, pa, hull.numpy(), flags)
    vi_g, vo_g = ctx.hull_intersect(dev, -u, u, hull.reshape(-1).cuda())
    assert np.array_equal(vi_g.cpu().numpy(), vi_o) and np.array_equal(vo_g.cpu().numpy(), vo_o)
    assert vi_o[5] == -1 and vi_o[6] == -1 and np.count_nonzero(vi_o >= 0) > 3000
    sl = cfg.nx * cfg.ny
    for G, ext in ((2, 1), (3, 2), (2, 0), (1, 0)):
        regs_o = regions_oracle.setup_image_regions(cfg.nz, G, ext)
        regs_g = binding.regions_setup(cfg.nz, G, ext)
        for ro, rg in zip(regs_o, regs_g):
            idx_o = regions_oracle.identify_protons_passing_region(vi_o, vo_o, sl, ro[0], ro[1])
            idx_g = ctx.region_members(vi_g, vo_g, rg)
            assert np.array_equal(idx_g.cpu().numpy(), idx_o)
            sub, b_sub = ctx.gather_histories(dev, -u, u, b_d, idx_g)
            for k in binding.PROTON_KEYS:
                assert np.array_equal(sub[k].cpu().numpy(), arrays[k][idx_o], equal_nan=True)
            assert np.array_equal(b_sub.cpu().numpy(), b_h[idx_o])
    # no hull mask (every voxel is hull): the entry / exit voxels are those of the grid box
    g2, p2, pa2, P2 = oracle_setup(oracle, cfg, dict(arrays), None)
    vi_o2, vo_o2 = regions_oracle.hull_ends(g2, p2, pa2, None, P2.rows()[3])
    vi_g2, vo_g2 = ctx.hull_intersect(dev, -u, u, None)
    assert np.array_equal(vi_g2.cpu().numpy(), vi_o2) and np.array_equal(vo_g2.cpu().numpy(), vo_o2)
    # empty input
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in binding.PROTON_KEYS}
    e_in, e_out = ctx.hull_intersect(empty, -u, u, None)
    assert e_in.numel() == 0 and ctx.region_members(e_in, e_out, binding.regions_setup(cfg.nz, 1, 0)[0]).numel() == 0


def test_hull_intersect_equals_the_ends_of_the_generated_rows(binding):
    """At a size the oracle's per-history loop cannot do: the voxels of pct_hull_intersect are the first and last voxel of the
    rows pct_generate_mlp produces (R10: the walk ends in the exit hull voxel unless END_MISMATCH is flagged)."""
    cfg = synth.scaled(synth.CONFIGS["head"], 300000)
    x_true, hull, shadow = synth.make_phantom(cfg, "cuda")
    pr = synth.generate_protons(cfg, x_true, shadow, device="cuda")
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    u = cfg.u_tracker
    hull_d = hull.reshape(-1).cuda().contiguous()
    v_in, v_out = ctx.hull_intersect(dev, -u, u, hull_d)
    paths = ctx.generate_mlp(dev, -u, u, hull_d)
    row_ptr, vox, ell, flags = ctx.paths_decode(paths)
    row_ptr, vox, flags = row_ptr.cpu().numpy(), vox.cpu().numpy(), flags.cpu().numpy()
    v_in, v_out = v_in.cpu().numpy(), v_out.cpu().numpy()
    a1_rej = (flags & (binding.REJ_MISS | binding.REJ_ORDER | binding.REJ_DEPTH | binding.REJ_NONFINITE)) != 0
    assert np.array_equal(v_in < 0, a1_rej) and np.array_equal(v_out < 0, a1_rej)
    has = (row_ptr[1:] > row_ptr[:-1])
    assert np.array_equal(vox[row_ptr[:-1][has]], v_in[has])
    ends_ok = has & ((flags & binding.END_MISMATCH) == 0)
    assert np.array_equal(vox[row_ptr[1:][ends_ok] - 1], v_out[ends_ok]) and np.count_nonzero(ends_ok) > 250000


@pytest.mark.parametrize("G,ext,block", [(2, 1, 1000), (3, 2, 4000), (2, 0, 700)])
def test_reconstruct_regions_matches_oracle(binding, oracle, regions_oracle, G, ext, block):
    cfg, ctx, dev, arrays, hull, b_d, b_h = case(binding, oracle, "tiny", 4000, nan_at=17)
    u = cfg.u_tracker
    g = oracle.make_geometry(**synth.geometry(cfg))
    p = oracle.make_params(**synth.mlp_params(cfg))
    x_o, mem_o, _ = regions_oracle.reconstruct(g, p, arrays, -u, u, hull.numpy(), b_h, None, G, ext, 2, block, cfg.lam)
    hull_d = hull.reshape(-1).cuda().contiguous()
    x_g, mem_g = ctx.reconstruct_regions(dev, -u, u, hull_d, b_d, None, G, ext, 2, block, cfg.lam)
    assert mem_g == [int(mm.size) for mm in mem_o]
    x_g = x_g.cpu().numpy()
    assert np.linalg.norm(x_g - x_o) / np.linalg.norm(x_o) <= REL_L2_TOL and np.abs(x_g - x_o).max() <= MAX_ABS_TOL
    assert np.abs(x_o - 1.0).max() > 0.05
    # one region per call, as one process per GPU would run it, into the same output image
    x_s = torch.full((ctx.n,), -7.0, dtype=torch.float32, device="cuda")
    for r in range(G):
        _, mem_r = ctx.reconstruct_regions(dev, -u, u, hull_d, b_d, None, G, ext, 2, block, cfg.lam, region_first=r, region_count=1, out=x_s)
        assert mem_r[r] == mem_g[r] and all(v == -1 for k, v in enumerate(mem_r) if k != r)
    x_s = x_s.cpu().numpy()
    assert np.abs(x_s - x_o).max() <= MAX_ABS_TOL
    # a given start image
    x0 = torch.full((ctx.n,), 0.9, dtype=torch.float32, device="cuda")
    x_o0, _, _ = regions_oracle.reconstruct(g, p, arrays, -u, u, hull.numpy(), b_h, x0.cpu().numpy(), G, ext, 1, block, cfg.lam)
    x_g0, _ = ctx.reconstruct_regions(dev, -u, u, hull_d, b_d, x0, G, ext, 1, block, cfg.lam)
    assert np.abs(x_g0.cpu().numpy() - x_o0).max() <= MAX_ABS_TOL
    with pytest.raises(binding.PctError):
        ctx.reconstruct_regions(dev, -u, u, hull_d, b_d, None, cfg.nz + 1, ext, 1, block, cfg.lam)
    with pytest.raises(binding.PctError):
        ctx.reconstruct_regions(dev, -u, u, hull_d, b_d, x0, G, ext, 1, block, cfg.lam, out=x0)


def test_regions_through_the_plan_path_reproduce_the_plain_solve(binding):
    """Property at a size where blocks take the solve plan (B = 100 k): with an extension that makes every region the whole
    volume, Algorithm 1 must give the plain reconstruction of the accepted histories (one block per sweep boundary-free: the
    same member list in every region)."""
    cfg = synth.scaled(synth.CONFIGS["head"], 300000)
    x_true, hull, shadow = synth.make_phantom(cfg, "cuda")
    pr = synth.generate_protons(cfg, x_true, shadow, device="cuda")
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    b = pr["wepl"].cuda().contiguous()
    u = cfg.u_tracker
    hull_d = hull.reshape(-1).cuda().contiguous()
    v_in, v_out = ctx.hull_intersect(dev, -u, u, hull_d)
    idx = ctx.region_members(v_in, v_out, binding.regions_setup(cfg.nz, 1, 0)[0])
    sub, b_sub = ctx.gather_histories(dev, -u, u, b, idx)
    paths = ctx.generate_mlp({k: v.contiguous() for k, v in sub.items()}, -u, u, hull_d)
    x_plain = ctx.solve(paths, b_sub.contiguous(), torch.ones(ctx.n, device="cuda"), 2, 100000, cfg.lam).cpu().numpy()
    x_r, mem = ctx.reconstruct_regions(dev, -u, u, hull_d, b, None, 2, cfg.nz, 2, 100000, cfg.lam)
    assert mem == [int(idx.numel())] * 2 and paths.plan_info()["n_groups"] > 0
    x_r = x_r.cpu().numpy()
    assert np.linalg.norm(x_r - x_plain) / np.linalg.norm(x_plain) <= REL_L2_TOL and np.abs(x_r - x_plain).max() <= MAX_ABS_TOL
    # and the paper's use: two regions with a small overlap agree with the joint solve away from the cut (Table I: a path hardly
    # moves along z).  One block per sweep, so that dropping far-away histories cannot move a block boundary.
    big = 400000
    x_joint = ctx.solve(paths, b_sub.contiguous(), torch.ones(ctx.n, device="cuda"), 2, big, cfg.lam).cpu().numpy()
    x_2, mem2 = ctx.reconstruct_regions(dev, -u, u, hull_d, b, None, 2, 4, 2, big, cfg.lam)
    assert 0 < mem2[0] < idx.numel() and 0 < mem2[1] < idx.numel() and mem2[0] + mem2[1] > idx.numel()
    sl = cfg.nx * cfg.ny
    x_2 = x_2.cpu().numpy()
    far = np.r_[0:(cfg.nz // 2 - 16) * sl, (cfg.nz // 2 + 16) * sl:cfg.nz * sl]
    assert np.abs(x_2[far] - x_joint[far]).max() <= MAX_ABS_TOL and np.abs(x_2 - 1.0).max() > 0.05


def test_one_process_runs_all_regions_through_the_distributed_entry(binding):
    """paper_1802_01070_b200.regions with a process group of one rank: that rank owns every region, the result is
    pct_reconstruct_regions' (the multi-rank slice assembly itself is covered on gloo in tests/test_oracle_regions.py)."""
    import socket
    import torch.distributed as dist
    from paper_1802_01070_b200 import regions
    cfg = synth.scaled(synth.CONFIGS["tiny"], 4000)
    x_true, hull, shadow = synth.make_phantom(cfg, "cuda")
    pr = synth.generate_protons(cfg, x_true, shadow, device="cuda")
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    b = pr["wepl"].cuda().contiguous()
    u = cfg.u_tracker
    hull_d = hull.reshape(-1).cuda().contiguous()
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        x_d, mem_d = regions.reconstruct_regions_distributed(ctx, dev, -u, u, hull_d, b, None, 1, 2, cfg.block, cfg.lam, n_regions=2)
    finally:
        dist.destroy_process_group()
    x_r, mem_r = ctx.reconstruct_regions(dev, -u, u, hull_d, b, None, 2, 1, 2, cfg.block, cfg.lam)
    assert mem_d == mem_r and all(v > 0 for v in mem_r)
    assert np.abs(x_d.cpu().numpy() - x_r.cpu().numpy()).max() <= MAX_ABS_TOL
