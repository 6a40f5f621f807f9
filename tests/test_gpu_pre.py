"""Parity of the preprocessing entry points and the solver options against the CPU oracle (through the C-ABI binding):
pct_fbp (R25), pct_hull_carve (R26), pct_solve_ex (R27).  SURVEY.md 8(f) rows 1-3.

Tolerances: the hull mask is byte work -> bit-exact.  The FBP image is FP64 inside on both sides, float32 out; what can
differ is a history whose (theta, s, z) lies within an ulp of a bin edge (libm vs CUDA atan2 / cos / sin) and lands in the
neighbouring bin: with ~10 histories per bin that moves a bin's mean by ~10 % of the WEPL noise, a handful of bins per
10^8 histories -> max-abs 1e-3 of the image scale is asserted at full size, 1e-6 relative L2 on the small cases where no
such flip occurs.  Weighted / clamped DROP: the north_star tolerance of the plain solver."""
import dataclasses
import os

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


def setup(binding, oracle, cfg, device="cuda", shadow_scale=None, noise=None):
    c = cfg if noise is None else dataclasses.replace(cfg, noise=noise)
    x_true, hull, shadow = synth.make_phantom(c, device)
    if shadow_scale:
        shadow = dict(shadow, a=shadow["a"] * shadow_scale, b=shadow["b"] * shadow_scale)
    pr = synth.generate_protons(c, x_true, shadow, device=device)
    ctx = binding.Context(synth.geometry(c), synth.mlp_params(c), 0)
    dev = {k: pr[k].cuda().contiguous() for k in binding.PROTON_KEYS}
    host = {k: pr[k].cpu().numpy() for k in binding.PROTON_KEYS}
    pa = oracle.ProtonArrays(host, -c.u_tracker, c.u_tracker)
    g = oracle.make_geometry(**synth.geometry(c))
    return c, ctx, dev, pa, g, pr["wepl"].cuda().contiguous(), pr["wepl"].cpu().numpy(), hull, x_true


@pytest.mark.parametrize("name,m,n_theta,n_s,ds,mc", [("tiny", 50000, 45, 24, 2.0, 1), ("tiny", 50000, 91, 50, 1.0, 2),
                                                        ("paperA", 300000, 60, 140, 2.0, 1), ("head", 200000, 36, 120, 2.0, 3)])
def test_fbp_matches_oracle(binding, oracle, name, m, n_theta, n_s, ds, mc):
    cfg = synth.scaled(synth.CONFIGS[name], m)
    if name != "tiny":          # a coarser grid keeps the oracle's voxel loop in seconds; same phantom, same beam
        cfg = dataclasses.replace(cfg, nx=cfg.nx // 4, ny=cfg.ny // 4, nz=cfg.nz // 4, h=4.0)
    c, ctx, dev, pa, g, b_d, b_h, hull, x_true = setup(binding, oracle, cfg)
    x_g = ctx.fbp(dev, -c.u_tracker, c.u_tracker, b_d, n_theta, n_s, ds, mc).cpu().numpy().reshape(c.nz, c.ny, c.nx)
    x_o = oracle.fbp(g, pa, b_h, n_theta, n_s, ds, mc)
    scale = np.abs(x_o).max()
    assert scale > 0.5
    assert np.linalg.norm(x_g - x_o) / np.linalg.norm(x_o) < 1e-6
    assert np.abs(x_g - x_o).max() < 2e-6 * scale
    # degenerate inputs: no histories -> zero image; a NaN record and a NaN WEPL are skipped
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in binding.PROTON_KEYS}
    assert torch.count_nonzero(ctx.fbp(empty, -c.u_tracker, c.u_tracker, torch.empty(0, device="cuda"), n_theta, n_s, ds)) == 0
    dev2 = {k: v.clone() for k, v in dev.items()}
    dev2["t_in"][7] = float("nan")
    b2 = b_d.clone(); b2[11] = float("nan")
    host2 = {k: v.cpu().numpy() for k, v in dev2.items()}
    x_g2 = ctx.fbp(dev2, -c.u_tracker, c.u_tracker, b2, n_theta, n_s, ds, mc).cpu().numpy().reshape(c.nz, c.ny, c.nx)
    x_o2 = oracle.fbp(g, oracle.ProtonArrays(host2, -c.u_tracker, c.u_tracker), b2.cpu().numpy(), n_theta, n_s, ds, mc)
    assert np.all(np.isfinite(x_g2)) and np.abs(x_g2 - x_o2).max() < 2e-6 * scale
    with pytest.raises(binding.PctError):
        ctx.fbp(dev, -c.u_tracker, c.u_tracker, b_d, 0, n_s, ds)


def test_fbp_and_carving_at_bench_geometry(binding, oracle):
    """pct_fbp and pct_hull_carve at config 2's full grid (256 x 256 x 128, the bins bench.py uses) on the first 6 M
    histories of the workload: whole image / whole mask against the oracle."""
    cfg = synth.scaled(synth.CONFIGS["paperA"], int(os.environ.get("PCT_TEST_PRE_M", 6_000_000)))
    c, ctx, dev, pa, g, b_d, b_h, hull, x_true = setup(binding, oracle, cfg)
    n_s = 2 * int(np.ceil(0.5 * np.hypot(c.nx, c.ny))) + 2
    x_g = ctx.fbp(dev, -c.u_tracker, c.u_tracker, b_d, 180, n_s, c.h).cpu().numpy().reshape(c.nz, c.ny, c.nx)
    x_o = oracle.fbp(g, pa, b_h, 180, n_s, c.h)
    scale = np.abs(x_o).max()
    # a history within an ulp of a bin edge may land in the neighbouring bin (libm vs CUDA atan2 / cos): the bins hold ~1
    # history each at this sample size, so such a flip moves two bins by a whole WEPL -- allow a handful of them
    diff = np.abs(x_g - x_o)
    assert np.linalg.norm(x_g - x_o) / np.linalg.norm(x_o) < 1e-4 and np.quantile(diff, 0.999) < 1e-6 * scale
    h_g = ctx.hull_carve(dev, -c.u_tracker, c.u_tracker, b_d, 1.0, 0.25 * c.h).cpu().numpy().reshape(c.nz, c.ny, c.nx)
    h_o = oracle.hull_carve(g, pa, b_h, 1.0, 0.25 * c.h)
    assert np.array_equal(h_g, h_o), int((h_g != h_o).sum())
    assert 0 < int((h_g == 0).sum())


@pytest.mark.parametrize("name,m,scale", [("tiny", 50000, 1.3), ("head", 300000, 1.15), ("paperB", 200000, 1.0)])
def test_hull_carve_matches_oracle(binding, oracle, name, m, scale):
    cfg = synth.scaled(synth.CONFIGS[name], m)
    if name != "tiny":
        cfg = dataclasses.replace(cfg, nx=cfg.nx // 2, ny=cfg.ny // 2, nz=cfg.nz // 2, h=2.0)
    c, ctx, dev, pa, g, b_d, b_h, hull, x_true = setup(binding, oracle, cfg, shadow_scale=scale, noise=0.0)
    for (air, chord) in ((0.5, 0.25 * c.h), (2.0, 0.05)):
        h_g = ctx.hull_carve(dev, -c.u_tracker, c.u_tracker, b_d, air, chord).cpu().numpy().reshape(c.nz, c.ny, c.nx)
        h_o = oracle.hull_carve(g, pa, b_h, air, chord)
        assert np.array_equal(h_g, h_o), int((h_g != h_o).sum())
        assert set(np.unique(h_g).tolist()) <= {0, 1}
        if scale > 1.0:
            assert (h_g == 0).sum() > 0.02 * c.n              # something was carved
    # no history below the threshold: nothing carved; empty input: all ones
    assert ctx.hull_carve(dev, -c.u_tracker, c.u_tracker, b_d, -1.0, 0.1).all()
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in binding.PROTON_KEYS}
    assert ctx.hull_carve(empty, -c.u_tracker, c.u_tracker, torch.empty(0, device="cuda"), 0.5, 0.1).all()


def test_carved_hull_feeds_the_hot_path(binding, oracle):
    """The data-derived hull in place of the analytic mask: pct_generate_mlp + pct_solve on it match the oracle run on the
    same mask (rows differ from the analytic-hull rows -- the hull decides where the MLP starts -- parity does not)."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 20000, block=5000, iters=2)
    c, ctx, dev, pa, g, b_d, b_h, hull, x_true = setup(binding, oracle, cfg, shadow_scale=1.3)
    carved = ctx.hull_carve(dev, -c.u_tracker, c.u_tracker, b_d, 1.0, 0.25)
    assert 0.2 * c.n < int(carved.sum()) < 0.9 * c.n
    paths = ctx.generate_mlp(dev, -c.u_tracker, c.u_tracker, carved)
    p = oracle.make_params(**synth.mlp_params(c))
    P = oracle.Paths(g, p, pa, carved.cpu().numpy())
    assert paths.total_visits == P.total_visits or paths.n_ties + P.n_ties > 0
    x_g = ctx.solve(paths, b_d, torch.ones(c.n, device="cuda"), c.iters, c.block, c.lam).cpu().numpy()
    x_o = P.solve(b_h, np.ones(c.n, np.float32), c.iters, c.block, c.lam)
    assert np.linalg.norm(x_g - x_o) / np.linalg.norm(x_o) <= REL_L2_TOL and np.abs(x_g - x_o).max() <= MAX_ABS_TOL


@pytest.mark.parametrize("mode,B", [(1, 3000), (2, 5000), (2, 1777)])
def test_weighted_clamped_solve_matches_oracle(binding, oracle, mode, B):
    """pct_solve_ex through the direct kernels (mode 1) and the windowed plan (mode 2, counting and cached-count sweeps)."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 20000)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    ctx = binding.Context(synth.geometry(cfg), synth.mlp_params(cfg), 0)
    dev = {k: pr[k].cuda() for k in binding.PROTON_KEYS}
    paths = ctx.generate_mlp(dev, -cfg.u_tracker, cfg.u_tracker, hull.reshape(-1).cuda())
    ctx.solve_config(mode)
    rng = np.random.default_rng(3)
    w = rng.uniform(0, 1, cfg.m).astype(np.float32)
    w[::5] = 0.0
    b = pr["wepl"]
    x0 = torch.ones(cfg.n, device="cuda")
    for (weights, clamp) in ((w, None), (None, (0.8, 1.25)), (w, (0.0, 1.1)), (w, (1.05, 1.5))):
        x_g = ctx.solve(paths, b.cuda(), x0, 3, B, 0.2, weights=None if weights is None else torch.from_numpy(weights).cuda(),
                        clamp=clamp).cpu().numpy()
        lo, hi = clamp if clamp else (1.0, 0.0)
        x_o = P.solve_ex(b.numpy(), np.ones(cfg.n, np.float32), weights, 3, B, 0.2, lo, hi)
        assert np.linalg.norm(x_g - x_o) / np.linalg.norm(x_o) <= REL_L2_TOL, (weights is None, clamp)
        assert np.abs(x_g - x_o).max() <= MAX_ABS_TOL
        assert np.abs(x_g - 1.0).max() > 0.02
    # options that change nothing reproduce pct_solve
    x_a = ctx.solve(paths, b.cuda(), x0, 2, B, 0.1).cpu().numpy()
    x_b = ctx.solve(paths, b.cuda(), x0, 2, B, 0.1, weights=torch.ones(cfg.m, device="cuda"), clamp=(-1e30, 1e30)).cpu().numpy()
    assert np.abs(x_a - x_b).max() <= 1e-5


def test_fbp_start_converges_faster(binding, oracle):
    """What the FBP iterate is for (PAPER.md:7; 3-5 sweeps in the paper, :113): after ONE sweep from x0 = FBP the residual
    is below what x0 = 1 reaches after three."""
    cfg = synth.scaled(synth.CONFIGS["paperA"], 3_000_000, block=200_000)       # bone shell, air cavities: x0 = 1 is far off
    cfg = dataclasses.replace(cfg, nx=128, ny=128, nz=64, h=2.0)
    c, ctx, dev, pa, g, b_d, b_h, hull, x_true = setup(binding, oracle, cfg)
    hull_d = hull.reshape(-1).cuda()
    paths = ctx.generate_mlp(dev, -c.u_tracker, c.u_tracker, hull_d)
    x_fbp = ctx.fbp(dev, -c.u_tracker, c.u_tracker, b_d, 60, 96, 3.0)           # ~8 histories per bin

    def rms(x):
        r = (ctx.forward_project(paths, x) - b_d)[:200_000]
        return float(torch.sqrt(torch.mean(r * r)))
    ones = torch.ones(c.n, device="cuda")
    r_fbp0, r_one0 = rms(x_fbp), rms(ones)
    r_fbp1 = rms(ctx.solve(paths, b_d, x_fbp, 1, c.block, c.lam))
    r_one3 = rms(ctx.solve(paths, b_d, ones, 3, c.block, c.lam))
    print(f"rms residual [mm]: x0=1 {r_one0:.3f} -> 3 sweeps {r_one3:.3f};  x0=FBP {r_fbp0:.3f} -> 1 sweep {r_fbp1:.3f}")
    assert r_fbp0 < 0.5 * r_one0 and r_fbp1 < r_one3
