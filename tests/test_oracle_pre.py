"""Pins for the oracle's preprocessing steps and solver options: FBP initial iterate (reading R25), hull by
space carving (R26), weighted / clamped DROP (PAPER.md:57 ref [9], R27).

The paper prints no number for any of them; they are pinned by mathematics: the ramp kernel's defining integral
(quadrature), the value FBP must give inside a uniform disc (centred and off-centre, parallel and diverging beams --
every sign convention of R25 is wrong-able there), an independent numpy restatement built on library routines
(np.convolve, np.interp), Siddon's exact chords for the carving, and dense-matrix DROP for the solver options.
"""
import dataclasses

import numpy as np
import pytest
from scipy import integrate

import synth
from helpers import oracle_setup
from test_oracle_walk import siddon
from test_oracle_solver import small_system

GRID = dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-fbp", nx=40, ny=40, nz=2, u_tracker=40.0)


def geometry_of(oracle, cfg):
    return oracle.make_geometry(**synth.geometry(cfg))


def chord_records(cfg, theta, s, z, sad=None, rng=None):
    """Tracker records of straight chords with direction angle theta and signed distance s from the axis (R25): built in
    the GRID frame from the definition (direction e = (cos, sin), normal n = (-sin, cos), points s n + r e), then expressed
    in a gantry frame phi that differs from theta when the beam diverges (sad given)."""
    theta, s, z = np.asarray(theta, float), np.asarray(s, float), np.asarray(z, float)
    m = theta.size
    alpha = np.zeros(m) if sad is None else rng.uniform(-0.06, 0.06, m)      # chord direction relative to the beam axis
    phi = theta - alpha
    ex, ey = np.cos(theta), np.sin(theta)
    nx_, ny_ = -np.sin(theta), np.cos(theta)
    cph, sph = np.cos(phi), np.sin(phi)
    out = {}
    for name, u_plane in (("in", -cfg.u_tracker), ("out", cfg.u_tracker)):
        # point of the chord whose gantry-frame depth is u_plane: (s n + r e) . (cph, sph) = u_plane
        r = (u_plane - s * (nx_ * cph + ny_ * sph)) / (ex * cph + ey * sph)
        px, py = s * nx_ + r * ex, s * ny_ + r * ey
        out["t_" + name] = -px * sph + py * cph
        out["v_" + name] = z.copy()
    slope = np.tan(alpha)
    return dict(phi=phi, t_in=out["t_in"], v_in=out["v_in"], dt_in=slope, dv_in=np.zeros(m), t_out=out["t_out"],
                v_out=out["v_out"], dt_out=slope, dv_out=np.zeros(m))


def disc_wepl(theta, s, centre, radius, rsp):
    """Line integral of a uniform disc along the chord (theta, s): 2 rsp sqrt(R^2 - d^2), d = distance of the centre."""
    d = s - (-centre[0] * np.sin(theta) + centre[1] * np.cos(theta))
    return (2.0 * rsp * np.sqrt(np.maximum(radius ** 2 - d ** 2, 0.0))).astype(np.float32)


def test_ramp_kernel_is_the_band_limited_ramp(oracle):
    """q = ds (p * h) with h(n) = int_{-1/(2 ds)}^{1/(2 ds)} |f| exp(2 pi i f n ds) df (the defining integral), by quadrature."""
    for ds in (1.0, 0.7):
        cfg = dataclasses.replace(GRID, h=ds)
        n_s = 33
        rec = chord_records(cfg, [0.3], [0.0], [-0.5 * ds])          # one history in the central s bin, slice 0
        pa = oracle.ProtonArrays(rec, -cfg.u_tracker, cfg.u_tracker)
        _, mean, filt = oracle.fbp(geometry_of(oracle, cfg), pa, [1.0], 12, n_s, ds, want_sinogram=True)
        it, js = np.argwhere(mean[0] == 1.0)[0]
        assert (mean != 0).sum() == 1 and js == n_s // 2
        for n in range(-8, 9):
            ref = 2.0 * integrate.quad(lambda f: f * np.cos(2 * np.pi * f * n * ds), 0.0, 0.5 / ds, epsabs=1e-14, epsrel=1e-12)[0]
            assert filt[0, it, js + n] == pytest.approx(ds * ref, abs=1e-12)


@pytest.mark.parametrize("centre,sad", [((0.0, 0.0), None), ((4.0, -3.0), None), ((4.0, -3.0), 2000.0), ((-5.0, 2.5), 2000.0)])
def test_uniform_disc_is_reconstructed(oracle, centre, sad):
    """FBP of the exact projections of a uniform disc returns its value inside and ~0 outside (scale factor, sign
    conventions of theta / s / back projection, rebinning of a diverging beam)."""
    cfg, R, rsp = GRID, 9.0, 1.3
    n_theta, n_s, ds = 120, 64, 1.0
    rng = np.random.default_rng(3)
    if sad is None:          # one history exactly in the middle of every bin
        th = (np.arange(n_theta) + 0.5) * 2 * np.pi / n_theta
        sc = (np.arange(n_s) + 0.5 - 0.5 * n_s) * ds
        theta, s = [a.reshape(-1) for a in np.meshgrid(th, sc, indexing="ij")]
    else:                    # random chords of a diverging beam: many per bin, gantry angle != chord angle
        m = 400_000
        theta, s = rng.uniform(0, 2 * np.pi, m), rng.uniform(-0.5 * n_s * ds, 0.5 * n_s * ds, m)
    z = np.full(theta.size, -0.5)
    rec = chord_records(cfg, theta, s, z, sad, rng)
    b = disc_wepl(theta, s, centre, R, rsp)
    pa = oracle.ProtonArrays(rec, -cfg.u_tracker, cfg.u_tracker)
    x0 = oracle.fbp(geometry_of(oracle, cfg), pa, b, n_theta, n_s, ds)
    lo = np.array(cfg.lo)
    xs = lo[0] + (np.arange(cfg.nx) + 0.5) * cfg.h
    ys = lo[1] + (np.arange(cfg.ny) + 0.5) * cfg.h
    r = np.hypot(xs[None, :] - centre[0], ys[:, None] - centre[1])
    img = x0[0]                                              # slice 0 holds z = -0.5
    tol = 0.02 if sad is None else 0.04
    assert np.abs(img[r < R - 2.0] - rsp).max() < tol * rsp
    out = img[r > R + 2.5]                                   # streaks of the sharp edge (one sample per 1 mm bin): small, zero-mean
    assert np.abs(out).max() < 0.12 * rsp and np.abs(out).mean() < 0.025 * rsp and abs(out.mean()) < 0.005 * rsp
    X, Y = np.meshgrid(xs, ys)
    assert abs((img * X).sum() / img.sum() - centre[0]) < 0.05 and abs((img * Y).sum() / img.sum() - centre[1]) < 0.05
    assert img.sum() * cfg.h ** 2 == pytest.approx(np.pi * R * R * rsp, rel=0.01)
    assert np.abs(x0[1]).max() == 0.0                        # nothing was binned into the other slice


def numpy_fbp(cfg, rec, b, n_theta, n_s, ds, min_count=1):
    """Independent restatement of R25 on library routines: np.add.at binning, np.convolve filtering, np.interp back projection."""
    alpha = np.arctan2(rec["t_out"] - rec["t_in"], 2 * cfg.u_tracker)
    theta = np.mod(rec["phi"] + alpha, 2 * np.pi)
    s = 0.5 * (rec["t_in"] + rec["t_out"]) * np.cos(alpha)
    z = 0.5 * (rec["v_in"] + rec["v_out"])
    it = np.minimum((theta / (2 * np.pi / n_theta)).astype(int), n_theta - 1)
    js = np.floor(s / ds + 0.5 * n_s).astype(int)
    iz = np.floor((z - cfg.lo[2]) / cfg.h).astype(int)
    ok = (js >= 0) & (js < n_s) & (iz >= 0) & (iz < cfg.nz)
    tot, cnt = np.zeros((cfg.nz, n_theta, n_s)), np.zeros((cfg.nz, n_theta, n_s))
    np.add.at(tot, (iz[ok], it[ok], js[ok]), b[ok].astype(np.float64))
    np.add.at(cnt, (iz[ok], it[ok], js[ok]), 1.0)
    mean = np.where(cnt >= min_count, tot / np.maximum(cnt, 1.0), 0.0)
    n = np.arange(-(n_s - 1), n_s)
    h = np.where(n == 0, 1.0 / (4 * ds * ds), np.where(n % 2 != 0, -1.0 / (np.pi ** 2 * n.astype(float) ** 2 * ds * ds + (n == 0)), 0.0))
    filt = np.array([[ds * np.convolve(mean[k, j], h)[n_s - 1:2 * n_s - 1] for j in range(n_theta)] for k in range(cfg.nz)])
    xs = cfg.lo[0] + (np.arange(cfg.nx) + 0.5) * cfg.h
    ys = cfg.lo[1] + (np.arange(cfg.ny) + 0.5) * cfg.h
    X, Y = np.meshgrid(xs, ys)
    centres = (np.arange(n_s) + 0.5 - 0.5 * n_s) * ds
    img = np.zeros((cfg.nz, cfg.ny, cfg.nx))
    for j in range(n_theta):
        th = (j + 0.5) * 2 * np.pi / n_theta
        sv = -X * np.sin(th) + Y * np.cos(th)
        for k in range(cfg.nz):
            img[k] += np.interp(sv, centres, filt[k, j], left=0.0, right=0.0)
    return np.pi / n_theta * img, mean, filt


def test_matches_numpy_restatement(oracle):
    cfg = synth.scaled(synth.CONFIGS["tiny"], 20000)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    rec = {k: v.numpy() for k, v in pr.items() if k != "wepl"}
    b = pr["wepl"].numpy()
    pa = oracle.ProtonArrays(rec, -cfg.u_tracker, cfg.u_tracker)
    for (n_theta, n_s, ds, mc) in ((90, 48, 1.0, 1), (45, 30, 1.5, 3)):
        x0, mean, filt = oracle.fbp(geometry_of(oracle, cfg), pa, b, n_theta, n_s, ds, mc, want_sinogram=True)
        ref, mean_r, filt_r = numpy_fbp(cfg, rec, b, n_theta, n_s, ds, mc)
        assert np.abs(mean - mean_r).max() < 1e-9
        assert np.abs(filt - filt_r).max() < 1e-9
        # np.interp returns 0 beyond the first / last bin CENTRE, R25 interpolates towards 0 over the last half bin: compare inside
        assert np.abs(x0 - ref)[:, 4:-4, 4:-4].max() < 1e-9
    # the image of the Tiny phantom: water ~1 in the body, inserts visible, ~0 outside
    # (bins wide enough for 20 k histories: 45 directions x 24 lateral bins of 2 mm x 8 slices, ~2 histories per bin)
    x0 = oracle.fbp(geometry_of(oracle, cfg), pa, b, 45, 24, 2.0)
    body = hull.numpy() == 1
    print("FBP of Tiny: median in the body", np.median(x0[body]), "outside", np.median(x0[~body]))
    assert abs(np.median(x0[body]) - 1.0) < 0.15 and abs(np.median(x0[~body])) < 0.1
    xt = x_true.numpy()
    assert x0[xt == 1.6].mean() > x0[xt == 1.0].mean() + 0.15 and x0[xt == 0.3].mean() < x0[xt == 1.0].mean() - 0.15


def test_fbp_is_linear_and_ignores_bad_records(oracle):
    cfg = GRID
    rng = np.random.default_rng(5)
    m = 3000
    theta, s = rng.uniform(0, 2 * np.pi, m), rng.uniform(-15, 15, m)
    rec = chord_records(cfg, theta, s, rng.uniform(-1, 1, m))
    b1, b2 = rng.uniform(0, 30, m).astype(np.float32), rng.uniform(0, 30, m).astype(np.float32)
    g = geometry_of(oracle, cfg)
    pa = oracle.ProtonArrays(rec, -cfg.u_tracker, cfg.u_tracker)
    f = lambda b: oracle.fbp(g, pa, b, 60, 40, 1.0)
    assert np.abs(f(b1 + b2) - f(b1) - f(b2)).max() < 1e-5          # float32 sum of the inputs
    rec2 = {k: np.concatenate([v, v[:3]]) for k, v in rec.items()}
    rec2["t_in"][-1] = np.nan; rec2["v_in"][-2] = 1e9; rec2["t_in"][-3] = 1e4       # non-finite, outside z, outside s
    rec2["t_out"][-3] = 1e4
    pa2 = oracle.ProtonArrays(rec2, -cfg.u_tracker, cfg.u_tracker)
    assert np.array_equal(oracle.fbp(g, pa2, np.concatenate([b1, [5, 5, 5]]).astype(np.float32), 60, 40, 1.0), f(b1))


# ---- space carving -------------------------------------------------------------------------------------------------
def test_carved_voxels_are_siddons_chords(oracle):
    """A history with WEPL below the threshold carves exactly the voxels Siddon's ray tracing gives a chord > min_chord."""
    cfg = dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-carve", nx=20, ny=24, nz=6, h=0.7, u_tracker=30.0)
    g = geometry_of(oracle, cfg)
    rays = {k: v.numpy() for k, v in synth.random_rays(60, cfg, seed=11).items()}
    rays["t_out"] = rays["t_out"] + np.random.default_rng(1).normal(0, 1.0, 60)      # chord != entry direction
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    for min_chord in (0.0, 0.05, 0.3):
        for i in range(60):
            one = {k: v[i:i + 1] for k, v in rays.items()}
            pa = oracle.ProtonArrays(one, -cfg.u_tracker, cfg.u_tracker)
            hull = oracle.hull_carve(g, pa, [0.2], 1.0, min_chord)
            c, s = np.cos(one["phi"][0]), np.sin(one["phi"][0])
            A = np.array([-cfg.u_tracker * c - one["t_in"][0] * s, -cfg.u_tracker * s + one["t_in"][0] * c, one["v_in"][0]])
            B = np.array([cfg.u_tracker * c - one["t_out"][0] * s, cfg.u_tracker * s + one["t_out"][0] * c, one["v_out"][0]])
            vox, chords = siddon(lo, cfg.h, n, A, B)
            carved = np.nonzero(hull.reshape(-1) == 0)[0]
            sure = set(vox[chords > min_chord + 1e-9].tolist())
            maybe = set(vox[chords > min_chord - 1e-9].tolist())
            assert sure <= set(carved.tolist()) <= maybe, (i, min_chord)
            assert oracle.hull_carve(g, pa, [1.0], 1.0, min_chord).all()          # WEPL not below the threshold: nothing carved


def test_carving_recovers_a_convex_body(oracle):
    cfg = synth.scaled(synth.CONFIGS["tiny"], 50000)
    x_true, hull, shadow = synth.make_phantom(cfg)
    wide = dict(shadow, a=15.5, b=15.5)                       # illuminate the air around the body too
    pr = synth.generate_protons(dataclasses.replace(cfg, noise=0.0), x_true, wide)
    rec = {k: v.numpy() for k, v in pr.items() if k != "wepl"}
    pa = oracle.ProtonArrays(rec, -cfg.u_tracker, cfg.u_tracker)
    carved = oracle.hull_carve(geometry_of(oracle, cfg), pa, pr["wepl"].numpy(), 0.5, 0.25)
    body = hull.numpy().astype(bool)
    # interior of the body (all 8 in-plane neighbours are body) is never carved; the air well outside is
    inner = body.copy()
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            inner &= np.roll(np.roll(body, dy, 1), dx, 2)
    assert carved[inner].all()
    z, y, x = np.meshgrid(np.arange(cfg.nz), np.arange(cfg.ny) - 15.5, np.arange(cfg.nx) - 15.5, indexing="ij")
    ring = (np.hypot(x, y) > 13.5) & (np.hypot(x, y) < 15.0)
    assert carved[ring].mean() < 0.02
    # more data never un-carves (monotone)
    half = {k: v[:25000] for k, v in rec.items()}
    c_half = oracle.hull_carve(geometry_of(oracle, cfg), oracle.ProtonArrays(half, -cfg.u_tracker, cfg.u_tracker),
                               pr["wepl"].numpy()[:25000], 0.5, 0.25)
    assert np.all(carved <= c_half)


# ---- weighted / clamped DROP -------------------------------------------------------------------------------------------
def dense_drop_ex(A, rows, ell, b, x0, w, iters, B, lam, lo, hi):
    x = x0.astype(np.float64).copy()
    m, n = A.shape
    for _ in range(iters):
        for i0 in range(0, m, B):
            upd, s = np.zeros(n), np.zeros(n)
            for i in range(i0, min(m, i0 + B)):
                if len(rows[i]) == 0:
                    continue
                li = float(ell[i])
                upd += w[i] * (float(b[i]) - A[i] @ x) / (len(rows[i]) * li * li) * A[i]
                np.add.at(s, rows[i], 1.0)
            x += lam * upd / np.maximum(1.0, s)
            if lo <= hi:
                x[s > 0] = np.clip(x[s > 0], lo, hi)
    return x


@pytest.mark.parametrize("B,lam,iters,clamp", [(7, 0.5, 3, (0.9, 1.1)), (40, 0.3, 4, (1.0, 0.0)), (160, 1.0, 2, (0.0, 1.05)), (1, 1.0, 1, (0.95, 1.3))])
def test_weighted_clamped_drop_matches_dense(oracle, B, lam, iters, clamp):
    cfg, P, rows, ell, A = small_system(oracle)
    rng = np.random.default_rng(2)
    b = (A @ rng.uniform(0.5, 1.5, cfg.n) * (1 + 0.05 * rng.normal(size=cfg.m))).astype(np.float32)
    x0 = rng.uniform(0.95, 1.05, cfg.n).astype(np.float32)
    w = rng.uniform(0.0, 1.0, cfg.m).astype(np.float32)
    w[::7] = 0.0
    x = P.solve_ex(b, x0, w, iters, B, lam, *clamp)
    ref = dense_drop_ex(A, rows, ell, b, x0, w.astype(np.float64), iters, B, lam, *clamp)
    assert np.abs(x - ref.astype(np.float32)).max() < 2e-6
    # unit weights, no clamp: the plain solver, bit for bit; zero-weight rows equal removed rows' corrections
    assert np.array_equal(P.solve_ex(b, x0, None, iters, B, lam), P.solve(b, x0, iters, B, lam))
    assert np.array_equal(P.solve_ex(b, x0, np.ones(cfg.m, np.float32), iters, B, lam), P.solve(b, x0, iters, B, lam))
    if clamp[0] <= clamp[1]:
        touched = np.zeros(cfg.n, bool)
        for r in rows:
            touched[r] = True
        assert x[touched].min() >= np.float32(clamp[0]) - 1e-7 and x[touched].max() <= np.float32(clamp[1]) + 1e-7
        assert np.array_equal(x[~touched], x0[~touched])
