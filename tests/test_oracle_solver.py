"""Pins for the oracle's projections and DROP solver (A4-A9): PAPER.md:98 (DROP, ref [11]), readings R12-R20.

References written here in numpy on DENSE matrices built from the visit lists: dense DROP, relaxed Kaczmarz
(B=1), the simultaneous step (B=m), fixed points, and brute-force dense least squares (north_star).
"""
import dataclasses

import numpy as np
import pytest

import synth
from helpers import oracle_setup, split_rows

SMALL = dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-small", nx=8, ny=8, nz=2, u_tracker=8.0, m=160)


def small_system(oracle, m=160, seed=7, hull=None):
    cfg = dataclasses.replace(SMALL, m=m)
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0, 2 * np.pi, m)
    t = rng.uniform(-3.9, 3.9, m)
    v = rng.uniform(-0.95, 0.95, m)
    dt = rng.normal(0, 0.02, m)
    dv = rng.normal(0, 0.005, m)
    du = 2 * cfg.u_tracker
    kick = rng.normal(0, 0.02, m)
    pr = dict(phi=phi, t_in=t, v_in=v, dt_in=dt, dv_in=dv, t_out=t + dt * du + 0.5 * kick * du, v_out=v + dv * du,
              dt_out=dt + kick, dv_out=dv)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    row_ptr, vox, ell, flags, length = P.rows()
    rows = split_rows(row_ptr, vox)
    A = np.zeros((m, cfg.n))
    for i, r in enumerate(rows):
        np.add.at(A[i], r, float(ell[i]))          # R12: value l_i on every visit
    return cfg, P, rows, ell, A


def dense_drop(A, rows, ell, b, x0, iters, B, lam):
    """x <- x + lam * U_t * sum_i (b_i - a_i.x)/||a_i||^2 a_i, ||a_i||^2 = N_i l_i^2, U_t = 1/max(1,s_j) (R13-R17)."""
    x = x0.astype(np.float64).copy()
    m, n = A.shape
    for _ in range(iters):
        for i0 in range(0, m, B):
            i1 = min(m, i0 + B)
            upd, s = np.zeros(n), np.zeros(n)
            for i in range(i0, i1):
                if len(rows[i]) == 0:
                    continue
                li = float(ell[i])
                r = (float(b[i]) - A[i] @ x) / (len(rows[i]) * li * li)
                upd += r * A[i]
                np.add.at(s, rows[i], 1.0)
            x += lam * upd / np.maximum(1.0, s)
    return x


def test_forward_project_and_counts(oracle):
    cfg, P, rows, ell, A = small_system(oracle)
    _, _, _, _, length = P.rows()
    ones = np.ones(cfg.n, np.float32)
    assert P.forward_project(ones) == pytest.approx(length.astype(np.float32), rel=2e-6)     # sum_j a_ij = L_i
    rng = np.random.default_rng(0)
    x = rng.uniform(0.2, 1.8, cfg.n).astype(np.float32)
    assert P.forward_project(x) == pytest.approx((A @ x.astype(np.float64)).astype(np.float32), rel=1e-6)
    for (i0, i1) in ((0, cfg.m), (10, 57), (5, 5)):
        c = P.column_counts(i0, i1)
        ref = np.zeros(cfg.n, np.int64)
        for r in rows[i0:i1]:
            np.add.at(ref, r, 1)
        assert np.array_equal(c.astype(np.int64), ref)
        assert c.sum() == sum(len(r) for r in rows[i0:i1])


@pytest.mark.parametrize("B,lam,iters", [(1, 1.0, 2), (7, 0.5, 3), (40, 0.1, 4), (160, 0.3, 3), (1000, 1.0, 2)])
def test_matches_dense_matrix_drop(oracle, B, lam, iters):
    cfg, P, rows, ell, A = small_system(oracle)
    rng = np.random.default_rng(1)
    b = (A @ rng.uniform(0.5, 1.5, cfg.n) * (1 + 0.01 * rng.normal(size=cfg.m))).astype(np.float32)
    x0 = rng.uniform(0.8, 1.2, cfg.n).astype(np.float32)
    x32, x64 = P.solve(b, x0, iters, B, lam, f64=True)
    ref = dense_drop(A, rows, ell, b, x0, iters, B, lam)
    assert np.max(np.abs(x64 - ref)) < 1e-12
    assert np.array_equal(x32, x64.astype(np.float32))


def test_kaczmarz_special_case(oracle):
    """B=1, lambda=1, a row without repeated voxels: after the step a_i.x = b_i exactly (textbook ART)."""
    cfg, P, rows, ell, A = small_system(oracle, m=1, seed=11)
    assert len(rows[0]) > 0 and len(set(rows[0].tolist())) == len(rows[0])
    b = np.array([7.25], np.float32)
    x0 = np.full(cfg.n, 0.9, np.float32)
    _, x = P.solve(b, x0, 1, 1, 1.0, f64=True)
    assert A[0] @ x == pytest.approx(7.25, rel=1e-13)
    li = float(ell[0])
    ref = x0.astype(np.float64) + (7.25 - A[0] @ x0.astype(np.float64)) / (A[0] @ A[0]) * A[0]
    assert np.max(np.abs(x - ref)) < 1e-13 and A[0] @ A[0] == pytest.approx(len(rows[0]) * li * li, rel=1e-12)


def test_exact_solution_is_a_fixed_point(oracle):
    cfg, P, rows, ell, A = small_system(oracle)
    rng = np.random.default_rng(2)
    xt = rng.uniform(0.3, 1.7, cfg.n)
    b = (A @ xt).astype(np.float32)
    for B, lam in ((1, 1.0), (13, 0.7), (160, 0.2)):
        _, x = P.solve(b, xt.astype(np.float32), 3, B, lam, f64=True)
        assert np.max(np.abs(x - xt)) < 5e-6           # b, x0 rounded to float32 -> residuals ~1e-7 relative


def test_consistent_system_converges_to_dense_least_squares(oracle):
    """north_star: noise-free consistent systems converge to the phantom / brute-force dense least squares."""
    cfg, P, rows, ell, A = small_system(oracle, m=900, seed=3)
    rng = np.random.default_rng(4)
    xt = rng.uniform(0.3, 1.7, cfg.n)
    b = (A @ xt).astype(np.float32)
    x0 = np.ones(cfg.n, np.float32)
    seen = A.sum(axis=0) > 0
    assert np.linalg.matrix_rank(A[:, seen]) == seen.sum()              # the data determine every seen voxel
    lsq = np.linalg.lstsq(A[:, seen], b.astype(np.float64) - A[:, ~seen] @ x0[~seen].astype(np.float64), rcond=None)[0]
    res = []
    for iters in (1, 20, 400):
        _, x = P.solve(b, x0, iters, 30, 1.0, f64=True)
        res.append(np.linalg.norm(A @ x - b))
    assert res[1] < 0.1 * res[0] and res[2] < 1e-3 * res[0]
    assert np.max(np.abs(x[seen] - lsq)) < 1e-3 and np.max(np.abs(x[seen] - xt[seen])) < 1e-3
    assert np.array_equal(x[~seen], x0[~seen].astype(np.float64))       # R16: untouched voxels keep x0


def test_tiny_phantom_noise_free_converges(oracle):
    """Config-0 phantom, b = A x_true: the sweep residual falls and x approaches the phantom inside the hull."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 20000, block=2000)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    xt = x_true.numpy().reshape(-1)
    b = P.forward_project(xt)
    x0 = np.ones(cfg.n, np.float32)
    inside = hull.numpy().reshape(-1) > 0
    err, res = [], []
    for iters in (0, 5, 40):
        x = P.solve(b, x0, iters, cfg.block, 0.5) if iters else x0
        err.append(np.sqrt(np.mean((x - xt)[inside] ** 2)))
        res.append(np.linalg.norm(P.forward_project(x) - b))
    assert res[1] < 0.2 * res[0] and res[2] < 0.05 * res[0]
    assert err[1] < 0.6 * err[0] and err[2] < 0.35 * err[0]
