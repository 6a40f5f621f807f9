"""Pins for the oracle's hull entry (A1) and voxel walk (A3): readings R3-R5, R9-R12.

Independent references written here: Siddon's exact ray tracing (sorted plane crossings + midpoints, a
different algorithm from the oracle's lazy stepping), a slab-clipping restatement of the box entry/exit, and
brute-force dense sampling of the polyline.
"""
import dataclasses

import numpy as np
import pytest

import synth
from helpers import oracle_setup, split_rows


def siddon(lo, h, n, A, B):
    """Ordered voxels with non-zero chord on segment A->B, and the chords (Siddon 1985)."""
    A, B = np.asarray(A, float), np.asarray(B, float)
    alphas = [0.0, 1.0]
    for a in range(3):
        if B[a] != A[a]:
            planes = lo[a] + h * np.arange(n[a] + 1)
            al = (planes - A[a]) / (B[a] - A[a])
            alphas.extend(al[(al > 0) & (al < 1)].tolist())
    al = np.unique(np.array(alphas))
    mid = 0.5 * (al[1:] + al[:-1])
    pts = A[None, :] + mid[:, None] * (B - A)[None, :]
    idx = np.floor((pts - np.asarray(lo)[None, :]) / h).astype(np.int64)
    ok = np.all((idx >= 0) & (idx < np.asarray(n)[None, :]), axis=1) & (np.diff(al) > 0)
    lin = idx[:, 0] + n[0] * (idx[:, 1] + n[1] * idx[:, 2])
    return lin[ok], (np.diff(al) * np.linalg.norm(B - A))[ok]


def dedupe(seq):
    seq = np.asarray(seq)
    if seq.size == 0:
        return seq
    keep = np.ones(seq.size, bool)
    keep[1:] = seq[1:] != seq[:-1]
    return seq[keep]


def polyline_siddon(lo, h, n, verts):
    out = []
    for k in range(len(verts) - 1):
        v, _ = siddon(lo, h, n, verts[k], verts[k + 1])
        out.extend(v.tolist())
    return dedupe(np.array(out, dtype=np.int64))


GRIDS = [
    dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-g0", nx=40, ny=36, nz=12, u_tracker=40.0),
    dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-g1", nx=24, ny=30, nz=10, h=0.7, u_tracker=30.0),
]


@pytest.mark.parametrize("cfg", GRIDS, ids=lambda c: c.name)
def test_straight_line_limit_equals_siddon(oracle, cfg):
    """north_star: 'the straight-line limit, where MLP with no scattering must equal exact Siddon chords'.
    hull = NULL (all voxels): the list is Siddon's ordered non-zero-chord set of the box chord, N*l = L =
    sum of Siddon chords = slab-clipped chord length (pins (i) and (v) of SURVEY 8(c))."""
    rays = synth.random_rays(400, cfg, seed=5)
    g, p, pa, P = oracle_setup(oracle, cfg, rays, hull=None)
    row_ptr, vox, ell, flags, length = P.rows()
    rows = split_rows(row_ptr, vox)
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    hi = lo + n * cfg.h
    checked = 0
    for i in range(rays["phi"].numel()):
        a = {k: float(v[i]) for k, v in rays.items()}
        c, s = np.cos(a["phi"]), np.sin(a["phi"])
        T = np.array([-cfg.u_tracker * c - a["t_in"] * s, -cfg.u_tracker * s + a["t_in"] * c, a["v_in"]])
        d = np.array([c - a["dt_in"] * s, s + a["dt_in"] * c, a["dv_in"]])
        with np.errstate(divide="ignore", invalid="ignore"):
            s1, s2 = (lo - T) / d, (hi - T) / d
        s_in, s_out = max(0.0, np.max(np.minimum(s1, s2))), np.min(np.maximum(s1, s2))
        if not s_in < s_out:
            assert len(rows[i]) == 0 and flags[i] & oracle.REJ_MISS
            continue
        if flags[i] & oracle.REJECT_MASK:
            continue
        A, B = T + s_in * d, T + s_out * d
        ref, chords = siddon(lo, cfg.h, n, A, B)
        assert length[i] == pytest.approx(np.linalg.norm(B - A), rel=1e-12)
        assert len(rows[i]) * float(ell[i]) == pytest.approx(chords.sum(), rel=1e-6)
        if flags[i] & oracle.TIE:
            continue
        # zero-measure differences only where Siddon sees a chord shorter than the MLP vertices' rounding noise
        ref = ref[chords > 1e-9]
        got = rows[i]
        if len(got) != len(ref) or np.any(got != ref):
            short = set(siddon(lo, cfg.h, n, A, B)[0][chords <= 1e-9].tolist())
            assert set(got.tolist()) ^ set(ref.tolist()) <= short, i
        checked += 1
    assert checked > 300


def test_curved_paths_equal_per_segment_siddon(oracle):
    """Pin (iv): for scattered histories the list equals exact per-segment ray tracing of the MLP polyline."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 900)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    row_ptr, vox, ell, flags, length = P.rows()
    rows = split_rows(row_ptr, vox)
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    hull_flat = hull.numpy().reshape(-1)
    checked = 0
    for i in range(0, cfg.m, 3):
        if flags[i] & (oracle.REJECT_MASK | oracle.TIE):
            continue
        verts, vs, ve = oracle.polyline(g, p, pa, i, hull.numpy())
        ref = polyline_siddon(lo, cfg.h, n, verts)
        got = rows[i]
        assert got[0] == vs and hull_flat[vs] == 1 and hull_flat[ve] == 1
        assert len(got) == len(ref) and np.all(got == ref), i
        assert length[i] == pytest.approx(np.linalg.norm(np.diff(verts, axis=0), axis=1).sum(), rel=1e-12)
        assert float(ell[i]) == pytest.approx(length[i] / len(got), rel=1e-6)
        if not flags[i] & oracle.END_MISMATCH:
            assert got[-1] == ve
        checked += 1
    assert checked > 250


def test_brute_force_dense_sampling(oracle):
    """Sample the polyline every 2e-4 mm; consecutive-deduped floor() voxels must be a subsequence of the
    list, missing at most corner clips shorter than the sampling step."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 90)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    row_ptr, vox, ell, flags, _ = P.rows()
    rows = split_rows(row_ptr, vox)
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    done = 0
    for i in range(0, cfg.m, 9):
        if flags[i] & oracle.REJECT_MASK:
            continue
        verts, vs, ve = oracle.polyline(g, p, pa, i, hull.numpy())
        seq = []
        for k in range(len(verts) - 1):
            L = np.linalg.norm(verts[k + 1] - verts[k])
            s = (np.arange(int(L / 2e-4) + 1) + 0.5) / (int(L / 2e-4) + 1)
            pts = verts[k][None] + s[:, None] * (verts[k + 1] - verts[k])[None]
            idx = np.floor((pts - lo[None]) / cfg.h).astype(np.int64)
            seq.append(dedupe(idx[:, 0] + n[0] * (idx[:, 1] + n[1] * idx[:, 2])))
        brute = dedupe(np.concatenate(seq))
        got = rows[i]
        j = 0
        for v in got:                     # subsequence check
            if j < len(brute) and brute[j] == v:
                j += 1
        assert j == len(brute), i
        assert len(got) - len(brute) <= max(1, len(got) // 20)
        done += 1
    assert done >= 8


def test_list_topology(oracle):
    """Pins (ii),(iii): consecutive entries are 6-neighbours; N-1 >= Manhattan(V_s,V_e) with equal parity."""
    cfg = synth.scaled(synth.CONFIGS["head"], 3000)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    row_ptr, vox, ell, flags, _ = P.rows()
    assert P.total_visits == row_ptr[-1] and P.n_rejected < 0.05 * cfg.m
    strides = {1, cfg.nx, cfg.nx * cfg.ny}
    zspan = []
    for r in split_rows(row_ptr, vox):
        if len(r) == 0:
            continue
        d = np.abs(np.diff(r.astype(np.int64)))
        assert set(np.unique(d).tolist()) <= strides
        c0 = np.array(np.unravel_index(r[0], (cfg.nz, cfg.ny, cfg.nx)))
        c1 = np.array(np.unravel_index(r[-1], (cfg.nz, cfg.ny, cfg.nx)))
        man = np.abs(c1 - c0).sum()
        assert len(r) - 1 >= man and (len(r) - 1 - man) % 2 == 0
        z = r // (cfg.nx * cfg.ny)
        zspan.append((z.max() * cfg.h) // 2.5 - (z.min() * cfg.h) // 2.5 + 1)
    # loose shape check against PAPER.md Table I (:47-55): paths barely move along z
    assert np.mean(np.array(zspan) <= 4) > 0.9


def test_hull_entry_point(oracle):
    """R3-R4: V_s is the first hull voxel on the tracker ray; P_0 lies on that ray and on a face of V_s."""
    cfg = synth.scaled(synth.CONFIGS["tiny"], 300)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    _, _, _, flags, _ = P.rows()
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    hull_flat = hull.numpy().reshape(-1)
    for i in range(cfg.m):
        if flags[i] & oracle.REJECT_MASK:
            continue
        verts, vs, ve = oracle.polyline(g, p, pa, i, hull.numpy())
        a = {k: float(v[i]) for k, v in pr.items()}
        c, s = np.cos(a["phi"]), np.sin(a["phi"])
        for (u, t, v, dt, dv, P0, V, sign) in ((-cfg.u_tracker, a["t_in"], a["v_in"], a["dt_in"], a["dv_in"], verts[0], vs, 1),
                                               (cfg.u_tracker, a["t_out"], a["v_out"], a["dt_out"], a["dv_out"], verts[-1], ve, -1)):
            T = np.array([u * c - t * s, u * s + t * c, v])
            d = sign * np.array([c - dt * s, s + dt * c, dv])
            w = P0 - T
            assert np.linalg.norm(np.cross(w, d)) / np.linalg.norm(d) < 1e-10          # on the ray
            assert np.dot(w, d) > 0
            ray_vox, _ = siddon(lo, cfg.h, n, T, P0)                                   # everything before is air
            assert not hull_flat[ray_vox[ray_vox != V]].any()
            cv = np.array([V % cfg.nx, (V // cfg.nx) % cfg.ny, V // (cfg.nx * cfg.ny)])
            f_lo, f_hi = lo + cv * cfg.h, lo + (cv + 1) * cfg.h
            assert np.all(P0 >= f_lo - 1e-12) and np.all(P0 <= f_hi + 1e-12)          # in the closed voxel
            assert np.any((P0 == f_lo) | (P0 == f_hi))                                 # exactly on one of its faces


def test_rejections(oracle):
    cfg = synth.scaled(synth.CONFIGS["tiny"], 6)
    x_true, hull, shadow = synth.make_phantom(cfg)
    z = np.zeros(6)
    pr = dict(phi=z.copy(), t_in=z.copy(), v_in=z.copy(), dt_in=z.copy(), dv_in=z.copy(), t_out=z.copy(),
              v_out=z.copy(), dt_out=z.copy(), dv_out=z.copy())
    pr["t_in"][1] = pr["t_out"][1] = 15.5          # inside the grid, misses the r=12 hull
    pr["t_in"][2] = pr["t_out"][2] = 40.0          # misses the grid box
    pr["t_in"][3] = np.nan                          # non-finite
    pr["dv_in"][4] = 0.5; pr["v_out"][4] = 22.0; pr["dv_out"][4] = 0.5   # leaves through the top: exit ray misses
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    row_ptr, vox, ell, flags, _ = P.rows()
    N = np.diff(row_ptr)
    assert N[0] == 24 and flags[0] == 0             # straight through the centre: 24 voxels of the r=12 cylinder
    assert N[1] == 0 and flags[1] == oracle.REJ_MISS
    assert N[2] == 0 and flags[2] == oracle.REJ_MISS
    assert N[3] == 0 and flags[3] == oracle.REJ_NONFINITE
    assert N[4] == 0 and flags[4] & oracle.REJECT_MASK
    assert N[5] == 24
    # capacity and depth limits
    g, p, pa, P2 = oracle_setup(oracle, cfg, pr, hull, params_override=dict(max_visits=10))
    assert P2.rows()[3][0] == oracle.REJ_CAPACITY
    g, p, pa, P3 = oracle_setup(oracle, cfg, pr, hull, params_override=dict(poly_max_depth_mm=20.0))
    assert P3.rows()[3][0] == oracle.REJ_DEPTH
    assert P.n_rejected == 4 and P.total_visits == 48
