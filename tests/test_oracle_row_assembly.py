"""Pin for the oracle's row assembly (compute_row): reading R8 (sampling) and R5 (end states) of DESIGN.md / SURVEY.md
8(c), i.e. everything between "hull entry/exit found" and "polyline handed to the walk" (tracker positions
and directions in, most likely path out).

The other walk tests take their vertices from pcto.polyline itself and the straight-line tests have equal entry and
exit slopes, so none of them sees (a) the number of MLP samples K = max(1, ceil(D / (step_frac h) - 1e-9)), (b) the
sample depths u0 + k D / K, (c) which tracker slope is paired with which end state in which plane, (d) the rotation of
(u, t_k, v_k) back to the grid frame.  Here every vertex is recomputed in numpy from the TRACKER RECORD: the hull entry
and exit points by an independent slab intersection with the first hull voxel found by Siddon's ray tracing, K and the
depths from R8, t_k and v_k from pcto.mlp_point (itself pinned in test_oracle_mlp.py) with (t0, dt_in) -> (t2, dt_out)
and (v0, dv_in) -> (v2, dv_out), and compared with pcto.polyline to 1e-10 mm.  Negative controls show that the
plausible mistakes (K from h instead of h/2, entry/exit slopes swapped, t/v planes swapped) move vertices by far more.
"""
import numpy as np

import synth
from helpers import oracle_setup
from test_oracle_walk import siddon


def first_hull_voxel(lo, h, n, hull_flat, T, d, reach):
    """First voxel with hull = 1 on the ray T + s d (Siddon order), and the point where the ray enters its box."""
    vox, _ = siddon(lo, h, n, T, T + reach * d)
    hit = vox[hull_flat[vox] != 0]
    if hit.size == 0:
        return None, None
    V = int(hit[0])
    c = np.array([V % n[0], (V // n[0]) % n[1], V // (n[0] * n[1])])
    f_lo, f_hi = lo + c * h, lo + (c + 1) * h
    with np.errstate(divide="ignore", invalid="ignore"):
        s1, s2 = (f_lo - T) / d, (f_hi - T) / d
    near = np.where(d != 0, np.minimum(s1, s2), -np.inf)
    a = int(np.argmax(near))
    P = T + near[a] * d
    P[a] = f_lo[a] if d[a] > 0 else f_hi[a]          # on the crossed face, exactly
    return V, P


def recompute_vertices(oracle, p, cfg, rec, hull_flat, step_h=None, swap_slopes=False, swap_planes=False):
    lo, n = np.array(cfg.lo), np.array([cfg.nx, cfg.ny, cfg.nz])
    c, s = np.cos(rec["phi"]), np.sin(rec["phi"])
    rot = lambda u, t, v: np.array([u * c - t * s, u * s + t * c, v])             # R1
    reach = 4.0 * cfg.u_tracker
    V_s, P0 = first_hull_voxel(lo, cfg.h, n, hull_flat, rot(-cfg.u_tracker, rec["t_in"], rec["v_in"]),
                               rot(1.0, rec["dt_in"], rec["dv_in"]), reach)
    V_e, PK = first_hull_voxel(lo, cfg.h, n, hull_flat, rot(cfg.u_tracker, rec["t_out"], rec["v_out"]),
                               -rot(1.0, rec["dt_out"], rec["dv_out"]), reach)
    if V_s is None or V_e is None:
        return None
    gan = lambda P: (P[0] * c + P[1] * s, -P[0] * s + P[1] * c, P[2])              # R1 inverse
    (u0, t0, v0), (u2, t2, v2) = gan(P0), gan(PK)
    D = u2 - u0
    step = 0.5 * (cfg.h if step_h is None else step_h)
    K = max(1, int(np.ceil(D / step - 1e-9)))                                      # R8
    dt_a, dt_b, dv_a, dv_b = rec["dt_in"], rec["dt_out"], rec["dv_in"], rec["dv_out"]
    if swap_slopes:
        dt_a, dt_b, dv_a, dv_b = dt_b, dt_a, dv_b, dv_a
    if swap_planes:
        dt_a, dv_a, dt_b, dv_b = dv_a, dt_a, dv_b, dt_b
    verts = [P0]
    for k in range(1, K):
        w1 = k * D / K
        tk = oracle.mlp_point(p, D, w1, (t0, dt_a), (t2, dt_b))[0]                 # R5: tracker slopes at both ends
        vk = oracle.mlp_point(p, D, w1, (v0, dv_a), (v2, dv_b))[0]
        verts.append(rot(u0 + w1, tk, vk))
    verts.append(PK)
    return np.array(verts), V_s, V_e, K


def test_row_assembly_matches_independent_recomputation(oracle):
    cfg = synth.scaled(synth.CONFIGS["tiny"], 1200)
    x_true, hull, shadow = synth.make_phantom(cfg)
    pr = synth.generate_protons(cfg, x_true, shadow)
    g, p, pa, P = oracle_setup(oracle, cfg, pr, hull)
    flags = P.rows()[3]
    hull_flat = hull.numpy().reshape(-1)
    checked, worst, n_interior = 0, 0.0, 0
    detect = dict(step=0, slopes=0, planes=0)
    for i in range(0, cfg.m, 3):
        if flags[i] & (oracle.REJECT_MASK | oracle.TIE):
            continue
        rec = {k: float(v[i]) for k, v in pr.items()}
        verts_o, vs, ve = oracle.polyline(g, p, pa, i, hull.numpy())
        verts, V_s, V_e, K = recompute_vertices(oracle, p, cfg, rec, hull_flat)
        assert (V_s, V_e) == (vs, ve), i
        assert len(verts_o) == K + 1, (i, len(verts_o), K)                         # the sample count of R8
        err = np.max(np.abs(verts - verts_o))
        worst = max(worst, err)
        assert err < 1e-10, (i, err)
        checked += 1
        n_interior += K - 1
        # negative controls: each plausible mistake must be visible at this tolerance
        wrong_k = recompute_vertices(oracle, p, cfg, rec, hull_flat, step_h=2.0 * cfg.h)
        detect["step"] += len(wrong_k[0]) != len(verts_o)
        for key, kw in (("slopes", dict(swap_slopes=True)), ("planes", dict(swap_planes=True))):
            w = recompute_vertices(oracle, p, cfg, rec, hull_flat, **kw)[0]
            detect[key] += len(w) == len(verts_o) and np.max(np.abs(w - verts_o)) > 1e-6
    assert checked >= 300 and n_interior > 20 * checked
    assert detect["step"] >= 0.95 * checked, detect      # a few chords are shorter than one step either way
    assert detect["slopes"] >= 0.9 * checked and detect["planes"] >= 0.9 * checked, detect


def test_sample_count_edge_cases(oracle):
    """R8 at the boundaries of ceil(): a chord of exactly k nominal steps gives K = k (the -1e-9 guard), slightly more
    gives k + 1; K = 1 for a chord shorter than one step (no interior vertex, the polyline is the segment P_0 P_K)."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["tiny"], name="tiny-slab", nx=16, ny=8, nz=4, m=4, u_tracker=20.0)
    lo = np.array(cfg.lo)
    # hull = slab of voxels ix in [4, 4 + w): a ray along +x (phi = 0, t = v = 0.3) has D = w exactly
    for w, expect in ((3, 6), (1, 2), (7, 14)):
        hull = np.zeros((cfg.nz, cfg.ny, cfg.nx), np.uint8)
        hull[:, :, 4:4 + w] = 1
        z = np.zeros(1)
        rays = dict(phi=z, t_in=z + 0.3, v_in=z + 0.3, dt_in=z, dv_in=z, t_out=z + 0.3, v_out=z + 0.3, dt_out=z, dv_out=z)
        g, p, pa, P = oracle_setup(oracle, dataclasses.replace(cfg, m=1), rays, hull)
        verts, vs, ve = oracle.polyline(g, p, pa, 0, hull)
        assert len(verts) == expect + 1
        assert verts[0][0] == lo[0] + 4 and verts[-1][0] == lo[0] + 4 + w
        assert np.allclose(np.diff(verts[:, 0]), 0.5, atol=1e-12)
    # oblique ray: D is not a multiple of the step -> K = ceil, uniform sub-steps D / K < step
    hull = np.zeros((cfg.nz, cfg.ny, cfg.nx), np.uint8)
    hull[:, :, 4:9] = 1
    phi = np.array([0.2])
    z = np.zeros(1)
    rays = dict(phi=phi, t_in=z, v_in=z + 0.3, dt_in=z, dv_in=z, t_out=z, v_out=z + 0.3, dt_out=z, dv_out=z)
    g, p, pa, P = oracle_setup(oracle, dataclasses.replace(cfg, m=1), rays, hull)
    verts, vs, ve = oracle.polyline(g, p, pa, 0, hull)
    D = 5.0 / np.cos(0.2)                                  # chord of the slab along the beam direction u
    K = int(np.ceil(D / 0.5))
    assert len(verts) == K + 1
    du = np.linalg.norm(np.diff(verts, axis=0), axis=1)
    assert np.allclose(du, D / K, rtol=1e-12) and D / K < 0.5
