"""Pins for the oracle's MLP (A2): the formalism of PAPER.md ref [3], readings R6-R8.

The paper prints no MLP number, so these pin the oracle to the mathematics: quadrature, the textbook cubic
Hermite special case, the maximum-likelihood definition itself (numerical chi^2 minimisation), invariances,
and the survey-time cross-check values in tests/golden/mlp_survey_values.txt.
"""
import os

import numpy as np
import pytest
from scipy import integrate, interpolate, optimize

import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "mlp_survey_values.txt")
POLY = synth.poly_mm(200.0, 200.0)
E0, X0 = 13.6, 361.0


def params(pcto, poly=POLY, log_coeff=0.038):
    return pcto.make_params(poly, 400.0, X0, log_coeff, 0.5, 1e-9, 2048)


def f_of(poly):
    return lambda w: sum(a * w ** i for i, a in enumerate(poly))


def sigma_quad(poly, w_a, w_b, W, log_coeff=0.038):
    """[[tt, tth],[tth, thth]] by adaptive quadrature of the definition."""
    f = f_of(poly)
    g = E0 ** 2 * (1 + log_coeff * np.log((w_b - w_a) / X0)) ** 2 / X0
    q = [integrate.quad(lambda w, k=k: (W - w) ** k * f(w), w_a, w_b, epsabs=0, epsrel=1e-13)[0] for k in (2, 1, 0)]
    return g * np.array([[q[0], q[1]], [q[1], q[2]]])


def golden():
    out = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def test_scatter_moments_match_quadrature(oracle):
    p = params(oracle)
    f = f_of(POLY)
    for (w_a, w_b, W) in [(0.0, 0.5, 0.5), (0.0, 100.0, 100.0), (100.0, 200.0, 200.0), (299.5, 300.0, 300.0),
                          (12.3, 77.7, 150.0), (0.0, 250.0, 250.0)]:
        got = oracle.scatter_moments(p, w_a, w_b, W)
        for k, idx in ((2, 0), (1, 1), (0, 2)):
            ref = integrate.quad(lambda w: (W - w) ** k * f(w), w_a, w_b, epsabs=0, epsrel=1e-13)[0]
            assert got[idx] == pytest.approx(ref, rel=1e-10), (w_a, w_b, W, k)


def test_survey_cross_check_values(oracle):
    """tests/golden/mlp_survey_values.txt (cm units) vs the oracle (mm units)."""
    gold = golden()
    p = params(oracle)

    def sig(w_a, w_b, W):
        m = oracle.scatter_moments(p, w_a, w_b, W)
        g = E0 ** 2 * (1 + 0.038 * np.log((w_b - w_a) / X0)) ** 2 / X0
        return g * m[0] / 100.0, g * m[1] / 10.0, g * m[2]          # mm^2 -> cm^2, mm -> cm
    s1, s2 = sig(0, 100, 100), sig(100, 200, 200)
    for got, key in zip(s1, ("tt", "tth", "thth")):
        assert got == pytest.approx(gold["sigma1_0_10cm_" + key], rel=2e-5)
    for got, key in zip(s2, ("tt", "tth", "thth")):
        assert got == pytest.approx(gold["sigma2_10_20cm_" + key], rel=2e-5)
    for w1, key in ((50.0, "mlp_t_5cm"), (100.0, "mlp_t_10cm"), (150.0, "mlp_t_15cm")):
        y = oracle.mlp_point(p, 200.0, w1, (0.0, 0.0), (2.0, 0.02))
        assert y[0] / 10.0 == pytest.approx(gold[key], rel=6e-6)   # printed to 6-7 digits


def test_constant_f_no_log_is_cubic_hermite(oracle):
    """poly=(c,0,..), log_coeff=0: the MLP is exactly the cubic Hermite interpolant of (t0,t0',t2,t2')."""
    p = params(oracle, poly=(3.3e-6, 0, 0, 0, 0, 0), log_coeff=0.0)
    rng = np.random.default_rng(1)
    for _ in range(20):
        D = rng.uniform(5, 300)
        y0 = (rng.uniform(-50, 50), rng.uniform(-0.1, 0.1))
        y2 = (rng.uniform(-50, 50), rng.uniform(-0.1, 0.1))
        spl = interpolate.CubicHermiteSpline([0.0, D], [y0[0], y2[0]], [y0[1], y2[1]])
        for w1 in rng.uniform(0.01 * D, 0.99 * D, 5):
            y = oracle.mlp_point(p, D, w1, y0, y2)
            assert y[0] == pytest.approx(float(spl(w1)), abs=1e-10)
            assert y[1] == pytest.approx(float(spl(w1, 1)), abs=1e-11)


def test_mlp_is_the_chi2_minimiser(oracle):
    """The defining property (maximum likelihood): y1 minimises
    (y1-R0 y0)^T S1^-1 (y1-R0 y0) + (y2-R1 y1)^T S2^-1 (y2-R1 y1), with S1,S2 from quadrature."""
    p = params(oracle)
    rng = np.random.default_rng(2)
    for _ in range(10):
        D = rng.uniform(20, 200)
        w1 = rng.uniform(0.1 * D, 0.9 * D)
        y0 = np.array([rng.uniform(-5, 5), rng.uniform(-0.05, 0.05)])
        y2 = np.array([rng.uniform(-5, 5), rng.uniform(-0.05, 0.05)])
        S1i = np.linalg.inv(sigma_quad(POLY, 0, w1, w1))
        S2i = np.linalg.inv(sigma_quad(POLY, w1, D, D))
        R0 = np.array([[1, w1], [0, 1.0]])
        R1 = np.array([[1, D - w1], [0, 1.0]])

        def chi2(y1):
            a, b = y1 - R0 @ y0, y2 - R1 @ y1
            return a @ S1i @ a + b @ S2i @ b
        y = oracle.mlp_point(p, D, w1, y0, y2)
        res = optimize.minimize(chi2, R0 @ y0, method="Nelder-Mead", options=dict(xatol=1e-10, fatol=1e-16, maxiter=4000))
        assert y[0] == pytest.approx(res.x[0], abs=2e-6)
        assert y[1] == pytest.approx(res.x[1], abs=2e-7)
        # and it is a stationary point: the gradient vanishes (much tighter than the simplex search)
        eps = np.array([1e-4, 1e-6])
        for k in range(2):
            d = np.zeros(2); d[k] = eps[k]
            assert chi2(y + d) > chi2(y) and chi2(y - d) > chi2(y)


def test_straight_line_identity(oracle):
    """If y2 = R1 R0 y0 (no scattering) the MLP is the straight line at every depth."""
    p = params(oracle)
    rng = np.random.default_rng(3)
    for _ in range(50):
        D = rng.uniform(1, 300)
        y0 = (rng.uniform(-100, 100), rng.uniform(-0.2, 0.2))
        y2 = (y0[0] + D * y0[1], y0[1])
        for w1 in rng.uniform(1e-3 * D, (1 - 1e-3) * D, 4):
            y = oracle.mlp_point(p, D, w1, y0, y2)
            assert y[0] == pytest.approx(y0[0] + w1 * y0[1], abs=1e-10)
            assert y[1] == pytest.approx(y0[1], abs=1e-11)


def test_endpoint_limits(oracle):
    """y_MLP(u0+eps) -> y0 and y_MLP(u2-eps) -> y2 (north_star: endpoints reproduce entry/exit)."""
    p = params(oracle)
    D, y0, y2 = 180.0, (3.0, 0.02), (9.5, -0.01)
    for eps in (1e-3, 1e-5):
        a = oracle.mlp_point(p, D, eps, y0, y2)
        b = oracle.mlp_point(p, D, D - eps, y0, y2)
        assert a[0] == pytest.approx(y0[0], abs=10 * eps) and a[1] == pytest.approx(y0[1], abs=10 * eps)
        assert b[0] == pytest.approx(y2[0], abs=10 * eps) and b[1] == pytest.approx(y2[1], abs=10 * eps)


def test_scale_invariance_of_poly(oracle):
    """Only ratios of Sigma matter (R7): scaling f by a constant leaves the path unchanged."""
    p1 = params(oracle)
    p2 = params(oracle, poly=tuple(7.5 * a for a in POLY))
    D, y0, y2 = 150.0, (-2.0, 0.03), (4.0, 0.05)
    for w1 in (10.0, 75.0, 140.0):
        a, b = oracle.mlp_point(p1, D, w1, y0, y2), oracle.mlp_point(p2, D, w1, y0, y2)
        assert a == pytest.approx(b, rel=1e-12, abs=1e-12)


def test_literal_form_equals_gaussian_conditioning_form(oracle):
    """Independent algebraic form: y = mu + S1 R1^T (R1 S1 R1^T + S2)^-1 (y2 - R1 mu), mu = R0 y0."""
    p = params(oracle)
    rng = np.random.default_rng(4)
    for _ in range(20):
        D = rng.uniform(10, 250)
        w1 = rng.uniform(0.02 * D, 0.98 * D)
        y0 = np.array([rng.uniform(-50, 50), rng.uniform(-0.1, 0.1)])
        y2 = np.array([rng.uniform(-50, 50), rng.uniform(-0.1, 0.1)])
        S1, S2 = sigma_quad(POLY, 0, w1, w1), sigma_quad(POLY, w1, D, D)
        R0, R1 = np.array([[1, w1], [0, 1.0]]), np.array([[1, D - w1], [0, 1.0]])
        mu = R0 @ y0
        ref = mu + S1 @ R1.T @ np.linalg.solve(R1 @ S1 @ R1.T + S2, y2 - R1 @ mu)
        y = oracle.mlp_point(p, D, w1, y0, y2)
        assert y[0] == pytest.approx(ref[0], abs=1e-9)
        assert y[1] == pytest.approx(ref[1], abs=1e-10)


def test_polynomial_tracks_bragg_kleeman():
    """R6: the 200 MeV coefficient set agrees with the closed-form 1/(beta^2 p^2) within 2.5 % on 0-200 mm
    (SURVEY quotes 1.6 % with slightly different constants), and the fitted 230 MeV set is positive and within 2 %."""
    d = np.linspace(0, 200, 201)
    f = f_of(POLY)(d)
    ref = synth.inv_beta2p2(synth.energy_at_depth(200.0, d))
    assert np.all(f > 0) and np.max(np.abs(f / ref - 1)) < 0.025
    cfg = synth.CONFIGS["paperB"]                       # 230 MeV: least-squares fit up to the largest chord
    poly = synth.poly_mm(cfg.energy, cfg.poly_max_depth)
    d = np.linspace(0, cfg.poly_max_depth, 611)
    ref = synth.inv_beta2p2(synth.energy_at_depth(230.0, d))
    assert np.all(f_of(poly)(d) > 0)
    assert np.max(np.abs(f_of(poly)(d) / ref - 1)) < 0.2
