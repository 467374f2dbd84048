"""Pins for the oracle's MLP (T64 definition and T32 rule mirror).  CPU only.

Each test pins the oracle to something other than itself: a closed form, a brute-force
optimisation of the likelihood, numerical quadrature, an invariance, kinematics, or the worked
example of SURVEY.md Appendix A (tests/golden/survey_appendix_a.json).
"""
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate, optimize

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_appendix_a.json")))

A_CM = [7.457e-6, 4.548e-7, -5.777e-8, 1.301e-8, -9.228e-10, 2.687e-11]


def f_ref(s_mm):
    """1/(beta^2 p^2) polynomial retyped here (depth in cm inside)."""
    s = s_mm / 10.0
    return sum(a * s ** k for k, a in enumerate(A_CM))


# ---------------------------------------------------------------- P1: closed form
@pytest.mark.parametrize("L", [3.0, 64.0, 200.0])
def test_p1_constant_scattering_is_cubic_hermite(oracle_mod, L):
    """With constant scattering power and no log factor the maximum-likelihood path is the cubic
    Hermite spline through (t0,th0),(t2,th2) (it minimises int t''^2)."""
    a = [3.3e-6, 0, 0, 0, 0, 0]
    rng = np.random.default_rng(1)
    for _ in range(20):
        t0, t2 = rng.normal(0, 2, 2)
        th0, th2 = rng.normal(0, 0.02, 2)
        s = rng.uniform(0.02, 0.98) * L
        y = oracle_mod.mlp_matrix_f64(s, L, [t0, th0], [t2, th2], a_mm=a, use_log=False)
        x = s / L
        h00, h10 = 2 * x ** 3 - 3 * x ** 2 + 1, x ** 3 - 2 * x ** 2 + x
        h01, h11 = -2 * x ** 3 + 3 * x ** 2, x ** 3 - x ** 2
        t_ref = h00 * t0 + h10 * L * th0 + h01 * t2 + h11 * L * th2
        d00, d10 = (6 * x ** 2 - 6 * x) / L, 3 * x ** 2 - 4 * x + 1
        d01, d11 = (-6 * x ** 2 + 6 * x) / L, 3 * x ** 2 - 2 * x
        th_ref = d00 * t0 + d10 * th0 + d01 * t2 + d11 * th2
        assert y[0] == pytest.approx(t_ref, abs=1e-11)
        assert y[1] == pytest.approx(th_ref, abs=1e-12)


# ---------------------------------------------------------------- brute force on the definition
def test_matrix_form_maximises_the_likelihood(oracle_mod):
    """The matrix formula must be the minimiser of the chi^2 it was derived from; chi^2 itself is
    checked against a numpy re-statement with scipy quadrature for the covariance integrals."""
    L, s1 = 180.0, 70.0
    y0, y2 = np.array([0.3, 0.012]), np.array([2.1, -0.004])
    y = oracle_mod.mlp_matrix_f64(s1, L, y0, y2)

    def K(d):
        return (1 + 0.038 * math.log(d / 361.0)) ** 2

    def cov(lo, hi, ref, k):
        q = lambda n: integrate.quad(lambda s: (ref - s) ** n * f_ref(s), lo, hi, epsabs=0, epsrel=1e-13)[0]
        return k * np.array([[q(2), q(1)], [q(1), q(0)]])

    S1, S2 = cov(0, s1, s1, K(s1)), cov(s1, L, L, K(L - s1))

    def chi2(v):
        e1 = v - np.array([y0[0] + s1 * y0[1], y0[1]])
        e2 = y2 - np.array([v[0] + (L - s1) * v[1], v[1]])
        return e1 @ np.linalg.solve(S1, e1) + e2 @ np.linalg.solve(S2, e2)

    assert oracle_mod.mlp_chi2_f64(s1, L, y0, y2, y) == pytest.approx(chi2(y), rel=1e-9)
    scale = chi2(y)
    res = optimize.minimize(lambda v: chi2(v * np.array([1.0, 1e-2])) / scale, y / np.array([1.0, 1e-2]) + 0.3,
                            method="Nelder-Mead", options=dict(xatol=1e-10, fatol=1e-14, maxiter=4000))
    best = res.x * np.array([1.0, 1e-2])
    assert best[0] == pytest.approx(y[0], abs=2e-6)
    assert best[1] == pytest.approx(y[1], abs=2e-7)
    for dv in ([1e-3, 0], [0, 1e-5], [-1e-3, 1e-5]):
        assert chi2(y + np.array(dv)) > chi2(y)


def test_scattering_integrals_match_quadrature(oracle_mod):
    for s1, L in [(1.0, 2.5), (50.0, 200.0), (199.0, 200.0), (128.0, 256.0), (255.0, 255.5)]:
        S1, S2 = oracle_mod.sigma_f64(s1, L)
        for n, (v1, v2) in zip((2, 1, 0), zip(S1, S2)):
            q1 = integrate.quad(lambda s: (s1 - s) ** n * f_ref(s), 0, s1, epsabs=0, epsrel=1e-13)[0]
            q2 = integrate.quad(lambda s: (L - s) ** n * f_ref(s), s1, L, epsabs=0, epsrel=1e-13)[0]
            assert v1 == pytest.approx(q1, rel=1e-10)
            assert v2 == pytest.approx(q2, rel=1e-10)


# ---------------------------------------------------------------- P6: constants vs kinematics
def test_p6_scattering_polynomial_vs_kinematics(oracle_mod):
    """1/(beta^2 p^2) of a 200 MeV proton after depth s in water, residual energy from the
    Bragg-Kleeman range R = 0.0022 E^1.77 cm; the fit is good to <10 % over 0..20 cm."""
    mp = 938.272
    r0 = 0.0022 * 200.0 ** 1.77
    for s_cm in (0.0, 5.0, 10.0, 15.0, 20.0):
        e = ((r0 - s_cm) / 0.0022) ** (1 / 1.77)
        pv = (e * e + 2 * e * mp) / (e + mp)
        assert oracle_mod.scatter_f(10.0 * s_cm) == pytest.approx(1.0 / pv ** 2, rel=0.10)
        assert oracle_mod.scatter_f(10.0 * s_cm) == pytest.approx(f_ref(10.0 * s_cm), rel=1e-13)
    s = np.linspace(0, 512, 2049)
    assert min(oracle_mod.scatter_f(v) for v in s) > 0  # positive over the supported hull chords


# ---------------------------------------------------------------- P2, P3, P5
def test_p2_shear_equivariance_and_straight_line(oracle_mod):
    L = 150.0
    rng = np.random.default_rng(2)
    for _ in range(10):
        y0 = np.array([rng.normal(0, 1), rng.normal(0, 0.01)])
        y2 = np.array([rng.normal(0, 1), rng.normal(0, 0.01)])
        a, b = rng.normal(0, 5), rng.normal(0, 0.05)
        s = rng.uniform(1, L - 1)
        y = oracle_mod.mlp_matrix_f64(s, L, y0, y2)
        ysh = oracle_mod.mlp_matrix_f64(s, L, y0 + [a, b], y2 + [a + b * L, b])
        assert ysh[0] == pytest.approx(y[0] + a + b * s, abs=1e-11)
        assert ysh[1] == pytest.approx(y[1] + b, abs=1e-13)
    # collinear data: the path is the straight line
    y = oracle_mod.mlp_matrix_f64(40.0, L, [1.0, 0.02], [1.0 + 0.02 * L, 0.02])
    assert y[0] == pytest.approx(1.0 + 0.02 * 40.0, abs=1e-12)
    assert y[1] == pytest.approx(0.02, abs=1e-14)


def test_p3_endpoints(oracle_mod):
    L, y0, y2 = 120.0, [0.7, 0.015], [2.2, -0.01]
    a = oracle_mod.mlp_matrix_f64(1e-6, L, y0, y2)
    b = oracle_mod.mlp_matrix_f64(L - 1e-6, L, y0, y2)
    assert a[0] == pytest.approx(y0[0], abs=1e-7) and a[1] == pytest.approx(y0[1], abs=1e-6)
    assert b[0] == pytest.approx(y2[0], abs=1e-7) and b[1] == pytest.approx(y2[1], abs=1e-6)


def test_p5_log_factor_cancels_at_mid_depth_and_rule_log(oracle_mod):
    L, y0, y2 = 200.0, [0.0, 0.01], [1.5, -0.005]
    a = oracle_mod.mlp_matrix_f64(100.0, L, y0, y2, use_log=True)
    b = oracle_mod.mlp_matrix_f64(100.0, L, y0, y2, use_log=False)
    assert a[0] == pytest.approx(b[0], abs=1e-13)
    c = oracle_mod.mlp_matrix_f64(50.0, L, y0, y2, use_log=True)
    d = oracle_mod.mlp_matrix_f64(50.0, L, y0, y2, use_log=False)
    assert abs(c[0] - d[0]) > 5e-4  # away from the middle the log factor matters
    for x in np.concatenate([np.geomspace(2 ** -10 / 361, 1.5, 4001), [0.5, 1.0, 0.70710678, 0.7071068]]):
        assert oracle_mod.rule_log(x) == pytest.approx(math.log(float(np.float32(x))), abs=4e-6)


# ---------------------------------------------------------------- P12: worked example (one plane)
def test_p12_survey_worked_example_one_plane(oracle_mod):
    g = GOLD["one_plane"]
    for s, t in g["t_log"].items():
        assert oracle_mod.mlp_matrix_f64(float(s), g["L"], g["y0"], g["y2"])[0] == pytest.approx(t, abs=2e-8)
    for s, t in g["t_nolog"].items():
        assert oracle_mod.mlp_matrix_f64(float(s), g["L"], g["y0"], g["y2"], use_log=False)[0] == pytest.approx(t, abs=2e-8)
    # chord-frame coefficients: t(s) = c0*alpha0 + c2*alpha2 for data (0,alpha0),(0,alpha2)
    for s, (c0, c2) in g["chord_coefs"].items():
        assert oracle_mod.mlp_matrix_f64(float(s), g["L"], [0, 1.0], [0, 0.0])[0] == pytest.approx(c0, abs=2e-6)
        assert oracle_mod.mlp_matrix_f64(float(s), g["L"], [0, 0.0], [0, 1.0])[0] == pytest.approx(c2, abs=2e-6)


# ---------------------------------------------------------------- T32 coefficients vs T64 definition
def test_rule_coefficients_match_definition(oracle_mod):
    """c0, c2 of the fp32 rule against the fp64 matrix form (chord-frame unit responses)."""
    geom = oracle_mod.Geometry(256, 256, 16, 1.0, -192.0, 192.0)
    worst = 0.0
    rng = np.random.default_rng(5)
    for _ in range(60):
        t_in = rng.uniform(-120, 120)
        h = oracle_mod.binding._Hist(t_in, 0.0, t_in + rng.normal(0, 1), 0.5, rng.normal(0, 0.003), 0.0,
                                     rng.normal(0, 0.01), 0.001, 1.0, 0.0)
        r = oracle_mod.row_f32(geom, h)
        _, hull = oracle_mod.path_f64(geom, h)
        if r["nseg"] == 0:
            continue
        L = float(hull[6])
        K = r["nseg"] - 1
        for k in range(1, K + 1):
            c0 = oracle_mod.mlp_matrix_f64(float(k), L, [0, 1.0], [0, 0.0])[0]
            c2 = oracle_mod.mlp_matrix_f64(float(k), L, [0, 0.0], [0, 1.0])[0]
            worst = max(worst, abs(r["coefs"][k, 0] - c0) / max(1.0, abs(c0)),
                        abs(r["coefs"][k, 1] - c2) / max(1.0, abs(c2)))
    assert worst < 2e-4  # x 30 mrad => < 1e-5 mm
