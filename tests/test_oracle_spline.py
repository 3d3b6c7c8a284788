"""Pins P1-P3 of the oracle's not-a-knot cubic spline."""
import numpy as np
from scipy.interpolate import CubicSpline

from oracle import spline


def log_knots(n, lo=1e-4, hi=1e-1):
    return np.geomspace(lo, hi, n)


def test_p1_cubic_polynomials_reproduced_exactly():
    # north_star pin: a cubic is reproduced by the not-a-knot spline to 1e-12 (a natural spline would fail)
    x = log_knots(64, 0.5, 3.0)
    rng = np.random.default_rng(1)
    for _ in range(5):
        c = rng.standard_normal(4)
        y = c[0] + x * (c[1] + x * (c[2] + x * c[3]))
        coef = spline.coefficients(x, y)
        f = rng.uniform(x[0], x[-1], 2000)
        exact = c[0] + f * (c[1] + f * (c[2] + f * c[3]))
        got = spline.evaluate(x, coef, f)
        assert np.max(np.abs(got - exact)) <= 1e-12 * np.max(np.abs(exact))
        # slopes are the exact derivative at the knots
        s = spline.notaknot_slopes(x, y)
        assert np.allclose(s, c[1] + x * (2 * c[2] + 3 * c[3] * x), rtol=1e-11, atol=1e-11)


def test_p2_matches_scipy_notaknot_coefficients():
    x = log_knots(257)
    rng = np.random.default_rng(2)
    y = np.sin(40.0 * x) + rng.standard_normal(x.size) * 0.1
    coef = spline.coefficients(x, y)
    cs = CubicSpline(x, y, bc_type="not-a-knot")
    ref = cs.c[::-1].T                      # scipy stores highest power first: -> [S-1, (y, s, c, d)]
    scale = np.max(np.abs(ref), axis=0)
    assert np.all(np.max(np.abs(coef - ref), axis=0) <= 1e-10 * scale)
    f = rng.uniform(x[0], x[-1], 5000)
    assert np.max(np.abs(spline.evaluate(x, coef, f) - cs(f))) <= 1e-12 * np.max(np.abs(y))


def test_p2_small_systems():
    rng = np.random.default_rng(3)
    for n in (4, 5, 8):
        x = np.sort(rng.uniform(0.0, 1.0, n))
        y = rng.standard_normal(n)
        cs = CubicSpline(x, y, bc_type="not-a-knot")
        f = np.linspace(x[0], x[-1], 101)
        assert np.max(np.abs(spline.evaluate(x, spline.coefficients(x, y), f) - cs(f))) < 1e-10


def test_p3_fourth_order_convergence():
    fun = lambda v: np.sin(3.0 * np.log(v)) / v ** 0.25
    f = np.geomspace(1.1e-3, 0.9e-1, 20001)
    errs = []
    for n in (129, 257, 513):
        x = log_knots(n, 1e-3, 1e-1)
        errs.append(np.max(np.abs(spline.evaluate(x, spline.coefficients(x, fun(x)), f) - fun(f))))
    assert 12.0 < errs[0] / errs[1] < 20.0
    assert 12.0 < errs[1] / errs[2] < 20.0


def test_right_continuous_interval_choice():
    x = np.array([1.0, 2.0, 3.0, 4.0, 5.0])
    y = np.array([0.0, 1.0, 0.0, 2.0, 1.0])
    coef = spline.coefficients(x, y)
    assert np.allclose(spline.evaluate(x, coef, x), y, atol=1e-14)
