"""Pins for the oracle's natural cubic spline ("cubic spline [6]")."""
import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I


def complex_knots(n, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(0.5, 2.0, n) * np.exp(1j * (np.pi * np.arange(n) / (n - 1) + 0.2 * rng.normal(size=n)))


@pytest.mark.parametrize("knots", [I.knots_uniform(10), I.knots_uniform(50), I.knots_config2()])
def test_passes_exactly_through_knots_and_natural_ends(knots):
    y = complex_knots(knots.size, 1)
    s = orc.spline_eval(knots, y, knots)
    assert np.array_equal(s, y)                              # A_0(s_k) = a_k e^{i phi_k}, bit-exact in NR form
    for part in (y.real, y.imag):
        ypp = orc.spline_second_derivs(knots, part)
        assert ypp[0] == 0.0 and ypp[-1] == 0.0              # natural end condition (reading P2)
        h = np.diff(knots)
        lhs = h[:-1] / 6 * ypp[:-2] + (h[:-1] + h[1:]) / 3 * ypp[1:-1] + h[1:] / 6 * ypp[2:]
        rhs = np.diff(part)[1:] / h[1:] - np.diff(part)[:-1] / h[:-1]
        assert np.max(np.abs(lhs - rhs)) < 1e-12 * max(1.0, np.max(np.abs(rhs)))


@pytest.mark.parametrize("knots", [I.knots_uniform(10), I.knots_uniform(30), I.knots_config2()])
def test_matches_scipy_natural_cubic_spline_including_extrapolation(knots):
    y = complex_knots(knots.size, 2)
    lo, hi = I.s_limits()
    s = np.concatenate([np.linspace(lo, hi, 2001), knots, [knots[0] - 1e-3, knots[-1] + 3.1e-4, knots[-1] + 1e-2]])
    ref = CubicSpline(knots, y.real, bc_type="natural")(s) + 1j * CubicSpline(knots, y.imag, bc_type="natural")(s)
    got = orc.spline_eval(knots, y, s)
    assert np.max(np.abs(got - ref)) < 2e-13
    assert (s > knots[-1]).sum() >= 2 and (s < knots[0]).sum() >= 1     # reading P3 exercised on both sides


def test_derivatives_continuous_at_interior_knots():
    knots = I.knots_config2()
    y = complex_knots(knots.size, 3).real
    ypp = orc.spline_second_derivs(knots, y)
    h = np.diff(knots)
    # first derivative from the left and right segment formulas (Numerical Recipes eq. 3.3.5)
    slope = np.diff(y) / h
    d_right = slope[1:] - h[1:] * (2 * ypp[1:-1] + ypp[2:]) / 6        # S'(x_i^+) on segment i
    d_left = slope[:-1] + h[:-1] * (ypp[:-2] + 2 * ypp[1:-1]) / 6       # S'(x_i^-) on segment i-1
    assert np.max(np.abs(d_right - d_left)) < 1e-10
    # numerically, through the evaluated spline
    eps = 1e-6
    for k, xk in enumerate(knots[1:-1], start=1):
        f = lambda s: orc.spline_eval(knots, y + 0j, [s])[0].real
        dl = (f(xk) - f(xk - eps)) / eps
        dr = (f(xk + eps) - f(xk)) / eps
        # one-sided differences differ by eps S''(x_k) when S' is continuous; a kink would show as O(1)
        assert dr - dl == pytest.approx(eps * ypp[k], abs=1e-3 * eps * abs(ypp[k]) + 2e-8)


def test_closed_forms():
    # N = 3 uniform: y''_1 = 3 (y0 - 2 y1 + y2) / (2 h^2)
    x = np.array([0.2, 0.7, 1.2])
    y = np.array([1.3, -0.4, 2.2])
    ypp = orc.spline_second_derivs(x, y)
    assert ypp[1] == pytest.approx(3 * (y[0] - 2 * y[1] + y[2]) / (2 * 0.25), rel=1e-14)
    assert ypp[0] == 0 and ypp[2] == 0
    # collinear data: y'' = 0 and the spline is the straight line, also outside the knots
    x = I.knots_config2()
    line = 0.3 - 1.7 * x
    assert np.max(np.abs(orc.spline_second_derivs(x, line))) < 1e-11
    s = np.linspace(0.0, 3.2, 101)
    assert np.max(np.abs(orc.spline_eval(x, line + 0j, s).real - (0.3 - 1.7 * s))) < 1e-12
    # N = 2: linear interpolation of the complex values
    got = orc.spline_eval([1.0, 3.0], [1 + 1j, 3 - 1j], [1.5, 4.0])
    assert np.allclose(got, [1.5 + 0.5j, 4 - 2j], rtol=0, atol=1e-15)
    # a cubic with vanishing second derivative at both ends is reproduced exactly: p(s) = (s-a)^3 - 3 (b-a)(s-a)^2 ... use
    # p'' = 6 (s-a) - 6 (s-a)^2/(b-a) is not cubic; instead check the interpolation error order: h^4 on a smooth function
    f = lambda s: np.sin(3 * s)
    errs = []
    for n in (20, 40, 80):
        xs = np.linspace(0.5, 2.5, n)
        mid = np.linspace(1.2, 1.8, 301)                      # away from the natural ends
        errs.append(np.max(np.abs(orc.spline_eval(xs, f(xs) + 0j, mid).real - f(mid))))
    assert errs[0] / errs[1] > 10 and errs[1] / errs[2] > 10  # ~16x per halving (4th order)


def test_real_and_imaginary_parts_are_splined_separately():
    """Reading P1: the spline acts on Re and Im of y_k, hence it is linear in the complex knot values."""
    knots = I.knots_uniform(12)
    y1, y2 = complex_knots(12, 4), complex_knots(12, 5)
    s = np.linspace(0.1, 2.9, 57)
    a, b = 0.7 - 0.2j, -1.1 + 0.5j
    lhs = orc.spline_eval(knots, a * y1 + b * y2, s)
    rhs = a * orc.spline_eval(knots, y1, s) + b * orc.spline_eval(knots, y2, s)
    assert np.max(np.abs(lhs - rhs)) < 1e-13
