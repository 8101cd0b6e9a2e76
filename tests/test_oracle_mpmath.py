"""Accuracy pin of the oracle's whole amplitude (SURVEY 8(c) pin table, "Whole amplitude": mpmath 40-digit evaluation of
O1-O6 on ~100 points).  The GPU parity bar is 1e-12 per event, so the oracle's own double-precision evaluation must be
good to ~1e-13: here |A|^2 from the C++ oracle is compared with the same definition carried out in 40-digit arithmetic
(mpmath: Kallen functions, Blatt-Weisskopf ratios, running width, Breit-Wigner, Zemach factors, natural cubic spline by
an exact-arithmetic tridiagonal solve), on seeded points chosen where double precision is at its worst: within 1e-6 of
the thresholds, beyond the last knot, on the rho(770) / phi(1020) poles, for equal and unequal daughter masses.

Tolerance (reading P15): |d|A|^2| <= 5e-14 x (sum_k |c_k B_k|)^2, the incoherent scale -- rounding errors scale with the
terms that are added, not with what is left after they interfere.  Within a relative 1e-5 of the threshold
(m1 + m2)^2 the bound is 5e-13: the oracle evaluates the Kallen function in its plain form a^2 + b^2 + c^2 - 2ab - ..
(it has to stay the plain definition), which cancels there; measured 9e-14 at 1e-6 from an unequal-mass threshold."""
import numpy as np
import pytest

mp = pytest.importorskip("mpmath")

from oracle import oracle as orc                      # noqa: E402
from paper_1703_03284_b200 import inputs as I         # noqa: E402

mp.mp.dps = 40
F = mp.mpf


def kallen(a, b, c):
    return a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c


def barrier(L, z, z0):
    if L == 0:
        return F(1)
    if L == 1:
        return mp.sqrt((1 + z0) / (1 + z))
    return mp.sqrt((9 + 3 * z0 + z0 * z0) / (9 + 3 * z + z * z))


def term(kin, r, x, y):
    """T_r(x, y) = F_D F_R Z_L BW, readings P9 / P10 of DESIGN.md, in 40-digit arithmetic"""
    M, m1, m2, m3 = (F(kin[k]) for k in ("M", "m1", "m2", "m3"))
    m0, g0, L = F(r["mass"]), F(r["width"]), int(r["spin"])
    rr, rp = F(r["r_res"]), F(r["r_parent"])
    q2 = lambda s: kallen(s, m1 * m1, m2 * m2) / (4 * s)
    p2 = lambda s: kallen(M * M, s, m3 * m3) / (4 * M * M)
    FR = barrier(L, rr * rr * q2(x), rr * rr * q2(m0 * m0))
    FD = barrier(L, rp * rp * p2(x), rp * rp * p2(m0 * m0))
    ratio = q2(x) / q2(m0 * m0)
    width = g0 * ratio ** L * mp.sqrt(ratio) * (m0 / mp.sqrt(x)) * FR * FR
    bw = 1 / mp.mpc(m0 * m0 - x, -m0 * width)
    s23 = M * M + m1 * m1 + m2 * m2 + m3 * m3 - x - y
    Z1 = y - s23 + (M * M - m3 * m3) * (m2 * m2 - m1 * m1) / x
    Z = F(1) if L == 0 else (Z1 if L == 1 else Z1 * Z1 - kallen(M * M, x, m3 * m3) * kallen(x, m1 * m1, m2 * m2) / (3 * x * x))
    return FD * FR * Z * bw


def natural_spline(xk, yk):
    """second derivatives of the natural cubic spline through (xk, yk): the tridiagonal system of Numerical Recipes"""
    n = len(xk)
    ypp = [mp.mpc(0)] * n
    if n < 3:
        return ypp
    A = mp.zeros(n - 2, n - 2)
    b = mp.zeros(n - 2, 1)
    for i in range(1, n - 1):
        if i > 1:
            A[i - 1, i - 2] = (xk[i] - xk[i - 1]) / 6
        A[i - 1, i - 1] = (xk[i + 1] - xk[i - 1]) / 3
        if i < n - 2:
            A[i - 1, i] = (xk[i + 1] - xk[i]) / 6
        b[i - 1] = (yk[i + 1] - yk[i]) / (xk[i + 1] - xk[i]) - (yk[i] - yk[i - 1]) / (xk[i] - xk[i - 1])
    sol = mp.lu_solve(A, b)
    for i in range(1, n - 1):
        ypp[i] = sol[i - 1]
    return ypp


def spline(xk, yk, ypp, s):
    n = len(xk)
    if n == 0:
        return mp.mpc(0)
    j = 0
    while j < n - 2 and s >= xk[j + 1]:
        j += 1
    h = xk[j + 1] - xk[j]
    a = (xk[j + 1] - s) / h
    b = 1 - a
    return a * yk[j] + b * yk[j + 1] + ((a ** 3 - a) * ypp[j] + (b ** 3 - b) * ypp[j + 1]) * h * h / 6


def amplitude_mp(kin, knots, resonances, params, s12, s13):
    """(A, incoherent scale sum_k |term_k|) of O6 in 40-digit arithmetic; doubles enter as the exact values they hold"""
    N, R = len(knots), len(resonances)
    xk = [F(float(k)) for k in knots]
    p = [F(float(v)) for v in params]
    yk = [p[k] * mp.mpc(mp.cos(p[N + k]), mp.sin(p[N + k])) for k in range(N)]
    ypp = natural_spline(xk, yk)
    shapes, f = [], 0
    for r in resonances:
        r = dict(r)
        if r.get("shape_floats"):
            r["mass"], r["width"] = p[2 * N + 2 * R + 2 * f], p[2 * N + 2 * R + 2 * f + 1]
            f += 1
        shapes.append(r)
    x, y = F(float(s12)), F(float(s13))
    parts = [spline(xk, yk, ypp, x), spline(xk, yk, ypp, y)]
    for i, r in enumerate(shapes):
        c = p[2 * N + 2 * i] * mp.mpc(mp.cos(p[2 * N + 2 * i + 1]), mp.sin(p[2 * N + 2 * i + 1]))
        parts.append(c * (mp.mpc(1) if r["spin"] == -1 else term(I_kin(kin), r, x, y) + term(I_kin(kin), r, y, x)))
    A = sum(parts, mp.mpc(0))
    return A, sum(abs(t) for t in parts)


def I_kin(kin):
    return kin


def _points(kin, knots, resonances, n_random, seed):
    """seeded interior points + the places where double precision is strained"""
    lo, hi = I.s_limits(kin)
    key = I.stream_key(seed, 40, 0)
    a, b = I.phase_space_points(n_random, key, kin)
    pts = list(zip(a, b))
    # along the boundary of s12 (within 1e-6 of both thresholds), s13 at the centre of its band
    for s in (lo * (1 + 1e-6), lo + 1e-9, hi * (1 - 1e-6), hi - 1e-9):
        c, h = I.s13_band(np.array([s]), kin)
        pts += [(s, float(c[0])), (float(c[0]), s)]
    # beyond the last knot and before the first one, when the knots do not cover the whole range
    if len(knots):
        for s in (0.5 * (knots[-1] + hi), 0.5 * (knots[0] + lo)):
            if lo < s < hi:
                c, h = I.s13_band(np.array([s]), kin)
                pts.append((s, float(c[0] + 0.3 * h[0])))
        k = len(knots) // 2                         # exactly on a knot, and one ulp either side
        for s in (knots[k], np.nextafter(knots[k], 0.0), np.nextafter(knots[k], 10.0)):
            c, h = I.s13_band(np.array([s]), kin)
            pts.append((float(s), float(c[0] - 0.2 * h[0])))
    # on the poles
    for r in resonances:
        if r["spin"] >= 0:
            s = float(r["mass"]) ** 2
            if lo < s < hi:
                c, h = I.s13_band(np.array([s]), kin)
                pts += [(s, float(c[0] + 0.5 * h[0])), (float(c[0] - 0.5 * h[0]), s)]
    return [(x, y) for x, y in pts if I.inside(np.array([x]), np.array([y]), kin)[0]]


def _check(kin, knots, resonances, params, n_random, seed):
    o = orc.Oracle(kin, knots, resonances)
    pts = _points(kin, knots, resonances, n_random, seed)
    assert len(pts) >= n_random
    s12 = np.array([p[0] for p in pts])
    s13 = np.array([p[1] for p in pts])
    got = o.abs2(params, s12, s13)
    lo, _ = I.s_limits(kin)
    worst = 0.0
    for (x, y), g in zip(pts, got):
        A, scale = amplitude_mp(kin, knots, resonances, params, x, y)
        ref = A.real ** 2 + A.imag ** 2
        err = abs(F(float(g)) - ref) / (scale * scale)
        worst = max(worst, float(err))
        near_threshold = min(x, y) < lo * (1 + 1e-5)
        assert err <= F("5e-13" if near_threshold else "5e-14"), (x, y, float(g), float(ref), float(err))
    return worst


def test_config1_amplitude_against_40_digit_arithmetic():
    """30 knots + rho(770) + f2(1270) on D+ -> pi+ pi+ pi- (BASELINE configs[1])"""
    c = I.Config(1)
    _check(c.kin, c.knots, c.resonances, c.perturbed(3), 60, 1)


def test_config3_floating_shape_against_40_digit_arithmetic():
    """50 knots + floating rho(770) + rho(1450) + f2(1270): the bench model, shapes taken from the parameter vector"""
    c = I.Config(3)
    _check(c.kin, c.knots, c.resonances, c.perturbed(7), 30, 2)


def test_kkk_phi1020_against_40_digit_arithmetic():
    """the paper's own decay D+ -> K+ K+ K-: 40 knots + the 4 MeV wide phi(1020) (config 5; pole value ~ 230)"""
    c = I.Config(5)
    _check(c.kin, c.knots, c.resonances, c.truth, 30, 3)


def test_unequal_masses_against_40_digit_arithmetic():
    """K- pi+ pi+ -like kinematics (m1 != m2): the general-mass q^2, Zemach and boundary forms; spins 0, 1, 2"""
    kin = {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}
    lo, hi = I.s_limits(kin)
    knots = np.linspace(lo * 1.01, hi * 0.98, 12)
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=1.5, r_parent=5.0),
           dict(mass=1.4324, width=0.109, spin=2, r_res=1.5, r_parent=5.0),
           dict(mass=1.425, width=0.27, spin=0, r_res=1.5, r_parent=5.0)]
    rng = np.random.default_rng(5)
    p = np.concatenate([rng.uniform(0.5, 2, 12), rng.uniform(0, 3, 12), [1.0, 0.2, 0.6, 2.0, 1.3, -1.0]])
    _check(kin, knots, res, p, 40, 4)


def test_isobar_model_against_40_digit_arithmetic():
    """Isobar S-wave: no spline, a constant non-resonant term, a scalar Breit-Wigner and phi(1020)"""
    c = I.Config(5)
    res = [dict(mass=1.35, width=0.25, spin=0, r_res=1.5, r_parent=5.0),
           dict(mass=1.019461, width=0.004249, spin=1, r_res=1.5, r_parent=5.0),
           dict(mass=0.0, width=0.0, spin=-1, r_res=0.0, r_parent=0.0)]
    p = np.array([1.2, 0.4, 0.15, 1.9, 0.8, -2.2])
    _check(c.kin, np.zeros(0), res, p, 40, 5)
