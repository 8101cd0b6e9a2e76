"""Pins for the oracle's kinematics, barrier, width, propagator and angular factors.

Every expected value here comes from something other than the oracle's own formula: exact decimal constants,
energy-momentum conservation in explicit frames, Lorentz boosts of explicit four-vectors, spherical Hankel
functions from scipy, closed forms at the pole, and the elastic unitarity bound.
"""
import math
import os

import mpmath
import numpy as np
import pytest
from scipy.special import spherical_jn, spherical_yn

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I

PIPI = dict(I.KIN)
KPIPI = {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}     # unequal m1: exercises the general terms
RHO = {"mass": 0.775, "width": 0.149, "spin": 1, "r_res": 1.5, "r_parent": 5.0}
F2 = {"mass": 1.2755, "width": 0.1867, "spin": 2, "r_res": 1.5, "r_parent": 5.0}
F0 = {"mass": 0.98, "width": 0.07, "spin": 0, "r_res": 1.5, "r_parent": 5.0}


def make(kin, res):
    return orc.Oracle(kin, I.knots_uniform(4), res)


def read_golden(path):
    out = {}
    for line in open(path):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


# --------------------------------------------------------------------------------------------------------------
# independent kinematics: D rest frame energies and the triangle criterion; explicit four-vectors and boosts
# --------------------------------------------------------------------------------------------------------------
def physical(kin, s12, s13):
    """A configuration exists iff the three D-frame momenta close into a triangle."""
    M, m1, m2, m3 = kin["M"], kin["m1"], kin["m2"], kin["m3"]
    s23 = M * M + m1 * m1 + m2 * m2 + m3 * m3 - s12 - s13
    E1, E2, E3 = (M * M + m1 * m1 - s23) / (2 * M), (M * M + m2 * m2 - s13) / (2 * M), (M * M + m3 * m3 - s12) / (2 * M)
    if E1 < m1 or E2 < m2 or E3 < m3:
        return False
    p1, p2, p3 = math.sqrt(E1 * E1 - m1 * m1), math.sqrt(E2 * E2 - m2 * m2), math.sqrt(E3 * E3 - m3 * m3)
    return abs(p1 - p2) <= p3 <= p1 + p2


def four_vectors(kin, s12, s13):
    """Explicit (E, px, py, pz) of particles 1, 2, 3 in the D rest frame for a physical (s12, s13)."""
    M, m1, m2, m3 = kin["M"], kin["m1"], kin["m2"], kin["m3"]
    s23 = M * M + m1 * m1 + m2 * m2 + m3 * m3 - s12 - s13
    E1, E2 = (M * M + m1 * m1 - s23) / (2 * M), (M * M + m2 * m2 - s13) / (2 * M)
    p1, p2 = math.sqrt(E1 * E1 - m1 * m1), math.sqrt(E2 * E2 - m2 * m2)
    cos12 = (E1 * E2 - 0.5 * (s12 - m1 * m1 - m2 * m2)) / (p1 * p2)
    sin12 = math.sqrt(max(0.0, 1.0 - cos12 * cos12))
    v1 = np.array([E1, 0.0, 0.0, p1])
    v2 = np.array([E2, p2 * sin12, 0.0, p2 * cos12])
    v3 = np.array([M, 0.0, 0.0, 0.0]) - v1 - v2
    return v1, v2, v3


def boost_to_rest(v, frame):
    """Lorentz-boost four-vector v into the rest frame of four-vector `frame`."""
    m = math.sqrt(frame[0] ** 2 - frame[1:] @ frame[1:])
    beta = frame[1:] / frame[0]
    b2 = beta @ beta
    if b2 == 0.0:
        return v.copy()
    gamma = frame[0] / m
    bp = beta @ v[1:]
    e = gamma * (v[0] - bp)
    p = v[1:] + ((gamma - 1.0) * bp / b2 - gamma * v[0]) * beta
    return np.concatenate([[e], p])


def interior_points(kin, n, seed):
    rng = np.random.default_rng(seed)
    lo, hi = (kin["m1"] + kin["m2"]) ** 2, (kin["M"] - kin["m3"]) ** 2
    lo13 = (kin["m1"] + kin["m3"]) ** 2
    pts = []
    while len(pts) < n:
        a, b = rng.uniform(lo, hi), rng.uniform(lo13, hi)
        if physical(kin, a, b):
            pts.append((a, b))
    return pts


# --------------------------------------------------------------------------------------------------------------
def test_golden_constants(golden_dir):
    g = read_golden(os.path.join(golden_dir, "kinematics.txt"))
    lo, hi = I.s_limits(PIPI)
    assert lo == pytest.approx(g["s_min"], rel=1e-15)
    assert hi == pytest.approx(g["s_max"], rel=1e-15)
    o = make(PIPI, [RHO])
    # the oracle's s12 range is exactly [s_min, s_max]
    assert o.inside([g["s_min"] * (1 + 1e-12)], [0.5 * (g["sigma"] - g["s_min"])])[0]
    assert not o.inside([g["s_min"] * (1 - 1e-9)], [1.0])[0]
    assert not o.inside([g["s_max"] * (1 + 1e-9)], [0.3])[0]


def test_grid_cell_count_matches_triangle_criterion(golden_dir):
    g = read_golden(os.path.join(golden_dir, "kinematics.txt"))
    lo, hi = I.s_limits(PIPI)
    h = (hi - lo) / 100
    c = lo + (np.arange(100) + 0.5) * h
    o = make(PIPI, [RHO])
    a, b = np.meshgrid(c, c, indexing="ij")
    brute = np.array([physical(PIPI, x, y) for x, y in zip(a.ravel(), b.ravel())])
    assert int(brute.sum()) == int(g["n_cells_100"])
    assert np.array_equal(o.inside(a.ravel(), b.ravel()), brute)
    assert np.array_equal(I.inside(a.ravel(), b.ravel(), PIPI), brute)


@pytest.mark.parametrize("kin", [PIPI, KPIPI])
def test_inside_matches_triangle_criterion_random(kin):
    rng = np.random.default_rng(5)
    lo, hi = (kin["m1"] + kin["m2"]) ** 2 * 0.9, (kin["M"] - kin["m3"]) ** 2 * 1.05
    a, b = rng.uniform(lo, hi, 4000), rng.uniform(lo, hi, 4000)
    o = make(kin, [RHO])
    brute = np.array([physical(kin, x, y) for x, y in zip(a, b)])
    assert np.array_equal(o.inside(a, b), brute)
    assert np.array_equal(I.inside(a, b, kin), brute)
    assert 500 < brute.sum() < 3500


def test_area_matches_mpmath_quadrature_of_oracle_limits():
    o = make(PIPI, [RHO])
    lo, hi = I.s_limits(PIPI)
    mpmath.mp.dps = 30

    def width(s):
        a, b = o.s13_limits(float(s))
        return b - a

    # split at interior points so the end-point square roots are handled by tanh-sinh
    area = mpmath.quad(width, [lo, 0.2, 1.0, 2.5, hi], method="tanh-sinh", maxdegree=10)
    assert float(area) == pytest.approx(I.dalitz_area(PIPI), rel=1e-9)
    # independent: cell counting on a fine grid converges to the same area
    g12, _, w = I.grid_points(1000, PIPI)
    assert g12.size * w[0] == pytest.approx(I.dalitz_area(PIPI), rel=2e-4)
    assert g12.size / 1e6 == pytest.approx(0.595714, abs=2e-6)      # SURVEY 8(c) pin table


@pytest.mark.parametrize("kin", [PIPI, KPIPI])
def test_momenta_match_energy_conservation(kin):
    o = make(kin, [RHO])
    M, m1, m2, m3 = kin["M"], kin["m1"], kin["m2"], kin["m3"]
    for x in np.linspace((m1 + m2) ** 2 * 1.001, (M - m3) ** 2 * 0.999, 23):
        e1 = (x + m1 * m1 - m2 * m2) / (2 * math.sqrt(x))             # daughter energy in the resonance frame
        assert o.q2(x) == pytest.approx(e1 * e1 - m1 * m1, rel=1e-11, abs=1e-15)
        e3 = (M * M + m3 * m3 - x) / (2 * M)                           # bachelor energy in the parent frame
        assert o.pstar2(x) == pytest.approx(e3 * e3 - m3 * m3, rel=1e-11, abs=1e-15)


@pytest.mark.parametrize("kin", [PIPI, KPIPI])
def test_momenta_match_boosted_four_vectors(kin):
    o = make(kin, [RHO])
    for s12, s13 in interior_points(kin, 40, 11):
        v1, v2, v3 = four_vectors(kin, s12, s13)
        r1 = boost_to_rest(v1, v1 + v2)
        assert o.q2(s12) == pytest.approx(r1[1:] @ r1[1:], rel=1e-9, abs=1e-13)
        assert o.pstar2(s12) == pytest.approx(v3[1:] @ v3[1:], rel=1e-9, abs=1e-13)


@pytest.mark.parametrize("kin", [PIPI, KPIPI])
def test_zemach_factors_match_four_vector_angles(kin):
    """Z_1 = -4 p.q and Z_2 = 16 p^2 q^2 (cos^2 - 1/3) with p, q in the resonance frame (Zemach tensors)."""
    o = make(kin, [RHO])
    seen_neg = seen_pos = False
    for s12, s13 in interior_points(kin, 60, 3):
        v1, v2, v3 = four_vectors(kin, s12, s13)
        q = boost_to_rest(v1, v1 + v2)[1:]          # daughter a = particle 1
        p = boost_to_rest(v3, v1 + v2)[1:]          # bachelor
        pq = p @ q
        cos = pq / math.sqrt((p @ p) * (q @ q))
        seen_neg |= cos < -0.3
        seen_pos |= cos > 0.3
        assert o.zemach(0, s12, s13) == 1.0
        assert o.zemach(1, s12, s13) == pytest.approx(-4.0 * pq, rel=1e-9, abs=1e-12)
        assert o.zemach(2, s12, s13) == pytest.approx(16.0 * (p @ p) * (q @ q) * (cos * cos - 1.0 / 3.0),
                                                      rel=1e-9, abs=1e-12)
    assert seen_neg and seen_pos


def test_zemach_symmetries_equal_masses():
    o = make(PIPI, [RHO])
    sigma = PIPI["M"] ** 2 + 3 * PIPI["m1"] ** 2
    for x in (0.4, 0.9, 1.7):
        y = 0.5 * (sigma - x)                        # s13 = s23: the two daughters are exchanged symmetric
        assert abs(o.zemach(1, x, y)) < 1e-14
    # exchanging the daughters (y <-> s23) flips Z_1 and keeps Z_2
    x, y = 0.8, 1.1
    s23 = sigma - x - y
    assert o.zemach(1, x, s23) == pytest.approx(-o.zemach(1, x, y), rel=1e-12)
    assert o.zemach(2, x, s23) == pytest.approx(o.zemach(2, x, y), rel=1e-12)


@pytest.mark.parametrize("L", [1, 2])
def test_barrier_matches_spherical_hankel(L):
    """Blatt-Weisskopf: penetrability z^L B_L(z)^2 is proportional to 1 / (rho^2 |h_L^(1)(rho)|^2), rho^2 = z."""
    def pen(z):
        rho = math.sqrt(z)
        h2 = spherical_jn(L, rho) ** 2 + spherical_yn(L, rho) ** 2
        return 1.0 / (z * h2)

    for z0 in (0.3, 1.7):
        for z in (1e-3, 0.2, 0.9, 3.0, 40.0, 900.0):
            expect = math.sqrt(pen(z) / pen(z0) * (z0 / z) ** L)
            assert orc.barrier(L, z, z0) == pytest.approx(expect, rel=1e-11)


def test_barrier_limits():
    assert orc.barrier(0, 3.0, 0.2) == 1.0
    for L in (1, 2):
        assert orc.barrier(L, 0.7, 0.7) == 1.0                         # normalised to 1 at the pole
        zs = np.geomspace(1e-3, 1e6, 50)
        b = np.array([orc.barrier(L, z, 0.5) for z in zs])
        assert np.all(np.diff(b) < 0)                                   # decreasing in z
        big = orc.barrier(L, 1e12, 0.5)
        const = math.sqrt(1.5) if L == 1 else math.sqrt(9 + 1.5 + 0.25)
        assert big == pytest.approx(const * (1e12) ** (-L / 2), rel=1e-5)


@pytest.mark.parametrize("res", [RHO, F2, F0])
def test_breit_wigner_pole_and_unitarity(res):
    o = make(PIPI, [res])
    m0, g0 = res["mass"], res["width"]
    assert o.running_width(0, m0 * m0) == pytest.approx(g0, rel=1e-14)
    pole = o.breit_wigner(0, m0 * m0)
    assert pole.real == pytest.approx(0.0, abs=1e-12)
    assert pole.imag == pytest.approx(1.0 / (m0 * g0), rel=1e-13)     # BW(m0^2) m0 Gamma0 = i: phase exactly 90 deg
    lo, hi = I.s_limits(PIPI)
    xs = np.linspace(lo * 1.0001, hi, 400)
    bw = np.array([o.breit_wigner(0, x) for x in xs])
    gam = np.array([o.running_width(0, x) for x in xs])
    circle = m0 * gam * np.abs(bw)                                     # = sin(delta) <= 1, = 1 only at the pole
    assert np.all(circle <= 1.0 + 1e-13)
    assert xs[np.argmax(circle)] == pytest.approx(m0 * m0, abs=2 * (xs[1] - xs[0]))
    phase = np.unwrap(np.angle(bw))
    assert np.all(np.diff(phase) > 0)                                  # phase rises monotonically through 90 deg
    assert phase[0] < math.pi / 2 < phase[-1] or res is F2 or res is F0
    # elastic-unitarity identity Im BW = m0 Gamma |BW|^2
    assert np.allclose(bw.imag, m0 * gam * np.abs(bw) ** 2, rtol=1e-12, atol=0)


@pytest.mark.parametrize("res", [RHO, F2, F0])
def test_running_width_threshold_power(res):
    """Gamma(x) ~ q^(2L+1)/sqrt(x) near threshold (barrier -> const)."""
    o = make(PIPI, [res])
    lo, _ = I.s_limits(PIPI)
    x1, x2 = lo * (1 + 1e-6), lo * (1 + 4e-6)
    q1, q2 = math.sqrt(x1 / 4 - PIPI["m1"] ** 2), math.sqrt(x2 / 4 - PIPI["m1"] ** 2)
    ratio = o.running_width(0, x2) / o.running_width(0, x1)
    assert ratio == pytest.approx((q2 / q1) ** (2 * res["spin"] + 1) * math.sqrt(x1 / x2), rel=1e-4)


def test_running_width_full_formula_against_hankel_penetrability():
    """Gamma(x)/Gamma0 = [rho P_L(rho)]-ratio x m0/sqrt(x): the textbook q P_L(qr) / (q0 P_L(q0 r)) form."""
    for res in (RHO, F2):
        o = make(PIPI, [res])
        L, r, m0 = res["spin"], res["r_res"], res["mass"]

        def qpen(x):
            q = math.sqrt(x / 4 - PIPI["m1"] ** 2)
            rho = q * r
            return q / (rho * rho * (spherical_jn(L, rho) ** 2 + spherical_yn(L, rho) ** 2))

        for x in (0.2, 0.5, 0.9, 1.8, 2.8):
            expect = res["width"] * qpen(x) / qpen(m0 * m0) * m0 / math.sqrt(x)
            assert o.running_width(0, x) == pytest.approx(expect, rel=1e-10)


@pytest.mark.parametrize("kin", [PIPI, KPIPI])
def test_resonance_term_is_product_of_pinned_pieces(kin):
    """T_r = F_D F_R Z_L BW with F_D from the parent-frame bachelor momentum (reading P10)."""
    for ri, res in enumerate((RHO, F2, F0)):
        o = make(kin, [RHO, F2, F0])
        m0s = res["mass"] ** 2
        for s12, s13 in interior_points(kin, 12, 8):
            fr = orc.barrier(res["spin"], res["r_res"] ** 2 * o.q2(s12), res["r_res"] ** 2 * o.q2(m0s))
            fd = orc.barrier(res["spin"], res["r_parent"] ** 2 * o.pstar2(s12), res["r_parent"] ** 2 * o.pstar2(m0s))
            expect = fd * fr * o.zemach(res["spin"], s12, s13) * o.breit_wigner(ri, s12)
            got = o.resonance_term(ri, s12, s13)
            assert got == pytest.approx(expect, rel=1e-14)
