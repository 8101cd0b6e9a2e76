"""Pins of the oracle's Isobar-model pieces (O6b: "a sum of a constant non-resonant term and Breit-Wigner
functions", "constant nonresonant amplitude"; reading P27).

  * constant term alone: |A|^2 = |c|^2 everywhere, hence NLL = n ln(sum_j w_j) whatever c is (closed form);
  * the constant term is what a two-knot spline with both knot values c/2 gives (S(s12) + S(s13) = c): two different
    code paths of the oracle, the spline one pinned against scipy in tests/test_oracle_spline.py;
  * n_knots = 0 is the model whose knot values all vanish;
  * scalar Breit-Wigner: pole value i / (m0 Gamma0) with no barrier and no angular factor (spin 0 of O5);
  * gradient with respect to the constant's (|c|, arg c): Richardson-extrapolated differences of the pinned NLL, and
    the Euler identities of the global scale and phase invariance, which now have to include the constant.
"""
import numpy as np

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I

KIN = I.KIN_KKK
NONRES = dict(mass=0.0, width=0.0, spin=-1, r_res=0.0, r_parent=0.0)
F0 = dict(mass=1.35, width=0.25, spin=0, r_res=1.5, r_parent=5.0)
PHI = dict(mass=1.019461, width=0.004249, spin=1, r_res=1.5, r_parent=5.0)


def _points(n_ev=400, n_nm=900, seed=3):
    e12, e13 = I.phase_space_points(n_ev, I.stream_key(seed, 50, 0), KIN)
    g12, g13 = I.phase_space_points(n_nm, I.stream_key(seed, 50, 1), KIN)
    w = np.full(n_nm, I.dalitz_area(KIN) / n_nm)
    return e12, e13, g12, g13, w


def test_constant_term_alone_is_flat_and_its_nll_is_n_ln_sum_w():
    o = orc.Oracle(KIN, np.zeros(0), [NONRES])
    assert o.n_params == 2
    e12, e13, g12, g13, w = _points()
    for mag, arg in ((1.0, 0.0), (0.37, 2.1), (5.5, -1.3)):
        p = np.array([mag, arg])
        a2 = o.abs2(p, e12, e13)
        assert np.allclose(a2, mag * mag, rtol=1e-15, atol=0)
        amp = o.amplitude(p, e12[:5], e13[:5])
        assert np.allclose(amp, mag * np.exp(1j * arg), rtol=1e-15)
        assert abs(o.nll(p, e12, e13, g12, g13, w) - e12.size * np.log(w.sum())) < 1e-9


def test_constant_term_equals_a_two_knot_spline_with_both_values_half_of_it():
    lo, hi = I.s_limits(KIN)
    e12, e13, g12, g13, w = _points()
    cmag, carg = 0.8, -2.2
    iso = orc.Oracle(KIN, np.zeros(0), [F0, PHI, NONRES])
    spl = orc.Oracle(KIN, np.array([lo, hi]), [F0, PHI])
    p_iso = np.array([1.2, 0.4, 0.15, 1.9, cmag, carg])
    p_spl = np.array([cmag / 2, cmag / 2, carg, carg, 1.2, 0.4, 0.15, 1.9])
    a, b = iso.amplitude(p_iso, e12, e13), spl.amplitude(p_spl, e12, e13)
    assert np.max(np.abs(a - b)) <= 4e-16 * np.max(np.abs(a))
    assert abs(iso.nll(p_iso, e12, e13, g12, g13, w) - spl.nll(p_spl, e12, e13, g12, g13, w)) < 1e-10


def test_no_knots_is_the_model_with_vanishing_knot_values():
    e12, e13, _, _, _ = _points()
    res = [F0, PHI]
    a = orc.Oracle(KIN, np.zeros(0), res).amplitude(np.array([1.2, 0.4, 0.15, 1.9]), e12, e13)
    knots = np.linspace(1.0, 1.8, 5)
    p = np.concatenate([np.zeros(5), np.linspace(0, 1, 5), [1.2, 0.4, 0.15, 1.9]])
    b = orc.Oracle(KIN, knots, res).amplitude(p, e12, e13)
    assert np.array_equal(a, b)


def test_scalar_breit_wigner_pole_value_and_flat_angular_dependence():
    o = orc.Oracle(KIN, np.zeros(0), [F0])
    m0s = F0["mass"] ** 2
    t = o.resonance_term(0, m0s, 1.3) if hasattr(o, "resonance_term") else None
    L = orc.lib()
    import ctypes as C
    re, im = C.c_double(), C.c_double()
    r = orc.res_array([F0])
    for y in (1.05, 1.3, 1.6):                              # spin 0: no dependence on the other invariant
        L.orc_resonance_term(C.byref(o.kin), r, m0s, y, C.byref(re), C.byref(im))
        assert abs(re.value) < 1e-12 / (F0["mass"] * F0["width"])
        assert abs(im.value - 1.0 / (F0["mass"] * F0["width"])) < 1e-12 / (F0["mass"] * F0["width"])
    del t


def _richardson(f, x, k, h):
    def d(hh):
        xp, xm = x.copy(), x.copy()
        xp[k] += hh; xm[k] -= hh
        return (f(xp) - f(xm)) / (2 * hh)
    return (4 * d(h / 2) - d(h)) / 3


def test_gradient_with_constant_term_differences_and_euler_identities():
    lo, hi = I.s_limits(KIN)
    knots = np.linspace(lo * 1.001, hi * 0.999, 6)
    res = [F0, NONRES, PHI]                                  # the constant in the middle of the list
    o = orc.Oracle(KIN, knots, res)
    rng = np.random.default_rng(9)
    p = np.concatenate([rng.uniform(0.5, 2, 6), rng.uniform(0, 3, 6), [1.2, 0.4, 0.7, -0.9, 0.15, 1.9]])
    e12, e13, g12, g13, w = _points(300, 700, 4)
    f = lambda q: o.nll(q, e12, e13, g12, g13, w)
    nll, g = o.nll_grad(p, e12, e13, g12, g13, w)
    assert abs(nll - f(p)) < 1e-9
    for k in (0, 7, 12, 13, 14, 15, 16, 17):                 # a knot, a knot phase, every resonance-block entry
        fd = _richardson(f, p, k, 2e-3)
        assert abs(g[k] - fd) <= 2e-7 * max(1.0, np.max(np.abs(g))), (k, g[k], fd)
    mags = list(range(6)) + [12, 14, 16]
    phases = list(range(6, 12)) + [13, 15, 17]
    assert abs(sum(p[k] * g[k] for k in mags)) <= 1e-9 * np.sum(np.abs(g))     # common scale of ALL coefficients
    assert abs(sum(g[k] for k in phases)) <= 1e-9 * np.sum(np.abs(g))          # common phase
    # basis row: the constant's basis function is 1, and A = sum_k c_k B_k holds with it
    B = o.basis(p, e12[:20], e13[:20])
    assert np.array_equal(B[:, 6 + 1], np.ones(20, dtype=complex))
