"""Pins of the oracle's shape derivatives (O10: d/d(mass, width) of a resonance term and of the NLL; SURVEY 8(f) f2,
not in the paper).  The resonance term and the NLL are pinned elsewhere (test_oracle_kinematics.py, test_oracle_nll.py);
here their analytic derivatives are checked against Richardson-extrapolated central differences of those functions,
and against two closed forms at the pole."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I

KIN_PIPIPI = dict(I.KIN)
KIN_KPIPI = {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}


def _richardson(f, x, h):
    d = lambda s: (f(x + s) - f(x - s)) / (2 * s)
    return (4 * d(h / 2) - d(h)) / 3


@pytest.mark.parametrize("kin", [KIN_PIPIPI, KIN_KPIPI])
@pytest.mark.parametrize("spin", [0, 1, 2])
def test_resonance_term_shape_derivatives_match_finite_differences(kin, spin):
    lo, hi = I.s_limits(kin)
    m0 = 0.5 * (np.sqrt(lo) + np.sqrt(hi)) * 0.93
    base = dict(mass=m0, width=0.11, spin=spin, r_res=1.5, r_parent=5.0)
    s12, s13 = I.phase_space_points(40, I.stream_key(7, 1, spin), kin)
    for x, y in zip(s12, s13):
        def T(mass=base["mass"], width=base["width"]):
            r = dict(base, mass=mass, width=width)
            return orc.Oracle(kin, np.array([lo, hi]), [r]).resonance_term(0, x, y)
        dm, dg = orc.Oracle(kin, np.array([lo, hi]), [base]).resonance_term_dshape(base, x, y)
        fm = _richardson(lambda v: T(mass=v), base["mass"], 2e-4)
        fg = _richardson(lambda v: T(width=v), base["width"], 2e-4)
        scale = abs(T()) / base["width"]
        assert abs(dm - fm) <= 2e-8 * max(abs(fm), scale)
        assert abs(dg - fg) <= 2e-8 * max(abs(fg), scale)


def test_width_derivative_at_the_pole_closed_form():
    """At x = m0^2: BW = i/(m0 Gamma0), F = 1, so T = Z i/(m0 Gamma0) and dT/dGamma0 = -T/Gamma0 exactly."""
    kin = KIN_PIPIPI
    r = dict(mass=0.775, width=0.149, spin=1, r_res=1.5, r_parent=5.0)
    o = orc.Oracle(kin, np.array([0.08, 2.99]), [r])
    x, y = r["mass"] ** 2, 1.3
    T = o.resonance_term(0, x, y)
    _, dg = o.resonance_term_dshape(r, x, y)
    assert abs(dg + T / r["width"]) <= 1e-13 * abs(T / r["width"])


def test_nll_shape_gradient_matches_finite_differences():
    """config 3's model (rho(770) mass and width in the parameter vector) on a small sample."""
    c = I.Config(3, n_ev=3000, n_norm=6000)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    e12, e13 = I.phase_space_points(3000, c.key(7), c.kin)
    g12, g13, w = c.norm_points()
    p = c.perturbed(2)
    nll, gs = o.nll_grad_shape(p, e12, e13, g12, g13, w)
    assert nll == pytest.approx(o.nll(p, e12, e13, g12, g13, w), rel=1e-14)
    assert gs.size == 2
    for t, h in ((0, 1e-4), (1, 1e-4)):
        idx = c.n_params - 2 + t

        def f(v):
            q = p.copy(); q[idx] = v
            return o.nll(q, e12, e13, g12, g13, w)
        fd = _richardson(f, p[idx], h)
        assert gs[t] == pytest.approx(fd, rel=2e-6, abs=1e-6 * abs(nll))


def test_nll_shape_gradient_two_floating_resonances_and_unweighted_norm():
    kin = KIN_KPIPI
    lo, hi = I.s_limits(kin)
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=1.5, r_parent=5.0, shape_floats=1),
           dict(mass=1.2, width=0.2, spin=0, r_res=1.5, r_parent=5.0, shape_floats=0),
           dict(mass=1.4324, width=0.109, spin=2, r_res=2.0, r_parent=4.0, shape_floats=1)]
    knots = np.linspace(lo - 1e-3, hi + 1e-3, 9)
    o = orc.Oracle(kin, knots, res)
    s12, s13 = I.phase_space_points(3000, I.stream_key(3, 12, 1), kin)
    rng = np.random.default_rng(3)
    p = np.concatenate([rng.uniform(0.5, 2, 9), rng.uniform(0, 3, 9), rng.uniform(0.3, 1.5, 6),
                        [0.8955, 0.047, 1.4324, 0.109]])
    nll, gs = o.nll_grad_shape(p, s12[:1000], s13[:1000], s12[1000:], s13[1000:], None)
    assert gs.size == 4
    for t in range(4):
        idx = p.size - 4 + t

        def f(v):
            q = p.copy(); q[idx] = v
            return o.nll(q, s12[:1000], s13[:1000], s12[1000:], s13[1000:], None)
        fd = _richardson(f, p[idx], 1e-4)
        assert gs[t] == pytest.approx(fd, rel=5e-6, abs=1e-6 * abs(nll))


def test_hessian_matches_differences_of_the_pinned_gradient_and_the_invariance_identities():
    """O11: the oracle's analytic Hessian against Richardson central differences of its (separately pinned) analytic
    gradient, its symmetry, and the two exact identities that follow from differentiating the Euler relations
    sum_b dNLL/dphi_b = 0 (global phase) and sum_b rho_b dNLL/drho_b = 0 (global scale):
        sum_b H[a, phi_b] = 0    and    sum_b rho_b H[a, rho_b] + [a is a magnitude] g_a = 0   for every a."""
    c = I.Config(1, n_ev=1500, n_norm=3000)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    e12, e13 = I.phase_space_points(1500, c.key(7), c.kin)
    g12, g13, w = c.norm_points()
    p = c.perturbed(3)
    H = o.nll_hessian(p, e12, e13, g12, g13, w)
    P, N, R = p.size, c.N, c.R
    assert H.shape == (P, P)
    scale = np.max(np.abs(H))
    assert np.max(np.abs(H - H.T)) <= 1e-12 * scale
    _, g = o.nll_grad(p, e12, e13, g12, g13, w)
    is_phi = np.zeros(P, dtype=bool); is_phi[N:2 * N] = True; is_phi[2 * N + 1::2] = True
    rho = np.where(is_phi, 0.0, p)
    assert np.max(np.abs(H[:, is_phi].sum(axis=1))) <= 1e-10 * scale
    assert np.max(np.abs(H @ rho + np.where(is_phi, 0.0, g))) <= 1e-10 * scale * np.max(np.abs(p))
    for a in (0, 3, N - 1, N + 2, 2 * N - 1, 2 * N, 2 * N + 1, 2 * N + 3):
        def grad_at(v):
            q = p.copy(); q[a] = v
            return o.nll_grad(q, e12, e13, g12, g13, w)[1]
        col = _richardson(grad_at, p[a], 1e-5)             # 1e-4 still leaves 5e-7 of truncation error (narrow rho)
        assert np.max(np.abs(col - H[a])) <= 1e-9 * scale


def test_gradient_parts_match_differences_of_the_two_sums_and_recombine():
    """O9b: the per-rank pieces grad_ev = d(-S)/dtheta and grad_nm = dI/dtheta against Richardson
    differences of S = sum ln|A|^2 and I as orc_nll returns them (pinned on their own), over every kind of parameter
    (knot magnitude and phase, resonance magnitude and phase, floating mass and width); grad_ev + (n/I) grad_nm must
    be the pinned gradients of O9 and O10; an empty event set leaves grad_ev = 0."""
    kin = KIN_KPIPI
    lo, hi = I.s_limits(kin)
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=1.5, r_parent=5.0, shape_floats=1),
           dict(mass=1.2, width=0.2, spin=0, r_res=1.5, r_parent=5.0, shape_floats=0),
           dict(mass=1.4324, width=0.109, spin=2, r_res=2.0, r_parent=4.0, shape_floats=1)]
    knots = np.linspace(lo - 1e-3, hi + 1e-3, 9)
    o = orc.Oracle(kin, knots, res)
    s12, s13 = I.phase_space_points(2500, I.stream_key(3, 13, 1), kin)
    rng = np.random.default_rng(5)
    e12, e13, g12, g13 = s12[:900], s13[:900], s12[900:], s13[900:]
    w = rng.uniform(0.5, 1.5, g12.size) / g12.size
    p = np.concatenate([rng.uniform(0.5, 2, 9), rng.uniform(0, 3, 9), rng.uniform(0.3, 1.5, 6),
                        [0.8955, 0.047, 1.4324, 0.109]])
    S, Iv, gev, gnm = o.nll_grad_parts(p, e12, e13, g12, g13, w)
    nll, S0, I0 = o.nll(p, e12, e13, g12, g13, w, parts=True)
    assert S == pytest.approx(S0, rel=1e-14) and Iv == pytest.approx(I0, rel=1e-14)
    assert gev.size == gnm.size == p.size == 28
    _, g_lin = o.nll_grad(p, e12, e13, g12, g13, w)
    _, g_shape = o.nll_grad_shape(p, e12, e13, g12, g13, w)
    total = gev + (e12.size / Iv) * gnm
    ref = np.concatenate([g_lin, g_shape])
    assert np.max(np.abs(total - ref)) <= 1e-13 * np.max(np.abs(ref))
    for idx in (0, 4, 8, 9, 13, 17, 18, 19, 22, 23, 24, 25, 26, 27):
        def parts_at(v):
            q = p.copy(); q[idx] = v
            _, s_, i_ = o.nll(q, e12, e13, g12, g13, w, parts=True)
            return np.array([-s_, i_])
        fd = _richardson(parts_at, p[idx], 1e-4)
        assert gev[idx] == pytest.approx(fd[0], rel=5e-6, abs=1e-7 * np.max(np.abs(gev)))
        assert gnm[idx] == pytest.approx(fd[1], rel=5e-6, abs=1e-7 * np.max(np.abs(gnm)))
    _, _, gev0, gnm0 = o.nll_grad_parts(p, e12[:0], e13[:0], g12, g13, w)
    assert not gev0.any() and np.array_equal(gnm0, gnm)
