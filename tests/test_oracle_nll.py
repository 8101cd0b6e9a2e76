"""Pins for the oracle's total amplitude, NLL, normalisation, fixed-shape identities, gradient and for the toy
generator (north_star invariants of BASELINE.json)."""
import math

import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I


@pytest.fixture(scope="module")
def cfg0():
    c = I.Config(0)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    f = lambda a, b: o.abs2(c.truth, a, b)
    env = I.envelope_of(f, c.kin, n_side=256)
    e12, e13 = c.events(f, env)
    g12, g13, w = c.norm_points()
    return c, o, (e12, e13, g12, g13, w)


@pytest.fixture(scope="module")
def cfg2_small():
    c = I.Config(2, n_ev=3000, n_norm=5000)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    f = lambda a, b: o.abs2(c.truth, a, b)
    e12, e13 = c.events(f, I.envelope_of(f, c.kin, n_side=128))
    g12, g13, w = c.norm_points()
    return c, o, (e12, e13, g12, g13, w)


def unpack(c, p):
    N, R = c.N, c.R
    y = p[:N] * np.exp(1j * p[N:2 * N])
    cr = np.array([p[2 * N + 2 * r] * np.exp(1j * p[2 * N + 2 * r + 1]) for r in range(R)])
    return y, cr


# ---- O6: assembly of Eq. 1 ------------------------------------------------------------------------------------------
def test_amplitude_is_spline_plus_symmetrised_resonances(cfg2_small):
    c, o, (e12, e13, *_rest) = cfg2_small
    y, cr = unpack(c, c.truth)
    sp = lambda s: CubicSpline(c.knots, y.real, bc_type="natural")(s) + 1j * CubicSpline(c.knots, y.imag, bc_type="natural")(s)
    A = o.amplitude(c.truth, e12[:200], e13[:200])
    for i in range(200):
        expect = sp(e12[i]) + sp(e13[i])
        for r in range(c.R):
            expect += cr[r] * (o.resonance_term(r, e12[i], e13[i]) + o.resonance_term(r, e13[i], e12[i]))
        assert A[i] == pytest.approx(expect, rel=1e-12)
    assert np.allclose(o.abs2(c.truth, e12[:200], e13[:200]), np.abs(A) ** 2, rtol=1e-15)


def test_bose_symmetry_is_bit_exact(cfg2_small):
    c, o, (e12, e13, g12, g13, _) = cfg2_small
    assert np.array_equal(o.abs2(c.truth, e12, e13), o.abs2(c.truth, e13, e12))
    assert np.array_equal(o.abs2(c.truth, g12, g13), o.abs2(c.truth, g13, g12))


def test_s_wave_only_model_equals_scipy_spline():
    c = I.Config(1)
    o = orc.Oracle(c.kin, c.knots, [])
    p = c.truth[:2 * c.N]
    y = p[:c.N] * np.exp(1j * p[c.N:])
    g12, g13 = I.phase_space_points(500, c.key(I.S_NORM))
    sp = lambda s: CubicSpline(c.knots, y.real, bc_type="natural")(s) + 1j * CubicSpline(c.knots, y.imag, bc_type="natural")(s)
    assert np.max(np.abs(o.amplitude(p, g12, g13) - (sp(g12) + sp(g13)))) < 1e-12


def test_floating_shape_parameters_replace_the_listed_ones():
    c3 = I.Config(3, n_ev=10, n_norm=10)
    assert c3.n_params == 2 * 50 + 2 * 3 + 2 and c3.resonances[0]["shape_floats"] == 1
    o3 = orc.Oracle(c3.kin, c3.knots, c3.resonances)
    fixed = [dict(r, shape_floats=0) for r in c3.resonances]
    fixed[0]["mass"], fixed[0]["width"] = 0.781, 0.153
    of = orc.Oracle(c3.kin, c3.knots, fixed)
    p = c3.truth.copy()
    p[-2:] = [0.781, 0.153]
    g12, g13 = I.phase_space_points(300, c3.key(I.S_NORM))
    assert np.array_equal(o3.abs2(p, g12, g13), of.abs2(p[:-2], g12, g13))
    assert not np.array_equal(o3.abs2(c3.truth, g12, g13), o3.abs2(p, g12, g13))


# ---- O7: NLL -------------------------------------------------------------------------------------------------------
def test_nll_is_minus_sum_log_plus_n_log_integral(cfg0):
    c, o, (e12, e13, g12, g13, w) = cfg0
    nll, slog, integ = o.nll(c.truth, e12, e13, g12, g13, w, parts=True)
    a2e, a2n = o.abs2(c.truth, e12, e13), o.abs2(c.truth, g12, g13)
    s_ref = math.fsum(np.log(a2e))
    i_ref = math.fsum(w * a2n)
    assert slog == pytest.approx(s_ref, rel=1e-14)
    assert integ == pytest.approx(i_ref, rel=1e-14)
    assert nll == pytest.approx(-s_ref + e12.size * math.log(i_ref), rel=1e-13)    # natural log, no factor 2
    # PDF integrates to one on the normalisation set
    assert math.fsum(w * a2n / integ) == pytest.approx(1.0, rel=1e-14)
    # w = NULL means w_j = 1/n_norm
    nll_u = o.nll(c.truth, e12, e13, g12, g13, None)
    assert nll_u == pytest.approx(nll + e12.size * math.log(1.0 / (w[0] * g12.size)), rel=1e-12)


def test_nll_closed_form_for_constant_s_wave():
    """R = 0 and all knots equal to y: |A|^2 = |2y|^2 everywhere, so NLL = n_ev ln(sum_j w_j)."""
    c = I.Config(0)
    o = orc.Oracle(c.kin, c.knots, [])
    p = np.concatenate([np.full(c.N, 1.37), np.full(c.N, 0.6)])
    e12, e13 = I.phase_space_points(2000, c.key(I.S_EVENTS))
    g12, g13, w = c.norm_points()
    assert np.allclose(o.abs2(p, e12, e13), (2 * 1.37) ** 2, rtol=1e-14)
    assert o.nll(p, e12, e13, g12, g13, w) == pytest.approx(2000 * math.log(w.sum()), rel=1e-13)
    assert w.sum() == pytest.approx(5954 * w[0], rel=1e-14)


def test_nll_invariant_under_global_phase_and_scale(cfg2_small):
    c, o, d = cfg2_small
    base = o.nll(c.truth, *d)
    N, R = c.N, c.R
    rot = c.truth.copy()
    rot[N:2 * N] += 0.83
    rot[2 * N + 1:2 * N + 2 * R:2] += 0.83
    assert o.nll(rot, *d) == pytest.approx(base, abs=1e-9 * abs(base) + 1e-8)
    sc = c.truth.copy()
    sc[:N] *= 1.9
    sc[2 * N:2 * N + 2 * R:2] *= 1.9
    assert o.nll(sc, *d) == pytest.approx(base, abs=1e-9 * abs(base) + 1e-8)
    # but not under a phase on the S-wave alone
    part = c.truth.copy()
    part[N:2 * N] += 0.83
    assert abs(o.nll(part, *d) - base) > 1.0


def test_truth_parameters_fit_better_than_perturbed(cfg0):
    c, o, d = cfg0
    base = o.nll(c.truth, *d)
    worse = 0
    for t in range(6):
        p = c.truth + 0.05 * I.normals(c.key(77), t * c.n_params, c.n_params)
        worse += o.nll(p, *d) > base
    assert worse >= 5                                       # events were generated from the truth model


# ---- normalisation ---------------------------------------------------------------------------------------------------
def test_grid_integral_converges_and_agrees_with_monte_carlo():
    c = I.Config(0)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    integ = {}
    for n in (50, 100, 200, 400, 1600):
        g12, g13, w = I.grid_points(n, c.kin)
        integ[n] = math.fsum(w * o.abs2(c.truth, g12, g13))
    ref = integ[1600]
    errs = [abs(integ[n] - ref) for n in (50, 100, 200, 400)]
    assert errs[0] > errs[2] and errs[1] > errs[3]          # finer grid -> better integral
    assert errs[3] / ref < 2e-3
    n = 400_000
    m12, m13 = I.phase_space_points(n, c.key(I.S_NORM))
    v = I.dalitz_area(c.kin) * o.abs2(c.truth, m12, m13)
    mc, se = v.mean(), v.std(ddof=1) / math.sqrt(n)
    assert abs(mc - ref) < 3.5 * se + 1e-3 * ref


# ---- O8: fixed-shape identities ---------------------------------------------------------------------------------------
def test_amplitude_is_linear_in_coefficients_and_gram_gives_integral(cfg2_small):
    c, o, (e12, e13, g12, g13, w) = cfg2_small
    y, cr = unpack(c, c.truth)
    coef = np.concatenate([y, cr])
    B = o.basis(c.truth, e12[:400], e13[:400])
    assert B.shape == (400, c.N + c.R)
    assert np.max(np.abs(B[:, :c.N].imag)) == 0.0           # spline columns are real
    A = o.amplitude(c.truth, e12[:400], e13[:400])
    assert np.max(np.abs(B @ coef - A) / np.abs(A)) < 1e-12
    # cardinal property: at a knot the spline column k is 1 for the channel that sits on it
    G = o.gram(c.truth, g12, g13, w)
    assert np.allclose(G, G.conj().T, rtol=1e-13, atol=1e-15)
    integ = o.nll(c.truth, e12, e13, g12, g13, w, parts=True)[2]
    assert (coef.conj() @ G @ coef).real == pytest.approx(integ, rel=1e-12)


# ---- O9: gradient -----------------------------------------------------------------------------------------------------
def test_gradient_matches_richardson_finite_differences(cfg2_small):
    c, o, d = cfg2_small
    p0 = c.perturbed(3)
    nll, grad = o.nll_grad(p0, *d)
    assert nll == pytest.approx(o.nll(p0, *d), rel=1e-14)
    assert grad.size == 2 * c.N + 2 * c.R
    rng = np.random.default_rng(0)
    idx = list(rng.choice(2 * c.N, 14, replace=False)) + list(range(2 * c.N, 2 * c.N + 2 * c.R))
    for k in idx:
        def d1(h):
            a, b = p0.copy(), p0.copy()
            a[k] += h; b[k] -= h
            return (o.nll(a, *d) - o.nll(b, *d)) / (2 * h)
        h = 2e-3
        fd = (4 * d1(h / 2) - d1(h)) / 3                     # Richardson: O(h^4)
        assert grad[k] == pytest.approx(fd, rel=2e-6, abs=2e-5 * np.max(np.abs(grad)))


def test_gradient_with_floating_shape_covers_linear_parameters_only():
    c = I.Config(3, n_ev=1500, n_norm=2500)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    f = lambda a, b: o.abs2(c.truth, a, b)
    e12, e13 = c.events(f, I.envelope_of(f, c.kin, n_side=128))
    g12, g13, w = c.norm_points()
    p0 = c.perturbed(1)
    _, grad = o.nll_grad(p0, e12, e13, g12, g13, w)
    assert grad.size == 106                                   # reading P16
    for k in (3, 57, 100, 101, 104):
        def d1(h):
            a, b = p0.copy(), p0.copy()
            a[k] += h; b[k] -= h
            return (o.nll(a, e12, e13, g12, g13, w) - o.nll(b, e12, e13, g12, g13, w)) / (2 * h)
        fd = (4 * d1(1e-3) - d1(2e-3)) / 3
        assert grad[k] == pytest.approx(fd, rel=2e-6, abs=2e-5 * np.max(np.abs(grad)))


def test_gradient_obeys_scale_and_phase_invariance(cfg2_small):
    c, o, d = cfg2_small
    p = c.perturbed(5)
    _, g = o.nll_grad(p, *d)
    N, R = c.N, c.R
    scale = np.dot(p[:N], g[:N]) + sum(p[2 * N + 2 * r] * g[2 * N + 2 * r] for r in range(R))
    phase = g[N:2 * N].sum() + sum(g[2 * N + 2 * r + 1] for r in range(R))
    big = np.abs(g).max() * N
    assert abs(scale) < 1e-10 * big and abs(phase) < 1e-10 * big


# ---- generator ---------------------------------------------------------------------------------------------------------
def test_events_are_inside_and_follow_the_density(cfg0):
    c, o, (e12, e13, g12, g13, w) = cfg0
    assert e12.size == c.n_ev == 10_000 and g12.size == 5954
    assert o.inside(e12, e13).all()                           # north_star invariant
    # chunking does not change the sample
    f = lambda a, b: o.abs2(c.truth, a, b)
    env = I.envelope_of(f, c.kin, n_side=256)
    a12, a13 = I.accept_reject(500, c.key(I.S_EVENTS), f, env, c.kin, chunk=1000)
    assert np.array_equal(a12, e12[:500]) and np.array_equal(a13, e13[:500])
    # chi2 of a coarse histogram against the integral of |A|^2 per bin (fine-grid estimate)
    lo, hi = I.s_limits(c.kin)
    edges = np.linspace(lo, hi, 9)
    obs, _, _ = np.histogram2d(e12, e13, bins=[edges, edges])
    f12, f13, fw = I.grid_points(800, c.kin)
    dens, _, _ = np.histogram2d(f12, f13, bins=[edges, edges], weights=fw * f(f12, f13))
    exp = dens / dens.sum() * e12.size
    m = exp > 20
    chi2 = ((obs[m] - exp[m]) ** 2 / exp[m]).sum()
    ndf = m.sum() - 1
    assert chi2 < ndf + 5 * math.sqrt(2 * ndf)
    assert obs[~m].sum() < 0.05 * e12.size


def test_config_recipes():
    for idx, (N, R, P) in enumerate([(10, 1, 22), (30, 2, 64), (40, 3, 86), (50, 3, 108), (50, 6, 112)]):
        c = I.Config(idx, n_ev=10, n_norm=10)
        assert (c.N, c.R, c.n_params) == (N, R, P)
        assert np.all(np.diff(c.knots) > 0)
        assert c.knots[0] == I.KNOT_LO and c.knots[-1] == pytest.approx(I.KNOT_HI, rel=1e-15)
        assert np.all((c.truth[:N] >= 0.5) & (c.truth[:N] <= 2.0))
    k2 = I.knots_config2()
    assert ((k2 >= 0.8) & (k2 <= 1.2)).sum() == 20           # half of the 40 knots (reading P17)
    c1 = I.Config(1, n_ev=10, n_norm=10)
    d = c1.perturbed(4) - c1.truth
    assert 2e-4 < d.std() < 3e-3 and np.array_equal(c1.perturbed(4), c1.perturbed(4))
    assert not np.array_equal(c1.perturbed(4), c1.perturbed(5))


def test_paper_toy_config_kkk():
    """Config 5 = the paper's own toy: D+ -> K+K+K-, 40 knots over the whole m^2(K+K-) range + phi(1020),
    100 K events, grid spacing 0.001 GeV^2.  Recipe checks + the oracle's invariants on the other kinematics."""
    c = I.Config(5, n_ev=4000)
    lo, hi = I.s_limits(c.kin)
    assert c.N == 40 and c.R == 1 and c.knots[0] == pytest.approx(lo) and c.knots[-1] == pytest.approx(hi)
    assert (hi - lo) / 918 == pytest.approx(0.001, rel=2e-3)                     # grid spacing of PAPER.md:47
    g12, g13, w = c.norm_points()
    assert w[0] == pytest.approx(((hi - lo) / 918) ** 2)
    assert g12.size * w[0] == pytest.approx(I.dalitz_area(c.kin), rel=2e-3)       # grid covers the Dalitz plot
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    f = lambda a, b: o.abs2(c.truth, a, b)
    e12, e13 = c.events(f, I.envelope_of(f, c.kin, n_side=512))
    assert o.inside(e12, e13).all()
    # phi(1020) band: a visible excess of events within 3 widths of the pole in either K+K- mass
    m0, g0 = c.resonances[0]["mass"], c.resonances[0]["width"]
    band = (np.abs(np.sqrt(e12) - m0) < 3 * g0) | (np.abs(np.sqrt(e13) - m0) < 3 * g0)
    flat = I.phase_space_points(20000, c.key(9), c.kin)
    band_flat = (np.abs(np.sqrt(flat[0]) - m0) < 3 * g0) | (np.abs(np.sqrt(flat[1]) - m0) < 3 * g0)
    assert band.mean() > 3 * band_flat.mean()
    assert np.array_equal(o.abs2(c.truth, e12, e13), o.abs2(c.truth, e13, e12))
    p = c.perturbed(0)
    nll, grad = o.nll_grad(p, e12, e13, g12[::40], g13[::40], w[::40] * 40)
    assert np.isfinite(nll) and abs(np.sum(grad[c.N:2 * c.N]) + grad[-1]) <= 1e-8 * np.max(np.abs(grad))
