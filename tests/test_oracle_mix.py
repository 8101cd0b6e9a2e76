"""Pins of the oracle's signal + background mixture likelihood (O12, "signal purity 90 %").
The pure-signal NLL and its gradient are pinned elsewhere; here the mixture must reduce to them at f_s = 1, be
independent of f_s when the background density equals the signal density, have the closed form of a constant S-wave,
and its analytic derivatives must match Richardson central differences of its own value."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I


def _richardson(f, x, h):
    d = lambda s: (f(x + s) - f(x - s)) / (2 * s)
    return (4 * d(h / 2) - d(h)) / 3


@pytest.fixture(scope="module")
def case():
    c = I.Config(1, n_ev=1200, n_norm=2500)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    e12, e13 = I.phase_space_points(1200, c.key(7), c.kin)
    g12, g13, w = c.norm_points()
    bkg = (0.5 + I.uniforms(c.key(21), 0, 1200)) / I.dalitz_area(c.kin)        # a bumpy density of the right scale
    return c, o, e12, e13, bkg, g12, g13, w


def test_pure_signal_limit(case):
    c, o, e12, e13, bkg, g12, g13, w = case
    p = c.perturbed(0)
    v, g, dfs = o.nll_mix(p, e12, e13, bkg, 1.0, g12, g13, w, grad=True)
    ref, gref = o.nll_grad(p, e12, e13, g12, g13, w)
    assert v == pytest.approx(ref, rel=1e-13)
    assert np.max(np.abs(g - gref)) <= 1e-11 * np.max(np.abs(gref))


def test_background_equal_to_signal_makes_the_fraction_irrelevant(case):
    c, o, e12, e13, bkg, g12, g13, w = case
    p = c.perturbed(1)
    _, _, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
    same = o.abs2(p, e12, e13) / integ
    v1, _, d1 = o.nll_mix(p, e12, e13, same, 0.3, g12, g13, w, grad=True)
    v2, _, d2 = o.nll_mix(p, e12, e13, same, 0.9, g12, g13, w, grad=True)
    assert v1 == pytest.approx(v2, rel=1e-13) and v1 == pytest.approx(o.nll(p, e12, e13, g12, g13, w), rel=1e-13)
    assert abs(d1) <= 1e-9 * e12.size and abs(d2) <= 1e-9 * e12.size


def test_constant_s_wave_closed_form():
    c = I.Config(0, n_ev=800)
    o = orc.Oracle(c.kin, c.knots, [])
    e12, e13 = I.phase_space_points(800, c.key(7), c.kin)
    g12, g13, w = c.norm_points()
    bkg = (0.2 + 1.6 * I.uniforms(c.key(22), 0, 800)) / w.sum()
    p = np.concatenate([np.full(c.N, 0.83), np.full(c.N, -0.4)])
    fs = 0.9
    want = -float(np.sum(np.log(fs / w.sum() + (1.0 - fs) * bkg)))
    assert o.nll_mix(p, e12, e13, bkg, fs, g12, g13, w) == pytest.approx(want, rel=1e-13)


def test_derivatives_match_finite_differences(case):
    c, o, e12, e13, bkg, g12, g13, w = case
    p = c.perturbed(2)
    fs = 0.9
    v, g, dfs = o.nll_mix(p, e12, e13, bkg, fs, g12, g13, w, grad=True)
    assert v == o.nll_mix(p, e12, e13, bkg, fs, g12, g13, w)
    scale = np.max(np.abs(g))
    for a in (0, 5, c.N - 1, c.N + 3, 2 * c.N, 2 * c.N + 1, 2 * c.N + 2, 2 * c.N + 3):
        def f(x):
            q = p.copy(); q[a] = x
            return o.nll_mix(q, e12, e13, bkg, fs, g12, g13, w)
        assert g[a] == pytest.approx(_richardson(f, p[a], 1e-4), abs=2e-7 * scale)
    fd = _richardson(lambda x: o.nll_mix(p, e12, e13, bkg, x, g12, g13, w), fs, 1e-4)
    assert dfs == pytest.approx(fd, rel=1e-7)
    # scale invariance survives the mixture (the signal PDF is normalised): sum_k rho_k dNLL/drho_k = 0
    rho_idx = list(range(c.N)) + [2 * c.N + 2 * r for r in range(c.R)]
    assert abs(sum(p[k] * g[k] for k in rho_idx)) <= 1e-9 * scale * np.max(np.abs(p))
