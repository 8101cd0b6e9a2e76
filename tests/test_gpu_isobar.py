"""GPU parity of the Isobar comparison model ("the S-wave is represented by a sum of a constant non-resonant
term and Breit-Wigner functions") through the C ABI against the oracle (O6b, pinned in
tests/test_oracle_isobar.py and tests/test_oracle_mpmath.py):

  * D+ -> K+ K+ K- with NO spline (n_knots = 0): a scalar Breit-Wigner + phi(1020) + the constant term;
  * the MIPWA spline WITH a constant term beside it (the constant rides on the spline tables inside the library);
  * a floating scalar shape (the run-time resonance loop and k_grad_shape).

Bars: per-event |A|^2 1e-12 (reading P15), NLL 1e-10 (P14) on every path, gradient 1e-11 of the largest component,
Hessian 1e-8 of its largest entry, basis rows 1e-12.
"""
import types

import numpy as np
import pytest

from tests.helpers import abs2_ok, incoherent_scale, nll_tol

pytestmark = pytest.mark.gpu

NONRES = dict(mass=0.0, width=0.0, spin=-1, r_res=0.0, r_parent=0.0)
F0 = dict(mass=1.35, width=0.25, spin=0, r_res=1.5, r_parent=5.0)
PHI = dict(mass=1.019461, width=0.004249, spin=1, r_res=1.5, r_parent=5.0)


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


def _model(knots, resonances, seed):
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    kin = I.KIN_KKK
    o = orc.Oracle(kin, knots, resonances)
    N, R = len(knots), len(resonances)
    rng = np.random.default_rng(seed)
    p = np.concatenate([rng.uniform(0.5, 2, N), rng.uniform(0, 3, N)])
    for r in resonances:
        p = np.concatenate([p, [rng.uniform(0.3, 1.5) * (0.05 if r["spin"] == 1 else 1.0), rng.uniform(-3, 3)]])
    for r in resonances:
        if r.get("shape_floats"):
            p = np.concatenate([p, [r["mass"] * 1.003, r["width"] * 0.98]])
    e12, e13 = I.phase_space_points(30_011, I.stream_key(seed, 60, 0), kin)
    g12, g13 = I.phase_space_points(20_003, I.stream_key(seed, 60, 1), kin)
    w = np.full(g12.size, I.dalitz_area(kin) / g12.size)
    c = types.SimpleNamespace(kin=kin, knots=np.asarray(knots, dtype=float), resonances=resonances, N=N, R=R)
    return c, o, p, (e12, e13, g12, g13, w)


def _check_paths(c, o, p, data, paths):
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    assert m.n_params == p.size
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    ref = o.abs2(p, data[0], data[1])
    ok, worst, plain = abs2_ok(m.eval_abs2(p, 0), ref, incoherent_scale(o, c, p, data[0], data[1]))
    assert ok, (worst, plain)
    nll_ref, sl, integ = o.nll(p, *data, parts=True)
    _, g_ref = o.nll_grad(p, *data)
    for path in paths:
        m.set_path(path)
        assert abs(m.nll(p) - nll_ref) <= nll_tol(nll_ref, sl, integ, data[0].size), path
        nll, g = m.nll_grad(p)
        assert abs(nll - nll_ref) <= nll_tol(nll_ref, sl, integ, data[0].size), path
        assert np.max(np.abs(g - g_ref)) <= 1e-11 * np.max(np.abs(g_ref)), (path, np.max(np.abs(g - g_ref)))
    m.prepare()
    m.set_path(paths[0])
    assert abs(m.nll(p) - nll_ref) <= nll_tol(nll_ref, sl, integ, data[0].size)
    return m


def test_isobar_model_without_spline():
    """n_knots = 0: scalar Breit-Wigner + phi(1020) + constant; value, gradient, Hessian and basis on every path"""
    B = _lib()
    c, o, p, data = _model([], [F0, PHI, NONRES], 21)
    m = _check_paths(c, o, p, data, [B.PATH_RECOMPUTE, B.PATH_CACHED, B.PATH_CACHED_COMPACT, B.PATH_AUTO])
    got = m.eval_basis(p, 0, 0, 300)
    refb = o.basis(p, data[0][:300], data[1][:300])
    assert got.shape == refb.shape == (300, 3)
    assert (np.abs(got - refb) / np.maximum(1.0, np.abs(refb))).max() < 1e-12
    assert np.array_equal(got[:, 2], np.ones(300, dtype=complex))
    H_ref = o.nll_hessian(p, *data)
    _, g, H = m.nll_hessian(p)
    assert H.shape == (6, 6)
    assert np.max(np.abs(H - H_ref)) <= 1e-8 * np.max(np.abs(H_ref))
    assert np.max(np.abs(H - H.T)) <= 1e-9 * np.max(np.abs(H))
    m.close()


def test_constant_term_alone_has_the_closed_form_nll():
    """R = 1 (the constant), no spline: NLL = n ln sum_j w_j whatever the coefficient is"""
    B = _lib()
    c, o, p, data = _model([], [NONRES], 22)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    for path in (B.PATH_RECOMPUTE, B.PATH_CACHED, B.PATH_CACHED_COMPACT):
        m.set_path(path)
        assert abs(m.nll(np.array([0.7, 1.1])) - data[0].size * np.log(data[4].sum())) < 1e-7
    nll, g = m.nll_grad(np.array([0.7, 1.1]))
    assert np.max(np.abs(g)) < 1e-7                         # flat direction: scale and phase of the only coefficient
    m.close()


def test_spline_with_a_constant_term_beside_it():
    """12 knots + phi(1020) + constant (in the middle of the list): the constant rides on the spline tables"""
    B = _lib()
    from paper_1703_03284_b200 import inputs as I
    lo, hi = I.s_limits(I.KIN_KKK)
    knots = np.linspace(lo * 1.001, hi * 0.999, 12)
    c, o, p, data = _model(knots, [F0, NONRES, PHI], 23)
    m = _check_paths(c, o, p, data, [B.PATH_RECOMPUTE, B.PATH_CACHED, B.PATH_CACHED_COMPACT])
    got = m.eval_basis(p, 1, 5, 200)
    refb = o.basis(p, data[2][5:205], data[3][5:205])
    assert (np.abs(got - refb) / np.maximum(1.0, np.abs(refb))).max() < 1e-12
    H_ref = o.nll_hessian(p, *data)
    _, g, H = m.nll_hessian(p)
    assert np.max(np.abs(H - H_ref)) <= 1e-8 * np.max(np.abs(H_ref))
    # mixture likelihood with the constant term in the model
    bkg = np.full(data[0].size, 1.0 / data[4].sum())
    m.set_event_background(bkg)
    ref, gref, dref = o.nll_mix(p, data[0], data[1], bkg, 0.85, data[2], data[3], data[4], grad=True)
    nll, g, dfs = m.nll_mix_grad(p, 0.85)
    assert abs(nll - ref) <= 1e-10 * max(abs(ref), data[0].size)
    assert np.max(np.abs(g - gref)) <= 1e-10 * np.max(np.abs(gref)) and abs(dfs - dref) <= 1e-9 * max(1.0, abs(dref))
    m.close()


def test_floating_scalar_shape_with_constant_term():
    """a floating spin-0 Breit-Wigner: run-time resonance loop, d/d(mass, width) through k_grad_shape, sharded pieces"""
    B = _lib()
    res = [dict(F0, shape_floats=1), PHI, NONRES]
    c, o, p, data = _model([], res, 24)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    nll_ref, sl, integ = o.nll(p, *data, parts=True)
    assert abs(m.nll(p) - nll_ref) <= nll_tol(nll_ref, sl, integ, data[0].size)
    _, g_lin = o.nll_grad(p, *data)
    _, g_shape = o.nll_grad_shape(p, *data)
    g_ref = np.concatenate([g_lin, g_shape])
    nll, g = m.nll_grad_full(p)
    assert g.shape == (8,)
    assert np.max(np.abs(g - g_ref)) <= 1e-10 * np.max(np.abs(g_ref)), np.abs(g - g_ref)
    S, Iv, gev, gnm = m.nll_grad_parts(p)
    S_o, I_o, gev_o, gnm_o = o.nll_grad_parts(p, *data)
    assert abs(S - S_o) <= 1e-10 * abs(S_o) and abs(Iv - I_o) <= 1e-12 * I_o
    assert np.max(np.abs(gev - gev_o)) <= 1e-10 * np.max(np.abs(gev_o))
    assert np.max(np.abs(gnm - gnm_o)) <= 1e-10 * np.max(np.abs(gnm_o))
    m.close()


def test_bad_isobar_models_are_refused():
    B = _lib()
    from paper_1703_03284_b200 import inputs as I
    with pytest.raises(B.MipwaError):
        B.Mipwa(I.KIN_KKK, [], [NONRES, NONRES])            # two constant terms
    with pytest.raises(B.MipwaError):
        B.Mipwa(I.KIN_KKK, [], [dict(NONRES, shape_floats=1)])
    with pytest.raises(B.MipwaError):
        B.Mipwa(I.KIN_KKK, [], [])                          # nothing at all
    with pytest.raises(B.MipwaError):
        B.Mipwa(I.KIN_KKK, [1.2], [PHI])                    # one knot is no spline
