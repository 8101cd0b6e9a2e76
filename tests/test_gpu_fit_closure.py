"""Closure test: the library used the way the paper uses its PDF (toy events generated from the PDF, then
an unbinned maximum-likelihood fit of the knot values).  scipy's L-BFGS-B is the CALLER here (the minimiser is outside
the hot path); mipwa_nll_grad supplies value and gradient.  Global phase and scale are unconstrained by the likelihood,
so the first knot is held fixed.  Checks: the fit converges to a stationary point below NLL(truth), and the fitted PDF
agrees with the generating PDF over the Dalitz plot within the statistical precision of the sample."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_fit_recovers_the_generating_pdf():
    from scipy.optimize import minimize
    from paper_1703_03284_b200 import binding as B
    from paper_1703_03284_b200 import inputs as I

    c = I.Config(0, n_ev=100_000)
    m = B.Mipwa(c.kin, c.knots, c.resonances)

    def abs2_fn(a, b):                                    # events from the library's own per-point hook
        m.set_events(np.ascontiguousarray(a), np.ascontiguousarray(b))
        return m.eval_abs2(c.truth, 0)
    e12, e13 = c.events(abs2_fn, I.envelope_of(abs2_fn, c.kin, n_side=512))
    g12, g13, w = I.grid_points(400, c.kin)               # finer grid than config 0: normalisation bias << stat. error
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w); m.prepare()

    N = c.N
    free = np.ones(c.n_params, dtype=bool)
    free[0] = free[N] = False                             # fix a_0 and phi_0: removes the scale / phase degeneracy
    x0 = c.truth + 0.15 * I.normals(c.key(11), 0, c.n_params)
    x0[~free] = c.truth[~free]

    def fun(x):
        p = c.truth.copy(); p[free] = x
        v, g = m.nll_grad(p)
        return v, g[free]

    nll_truth = m.nll(c.truth)
    nll_start = fun(x0[free])[0]
    res = minimize(fun, x0[free], jac=True, method="L-BFGS-B", options=dict(maxiter=2000, maxfun=4000, ftol=1e-14, gtol=1e-6))
    fit = c.truth.copy(); fit[free] = res.x
    nll_fit = m.nll(fit)
    assert nll_start > nll_truth + 100.0                  # the start really was displaced
    assert nll_fit <= nll_truth + 1e-6                    # a minimum lies at or below the truth's NLL ...
    assert nll_truth - nll_fit < 3 * free.sum()           # ... by about half a unit per free parameter, not more
    _, g = m.nll_grad(fit)
    assert np.max(np.abs(g[free])) < 1e-2 * np.max(np.abs(fun(x0[free])[1]))
    # fitted vs generating PDF on the normalisation grid
    m.set_events(g12, g13)
    pt, pf = m.eval_abs2(c.truth, 0), m.eval_abs2(fit, 0)
    pt, pf = pt / np.sum(w * pt), pf / np.sum(w * pf)
    l1 = float(np.sum(w * np.abs(pf - pt)))              # integral |pdf_fit - pdf_truth|
    assert l1 < 0.03, l1                                  # ~ sqrt(n_free / n_ev) = 0.015 scale
    m.close()


def test_fit_with_floating_mass_and_width_recovers_the_pole():
    """Closure of mipwa_generate + mipwa_nll_grad_full: 200 K events generated on the device from a 12-knot S-wave +
    rho(770) (mass and width floating) + f2(1270); all 28 free parameters incl. the rho mass and width are fitted from
    a displaced start.  The pole parameters come back within 4 standard errors (errors from central differences of the
    analytic gradient), and the NLL drops below its value at the truth by about half a unit per free parameter."""
    from scipy.optimize import minimize
    from paper_1703_03284_b200 import binding as B
    from paper_1703_03284_b200 import inputs as I

    res = [dict(mass=0.775, width=0.149, spin=1, r_res=1.5, r_parent=5.0, shape_floats=1),
           dict(mass=1.2755, width=0.1867, spin=2, r_res=1.5, r_parent=5.0, shape_floats=0)]
    N = 12
    m = B.Mipwa(I.KIN, I.knots_uniform(N), res)
    key = I.stream_key(1, 40, 0)
    truth = np.concatenate([0.5 + 1.5 * I.uniforms(key, 0, N), np.pi * np.arange(N) / (N - 1) + 0.2 * I.normals(key, 100, N),
                            [1.0, 0.4, 0.6, 2.0], [0.775, 0.149]])
    e12, e13, _ = m.generate(truth, I.stream_key(1, 40, 1), 200_000, device=True)
    g12, g13, w = I.grid_points(500, I.KIN)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w); m.prepare()
    free = np.ones(truth.size, dtype=bool)
    free[0] = free[N] = False
    x0 = truth + 0.05 * I.normals(key, 200, truth.size)
    x0[~free] = truth[~free]
    x0[-2:] = [0.79, 0.13]

    def fun(x):
        p = truth.copy(); p[free] = x
        v, g = m.nll_grad_full(p)
        return v, g[free]
    bounds = [(None, None)] * (int(free.sum()) - 2) + [(0.5, 1.2), (0.02, 0.5)]
    r = minimize(fun, x0[free], jac=True, method="L-BFGS-B", bounds=bounds,
                 options=dict(maxiter=5000, maxfun=10000, ftol=1e-15, gtol=1e-6))
    nfree = int(free.sum())
    drop = r.fun - m.nll(truth)
    assert -3.0 * nfree < drop <= 1e-6, drop
    H = np.zeros((nfree, nfree))
    for a in range(nfree):
        xp, xm = r.x.copy(), r.x.copy()
        xp[a] += 1e-5; xm[a] -= 1e-5
        H[a] = (fun(xp)[1] - fun(xm)[1]) / 2e-5
    cov = np.linalg.inv(0.5 * (H + H.T))
    sm, sg = np.sqrt(cov[-2, -2]), np.sqrt(cov[-1, -1])
    assert 1e-4 < sm < 2e-3 and 2e-4 < sg < 4e-3, (sm, sg)            # ~0.4 MeV and ~0.8 MeV at 200 K events
    assert abs(r.x[-2] - 0.775) < 4 * sm and abs(r.x[-1] - 0.149) < 4 * sg, (r.x[-2:], sm, sg)
    m.close()


def test_mixture_fit_recovers_the_signal_fraction():
    """Closure of the mixture likelihood (purity about 90 %): 90 K signal events generated on the device
    from config 0's PDF plus 10 K background events uniform in phase space (density 1 / area); the knot values, the
    rho(770) coefficient and the signal fraction are fitted with mipwa_nll_mix_grad.  The fraction comes back within 4
    standard errors (error from the second difference of the likelihood in f_s at the minimum)."""
    from scipy.optimize import minimize
    from paper_1703_03284_b200 import binding as B
    from paper_1703_03284_b200 import inputs as I

    c = I.Config(0)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    s12, s13, _ = m.generate(c.truth, c.key(50), 90_000)
    b12, b13 = I.phase_space_points(10_000, c.key(51), c.kin)
    e12, e13 = np.concatenate([s12, b12]), np.concatenate([s13, b13])
    perm = np.argsort(I.uniforms(c.key(52), 0, e12.size))           # shuffle signal and background together
    e12, e13 = e12[perm].copy(), e13[perm].copy()
    bkg = np.full(e12.size, 1.0 / I.dalitz_area(c.kin))
    g12, g13, w = I.grid_points(400, c.kin)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w); m.set_event_background(bkg); m.prepare()
    N = c.N
    free = np.ones(c.n_params, dtype=bool)
    free[0] = free[N] = False
    x0 = np.concatenate([(c.truth + 0.1 * I.normals(c.key(53), 0, c.n_params))[free], [0.8]])

    def fun(x):
        p = c.truth.copy(); p[free] = x[:-1]
        v, g, dfs = m.nll_mix_grad(p, x[-1])
        return v, np.concatenate([g[free], [dfs]])
    bounds = [(None, None)] * int(free.sum()) + [(0.05, 1.0)]
    r = minimize(fun, x0, jac=True, method="L-BFGS-B", bounds=bounds, options=dict(maxiter=3000, maxfun=6000, ftol=1e-15, gtol=1e-6))
    fs = r.x[-1]
    h = 1e-3
    xp, xm = r.x.copy(), r.x.copy()
    xp[-1] += h; xm[-1] -= h
    curv = (fun(xp)[0] - 2 * r.fun + fun(xm)[0]) / h ** 2           # d2NLL/df_s^2 at fixed other parameters
    sigma = 1.0 / np.sqrt(curv)
    assert 5e-4 < sigma < 1e-2, sigma
    assert abs(fs - 0.9) < 4 * sigma + 2e-3, (fs, sigma)             # + the profile-vs-fixed difference of the error
    p_truth = np.concatenate([c.truth[free], [0.9]])
    assert r.fun <= fun(p_truth)[0] + 1e-6
    m.close()
