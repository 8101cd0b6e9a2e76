"""GPU parity: recompute path (k_nll_recompute, k_abs2) through the C ABI against the CPU oracle.

Tolerances (north_star; readings P14, P15): per-event |A|^2 relative 1e-12, NLL relative 1e-10.
"""
import math

import numpy as np
import pytest

from tests.helpers import abs2_ok, incoherent_scale, make_case, nll_tol

pytestmark = pytest.mark.gpu


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


def _ctx(c, data, device_arrays=False):
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    e12, e13, g12, g13, w = data
    if device_arrays:
        import torch
        t = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (e12, e13, g12, g13, w)]
        m.set_events(t[0], t[1])
        m.set_norm_points(t[2], t[3], t[4])
    else:
        m.set_events(e12, e13)
        m.set_norm_points(g12, g13, w)
    m.set_path(B.PATH_RECOMPUTE)
    return m


CASES = {
    0: dict(),                                    # full config 0: 10k events, 5954-cell grid
    1: dict(n_ev=40_000, n_norm=50_000),          # several tiles + ragged tail
    2: dict(n_ev=30_011, n_norm=20_003),          # non-uniform knots, three resonances
    3: dict(n_ev=25_000, n_norm=25_000),          # floating rho(770) shape
    4: dict(n_ev=20_000, n_norm=20_000),          # six resonances incl. a narrow one
    5: dict(n_ev=30_000),                         # the paper's own toy: D+ -> K+K+K-, 40 knots + phi(1020), 0.001 GeV^2 grid
}


@pytest.fixture(scope="module", params=sorted(CASES))
def case(request):
    c, o, data = make_case(request.param, **CASES[request.param])
    return c, o, data


def test_per_event_abs2_matches_oracle(case):
    c, o, data = case
    m = _ctx(c, data)
    for t in (0, 1):
        p = c.truth if t == 0 else c.perturbed(t)
        for which, (a, b) in enumerate([(data[0], data[1]), (data[2], data[3])]):
            got = m.eval_abs2(p, which)
            ref = o.abs2(p, a, b)
            ok, worst, plain = abs2_ok(got, ref, incoherent_scale(o, c, p, a, b))
            assert ok, f"config {c.idx} slot {which}: worst ratio {worst}, plain rel {plain}"
            assert plain < 1e-10
    m.close()


def test_nll_matches_oracle(case):
    c, o, data = case
    m = _ctx(c, data)
    for t in range(3):
        p = c.perturbed(t)
        ref, sl, integ = o.nll(p, *data, parts=True)
        got, gsl, ginteg = m.nll_parts(p)
        tol = nll_tol(ref, sl, integ, data[0].size)
        assert abs(got - ref) <= tol, (got, ref, tol)
        assert gsl == pytest.approx(sl, rel=1e-12)
        assert ginteg == pytest.approx(integ, rel=1e-12)
        assert m.nll(p) == got                      # bit-reproducible call to call
    m.close()


def test_borrowed_device_arrays_and_uniform_weights(case):
    c, o, data = case
    if c.idx not in (0, 2):
        pytest.skip("covered on two configs")
    m = _ctx(c, data, device_arrays=True)
    p = c.perturbed(7)
    ref, sl, integ = o.nll(p, *data, parts=True)
    assert abs(m.nll(p) - ref) <= nll_tol(ref, sl, integ, data[0].size)
    # w = NULL means w_j = 1/n
    m.set_norm_points(data[2], data[3], None)
    ref_u, sl_u, integ_u = o.nll(p, data[0], data[1], data[2], data[3], None, parts=True)
    assert abs(m.nll(p) - ref_u) <= nll_tol(ref_u, sl_u, integ_u, data[0].size)
    m.close()


def test_edge_cases():
    B = _lib()
    c, o, (e12, e13, g12, g13, w) = make_case(0, n_ev=300, n_norm=40)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    with pytest.raises(B.MipwaError) as ei:
        m.nll(c.truth)
    assert ei.value.code == B.ERR_STATE
    m.set_norm_points(g12, g13, w)
    # empty event sample: NLL = 0 * ln I = 0
    m.set_events(np.empty(0), np.empty(0))
    assert m.nll(c.truth) == 0.0
    # single event, ragged sizes
    for n in (1, 31, 33, 257, 300):
        m.set_events(e12[:n], e13[:n])
        ref, sl, integ = o.nll(c.truth, e12[:n], e13[:n], g12, g13, w, parts=True)
        assert abs(m.nll(c.truth) - ref) <= nll_tol(ref, sl, integ, n)
    # a point outside the boundary is refused and leaves the slot empty
    bad12, bad13 = e12[:10].copy(), e13[:10].copy()
    bad13[4] = 3.4
    with pytest.raises(B.MipwaError) as ei:
        m.set_events(bad12, bad13)
    assert ei.value.code == B.ERR_DOMAIN
    with pytest.raises(B.MipwaError):
        m.nll(c.truth)
    with pytest.raises(B.MipwaError) as ei:
        m.set_events(np.array([np.nan]), np.array([1.0]))
    assert ei.value.code == B.ERR_DOMAIN
    # wrong parameter count, non-finite parameter
    m.set_events(e12, e13)
    with pytest.raises(B.MipwaError) as ei:
        m.nll(c.truth[:-1])
    assert ei.value.code == B.ERR_ARG
    p = c.truth.copy(); p[3] = math.inf
    with pytest.raises(B.MipwaError):
        m.nll(p)
    # points exactly on knots and beyond the last knot (reading P3) agree with the oracle
    lo, hi = 0.0779191396, 2.9932114081
    s12 = np.concatenate([c.knots[1:-1], [2.9930, 2.99315, 0.07792]])
    s13 = np.full_like(s12, 0.3)
    s13[-3:] = [0.28, 0.2805, 1.74]
    keep = o.inside(s12, s13)
    assert keep.sum() >= 6 and keep[-3:].any()
    m.set_events(s12[keep], s13[keep])
    got, ref = m.eval_abs2(c.truth, 0), o.abs2(c.truth, s12[keep], s13[keep])
    assert np.max(np.abs(got - ref) / ref) < 1e-12
    m.close()
    # model validation
    with pytest.raises(B.MipwaError):
        B.Mipwa(c.kin, c.knots[::-1], c.resonances)
    with pytest.raises(B.MipwaError):
        B.Mipwa(c.kin, c.knots, [dict(c.resonances[0], spin=3)])


def test_degenerate_models():
    """R = 0 (pure S-wave, closed form NLL = n ln sum w for a constant spline), N = 2 (linear), spin-0 resonance."""
    B = _lib()
    c, o, (e12, e13, g12, g13, w) = make_case(0, n_ev=2000)
    m = B.Mipwa(c.kin, c.knots, [])
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
    p = np.concatenate([np.full(c.N, 1.37), np.full(c.N, 0.6)])
    assert m.nll(p) == pytest.approx(2000 * math.log(w.sum()), rel=1e-12)
    m.close()
    from oracle import oracle as orc
    res = [dict(mass=0.98, width=0.07, spin=0, r_res=1.5, r_parent=5.0),
           dict(mass=1.2755, width=0.1867, spin=2, r_res=3.0, r_parent=1.0)]
    knots = np.array([0.05, 3.1])
    o2 = orc.Oracle(c.kin, knots, res)
    m2 = B.Mipwa(c.kin, knots, res)
    m2.set_events(e12, e13); m2.set_norm_points(g12, g13, w)
    p2 = np.array([1.1, 0.7, 0.2, 1.9, 0.8, 0.4, 1.3, -2.0])
    got, ref = m2.eval_abs2(p2, 0), o2.abs2(p2, e12, e13)
    assert np.max(np.abs(got - ref) / ref) < 1e-12
    ref_n, sl, integ = o2.nll(p2, e12, e13, g12, g13, w, parts=True)
    assert abs(m2.nll(p2) - ref_n) <= nll_tol(ref_n, sl, integ, e12.size)
    m2.close()


def test_unequal_mass_kinematics():
    """m1 != m2 = m3 (K- pi+ pi+ like): exercises kappa and the general lambda terms."""
    B = _lib()
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    kin = {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=1.5, r_parent=5.0),
           dict(mass=1.4324, width=0.109, spin=2, r_res=1.5, r_parent=5.0)]
    lo, hi = I.s_limits(kin)
    knots = np.linspace(lo - 1e-3, hi + 1e-3, 17)
    g12, g13 = I.phase_space_points(6000, I.stream_key(3, 9, 1), kin)
    o = orc.Oracle(kin, knots, res)
    rng = np.random.default_rng(1)
    p = np.concatenate([rng.uniform(0.5, 2, 17), rng.uniform(0, 3, 17), [0.7, 0.3, 1.4, 2.2]])
    m = B.Mipwa(kin, knots, res)
    m.set_events(g12[:3000], g13[:3000]); m.set_norm_points(g12[3000:], g13[3000:])
    got, ref = m.eval_abs2(p, 0), o.abs2(p, g12[:3000], g13[:3000])
    assert np.max(np.abs(got - ref) / ref) < 1e-11
    ref_n, sl, integ = o.nll(p, g12[:3000], g13[:3000], g12[3000:], g13[3000:], None, parts=True)
    assert abs(m.nll(p) - ref_n) <= nll_tol(ref_n, sl, integ, 3000)
    m.close()


def test_prepare_keeps_results_and_hook_order(case):
    """mipwa_prepare: cell-sorted internal copies change only the summation order; hooks keep the caller's order;
    a new mipwa_set_* drops the sorted copy of that slot."""
    c, o, data = case
    B = _lib()
    m = _ctx(c, data, device_arrays=(c.idx % 2 == 0))
    p = c.perturbed(5)
    ref, sl, integ = o.nll(p, *data, parts=True)
    tol = nll_tol(ref, sl, integ, data[0].size)
    before = m.nll(p)
    m.prepare()
    after = m.nll(p)
    assert abs(after - ref) <= tol and abs(before - ref) <= tol
    assert m.nll(p) == after
    got = m.eval_abs2(p, 0)                                  # still in the caller's order
    refa = o.abs2(p, data[0], data[1])
    assert np.max(np.abs(got - refa) / refa) < 1e-10
    if not any(r.get("shape_floats") for r in c.resonances):
        for path in (B.PATH_CACHED, B.PATH_CACHED_COMPACT):
            m.set_path(path)
            assert abs(m.nll(p) - ref) <= tol
        m.set_path(B.PATH_RECOMPUTE)
    n2 = data[0].size // 2
    m.set_events(data[0][:n2], data[1][:n2])                # events change, normalisation copy stays sorted
    ref2, sl2, integ2 = o.nll(p, data[0][:n2], data[1][:n2], data[2], data[3], data[4], parts=True)
    assert abs(m.nll(p) - ref2) <= nll_tol(ref2, sl2, integ2, n2)
    m.close()
    m2 = B.Mipwa(c.kin, c.knots, c.resonances)
    with pytest.raises(B.MipwaError) as ei:
        m2.prepare()
    assert ei.value.code == B.ERR_STATE
    m2.close()


def test_hybrid_path_matches_oracle():
    """MIPWA_PATH_HYBRID (k_nll_hybrid): floating resonances recomputed, fixed ones cached for events and
    normalisation points.  configs[3] (rho(770) floats) and models with two floating resonances / spin 2 floating."""
    B = _lib()
    from oracle import oracle as orc
    c, o, data = make_case(3, n_ev=30_011, n_norm=20_003)
    models = [c.resonances,
              [dict(c.resonances[0], shape_floats=1), dict(c.resonances[1], shape_floats=1), dict(c.resonances[2])],
              [dict(c.resonances[0], shape_floats=0), dict(c.resonances[1]), dict(c.resonances[2], shape_floats=1)]]
    rng = np.random.default_rng(2)
    for res in models:
        oo = orc.Oracle(c.kin, c.knots, res)
        F = sum(r.get("shape_floats", 0) for r in res)
        shapes = []
        for r in res:
            if r.get("shape_floats"):
                shapes += [r["mass"] * (1 + 0.01 * rng.normal()), r["width"] * (1 + 0.05 * rng.normal())]
        p = np.concatenate([c.perturbed(1)[:2 * c.N + 2 * c.R], shapes])
        assert p.size == 2 * c.N + 2 * c.R + 2 * F
        ref, sl, integ = oo.nll(p, *data, parts=True)
        tol = nll_tol(ref, sl, integ, data[0].size)
        for prepared in (False, True):
            m = B.Mipwa(c.kin, c.knots, res)
            m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
            if prepared:
                m.prepare()
            m.set_path(B.PATH_HYBRID)
            got, gsl, ginteg = m.nll_parts(p)
            assert abs(got - ref) <= tol, (got, ref)
            assert gsl == pytest.approx(sl, rel=1e-12) and ginteg == pytest.approx(integ, rel=1e-12)
            assert m.nll(p) == got
            p2 = p.copy(); p2[-2:] *= 1.003                  # shapes move between calls: nothing stale in the cache
            ref2, sl2, integ2 = oo.nll(p2, *data, parts=True)
            assert abs(m.nll(p2) - ref2) <= nll_tol(ref2, sl2, integ2, data[0].size)
            m.set_path(B.PATH_AUTO)                          # AUTO picks the hybrid path here
            assert m.basis_bytes() > 0 and abs(m.nll(p) - ref) <= tol
            _, g = m.nll_grad(p)                             # AUTO: gradients stay on k_grad_recompute
            m.set_path(B.PATH_HYBRID)
            _, gh = m.nll_grad(p)                            # explicit hybrid path: k_grad_hybrid
            m.set_path(B.PATH_AUTO)
            _, ref_g = oo.nll_grad(p, *data)
            assert np.max(np.abs(g - ref_g)) <= 1e-9 * np.max(np.abs(ref_g))
            assert np.max(np.abs(gh - ref_g)) <= 1e-9 * np.max(np.abs(ref_g))
            m.set_norm_points(data[2][:5000], data[3][:5000], None)     # uniform weights, new normalisation cache
            ref3, sl3, integ3 = oo.nll(p, data[0], data[1], data[2][:5000], data[3][:5000], None, parts=True)
            assert abs(m.nll(p) - ref3) <= nll_tol(ref3, sl3, integ3, data[0].size)
            m.close()
    # not available without a fixed-shape or without a floating resonance
    c1, _, _ = make_case(1, n_ev=100, n_norm=100)
    m = B.Mipwa(c1.kin, c1.knots, c1.resonances)
    with pytest.raises(B.MipwaError) as ei:
        m.set_path(B.PATH_HYBRID)
    assert ei.value.code == B.ERR_STATE
    m.close()
    m = B.Mipwa(c.kin, c.knots, [dict(r, shape_floats=1) for r in c.resonances])
    with pytest.raises(B.MipwaError):
        m.set_path(B.PATH_HYBRID)
    m.close()


@pytest.mark.parametrize("n_fixed", [1, 2, 3, 4, 5])
def test_hybrid_ring_ragged_sizes(n_fixed):
    """k_nll_hybrid stages its cache columns through a cp.async ring, 1024 (RC <= 3: two points per thread) or 512
    points per block and iteration, two to four stages deep.  Sizes around the 256-point tile and the block iteration,
    fewer points than one block, more iterations than stages, an empty event set, both kinematics (equal and unequal
    daughter masses): NLL pieces against the oracle, and against the recompute kernel on the same context."""
    B = _lib()
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    fixed = [I._res(*I.RHO1450), I._res(*I.F2_1270), I._res(*I.SYN_A), I._res(*I.SYN_B), I._res(*I.SYN_C)][:n_fixed]
    for kin in (I.KIN, {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}):
        lo, hi = I.s_limits(kin)
        knots = np.linspace(lo - 1e-3, hi + 1e-3, 12)
        res = [I._res(*I.RHO770, shape_floats=1)] + fixed
        o = orc.Oracle(kin, knots, res)
        rng = np.random.default_rng(10 + n_fixed)
        p = np.concatenate([rng.uniform(0.5, 2, 12), rng.uniform(0, 3, 12), rng.uniform(0.3, 1.5, 2 * len(res)),
                            [0.78, 0.15]])
        s12, s13 = I.phase_space_points(400_000, I.stream_key(5, 20 + n_fixed, 1), kin)
        m = B.Mipwa(kin, knots, res)
        for n_ev, n_norm in ((0, 1), (1, 255), (257, 256), (1023, 1025), (513, 2049), (3, 5000), (160_001, 239_999)):
            e12, e13, g12, g13 = s12[:n_ev], s13[:n_ev], s12[n_ev:n_ev + n_norm], s13[n_ev:n_ev + n_norm]
            w = rng.uniform(0.5, 1.5, n_norm) / n_norm
            m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
            ref, sl, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
            m.set_path(B.PATH_HYBRID)
            got, gsl, ginteg = m.nll_parts(p)
            assert abs(got - ref) <= nll_tol(ref, sl, integ, n_ev), (n_ev, n_norm, got, ref)
            assert gsl == pytest.approx(sl, rel=1e-12, abs=1e-12) and ginteg == pytest.approx(integ, rel=1e-12)
            m.set_path(B.PATH_RECOMPUTE)
            rec, rsl, rinteg = m.nll_parts(p)
            assert gsl == pytest.approx(rsl, rel=1e-13, abs=1e-12) and ginteg == pytest.approx(rinteg, rel=1e-13)
            if n_ev in (257, 513, 160_001):                  # k_grad_hybrid + k_grad_shape: all 2N + 2R + 2 derivatives
                m.set_path(B.PATH_HYBRID)
                hn, hg = m.nll_grad_full(p)
                _, g_lin = o.nll_grad(p, e12, e13, g12, g13, w)
                _, g_shape = o.nll_grad_shape(p, e12, e13, g12, g13, w)
                ref_g = np.concatenate([g_lin, g_shape])
                assert abs(hn - ref) <= nll_tol(ref, sl, integ, n_ev)
                assert np.max(np.abs(hg - ref_g)) <= 1e-9 * np.max(np.abs(ref_g)), (n_ev, n_fixed)
        m.close()


@pytest.mark.gpu
@pytest.mark.parametrize("equal_masses", [True, False])
@pytest.mark.parametrize("shared_radii", [True, False])
def test_model_flag_variants(equal_masses, shared_radii):
    """The recompute, |A|^2 and gradient kernels are specialised on two model flags (equal daughter masses m1 == m2;
    radii shared by all resonances of one spin).  Two spin-1 and two spin-2 resonances make both flags matter; every
    one of the four kernel variants must match the oracle, which knows nothing of the flags."""
    B = _lib()
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    kin = {"M": 1.86966, "m1": 0.13957 if equal_masses else 0.493677, "m2": 0.13957, "m3": 0.13957}
    rr = (1.5, 1.5, 1.5, 1.5) if shared_radii else (1.5, 2.5, 1.5, 3.0)
    rp = (5.0, 5.0, 5.0, 5.0) if shared_radii else (5.0, 4.0, 5.0, 5.0)
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=rr[0], r_parent=rp[0]),
           dict(mass=1.2755, width=0.1867, spin=2, r_res=rr[2], r_parent=rp[2]),
           dict(mass=1.414, width=0.232, spin=1, r_res=rr[1], r_parent=rp[1]),
           dict(mass=1.5174, width=0.086, spin=2, r_res=rr[3], r_parent=rp[3])]
    lo, hi = I.s_limits(kin)
    knots = np.linspace(lo - 1e-3, hi + 1e-3, 23)
    s12, s13 = I.phase_space_points(9000, I.stream_key(3, 11, 1), kin)
    e12, e13, g12, g13 = s12[:4001], s13[:4001], s12[4001:], s13[4001:]
    w = np.full(g12.size, 0.37 / g12.size)
    o = orc.Oracle(kin, knots, res)
    rng = np.random.default_rng(5)
    p = np.concatenate([rng.uniform(0.5, 2, 23), rng.uniform(0, 3, 23), rng.uniform(0.3, 1.5, 8)])
    m = B.Mipwa(kin, knots, res)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w); m.set_path(B.PATH_RECOMPUTE)
    got, ref = m.eval_abs2(p, 0), o.abs2(p, e12, e13)
    assert np.max(np.abs(got - ref) / ref) < 1e-11
    ref_n, sl, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
    assert abs(m.nll(p) - ref_n) <= nll_tol(ref_n, sl, integ, e12.size)
    v, g = m.nll_grad(p)
    _, gref = o.nll_grad(p, e12, e13, g12, g13, w)
    assert abs(v - ref_n) <= nll_tol(ref_n, sl, integ, e12.size)
    assert np.max(np.abs(g - gref)) <= 1e-9 * np.max(np.abs(gref))
    m.close()
