"""GPU parity: analytic gradient on the recompute path (k_cell_keys, k_gather, k_grad_recompute) through the C ABI
against the oracle's O9 gradient (dense cardinal-spline form), which tests/test_oracle_nll.py pins to finite
differences and to the scale / phase Euler identities.

Tolerance (reading P26): every component within 1e-11 of the LARGEST gradient component.  Each
component is a sum of n_ev + n_norm terms of mixed sign whose partial sums are O(max component); fp64 summation in a
different order than the oracle's long-double accumulation leaves ~1e-13 relative to that scale (observed <= 2e-12), so
1e-11 has a decade of room for arithmetic and catches a wrong small component the earlier 1e-9 would have let through.
"""
import numpy as np
import pytest

from tests.helpers import make_case, nll_tol

pytestmark = pytest.mark.gpu


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


CASES = {
    0: dict(),
    1: dict(n_ev=40_000, n_norm=50_000),
    2: dict(n_ev=30_011, n_norm=20_003),          # non-uniform knots
    3: dict(n_ev=25_000, n_norm=25_000),          # floating rho(770) shape: gradient over the first 2N + 2R
    5: dict(n_ev=30_000),                         # the paper's own toy (K+K+K-, phi(1020), 0.001 GeV^2 grid)
    4: dict(n_ev=20_000, n_norm=20_000),          # six resonances (run-time resonance loop)
}


@pytest.fixture(scope="module", params=sorted(CASES))
def case(request):
    return make_case(request.param, **CASES[request.param])


def _check(got, ref):
    scale = np.max(np.abs(ref))
    err = np.max(np.abs(got - ref))
    assert err <= 1e-11 * scale, (err, scale, int(np.argmax(np.abs(got - ref))))


def test_gradient_matches_oracle(case):
    c, o, data = case
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    m.set_path(B.PATH_RECOMPUTE)
    for t in range(2):
        p = c.perturbed(t)
        ref_nll, ref_g = o.nll_grad(p, *data)
        nll, g = m.nll_grad(p)
        assert g.shape == (2 * c.N + 2 * c.R,)
        _, sl, integ = o.nll(p, *data, parts=True)
        assert abs(nll - ref_nll) <= nll_tol(ref_nll, sl, integ, data[0].size)
        _check(g, ref_g)
        assert abs(nll - m.nll(p)) <= nll_tol(ref_nll, sl, integ, data[0].size)      # value path agrees
    m.close()


def test_gradient_invariances_and_uniform_weights(case):
    """Euler identities (scale and global phase leave the NLL unchanged) hold for the GPU gradient itself."""
    c, o, data = case
    if c.idx not in (1, 3):
        pytest.skip("covered on two configs")
    B = _lib()
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], None)         # w = NULL -> 1/n
    p = c.perturbed(3)
    _, g = m.nll_grad(p)
    N, R = c.N, c.R
    mags = np.concatenate([p[:N], p[2 * N:2 * N + 2 * R:2]])
    gm = np.concatenate([g[:N], g[2 * N:2 * N + 2 * R:2]])
    gph = np.concatenate([g[N:2 * N], g[2 * N + 1:2 * N + 2 * R:2]])
    scale = np.max(np.abs(g))
    assert abs(np.dot(mags, gm)) <= 1e-9 * scale * mags.size
    assert abs(np.sum(gph)) <= 1e-9 * scale * mags.size
    _, ref_g = o.nll_grad(p, data[0], data[1], data[2], data[3], None)
    _check(g, ref_g)
    m.close()


def test_gradient_edge_cases():
    B = _lib()
    c, o, (e12, e13, g12, g13, w) = make_case(0, n_ev=700, n_norm=300)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    with pytest.raises(B.MipwaError) as ei:
        m.nll_grad(c.truth)
    assert ei.value.code == B.ERR_STATE
    m.set_norm_points(g12, g13, w)
    for n in (1, 31, 33, 700):                    # fewer points than warps in the grid; ragged chunks
        m.set_events(e12[:n], e13[:n])
        ref_nll, ref_g = o.nll_grad(c.truth, e12[:n], e13[:n], g12, g13, w)
        nll, g = m.nll_grad(c.truth)
        assert nll == pytest.approx(ref_nll, rel=1e-10)
        _check(g, ref_g)
    # a new event set must invalidate the sorted copy
    m.set_events(e12[100:400], e13[100:400])
    _, ref_g = o.nll_grad(c.truth, e12[100:400], e13[100:400], g12, g13, w)
    _check(m.nll_grad(c.truth)[1], ref_g)
    # empty sample: NLL = 0 and a zero gradient
    m.set_events(np.empty(0), np.empty(0))
    nll, g = m.nll_grad(c.truth)
    assert nll == 0.0 and np.all(g == 0.0)
    m.close()
    # pure S-wave model (R = 0) and N = 2 knots
    from oracle import oracle as orc
    knots = np.array([0.05, 3.1])
    o2 = orc.Oracle(c.kin, knots, [])
    m2 = B.Mipwa(c.kin, knots, [])
    m2.set_events(e12, e13); m2.set_norm_points(g12, g13, w)
    p2 = np.array([1.1, 0.7, 0.2, 1.9])
    _, ref_g = o2.nll_grad(p2, e12, e13, g12, g13, w)
    _check(m2.nll_grad(p2)[1], ref_g)
    m2.close()


def test_gradient_on_the_compact_cached_path(case):
    """Fixed shapes: mipwa_nll_grad under MIPWA_PATH_CACHED_COMPACT / AUTO streams the compact cache (k_grad_compact)
    and takes the normalisation part from the Gram matrix; under MIPWA_PATH_CACHED it recomputes.  All must agree
    with the oracle."""
    c, o, data = case
    B = _lib()
    if any(r.get("shape_floats") for r in c.resonances):
        pytest.skip("floating shapes cannot be cached")
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    p = c.perturbed(4)
    ref_nll, ref_g = o.nll_grad(p, *data)
    _, sl, integ = o.nll(p, *data, parts=True)
    tol = nll_tol(ref_nll, sl, integ, data[0].size)
    for path in (B.PATH_CACHED_COMPACT, B.PATH_AUTO, B.PATH_CACHED, B.PATH_RECOMPUTE, B.PATH_CACHED_COMPACT):
        m.set_path(path)
        nll, g = m.nll_grad(p)
        assert abs(nll - ref_nll) <= tol, path
        _check(g, ref_g)
        assert abs(m.nll(p) - ref_nll) <= tol
    # ragged and tiny samples on the cached gradient
    m.set_path(B.PATH_CACHED_COMPACT)
    for n in (1, 33, 257):
        m.set_events(data[0][:n], data[1][:n])
        _, ref_g = o.nll_grad(p, data[0][:n], data[1][:n], data[2], data[3], data[4])
        _check(m.nll_grad(p)[1], ref_g)
    m.close()


def test_full_gradient_with_floating_shapes_matches_oracle():
    """mipwa_nll_grad_full: the 2N + 2R coefficient derivatives plus d/d(mass, width) of every floating resonance
    (k_grad_shape) against the oracle's O10, which tests/test_oracle_shape.py pins to finite differences.
    Config 3 (rho(770) floats; ragged sizes) and a K- pi+ pi+ like model with two floating resonances of spin 1
    and 2 next to a fixed scalar, unweighted normalisation points."""
    B = _lib()
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    c, o, (e12, e13, g12, g13, w) = make_case(3, n_ev=25_003, n_norm=31_001)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w); m.set_path(B.PATH_RECOMPUTE)
    p = c.perturbed(1)
    v, g = m.nll_grad_full(p)
    ref_n, gref = o.nll_grad(p, e12, e13, g12, g13, w)
    _, gs = o.nll_grad_shape(p, e12, e13, g12, g13, w)
    full = np.concatenate([gref, gs])
    assert g.size == c.n_params == full.size
    _, sl, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
    assert abs(v - ref_n) <= nll_tol(ref_n, sl, integ, e12.size)
    assert np.max(np.abs(g - full)) <= 1e-9 * np.max(np.abs(full))
    assert np.max(np.abs(g[-2:] - gs)) <= 1e-9 * np.max(np.abs(gs))       # the shape entries on their own scale
    m.close()

    kin = {"M": 1.86966, "m1": 0.493677, "m2": 0.13957, "m3": 0.13957}
    lo, hi = I.s_limits(kin)
    res = [dict(mass=0.8955, width=0.047, spin=1, r_res=1.5, r_parent=5.0, shape_floats=1),
           dict(mass=1.2, width=0.2, spin=0, r_res=1.5, r_parent=5.0, shape_floats=0),
           dict(mass=1.4324, width=0.109, spin=2, r_res=2.0, r_parent=4.0, shape_floats=1)]
    knots = np.linspace(lo - 1e-3, hi + 1e-3, 9)
    o2 = orc.Oracle(kin, knots, res)
    s12, s13 = I.phase_space_points(9000, I.stream_key(3, 12, 1), kin)
    e12, e13, g12, g13 = s12[:4001], s13[:4001], s12[4001:], s13[4001:]
    rng = np.random.default_rng(3)
    p = np.concatenate([rng.uniform(0.5, 2, 9), rng.uniform(0, 3, 9), rng.uniform(0.3, 1.5, 6),
                        [0.8955, 0.047, 1.4324, 0.109]])
    m2 = B.Mipwa(kin, knots, res)
    m2.set_events(e12, e13); m2.set_norm_points(g12, g13, None); m2.set_path(B.PATH_RECOMPUTE)
    v, g = m2.nll_grad_full(p)
    ref_n, gref = o2.nll_grad(p, e12, e13, g12, g13, None)
    _, gs = o2.nll_grad_shape(p, e12, e13, g12, g13, None)
    full = np.concatenate([gref, gs])
    assert np.max(np.abs(g - full)) <= 1e-9 * np.max(np.abs(full))
    assert np.max(np.abs(g[-4:] - gs)) <= 1e-9 * np.max(np.abs(gs))
    m2.close()

    # no floating shape: the same call as mipwa_nll_grad (shared-memory flush order may differ in the last bits)
    c0, o0, (e12, e13, g12, g13, w) = make_case(0)
    m0 = B.Mipwa(c0.kin, c0.knots, c0.resonances)
    m0.set_events(e12, e13); m0.set_norm_points(g12, g13, w)
    va, ga = m0.nll_grad(c0.truth)
    vb, gb = m0.nll_grad_full(c0.truth)
    assert va == vb and np.max(np.abs(ga - gb)) <= 1e-12 * np.max(np.abs(ga))
    m0.close()


@pytest.mark.parametrize("idx,kw", [(0, dict()), (1, dict(n_ev=20_011, n_norm=30_000)), (4, dict(n_ev=4_000, n_norm=6_000))])
def test_hessian_matches_oracle(idx, kw):
    """mipwa_nll_hessian (k_gram in HESS mode over the events + Gram matrix + host assembly) against the oracle's O11
    Hessian, which tests/test_oracle_shape.py pins to differences of the gradient and to the invariance identities.
    Every entry within 1e-9 of the largest entry (same reasoning as the gradient tolerance, reading P26)."""
    B = _lib()
    c, o, (e12, e13, g12, g13, w) = make_case(idx, **kw)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
    p = c.perturbed(1)
    v, g, H = m.nll_hessian(p)
    Href = o.nll_hessian(p, e12, e13, g12, g13, w)
    ref_n, gref = o.nll_grad(p, e12, e13, g12, g13, w)
    _, sl, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
    assert abs(v - ref_n) <= nll_tol(ref_n, sl, integ, e12.size)
    _check(g, gref)
    scale = np.max(np.abs(Href))
    assert H.shape == Href.shape
    assert np.max(np.abs(H - Href)) <= 1e-9 * scale, np.max(np.abs(H - Href)) / scale
    assert np.max(np.abs(H - H.T)) <= 1e-11 * scale
    m.close()


def test_hessian_needs_fixed_shapes():
    B = _lib()
    c, o, (e12, e13, g12, g13, w) = make_case(3, n_ev=2_000, n_norm=2_000)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
    with pytest.raises(B.MipwaError) as e:
        m.nll_hessian(c.truth)
    assert e.value.code == B.ERR_STATE
    m.close()


def test_gradient_is_bit_reproducible():
    """Two calls with the same arguments return the same bits (per-warp segment bins summed in warp order, block
    partials in block order: no floating-point atomics anywhere), on the recompute path with the shape derivatives
    folded in, on the compact cached path and for the mixture likelihood."""
    B = _lib()
    c, o, data = make_case(3, n_ev=60_000, n_norm=50_000)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    p = c.perturbed(1)
    for call in (m.nll_grad, m.nll_grad_full):
        a, b = call(p), call(p)
        assert a[0] == b[0] and np.array_equal(a[1], b[1])
    m.nll_grad(c.perturbed(2))                                   # another point in between must leave no trace
    assert np.array_equal(m.nll_grad_full(p)[1], m.nll_grad_full(p)[1])
    m.set_event_background(np.full(data[0].size, 0.2))
    a, b = m.nll_mix_grad(p, 0.9), m.nll_mix_grad(p, 0.9)
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and a[2] == b[2]
    m.close()
    fixed = [dict(r, shape_floats=0) for r in c.resonances]
    mc = B.Mipwa(c.kin, c.knots, fixed)
    mc.set_events(data[0], data[1]); mc.set_norm_points(data[2], data[3], data[4])
    mc.set_path(B.PATH_CACHED_COMPACT)
    pc = p[:2 * c.N + 2 * c.R]
    a, b = mc.nll_grad(pc), mc.nll_grad(pc)
    assert a[0] == b[0] and np.array_equal(a[1], b[1])
    mc.close()


def test_full_hessian_with_floating_mass_and_width():
    """mipwa_nll_hessian_full at config 3 (rho(770) mass and width float, 108 parameters).  Block of the linear
    coefficients against the oracle's analytic Hessian O11 evaluated at the same (perturbed) shapes; the two shape rows
    against Richardson-extrapolated central differences of the ORACLE's pinned analytic gradient (O9 + O10)."""
    B = _lib()
    c, o, data = make_case(3, n_ev=6_000, n_norm=8_000)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    p = c.perturbed(1)
    P, Pl = p.size, 2 * c.N + 2 * c.R
    nll, g, H = m.nll_hessian_full(p)
    assert H.shape == (P, P) and np.max(np.abs(H - H.T)) <= 1e-9 * np.max(np.abs(H))
    H_lin = o.nll_hessian(p, *data)
    assert np.max(np.abs(H[:Pl, :Pl] - H_lin)) <= 1e-8 * np.max(np.abs(H_lin))

    def g_or(q):
        return np.concatenate([o.nll_grad(q, *data)[1], o.nll_grad_shape(q, *data)[1]])
    _check(g, g_or(p))
    for s in (Pl, Pl + 1):
        h = 1e-3 * p[Pl + 1]
        def d(hh):
            qp, qm = p.copy(), p.copy()
            qp[s] += hh; qm[s] -= hh
            return (g_or(qp) - g_or(qm)) / (2 * hh)
        ref = (4 * d(h / 2) - d(h)) / 3
        assert np.max(np.abs(H[s] - ref)) <= 1e-6 * np.max(np.abs(ref)), (s, np.max(np.abs(H[s] - ref)), np.max(np.abs(ref)))
    # a Newton step from a displaced shape lands on the minimum of the quadratic model: the error matrix is usable
    assert np.all(np.isfinite(H))
    m.close()
