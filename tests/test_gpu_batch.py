"""mipwa_nll_batch (include/mipwa.h): n_batch parameter vectors on the same sample, kernels enqueued back to back, one wait.
Same kernels and launch shape as mipwa_nll, so every value must have the bits of the blocking call, on every path; and the
oracle's value (O7) within the NLL tolerance of reading P14."""
import numpy as np
import pytest

from tests.helpers import make_case, nll_tol

pytestmark = pytest.mark.gpu


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


@pytest.mark.parametrize("idx", [2, 3])
def test_batch_has_the_bits_of_blocking_calls_on_every_path(idx):
    B = _lib()
    c, o, data = make_case(idx, n_ev=30_011, n_norm=20_003)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    ps = np.array([c.perturbed(t) for t in range(9)])
    fixed = not any(r.get("shape_floats") for r in c.resonances)
    paths = [B.PATH_RECOMPUTE, B.PATH_AUTO] + ([B.PATH_CACHED, B.PATH_CACHED_COMPACT, B.PATH_CACHED_REAL] if fixed else [])
    for path in paths:
        m.set_path(path)
        got, S, Iv = m.nll_batch(ps, parts=True)
        one = [m.nll_parts(p) for p in ps]
        assert np.array_equal(got, np.array([v[0] for v in one])), path
        assert np.array_equal(S, np.array([v[1] for v in one])) and np.array_equal(Iv, np.array([v[2] for v in one])), path
        again = m.nll_batch(ps[::-1])                      # the mapped block is reused: no value of the first call may survive
        assert np.array_equal(again, got[::-1]), path
    m.set_path(B.PATH_RECOMPUTE)
    got = m.nll_batch(ps)
    for p, v in zip(ps, got):
        ref, sl, integ = o.nll(p, *data, parts=True)
        assert abs(v - ref) <= nll_tol(ref, sl, integ, data[0].size)
    m.prepare()                                            # cell-sorted copies: same values within the tolerance
    srt = m.nll_batch(ps)
    assert np.max(np.abs(srt - got)) <= 1e-10 * np.max(np.abs(got))
    m.close()


def test_batch_sizes_unweighted_points_and_errors():
    B = _lib()
    c, o, data = make_case(1, n_ev=2_001, n_norm=3_003)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    with pytest.raises(B.MipwaError):
        m.nll_batch(np.array([c.perturbed(0)]))            # before the point sets
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], None)   # w_j = 1 / n
    m.set_path(B.PATH_RECOMPUTE)
    assert m.nll_batch(np.empty((0, c.n_params))).size == 0
    ps = np.array([c.perturbed(t % 7) for t in range(300)])  # more than the first allocation's 256 slots
    got = m.nll_batch(ps)
    assert np.array_equal(got[:7], np.array([m.nll(p) for p in ps[:7]]))
    assert np.array_equal(got[7:14], got[:7]) and np.array_equal(got[293:300], got[6:13])
    bad = ps[:5].copy(); bad[3, 0] = np.nan
    with pytest.raises(B.MipwaError):
        m.nll_batch(bad)
    with pytest.raises(B.MipwaError):
        m.nll_batch(ps[:, :-1])
    assert m.nll(ps[0]) == got[0]                          # the context is usable after a failed batch
    m.close()


@pytest.mark.parametrize("idx,n_ev,n_norm", [(1, 300, 500), (3, 700, 900), (2, 1, 40)])
def test_overlapped_launches_of_tiny_kernels(idx, n_ev, n_norm):
    """From the second vector on, the kernels of a batch are launched with programmatic stream serialisation: a kernel's
    blocks may be resident while its predecessor is still in its epilogue and wait (griddepcontrol.wait) before they touch the
    shared partials.  Samples of one or two blocks make every kernel catch up with its predecessor; random batch sizes,
    gradient and blocking calls in between.  Every value must keep the bits of the blocking call."""
    B = _lib()
    c, _, data = make_case(idx, n_ev=n_ev, n_norm=n_norm)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
    m.prepare()                                            # the order every later call uses (mipwa_nll_grad implies it)
    fixed = not any(r.get("shape_floats") for r in c.resonances)
    paths = [B.PATH_RECOMPUTE] + ([B.PATH_CACHED_COMPACT] if fixed else [B.PATH_AUTO])      # AUTO: the hybrid kernel
    ps = np.array([c.perturbed(t) for t in range(32)])
    ref = {}
    for path in paths:
        m.set_path(path)
        ref[path] = np.array([m.nll(p) for p in ps])
    rng = np.random.default_rng(idx)
    for it in range(60):
        path = paths[rng.integers(len(paths))]
        m.set_path(path)
        sel = rng.integers(0, 32, size=int(rng.integers(1, 300)))
        assert np.array_equal(m.nll_batch(ps[sel]), ref[path][sel]), (it, path, sel.size)
        if it % 7 == 0:
            m.nll_grad(ps[it % 32])
        if it % 11 == 0:
            assert m.nll(ps[3]) == ref[path][3]
    m.close()
