"""GPU parity of mipwa_nll_grad_parts (the pieces one rank of a sharded likelihood contributes) against
the oracle's O9b, which tests/test_oracle_shape.py pins to Richardson differences of S and I, and the two-rank
combine of sharding.combine_grad_parts run on ONE GPU as two independent contexts, one per slice, one after the other
(the ranks of a sharded likelihood never wait on each other: the only exchange is the host-side all_gather).

Tolerance: reading P26 per piece (every component within 1e-9 of the piece's largest component)."""
import numpy as np
import pytest

from tests.helpers import make_case
from paper_1703_03284_b200 import sharding

pytestmark = pytest.mark.gpu

CASES = {
    3: dict(n_ev=25_013, n_norm=25_001),          # floating rho(770): recompute + k_grad_shape, 108 parameters
    2: dict(n_ev=30_011, n_norm=20_003),          # fixed shapes: compact cache + Gram matrix (AUTO) and recompute
}


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


def _close(got, ref, tol=1e-9):
    scale = np.max(np.abs(ref))
    err = np.max(np.abs(got - ref))
    assert err <= tol * scale, (err, scale, int(np.argmax(np.abs(got - ref))))


@pytest.fixture(scope="module", params=sorted(CASES))
def case(request):
    return make_case(request.param, **CASES[request.param])


def _paths(B, c):
    if any(r.get("shape_floats") for r in c.resonances):
        return [B.PATH_RECOMPUTE, B.PATH_HYBRID]           # k_grad_recompute / k_grad_hybrid, both followed by k_grad_shape
    return [B.PATH_RECOMPUTE, B.PATH_AUTO]                 # AUTO: compact cache + Gram matrix


def test_parts_match_oracle(case):
    c, o, data = case
    B = _lib()
    p = c.perturbed(1)
    S0, I0, gev0, gnm0 = o.nll_grad_parts(p, *data)
    for path in _paths(B, c):
        m = B.Mipwa(c.kin, c.knots, c.resonances)
        m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], data[4])
        m.set_path(path)
        S, Iv, gev, gnm = m.nll_grad_parts(p)
        assert gev.shape == gnm.shape == p.shape
        assert abs(S - S0) <= 1e-11 * abs(S0) and abs(Iv - I0) <= 1e-11 * abs(I0)
        _close(gev, gev0); _close(gnm, gnm0)
        nll, g = m.nll_grad_full(p)                      # the single-GPU gradient is the recombination
        _close(gev + (data[0].size / Iv) * gnm, g, 1e-12)
        m.close()


def test_parts_with_uniform_weights_and_empty_event_slice(case):
    c, o, data = case
    B = _lib()
    p = c.perturbed(2)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0][:0], data[1][:0]); m.set_norm_points(data[2], data[3], None)      # w = NULL -> 1/n
    m.set_path(B.PATH_RECOMPUTE)
    S, Iv, gev, gnm = m.nll_grad_parts(p)
    S0, I0, gev0, gnm0 = o.nll_grad_parts(p, data[0][:0], data[1][:0], data[2], data[3], None)
    assert S == 0.0 and not gev.any() and not gev0.any()
    assert abs(Iv - I0) <= 1e-11 * abs(I0)
    _close(gnm, gnm0)
    with pytest.raises(B.MipwaError):
        m.nll_grad_parts(p[:-1])
    m.close()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_combine_equals_whole_sample(case, world):
    c, o, data = case
    B = _lib()
    p = c.perturbed(3)
    e12, e13, g12, g13, w = data
    for path in _paths(B, c):
        tot = None
        for rank in range(world):                        # one context per slice, whole-sample weights
            lo, hi = sharding.shard_range(e12.size, rank, world)
            glo, ghi = sharding.shard_range(g12.size, rank, world)
            m = B.Mipwa(c.kin, c.knots, c.resonances)
            m.set_events(e12[lo:hi], e13[lo:hi]); m.set_norm_points(g12[glo:ghi], g13[glo:ghi], w[glo:ghi])
            m.set_path(path)
            S, Iv, gev, gnm = m.nll_grad_parts(p)
            m.close()
            part = np.concatenate([[S, Iv, hi - lo], gev, gnm])
            tot = part if tot is None else tot + part    # rank order, as combine_grad_parts adds them
        P = p.size
        nll, grad, S, Iv, n = sharding.combine_grad_parts(tot[0], tot[1], int(tot[2]), tot[3:3 + P], tot[3 + P:])
        assert n == e12.size
        ref_nll, g_lin = o.nll_grad(p, *data)
        _, g_shape = o.nll_grad_shape(p, *data)
        _, sl, integ = o.nll(p, *data, parts=True)
        assert abs(nll - ref_nll) <= 1e-10 * max(abs(ref_nll), abs(sl) + n * abs(np.log(integ)))
        _close(grad, np.concatenate([g_lin, g_shape]))
