"""GPU parity: signal + background mixture likelihood (mipwa_set_event_background, mipwa_nll_mix, mipwa_nll_mix_grad;
SURVEY 8(f) f4) against the oracle's O12, which tests/test_oracle_mix.py pins.  Same tolerances as the pure-signal
NLL (reading P14) and gradient (reading P26)."""
import numpy as np
import pytest

from tests.helpers import make_case, nll_tol
from paper_1703_03284_b200 import inputs as I

pytestmark = pytest.mark.gpu

CASES = {0: dict(), 1: dict(n_ev=40_003, n_norm=50_000), 3: dict(n_ev=25_000, n_norm=25_001), 4: dict(n_ev=9_000, n_norm=9_000)}


@pytest.mark.parametrize("idx", sorted(CASES))
@pytest.mark.parametrize("f_sig", [0.9, 0.35])
def test_mixture_value_and_gradient_match_oracle(idx, f_sig):
    from paper_1703_03284_b200 import binding as B
    c, o, (e12, e13, g12, g13, w) = make_case(idx, **CASES[idx])
    bkg = (0.3 + 1.4 * I.uniforms(c.key(21), 0, e12.size)) / I.dalitz_area(c.kin)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
    m.set_event_background(bkg)
    p = c.perturbed(1)
    ref, gref, dref = o.nll_mix(p, e12, e13, bkg, f_sig, g12, g13, w, grad=True)
    _, sl, integ = o.nll(p, e12, e13, g12, g13, w, parts=True)
    tol = nll_tol(ref, sl, integ, e12.size)
    v = m.nll_mix(p, f_sig)                                # before prepare: the caller's event order
    assert abs(v - ref) <= tol, (v, ref)
    v2, g, dfs = m.nll_mix_grad(p, f_sig)                  # cell-sorted copies carry the densities along
    assert abs(v2 - ref) <= tol
    assert np.max(np.abs(g - gref)) <= 1e-9 * np.max(np.abs(gref))
    assert abs(dfs - dref) <= 1e-9 * max(abs(dref), e12.size)
    assert abs(m.nll_mix(p, f_sig) - ref) <= tol           # and the value path on the sorted copies
    m.close()


def test_mixture_limits_and_errors():
    from paper_1703_03284_b200 import binding as B
    import torch
    c, o, (e12, e13, g12, g13, w) = make_case(0)
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(e12, e13); m.set_norm_points(g12, g13, w)
    with pytest.raises(B.MipwaError) as e:
        m.nll_mix(c.truth, 0.9)                            # densities not set
    assert e.value.code == B.ERR_STATE
    bkg = torch.full((e12.size,), 1.0 / I.dalitz_area(c.kin), dtype=torch.float64, device="cuda")
    m.set_event_background(bkg)                            # borrowed device array
    m.set_path(B.PATH_RECOMPUTE)
    assert m.nll_mix(c.truth, 1.0) == pytest.approx(m.nll(c.truth), rel=1e-13)       # pure signal
    for bad in (0.0, -0.1, 1.5, float("nan")):
        with pytest.raises(B.MipwaError) as e:
            m.nll_mix(c.truth, bad)
        assert e.value.code == B.ERR_ARG
    m.set_events(e12, e13)                                 # new events drop the densities
    with pytest.raises(B.MipwaError) as e:
        m.nll_mix_grad(c.truth, 0.9)
    assert e.value.code == B.ERR_STATE
    m.close()
