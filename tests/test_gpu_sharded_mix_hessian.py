"""GPU parity of the sharded forms of the mixture likelihood and of the Hessian, and of the
device-side combine.  The slices of a 3-way split run as independent contexts on ONE GPU, one after the other (the ranks
of a sharded likelihood never wait on each other); their pieces are combined by the C library's rank-ordered sums and
must give what the ORACLE computes on the whole sample: O12 (mixture value, gradient, d/df_s), O11 (Hessian), O7 (NLL)."""
import numpy as np
import pytest

from tests.helpers import make_case, nll_tol
from paper_1703_03284_b200 import sharding

pytestmark = pytest.mark.gpu


def _lib():
    from paper_1703_03284_b200 import binding
    return binding


@pytest.fixture(scope="module")
def case():
    return make_case(2, n_ev=30_011, n_norm=20_003)          # fixed shapes, non-uniform knots, ragged sizes


def _slices(B, c, data, world, bkg=None):
    e12, e13, g12, g13, w = data
    ctxs = []
    for r in range(world):
        lo, hi = sharding.shard_range(e12.size, r, world)
        glo, ghi = sharding.shard_range(g12.size, r, world)
        m = B.Mipwa(c.kin, c.knots, c.resonances)
        m.set_events(e12[lo:hi], e13[lo:hi]); m.set_norm_points(g12[glo:ghi], g13[glo:ghi], w[glo:ghi])
        if bkg is not None:
            m.set_event_background(bkg[lo:hi])
        ctxs.append((m, hi - lo))
    return ctxs


def test_sharded_mixture_matches_whole_sample_oracle(case):
    c, o, data = case
    B = _lib()
    rng = np.random.default_rng(8)
    bkg = rng.uniform(0.05, 0.4, data[0].size)
    p, f_sig, P, world = c.perturbed(1), 0.9, 2 * c.N + 2 * c.R, 3
    ref, gref, dref = o.nll_mix(p, data[0], data[1], bkg, f_sig, data[2], data[3], data[4], grad=True)
    ctxs = _slices(B, c, data, world, bkg)
    norm_rows = []
    for m, n in ctxs:                                        # phase 1 on every "rank"
        I_r, gnm = m.norm_parts(p)
        norm_rows.append(np.concatenate([[I_r], gnm]))
    integral = 0.0
    for row in norm_rows:
        integral += row[0]
    _, _, I_or = o.nll(p, *data, parts=True)
    assert abs(integral - I_or) <= 1e-12 * I_or
    ev_rows = []
    for m, n in ctxs:                                        # phase 2 with the whole-sample integral
        S, Q, gev = m.nll_mix_parts(p, f_sig, integral)
        ev_rows.append(np.concatenate([[S, Q, n], gev]))
    nll, g, dfs = B.combine_mix_parts(np.array(norm_rows), np.array(ev_rows), P, f_sig)
    assert abs(nll - ref) <= 1e-10 * max(abs(ref), data[0].size)
    assert np.max(np.abs(g - gref)) <= 1e-10 * np.max(np.abs(gref))
    assert abs(dfs - dref) <= 1e-9 * max(1.0, abs(dref))
    # the single-context call is the world = 1 case of the same formulas
    m1 = B.Mipwa(c.kin, c.knots, c.resonances)
    m1.set_events(data[0], data[1]); m1.set_norm_points(data[2], data[3], data[4]); m1.set_event_background(bkg)
    nll1, g1, dfs1 = m1.nll_mix_grad(p, f_sig)
    assert abs(nll1 - nll) <= 1e-10 * max(abs(ref), data[0].size) and np.max(np.abs(g1 - g)) <= 1e-10 * np.max(np.abs(g))
    nll_s, g_s, dfs_s = sharding.nll_mix_sharded(m1, p, f_sig, data[0].size)    # no process group: one rank
    assert nll_s == pytest.approx(nll1, rel=1e-13) and np.max(np.abs(g_s - g1)) <= 1e-12 * np.max(np.abs(g1))
    for m, _ in ctxs:
        m.close()
    m1.close()


def test_sharded_hessian_matches_whole_sample_oracle(case):
    c, o, data = case
    B = _lib()
    p, world = c.perturbed(2), 3
    H_ref = o.nll_hessian(p, *data)
    ctxs = _slices(B, c, data, world)
    rows, Ms, Gs = [], [], []
    for m, n in ctxs:
        S, Iv, gev, gnm = m.nll_grad_parts(p)
        rows.append(np.concatenate([[S, Iv, n], gev, gnm]))
        M, G = m.hessian_parts(p)
        Ms.append(M); Gs.append(G)
    nll, grad, S, Iv, n_tot = B.combine_grad_parts(np.array(rows), p.size)
    ref_nll, sl, integ = o.nll(p, *data, parts=True)
    assert n_tot == data[0].size and abs(nll - ref_nll) <= nll_tol(ref_nll, sl, integ, n_tot)
    Mt, Gt = np.zeros_like(Ms[0]), np.zeros_like(Gs[0])
    for M, G in zip(Ms, Gs):
        Mt += M; Gt += G
    H = ctxs[0][0].hessian_assemble(p, n_tot, Mt, Gt, grad)
    assert np.max(np.abs(H - H_ref)) <= 1e-8 * np.max(np.abs(H_ref))
    m1 = B.Mipwa(c.kin, c.knots, c.resonances)               # one context over the whole sample: same matrix
    m1.set_events(data[0], data[1]); m1.set_norm_points(data[2], data[3], data[4])
    _, _, H1 = m1.nll_hessian(p)
    assert np.max(np.abs(H - H1)) <= 1e-9 * np.max(np.abs(H1))
    H2 = sharding.hessian_sharded(m1, p, n_tot, grad)        # no process group: one rank
    assert np.max(np.abs(H2 - H1)) <= 1e-12 * np.max(np.abs(H1))
    for m, _ in ctxs:
        m.close()
    m1.close()


def test_device_side_combine_matches_host_combine(case):
    """mipwa_nll_parts_device leaves (S, I, n) on the device; mipwa_combine_parts_device adds the gathered pieces in rank
    order in one tiny kernel and applies A7: same numbers as the host route, for every path, weights or not."""
    import torch
    c, o, data = case
    B = _lib()
    p, world = c.perturbed(0), 3
    ref_nll, sl, integ = o.nll(p, *data, parts=True)
    ctxs = _slices(B, c, data, world)
    gathered = torch.empty(3 * world, dtype=torch.float64, device="cuda")
    for path in (B.PATH_RECOMPUTE, B.PATH_CACHED_COMPACT, B.PATH_CACHED):
        host_rows = []
        for r, (m, n) in enumerate(ctxs):
            m.set_path(path)
            m.nll_parts_device(p, gathered[3 * r:3 * r + 3])
            _, S, Iv = m.nll_parts(p)
            host_rows.append([S, Iv, n])
        nll_d, S_d, I_d, n_d = ctxs[0][0].combine_parts_device(gathered, world)
        nll_h, S_h, I_h, n_h = B.combine_parts(np.array(host_rows))
        assert (S_d, I_d, n_d) == (S_h, I_h, n_h)             # same pieces, same rank-ordered sums: same bits
        assert abs(nll_d - nll_h) <= 1e-15 * abs(nll_h) * 4    # log on the device and in libm may differ by an ulp
        assert abs(nll_d - ref_nll) <= nll_tol(ref_nll, sl, integ, n_d)
    # normalisation points without weights (w_j = 1 / n): the device route applies the 1 / n itself
    m = B.Mipwa(c.kin, c.knots, c.resonances)
    m.set_events(data[0], data[1]); m.set_norm_points(data[2], data[3], None); m.set_path(B.PATH_RECOMPUTE)
    nll_s = sharding.nll_sharded_device(m, p)[0]
    assert abs(nll_s - m.nll(p)) <= 1e-15 * abs(nll_s) * 4
    m.close()
    for m, _ in ctxs:
        m.close()
