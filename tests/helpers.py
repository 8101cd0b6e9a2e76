"""Shared test helpers: build a config's inputs with the ORACLE as the accept-reject density, and the tolerance
definitions of DESIGN.md section 3 (readings P14, P15).  Imports the oracle and the input generator only."""
import numpy as np

from oracle import oracle as orc
from paper_1703_03284_b200 import inputs as I


def make_case(idx, n_ev=None, n_norm=None, env_side=256):
    """(config, oracle, (e12, e13, g12, g13, w)) with events drawn from the oracle's |A|^2 at the truth."""
    c = I.Config(idx, n_ev=n_ev, n_norm=n_norm)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    f = lambda a, b: o.abs2(c.truth, a, b)
    e12, e13 = c.events(f, I.envelope_of(f, c.kin, n_side=env_side))
    g12, g13, w = c.norm_points()
    return c, o, (e12, e13, g12, g13, w)


def incoherent_scale(o, c, params, s12, s13):
    """(sum_k |c_k B_k|)^2 per point: the scale rounding errors follow when the coherent sum cancels (P15)."""
    N, R = c.N, c.R
    y = params[:N] * np.exp(1j * params[N:2 * N])
    cr = np.array([params[2 * N + 2 * r] * np.exp(1j * params[2 * N + 2 * r + 1]) for r in range(R)])
    B = o.basis(params, s12, s13)
    return (np.abs(B) @ np.abs(np.concatenate([y, cr]))) ** 2


def abs2_ok(got, ref, scale, rtol=1e-12, eps_c=1e-3):
    """P15: |got - ref| <= rtol * max(ref, eps_c * incoherent scale).  Returns (ok, worst ratio, plain max rel)."""
    bound = rtol * np.maximum(ref, eps_c * scale)
    ratio = np.abs(got - ref) / bound
    plain = np.max(np.abs(got - ref) / ref)
    return bool(np.all(ratio <= 1.0)), float(ratio.max()), float(plain)


def nll_tol(nll_ref, sum_log, integral, n_ev, rtol=1e-10):
    """P14: the two O(n_ev) pieces can cancel, so the bound follows their sizes."""
    return rtol * max(abs(nll_ref), abs(sum_log) + n_ev * abs(np.log(integral)))
