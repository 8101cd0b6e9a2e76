"""Multi-GPU host logic: events and normalisation points are independent units, so rank g of G holds a
slice of each and evaluates its partial sums with its own libmipwa context.  The only exchange per likelihood call
is three doubles per rank (sum ln|A|^2, sum w|A|^2, n_ev), plus two gradient vectors when the minimiser wants
derivatives (3 + 2 n_params doubles, < 2 KB) - latency bound, so it goes through torch.distributed (NCCL over NVLink
on GPUs, gloo in the CPU tests); partials are gathered and added in rank order so that the result does not depend on
the reduction tree.
"""
import math


def shard_range(n, rank, world):
    """Contiguous slice [lo, hi) of n units owned by `rank` (sizes differ by at most one)."""
    return (n * rank) // world, (n * (rank + 1)) // world


def combine_parts(sum_log, integral, n_ev, group=None, device=None):
    """NLL of the whole sample from one rank's (sum_i ln|A_i|^2, sum_j w_j|A_j|^2, n_ev).

    The normalisation weights must already be those of the WHOLE sample (w_j = Area / n_norm_total), so that the
    per-rank integrals add.  Without an initialised process group this is the single-GPU combine (step A7).
    Returns (nll, total_sum_log, total_integral, total_n_ev).
    """
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        t = torch.tensor([sum_log, integral, float(n_ev)], dtype=torch.float64, device=device or "cpu")
        parts = [torch.empty_like(t) for _ in range(dist.get_world_size(group))]
        dist.all_gather(parts, t, group=group)
        S = I = n = 0.0
        for p in parts:                                  # rank order: bit-reproducible
            s_r, i_r, n_r = p.tolist()
            S += s_r; I += i_r; n += n_r
    else:
        S, I, n = sum_log, integral, float(n_ev)
    nll = -S + n * math.log(I) if n > 0 else 0.0
    return nll, S, I, int(n)


def combine_grad_parts(sum_log, integral, n_ev, grad_ev, grad_nm, group=None, device=None):
    """NLL and gradient of the whole sample from one rank's mipwa_nll_grad_parts output
    (S_r = sum_i ln|A_i|^2, I_r, n_r, grad_ev_r = d(-S_r)/dtheta, grad_nm_r = dI_r/dtheta):

        NLL = -sum_r S_r + n ln I,   dNLL/dtheta = sum_r grad_ev_r + (n / I) sum_r grad_nm_r,   n = sum_r n_r, I = sum_r I_r.

    A rank's own mipwa_nll_grad cannot be used here: it carries n_r / I_r.  One all_gather of 3 + 2 n_params doubles;
    the sum runs in rank order on every rank (same bits everywhere).  Returns (nll, grad, S, I, n).
    """
    import numpy as np
    import torch
    import torch.distributed as dist
    ge = np.ascontiguousarray(grad_ev, dtype=np.float64)
    gn = np.ascontiguousarray(grad_nm, dtype=np.float64)
    if ge.shape != gn.shape or ge.ndim != 1:
        raise ValueError("grad_ev and grad_nm must be vectors of the same length")
    P = ge.size
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        t = torch.from_numpy(np.concatenate([[sum_log, integral, float(n_ev)], ge, gn])).to(device or "cpu")
        parts = [torch.empty_like(t) for _ in range(dist.get_world_size(group))]
        dist.all_gather(parts, t, group=group)
        S = I = n = 0.0
        Ge, Gn = np.zeros(P), np.zeros(P)
        for p in parts:                                  # rank order: bit-reproducible
            v = p.cpu().numpy()
            S += float(v[0]); I += float(v[1]); n += float(v[2])
            Ge += v[3:3 + P]; Gn += v[3 + P:]
    else:
        S, I, n, Ge, Gn = sum_log, integral, float(n_ev), ge, gn
    if n > 0:
        return -S + n * math.log(I), Ge + (n / I) * Gn, S, I, int(n)
    return 0.0, np.zeros(P), S, I, 0
