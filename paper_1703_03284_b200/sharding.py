"""Multi-GPU host logic: events and normalisation points are independent units, so rank g of G holds a
slice of each and evaluates its partial sums with its own libmipwa context.  The only exchange per likelihood call is
three doubles per rank (sum ln|A|^2, sum w|A|^2, n_ev), plus two gradient vectors when the minimiser wants derivatives
(3 + 2 n_params doubles, < 2 KB) - latency bound, so it goes through torch.distributed (NCCL over NVLink on GPUs, gloo in
the CPU tests).  This module only moves the pieces; the sums themselves (always in rank order, so that every rank forms
the same bits) and step A7 are done by the C library: mipwa_combine_parts / mipwa_combine_grad_parts /
mipwa_combine_mix_parts on host data, mipwa_combine_parts_device on the GPU.

Three routes for the value:
  combine_parts          the pieces come from the host (mipwa_nll_parts); gloo, or NCCL through a staging tensor
  combine_parts_batch    B parameter vectors at once (mipwa_nll_batch): one all_gather for the whole batch
  nll_sharded_device     nothing touches the host between the likelihood kernel and the result: mipwa_nll_parts_device
                         leaves (S, I, n) in device memory, one all_gather on the same stream, mipwa_combine_parts_device
"""
import numpy as np

from . import binding


def shard_range(n, rank, world):
    """Contiguous slice [lo, hi) of n units owned by `rank` (sizes differ by at most one)."""
    return (n * rank) // world, (n * (rank + 1)) // world


def _world(group):
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        return dist.get_world_size(group)
    return 1


def _gather_rows(row, group, device):
    """all_gather one float64 vector per rank -> (world, len) numpy array, rows in rank order"""
    import torch
    import torch.distributed as dist
    world = _world(group)
    row = np.ascontiguousarray(row, dtype=np.float64)
    if world == 1:
        return row[None, :]
    t = torch.from_numpy(row).to(device or "cpu")
    parts = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(parts, t, group=group)
    return torch.stack(parts).cpu().numpy()


def combine_parts(sum_log, integral, n_ev, group=None, device=None):
    """NLL of the whole sample from one rank's (sum_i ln|A_i|^2, sum_j w_j|A_j|^2, n_ev).

    The normalisation weights must already be those of the WHOLE sample (w_j = Area / n_norm_total), so that the
    per-rank integrals add.  Without an initialised process group this is the single-GPU combine (step A7).
    Returns (nll, total_sum_log, total_integral, total_n_ev).
    """
    rows = _gather_rows([sum_log, integral, float(n_ev)], group, device)
    return binding.combine_parts(rows)


def combine_parts_batch(sum_log, integral, n_ev, group=None, device=None):
    """NLL of the whole sample at every one of B parameter vectors from one rank's pieces (mipwa_nll_batch with
    parts: sum_log[b], integral[b]): ONE all_gather of 2 B + 1 doubles per rank, then step A7 per vector in the C library
    (mipwa_combine_parts_batch: rank-ordered sums, the same bits on every rank).  Returns the B values."""
    S = np.ascontiguousarray(sum_log, dtype=np.float64)
    Iv = np.ascontiguousarray(integral, dtype=np.float64)
    if S.shape != Iv.shape or S.ndim != 1:
        raise ValueError("sum_log and integral must be vectors of the same length")
    rows = _gather_rows(np.concatenate([S, Iv, [float(n_ev)]]), group, device)
    return binding.combine_parts_batch(rows, S.size)


def combine_grad_parts(sum_log, integral, n_ev, grad_ev, grad_nm, group=None, device=None):
    """NLL and gradient of the whole sample from one rank's mipwa_nll_grad_parts output
    (S_r = sum_i ln|A_i|^2, I_r, n_r, grad_ev_r = d(-S_r)/dtheta, grad_nm_r = dI_r/dtheta):

        NLL = -sum_r S_r + n ln I,   dNLL/dtheta = sum_r grad_ev_r + (n / I) sum_r grad_nm_r,   n = sum_r n_r, I = sum_r I_r.

    A rank's own mipwa_nll_grad cannot be used here: it carries n_r / I_r.  One all_gather of 3 + 2 n_params doubles;
    the sums run in rank order on every rank (same bits everywhere).  Returns (nll, grad, S, I, n).
    """
    ge = np.ascontiguousarray(grad_ev, dtype=np.float64)
    gn = np.ascontiguousarray(grad_nm, dtype=np.float64)
    if ge.shape != gn.shape or ge.ndim != 1:
        raise ValueError("grad_ev and grad_nm must be vectors of the same length")
    rows = _gather_rows(np.concatenate([[sum_log, integral, float(n_ev)], ge, gn]), group, device)
    return binding.combine_grad_parts(rows, ge.size)


def nll_sharded_device(m, params, buffers=None, group=None):
    """One sharded likelihood step that stays on the device between the kernel and the result.

    m: this rank's binding.Mipwa, whose stream must be torch's CURRENT stream (the collective is enqueued behind the
    kernel on it).  buffers: optional (mine, gathered) float64 CUDA tensors of 3 and 3 x world elements, reused call to call.
    Returns (nll, S, I, n_ev) of the whole sample, identical on every rank.
    """
    import torch
    import torch.distributed as dist
    world = _world(group)
    if buffers is None:
        dev = torch.device("cuda", m.device)
        buffers = (torch.empty(3, dtype=torch.float64, device=dev), torch.empty(3 * world, dtype=torch.float64, device=dev))
    mine, gathered = buffers
    m.nll_parts_device(params, mine)
    if world > 1:
        dist.all_gather_into_tensor(gathered, mine, group=group)
    else:
        gathered = mine
    return m.combine_parts_device(gathered, world)


def nll_mix_sharded(m, params, f_sig, n_ev, grad=True, group=None, device=None):
    """Signal + background mixture likelihood of a sharded sample (two phases, include/mipwa.h):
    phase 1 gathers (I_r, dI_r/dtheta), phase 2 runs with I = sum_r I_r and gathers (S_r, Q_r, n_r, d(-S_r)/dtheta).
    Returns (nll, grad or None, dnll/df_sig) of the whole sample, identical on every rank."""
    P = 2 * m.N + 2 * m.R
    I_r, gnm = m.norm_parts(params, grad=grad)
    norm_rows = _gather_rows(np.concatenate([[I_r], gnm if grad else np.zeros(P)]), group, device)
    integral = 0.0
    for r in range(norm_rows.shape[0]):                  # rank order, the sum mipwa_combine_mix_parts forms as well
        integral += float(norm_rows[r, 0])
    S, Q, gev = m.nll_mix_parts(params, f_sig, integral, grad=grad)
    ev_rows = _gather_rows(np.concatenate([[S, Q, float(n_ev)], gev if grad else np.zeros(P)]), group, device)
    nll, g, dfs = binding.combine_mix_parts(norm_rows, ev_rows, P, f_sig)
    return nll, (g if grad else None), dfs


def hessian_sharded(m, params, n_ev, grad_total, group=None, device=None):
    """Hessian of a sharded fixed-shape likelihood in the 2N + 2R linear-coefficient parameters: every rank's event sum M_r
    and Gram matrix G_r (mipwa_hessian_parts) are gathered and added in rank order, then assembled on the host with the
    whole-sample gradient `grad_total` (combine_grad_parts)."""
    M, G = m.hessian_parts(params)
    rows = _gather_rows(np.concatenate([[float(n_ev)], M, G]), group, device)
    n_tot, Mt, Gt = 0.0, np.zeros_like(M), np.zeros_like(G)
    for r in range(rows.shape[0]):
        n_tot += rows[r, 0]
        Mt += rows[r, 1:1 + M.size]
        Gt += rows[r, 1 + M.size:]
    return m.hessian_assemble(params, int(n_tot), Mt, Gt, grad_total)
