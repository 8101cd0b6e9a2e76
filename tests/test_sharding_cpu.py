"""Multi-GPU host logic on CPU (gloo, world_size 2): the per-rank partial sums of a sharded likelihood combine to the
single-process NLL.  The per-rank partials come from the ORACLE here (no GPU in this suite); on GPUs
bench.py feeds the same helper with the partials of mipwa_nll_parts."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_1703_03284_b200 import sharding


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 100, 1_000_003):
        for world in (1, 2, 3, 8):
            cuts = [sharding.shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = I.Config(1, n_ev=4001, n_norm=3001)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    g12, g13, w = c.norm_points()                      # weights of the WHOLE sample (Area / n_norm)
    e12, e13 = I.phase_space_points(c.n_ev, c.key(I.S_EVENTS))
    p = c.perturbed(1)
    full = o.nll(p, e12, e13, g12, g13, w, parts=True)
    lo, hi = sharding.shard_range(c.n_ev, rank, world)
    glo, ghi = sharding.shard_range(g12.size, rank, world)
    _, S, Iv = o.nll(p, e12[lo:hi], e13[lo:hi], g12[glo:ghi], g13[glo:ghi], w[glo:ghi], parts=True)
    nll, St, It, nt = sharding.combine_parts(S, Iv, hi - lo)
    # the batched form (mipwa_nll_batch pieces): three parameter vectors, ONE all_gather
    ps = [p, c.perturbed(2), c.perturbed(3)]
    pieces = [o.nll(v, e12[lo:hi], e13[lo:hi], g12[glo:ghi], g13[glo:ghi], w[glo:ghi], parts=True) for v in ps]
    batch = sharding.combine_parts_batch([v[1] for v in pieces], [v[2] for v in pieces], hi - lo)
    batch_ref = [o.nll(v, e12, e13, g12, g13, w) for v in ps]
    q.put((rank, nll, St, It, nt, full, list(batch), batch_ref))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_combine_matches_single_process():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = [q.get(timeout=240) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nlls = set()
    batches = set()
    for rank, nll, St, It, nt, (full, fS, fI), batch, batch_ref in out:
        assert nt == 4001
        assert abs(St - fS) <= 1e-11 * abs(fS) and abs(It - fI) <= 1e-12 * abs(fI)
        assert abs(nll - full) <= 1e-10 * max(abs(full), abs(fS) + nt * abs(np.log(fI)))
        nlls.add(nll)
        assert batch[0] == nll                         # vector 0 of the batch is the single call
        for got, ref in zip(batch, batch_ref):
            assert abs(got - ref) <= 1e-10 * max(abs(ref), abs(fS) + nt * abs(np.log(fI)))
        batches.add(tuple(batch))
    assert len(nlls) == 1                              # every rank forms the same bits (rank-ordered sum)
    assert len(batches) == 1


def test_combine_without_process_group_is_step_a7():
    nll, S, Iv, n = sharding.combine_parts(12.5, 3.0, 7)
    assert (S, Iv, n) == (12.5, 3.0, 7) and nll == -12.5 + 7 * np.log(3.0)
    batch = sharding.combine_parts_batch([12.5, -4.0], [3.0, 0.5], 7)
    assert list(batch) == [-12.5 + 7 * np.log(3.0), 4.0 + 7 * np.log(0.5)]


def _grad_worker(rank, world, port, q):
    import torch.distributed as dist
    from oracle import oracle as orc
    from paper_1703_03284_b200 import inputs as I
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = I.Config(3, n_ev=1501, n_norm=2001)            # rho(770) floats: 108 parameters, shape derivatives included
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    g12, g13, w = c.norm_points()
    e12, e13 = I.phase_space_points(c.n_ev, c.key(I.S_EVENTS))
    p = c.perturbed(2)
    lo, hi = sharding.shard_range(c.n_ev, rank, world)
    glo, ghi = sharding.shard_range(g12.size, rank, world)
    S, Iv, gev, gnm = o.nll_grad_parts(p, e12[lo:hi], e13[lo:hi], g12[glo:ghi], g13[glo:ghi], w[glo:ghi])
    nll, grad, St, It, nt = sharding.combine_grad_parts(S, Iv, hi - lo, gev, gnm)
    ref_nll, g_lin = o.nll_grad(p, e12, e13, g12, g13, w)
    _, g_shape = o.nll_grad_shape(p, e12, e13, g12, g13, w)
    q.put((rank, nll, grad, nt, ref_nll, np.concatenate([g_lin, g_shape])))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gradient_combine_matches_single_process():
    """grad = sum_r grad_ev_r + (n / I) sum_r grad_nm_r against the oracle's whole-sample gradient (O9 + O10)."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_grad_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = [q.get(timeout=240) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    grads = []
    for rank, nll, grad, nt, ref_nll, ref_grad in out:
        assert nt == 1501 and grad.size == 108
        assert abs(nll - ref_nll) <= 1e-10 * max(abs(ref_nll), 1.0) * 50
        assert np.max(np.abs(grad - ref_grad)) <= 1e-11 * np.max(np.abs(ref_grad))
        grads.append(grad)
    assert np.array_equal(grads[0], grads[1])          # every rank forms the same bits


def test_gradient_combine_without_process_group():
    ge, gn = np.array([1.0, -2.0]), np.array([0.5, 4.0])
    nll, g, S, Iv, n = sharding.combine_grad_parts(12.5, 3.0, 7, ge, gn)
    assert nll == -12.5 + 7 * np.log(3.0) and np.array_equal(g, ge + (7 / 3.0) * gn) and n == 7
    assert sharding.combine_grad_parts(0.0, 3.0, 0, ge, gn)[0] == 0.0


def test_mixture_combine_matches_the_whole_sample_oracle():
    """mipwa_combine_mix_parts (C library, host only) on per-slice pieces built from the ORACLE's pinned quantities:
    phase 1 (I_r, dI_r/dtheta) = O9b, phase 2 (S_r, Q_r, d(-S_r)/dtheta at fixed kappa) from the oracle's mixture NLL of
    the slice with the WHOLE-sample integral forced through its weights.  The combination must give the oracle's
    whole-sample mixture likelihood O12 (value, gradient and d/df_s)."""
    from oracle import oracle as orc
    from paper_1703_03284_b200 import binding, inputs as I
    c = I.Config(1, n_ev=901, n_norm=1201)
    o = orc.Oracle(c.kin, c.knots, c.resonances)
    g12, g13, w = c.norm_points()
    e12, e13 = I.phase_space_points(c.n_ev, c.key(I.S_EVENTS))
    rng = np.random.default_rng(3)
    bkg = rng.uniform(0.05, 0.4, c.n_ev)
    p, f_sig, P, world = c.perturbed(0), 0.85, 2 * c.N + 2 * c.R, 3
    ref, gref, dref = o.nll_mix(p, e12, e13, bkg, f_sig, g12, g13, w, grad=True)
    _, _, I_tot = o.nll(p, e12, e13, g12, g13, w, parts=True)
    kappa = I_tot * (1 - f_sig) / f_sig
    norm_rows, ev_rows = [], []
    for r in range(world):
        lo, hi = sharding.shard_range(c.n_ev, r, world)
        glo, ghi = sharding.shard_range(g12.size, r, world)
        _, I_r, _, gnm = o.nll_grad_parts(p, e12[:1], e13[:1], g12[glo:ghi], g13[glo:ghi], w[glo:ghi])
        norm_rows.append(np.concatenate([[I_r], gnm[:P]]))
        # event pieces of the slice: D_i = |A_i|^2 + kappa b_i;  d(-S)/dtheta at fixed kappa = -sum (d|A_i|^2/dtheta) / D_i,
        # taken from the oracle's O9b event gradient of a sample re-weighted event by event: -sum_i dln|A_i|^2 * (|A_i|^2/D_i)
        a2 = o.abs2(p, e12[lo:hi], e13[lo:hi])
        D = a2 + kappa * bkg[lo:hi]
        gev = np.zeros(P)
        for i in range(lo, hi):                             # one event at a time: d(-ln|A_i|^2)/dtheta from O9b
            _, _, gi, _ = o.nll_grad_parts(p, e12[i:i + 1], e13[i:i + 1], g12[:1], g13[:1], w[:1])
            gev += gi[:P] * (a2[i - lo] / D[i - lo])
        ev_rows.append(np.concatenate([[np.sum(np.log(D)), np.sum(bkg[lo:hi] / D), hi - lo], gev]))
    nll, g, dfs = binding.combine_mix_parts(np.array(norm_rows), np.array(ev_rows), P, f_sig)
    assert abs(nll - ref) <= 1e-10 * max(abs(ref), c.n_ev)
    assert np.max(np.abs(g - gref)) <= 1e-9 * np.max(np.abs(gref))
    assert abs(dfs - dref) <= 1e-9 * max(1.0, abs(dref))
