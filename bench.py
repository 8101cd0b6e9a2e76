#!/usr/bin/env python
"""bench.py -- one JSON line for the MIPWA NLL hot path on B200 (contract: task prompt "Measurement").

A "step" is one likelihood evaluation mipwa_nll(params) over the whole sample: every event and every
normalisation point goes through the fused amplitude + reduction kernel once.
Workload at N = 1: BASELINE.json configs[3] (the configuration the metric "at 10M events" is quoted on):
50 knots + rho(770) [mass, width floating] + rho(1450) + f2(1270), 10 M events + 10 M normalisation points, fp64,
full recompute every call.  N > 1: every rank holds its own 10 M + 10 M shard (weak scaling); the only exchange
is three doubles per rank per call (paper_1703_03284_b200/sharding.py).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--events E] [--norm-points G]

--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1703_03284_b200 import inputs as I  # noqa: E402

METRIC = "MIPWA NLL events/s (full recompute, 10M events + 10M normalisation points per GPU, fp64)"
UNIT = "events/s"


# ---- algorithmic work per point: flops of the plain formulas, one per add / mul /
# div / sqrt / log, fma = 2: two channels x [10 shared kinematics + 14 spline + 37 R] + 4, plus 2 (1 + 3R) divisions,
# 2 (2 + R) square roots and one log = 59 + 82 R (305 at R = 3).  The kernel as built executes 261 at config 3
# (ncu-counted dadd + dmul + 2 dfma per point, profiles/r1_k_nll_recompute_ncu.md: the equal-mass and shared-radii
# specialisations and one reciprocal (square root) per resonance and channel do the same arithmetic in fewer
# operations), so nothing is padded; "executed_flops_per_point" in the roofline object gives the executed rate. ------
def flops_per_point(resonances):
    return 59 + 82 * len(resonances)


# dram__bytes_read.sum + dram__bytes_write.sum per k_nll_recompute launch at the bench size (10M events + 10M weighted
# normalisation points), from the one `ncu --set full` capture summarised in profiles/r1_k_nll_recompute_ncu.md
NCU_TRAFFIC_BYTES = {(10_000_000, 10_000_000): 445.3e6}
# executed FP64 flops per point in that capture (config 3's model): (dadd + dmul + 2 dfma) / points
NCU_EXECUTED_FLOPS_PER_POINT = {(10_000_000, 10_000_000): 260.7}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def stop(self):
        if self.proc:
            self.proc.terminate()

    def summary(self, t0, t1):
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": float(np.median([float(r[0]) for r in rows])), "sm_max_mhz": float(rows[0][1]),
                "power_w_max": max(float(r[2]) for r in rows), "samples": len(rows), "reasons": reasons}


def oracle_sample(cfg, n_ev, n_norm):
    """Inputs for the oracle legs: generated with the oracle itself as the accept-reject density (no CUDA)."""
    from oracle import oracle as orc
    o = orc.Oracle(cfg.kin, cfg.knots, cfg.resonances)
    f = lambda a, b: o.abs2(cfg.truth, a, b)
    e12, e13 = cfg.events(f, I.envelope_of(f, cfg.kin), n=n_ev)
    g12, g13 = I.phase_space_points(n_norm, cfg.key(I.S_NORM), cfg.kin)
    w = np.full(n_norm, I.dalitz_area(cfg.kin) / n_norm)
    return o, (e12, e13, g12, g13, w)


def time_oracle(cfg, n_ev, n_norm, steps, warmup):
    from oracle import oracle as orc
    o, data = oracle_sample(cfg, n_ev, n_norm)
    for t in range(warmup):
        o.nll(cfg.perturbed(t), *data)
    t0 = time.perf_counter()
    for t in range(steps):
        o.nll(cfg.perturbed(warmup + t), *data)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    return {"value": n_ev / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "seconds_per_call": dt,
            "sample": f"first {n_ev} events + {n_norm} normalisation points of the workload, {steps} NLL call(s), "
                      f"OpenMP over all host threads"}


def run_reference(args, cfg, workload):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # exactly K timed steps; each step is one oracle NLL call on a bounded sample of the workload, sized so that
    # K + W calls end within a few minutes (the oracle does ~1e7 points/s on 8-16 host threads)
    steps, warmup = max(1, args.steps), args.warmup
    per_set = int(max(10_000, min(400_000, 0.7e9 / (steps + warmup))))
    n_ev = min(cfg.n_ev, per_set)
    n_norm = min(cfg.norm_size, per_set)
    cb = time_oracle(cfg, n_ev, n_norm, steps, warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * cb["seconds_per_call"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload, sample_events=n_ev, sample_norm_points=n_norm),
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def gpu_inputs(cfg, m, B, torch, rank):
    """Events by accept-reject on the device (mipwa_generate: the recipe of DESIGN.md section 4 / reading P22, the
    same stream key inputs.Config.events uses), normalisation points uniform in phase space; both end up resident
    in HBM as torch tensors."""
    e12, e13, _ = m.generate(cfg.truth, cfg.key(I.S_EVENTS + 16 * rank), cfg.n_ev, n_side=1024, n_coarse=64)
    g12, g13, w = cfg.norm_points(stream=rank)
    host = [np.ascontiguousarray(a) for a in (e12, e13, g12, g13, w)]
    dev = [torch.from_numpy(a).cuda() for a in host]
    return host, dev


def m_grad_full_ref(m, B, p):
    """the same gradient through the full-recompute kernels (cross-check of the hybrid gradient leg)"""
    m.set_path(B.PATH_RECOMPUTE)
    g = m.nll_grad_full(p)[1]
    m.set_path(B.PATH_HYBRID)
    return g


def run_ours(args, cfg, workload):
    import torch
    import torch.distributed as dist
    from paper_1703_03284_b200 import binding as B
    from paper_1703_03284_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    m = B.Mipwa(cfg.kin, cfg.knots, cfg.resonances, device=local)
    stream = torch.cuda.Stream(device=dev)
    m.set_stream(stream)
    t_gen = time.perf_counter()
    host, d = gpu_inputs(cfg, m, B, torch, rank)
    t_gen = time.perf_counter() - t_gen
    if world > 1:                                    # whole-sample weights so that per-rank integrals add
        d[4] = d[4] / world
        host[4] = host[4] / world
    m.set_events(d[0], d[1])
    m.set_norm_points(d[2], d[3], d[4])
    m.set_path(B.PATH_RECOMPUTE)
    t_prep = time.perf_counter()
    m.prepare()                                      # once per sample: cell-sorted copies (a fit reuses them every call)
    torch.cuda.synchronize(dev)
    t_prep = time.perf_counter() - t_prep
    m.enable_timing(True)
    n_ev, n_norm = d[0].numel(), d[2].numel()

    params = [cfg.perturbed(t) for t in range(args.warmup + args.steps)]

    def step(p):
        _, S, Iv = m.nll_parts(p)
        return sharding.combine_parts(S, Iv, n_ev, device=dev)[0]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for t in range(args.warmup):
        step(params[t])

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = m.launch_count()
    kernel_ms = []
    w0 = time.perf_counter()
    ev0.record(stream)
    for t in range(args.steps):
        nll = step(params[args.warmup + t])
        kernel_ms.append(m.last_kernel_ms())
    ev1.record(stream)
    barrier()
    w1 = time.perf_counter()
    launches = m.launch_count() - launches0
    ms_total = ev0.elapsed_time(ev1)
    if world > 1:
        tt = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    ms_step = ms_total / args.steps

    # ---- e2e: the same evaluation through the C ABI from HOST buffers: H2D of the step's inputs (pinned), the
    # boundary check, the NLL kernel and the D2H of the result are all inside the timed region -----------------------
    pinned = [torch.from_numpy(a).pin_memory() for a in host]
    ph = [t.numpy() for t in pinned]
    e2e_steps = max(3, min(args.steps, 10))
    def e2e_step(p):
        m.set_events(ph[0], ph[1])
        m.set_norm_points(ph[2], ph[3], ph[4])
        _, S, Iv = m.nll_parts(p)
        return sharding.combine_parts(S, Iv, n_ev, device=dev)[0]
    e2e_step(params[0]); e2e_step(params[1])
    barrier()
    t0 = time.perf_counter()
    for t in range(e2e_steps):
        nll_e2e = e2e_step(params[args.warmup + t % args.steps])
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        tt = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    h2d = sum(a.nbytes for a in ph) + params[0].nbytes
    d2h = 16 + 16                                     # two boundary-check counters + (sum ln|A|^2, I)
    # back to resident device arrays for the fit-step latency number
    m.set_events(d[0], d[1]); m.set_norm_points(d[2], d[3], d[4]); m.prepare()
    t0 = time.perf_counter()
    for t in range(args.steps):
        step(params[args.warmup + t])
    fit_step_s = (time.perf_counter() - t0) / args.steps

    # ---- A8: value + analytic gradient (BASELINE configs[3]: "plus analytic gradient w.r.t. all 2N+2*3 parameters") ----
    sub_steps = max(3, min(args.steps, 30))
    for t in range(3):
        m.nll_grad(params[t])
    grad_ms = []
    barrier()
    t0 = time.perf_counter()
    for t in range(sub_steps):
        nll_g, grad = m.nll_grad(params[args.warmup + t % args.steps])
        grad_ms.append(m.last_kernel_ms())
    barrier()
    grad_wall = (time.perf_counter() - t0) / sub_steps
    grad_info = {"ms_per_call": 1e3 * grad_wall, "kernel_ms": float(np.mean(grad_ms)),
                 "events_per_s": n_ev * world / grad_wall, "n_grad": int(grad.size), "nll": nll_g,
                 "what": "mipwa_nll_grad: NLL + d/d(a_k, phi_k, |c_r|, arg c_r), same sample, k_grad_recompute"}
    # all n_params derivatives, incl. d/d(mass, width) of the floating rho(770) (k_grad_shape, one extra pass)
    for t in range(2):
        m.nll_grad_full(params[t])
    full_ms = []
    barrier()
    t0 = time.perf_counter()
    for t in range(sub_steps):
        nll_f, grad_f = m.nll_grad_full(params[args.warmup + t % args.steps])
        full_ms.append(m.last_kernel_ms())
    barrier()
    full_wall = (time.perf_counter() - t0) / sub_steps
    grad_info["full"] = {"ms_per_call": 1e3 * full_wall, "kernel_ms": float(np.mean(full_ms)), "n_grad": int(grad_f.size),
                         "d_mass_d_width": [float(x) for x in grad_f[grad.size:]],
                         "what": "mipwa_nll_grad_full: the above + d/d(mass, width) of every floating resonance"}

    # the sharded form of the same call: per-rank pieces, one all_gather of 3 + 2 n_params doubles, combine
    for t in range(2):
        m.nll_grad_parts(params[t])
    barrier()
    t0 = time.perf_counter()
    for t in range(sub_steps):
        S_p, I_p, g_ev, g_nm = m.nll_grad_parts(params[args.warmup + t % args.steps])
        nll_s, grad_s = sharding.combine_grad_parts(S_p, I_p, n_ev, g_ev, g_nm, device=dev)[:2]
    barrier()
    sh_wall = (time.perf_counter() - t0) / sub_steps
    grad_info["sharded"] = {"ms_per_call": 1e3 * sh_wall, "events_per_s": n_ev * world / sh_wall, "n_grad": int(grad_s.size),
                            "nll": nll_s, "max_abs_diff_vs_full_at_1gpu": (float(np.max(np.abs(grad_s - grad_f))) if world == 1 else None),
                            "what": "mipwa_nll_grad_parts + sharding.combine_grad_parts: whole-job NLL and all n_params "
                                    "derivatives from per-rank (S, I, d(-S), dI); 3 + 2 n_params doubles all-gathered per call"}

    # ---- signal + background mixture (purity 90 %): flat background density, two launches per call ----------
    m.set_event_background(torch.full((n_ev,), 1.0 / I.dalitz_area(cfg.kin), dtype=torch.float64, device=dev))
    for t in range(3):
        m.nll_mix(params[t], 0.9)
    mix_ms = []
    for t in range(sub_steps):
        nll_mix = m.nll_mix(params[args.warmup + t % args.steps], 0.9)
        mix_ms.append(m.last_kernel_ms())
    for t in range(2):
        m.nll_mix_grad(params[t], 0.9)
    mixg_ms = []
    for t in range(sub_steps):
        nll_mixg, g_mix, dfs_mix = m.nll_mix_grad(params[args.warmup + t % args.steps], 0.9)
        mixg_ms.append(m.last_kernel_ms())
    mix_info = {"f_sig": 0.9, "value_kernel_ms": float(np.mean(mix_ms)), "grad_kernel_ms": float(np.mean(mixg_ms)),
                "nll": nll_mix, "nll_grad_path": nll_mixg, "dnll_dfsig": dfs_mix,
                "what": "mipwa_nll_mix / mipwa_nll_mix_grad: -sum ln(f_s |A|^2 / I + (1 - f_s) b), normalisation launch then "
                        "event launch (kernel_ms spans both and the host read of I between them)"}
    m.set_event_background(None)

    # ---- hybrid path (AUTO's choice for this model): rho(770) recomputed, rho(1450) and f2(1270) cached per point -------
    hybrid_info = None
    try:
        m.set_path(B.PATH_HYBRID)
        t0 = time.perf_counter(); m.nll(params[0]); setup_s = time.perf_counter() - t0
        for t in range(3):
            m.nll(params[t])
        kms = []
        barrier()
        t0 = time.perf_counter()
        for t in range(sub_steps):
            nll_h = m.nll(params[args.warmup + t % args.steps])
            kms.append(m.last_kernel_ms())
        barrier()
        wall = (time.perf_counter() - t0) / sub_steps
        for t in range(3):
            m.nll_grad_full(params[t])
        gms = []
        for t in range(sub_steps):
            nll_hg, grad_hg = m.nll_grad_full(params[args.warmup + t % args.steps])
            gms.append(m.last_kernel_ms())
        hybrid_info = {"ms_per_call": 1e3 * wall, "kernel_ms": float(np.mean(kms)), "events_per_s": n_ev * world / wall,
                       "grad_full_kernel_ms": float(np.mean(gms)), "grad_full_nll": nll_hg,
                       "grad_full_max_abs_diff_vs_recompute": float(np.max(np.abs(
                           grad_hg - m_grad_full_ref(m, B, params[args.warmup + (sub_steps - 1) % args.steps])))),
                       "cache_bytes": m.basis_bytes(), "first_call_s": setup_s, "nll": nll_h,
                       "what": "MIPWA_PATH_HYBRID: floating resonances and spline recomputed, fixed-shape resonance terms "
                               "streamed from a per-point cache (not the headline: part of the work is cached); grad_full_*: "
                               "mipwa_nll_grad_full under an explicit MIPWA_PATH_HYBRID (k_grad_hybrid + k_grad_shape), "
                               "cross-checked against the full-recompute gradient"}
    except B.MipwaError:
        pass
    m.set_path(B.PATH_RECOMPUTE)

    # ---- A9/A10: fixed-shape cached paths on the SAME events (all shapes fixed at their listed values) ------------------
    cached_info = {}
    fixed = [dict(r, shape_floats=0) for r in cfg.resonances]
    mc = B.Mipwa(cfg.kin, cfg.knots, fixed, device=local)
    mc.set_stream(stream)
    mc.set_events(d[0], d[1]); mc.set_norm_points(d[2], d[3], d[4])
    mc.prepare()
    mc.enable_timing(True)
    pc = [p[:2 * cfg.N + 2 * cfg.R] for p in params]
    for name, path in (("dense", B.PATH_CACHED), ("compact", B.PATH_CACHED_COMPACT)):
        mc.set_path(path)
        t0 = time.perf_counter(); mc.nll(pc[0]); setup_s = time.perf_counter() - t0
        for t in range(3):
            mc.nll(pc[t])
        kms = []
        barrier()
        t0 = time.perf_counter()
        for t in range(sub_steps):
            nll_c = mc.nll(pc[args.warmup + t % args.steps])
            kms.append(mc.last_kernel_ms())
        barrier()
        wall = (time.perf_counter() - t0) / sub_steps
        nbytes = mc.basis_bytes()
        k = float(np.mean(kms))
        cached_info[name] = {"ms_per_call": 1e3 * wall, "kernel_ms": k, "events_per_s": n_ev * world / wall,
                             "bytes_per_event": nbytes / max(n_ev, 1), "cache_bytes": nbytes,
                             "first_call_s": setup_s, "nll": nll_c,
                             "roofline": {"bound": "hbm", "kernel": "k_nll_dense" if name == "dense" else "k_nll_compact",
                                          "achieved": nbytes / (k * 1e-3) * 1e-9, "unit": "GB/s", "traffic": None}}
    mc.set_path(B.PATH_CACHED_COMPACT)                 # gradient from the compact cache + Gram matrix (k_grad_compact)
    for t in range(3):
        mc.nll_grad(pc[t])
    kms = []
    barrier()
    t0 = time.perf_counter()
    for t in range(sub_steps):
        nll_cg, grad_c = mc.nll_grad(pc[args.warmup + t % args.steps])
        kms.append(mc.last_kernel_ms())
    barrier()
    wall = (time.perf_counter() - t0) / sub_steps
    cached_info["compact_grad"] = {"ms_per_call": 1e3 * wall, "kernel_ms": float(np.mean(kms)),
                                   "events_per_s": n_ev * world / wall, "nll": nll_cg, "n_grad": int(grad_c.size)}
    mc.set_path(B.PATH_RECOMPUTE)
    cached_info["recompute_same_model_nll"] = mc.nll(pc[args.warmup + (sub_steps - 1) % args.steps])
    mc.close()

    if rank == 0:
        time.sleep(0.2)
        sampler.stop()
    clocks = sampler.summary(w0, w1) if rank == 0 else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel of the step (k_nll_recompute): plain FP64 ALU work -----------------------------
    peak, peak_3reg = B.measure_fp64_peak(local, 3.0)
    fl = flops_per_point(cfg.resonances) * (n_ev + n_norm)
    k_ms = float(np.mean(kernel_ms))
    achieved = fl / (k_ms * 1e-3) * 1e-12
    nominal = None
    if clocks and clocks.get("sm_max_mhz"):
        nominal = 148 * 64 * 2 * clocks["sm_max_mhz"] * 1e6 * 1e-12
    roofline = {"bound": "alu", "kernel": "k_nll_recompute", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get((n_ev, n_norm)),
                "traffic_source": "profiles/r1_k_nll_recompute_ncu.md (ncu --set full, bytes per launch); algorithmic bytes "
                                  "per launch = 18 B x events + 26 B x weighted normalisation points (s12, s13, (w), 2-byte segment pair)",
                "peak_source": "measured on this GPU by mipwa_measure_fp64_peak (register-resident DFMA, 2 s sustained); "
                               "MEASURED_PEAKS.json has no FP64 entry; DESIGN.md section 6 derives the nominal peak",
                "nominal_peak": nominal, "flops_per_point": flops_per_point(cfg.resonances),
                "points_per_launch": n_ev + n_norm, "kernel_ms": k_ms,
                "executed_flops_per_point": NCU_EXECUTED_FLOPS_PER_POINT.get((n_ev, n_norm)),
                "algorithmic_bytes": 18.0 * n_ev + 26.0 * n_norm,
                "hbm_gbs": (18.0 * n_ev + 26.0 * n_norm) / (k_ms * 1e-3) * 1e-9}
    hbm_peak, hbm_src = 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_peak, hbm_src = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy, read+write)"
    except (OSError, KeyError, ValueError):
        pass
    for name in ("dense", "compact"):
        r = cached_info[name]["roofline"]
        r.update(peak=hbm_peak, frac=r["achieved"] / hbm_peak, peak_source=hbm_src)

    cpu = None
    if world == 1:
        cpu = time_oracle(cfg, min(n_ev, 4_000_000), min(n_norm, 4_000_000), 3, 1)

    total_events = n_ev * world
    line = {"metric": METRIC, "value": total_events / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload, events_per_gpu=n_ev, norm_points_per_gpu=n_norm,
                           l2="inputs read per step (18 B x 10M events + 26 B x 10M weighted normalisation points = 440 MB) exceed the "
                              "126 MB L2; no flush needed",
                           parallelism=f"dp{world} (events and normalisation points sharded; 3 doubles all-gathered per call)"),
            "nll_evals_per_s": 1e3 / ms_step, "points_per_s": (n_ev + n_norm) * world / (ms_step * 1e-3),
            "nll": nll, "clocks": clocks, "gpu_launches": int(launches) * world,
            "e2e": {"value": total_events / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                    "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * e2e_s, "nll": nll_e2e,
                    "what": "mipwa_set_events + mipwa_set_norm_points from pinned HOST arrays + mipwa_nll, every step"},
            "fit_step": {"ms_per_call": 1e3 * fit_step_s, "nll_evals_per_s": 1.0 / fit_step_s,
                         "what": "wall clock of mipwa_nll(host params) -> host fp64 with events resident (what a minimiser sees)"},
            "prepare_s": t_prep, "roofline": roofline, "grad": grad_info, "mixture": mix_info, "hybrid": hybrid_info, "cached": cached_info, "cpu_baseline": cpu, "input_generation_s": t_gen, "wall_ms_per_step": 1e3 * (w1 - w0) / args.steps}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---- secondary measurements behind the numbers in BASELINE.md / profiles (not the driver's bench line) --------------
def run_probe(args):
    """--probe resonances | hybrid | recompute-shape | grid-bias | sweep4 | latency : prints one JSON line per row (kernel times: CUDA events in the library,
    median over the calls after warm-up).  Phase-space points stand in for events where only the work per point
    matters; every mode cross-checks its NLL against another path."""
    import torch
    from paper_1703_03284_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --probe needs a CUDA device")

    def timed(m, p, calls=25, skip=5, grad=False):
        ms, v = [], None
        for _ in range(calls):
            v = m.nll_grad(p)[0] if grad else m.nll(p)
            ms.append(m.last_kernel_ms())
        return float(np.median(ms[skip:])), v

    if args.probe == "resonances":
        # recompute kernel time against the number and spin of the resonances, 10 M + 10 M points, N = 50:
        # the marginal cost of one resonance against the 2 clk per FP64 instruction of the pipe
        c = I.Config(3)
        n = args.events or 10_000_000
        e12, e13 = I.phase_space_points(n, c.key(7)); g12, g13 = I.phase_space_points(n, c.key(8))
        d = [torch.from_numpy(a).cuda() for a in (e12, e13, g12, g13)]
        L1 = [I._res(*I.RHO770), I._res(*I.RHO1450), I._res(*I.SYN_A), I._res(*I.SYN_C)]
        L2 = [I._res(*I.F2_1270), I._res(*I.SYN_B)]
        for name, res in (("R=0", []), ("1xL1", L1[:1]), ("2xL1", L1[:2]), ("3xL1", L1[:3]), ("4xL1", L1[:4]),
                          ("1xL2", L2[:1]), ("2xL2", L2[:2]), ("2xL1+1xL2", L1[:2] + L2[:1])):
            m = B.Mipwa(c.kin, c.knots, res)
            m.set_events(d[0], d[1]); m.set_norm_points(d[2], d[3], None); m.set_path(B.PATH_RECOMPUTE)
            m.prepare(); m.enable_timing(True)
            p = np.concatenate([c.truth[:100], np.tile([1.0, 0.3], len(res))])
            k, v = timed(m, p)
            print(json.dumps({"probe": "resonances", "model": name, "points": 2 * n, "kernel_ms": k, "nll": v,
                              "clk_per_warp_point_per_smsp_at_1965MHz": k * 1e-3 * 1.965e9 * 592 / (2 * n / 32)}), flush=True)
            m.close()
    elif args.probe == "hybrid":
        # the rule behind MIPWA_PATH_AUTO when some shapes float: rho(770) floating + k fixed-shape resonances,
        # full recompute against the hybrid path (fixed terms streamed from the per-point cache), 10 M + 10 M points
        c = I.Config(3)
        n = args.events or 10_000_000
        e12, e13 = I.phase_space_points(n, c.key(7)); g12, g13 = I.phase_space_points(n, c.key(8))
        d = [torch.from_numpy(a).cuda() for a in (e12, e13, g12, g13)]
        fixed = [I._res(*I.RHO1450), I._res(*I.F2_1270), I._res(*I.SYN_A), I._res(*I.SYN_B), I._res(*I.SYN_C)]
        for k in range(1, 6):
            res = [I._res(*I.RHO770, shape_floats=1)] + fixed[:k]
            m = B.Mipwa(c.kin, c.knots, res)
            m.set_events(d[0], d[1]); m.set_norm_points(d[2], d[3], None)
            m.prepare(); m.enable_timing(True)
            p = np.concatenate([c.truth[:100], np.tile([1.0, 0.3], len(res)), [0.775, 0.149]])
            row = {"probe": "hybrid", "fixed": k, "spins": [r["spin"] for r in res], "points": 2 * n}
            for name, path in (("recompute", B.PATH_RECOMPUTE), ("hybrid", B.PATH_HYBRID), ("auto", B.PATH_AUTO)):
                try:
                    m.set_path(path)
                    row[name + "_ms"], row[name + "_nll"] = timed(m, p)
                except B.MipwaError as e:
                    row[name + "_ms"] = None
            print(json.dumps(row), flush=True)
            m.close()
    elif args.probe == "recompute-shape":
        # kernel time of k_nll_recompute (value) and k_grad_recompute at configs[3]'s model on 10 M + 10 M weighted,
        # cell-sorted phase-space points; MIPWA_LIB_PATH selects a library rebuilt with other -DMIPWA_REC_* switches
        # (profiles/r1_recompute_shape.md)
        c = I.Config(3)
        n = args.events or 10_000_000
        e12, e13 = I.phase_space_points(n, c.key(7)); g12, g13 = I.phase_space_points(n, c.key(8))
        w = np.full(n, 5.06 / n)
        d = [torch.from_numpy(a).cuda() for a in (e12, e13, g12, g13, w)]
        m = B.Mipwa(c.kin, c.knots, c.resonances)
        m.set_events(d[0], d[1]); m.set_norm_points(d[2], d[3], d[4]); m.set_path(B.PATH_RECOMPUTE)
        m.prepare(); m.enable_timing(True)
        k, v = timed(m, c.perturbed(0), calls=60, skip=10)
        kg, vg = timed(m, c.perturbed(0), calls=30, skip=10, grad=True)
        print(json.dumps({"probe": "recompute-shape", "library": os.environ.get("MIPWA_LIB_PATH", "default"),
                          "points": 2 * n, "kernel_ms": k, "grad_kernel_ms": kg, "nll": v, "nll_grad_path": vg}), flush=True)
        m.close()
    elif args.probe == "grid-bias":
        # The paper's own experiment (PAPER.md:47, :61 Fig. 2, :49-55 Table 1) as far as it is described: a 100 K-event
        # toy of D+ -> K+K+K- (40 knots + phi(1020), config 5 of inputs.py; the parameter values are this repo's, the
        # paper prints none) generated from the PDF, then unbinned maximum-likelihood fits of all knot values and the
        # phi(1020) coefficient with the normalisation integral on grids of spacing 0.01 / 0.004 / 0.001 GeV^2.
        # scipy's L-BFGS-B is the caller (the minimiser is outside the hot path); a_0 and phi_0 are fixed (global
        # scale and phase are not constrained by the likelihood).  Reported: fitted - input knot values and the
        # wall-clock time of the whole fit.
        from scipy.optimize import minimize
        c = I.Config(5)
        m = B.Mipwa(c.kin, c.knots, c.resonances)

        t0 = time.perf_counter()
        e12, e13, _ = m.generate(c.truth, c.key(I.S_EVENTS), c.n_ev, n_side=2048, n_coarse=128, device=True)
        torch.cuda.synchronize()
        gen_s = time.perf_counter() - t0
        d_ev = [e12, e13]
        lo, hi = I.s_limits(c.kin)
        N = c.N
        free = np.ones(c.n_params, dtype=bool)
        free[0] = free[N] = False
        x0 = c.truth + 0.1 * I.normals(c.key(11), 0, c.n_params)
        x0[~free] = c.truth[~free]
        fits = {}
        for spacing in (0.01, 0.004, 0.001):
            n_side = int(round((hi - lo) / spacing))
            g12, g13, w = I.grid_points(n_side, c.kin)
            d_nm = [torch.from_numpy(a).cuda() for a in (g12, g13, w)]
            m.set_events(d_ev[0], d_ev[1]); m.set_norm_points(d_nm[0], d_nm[1], d_nm[2]); m.prepare()
            calls = [0]

            def fun(x):
                p = c.truth.copy(); p[free] = x
                v, g = m.nll_grad(p)
                calls[0] += 1
                return v, g[free]
            nll_truth = m.nll(c.truth)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            res = minimize(fun, x0[free], jac=True, method="L-BFGS-B",
                           options=dict(maxiter=5000, maxfun=20000, ftol=1e-15, gtol=1e-7))
            fit_s = time.perf_counter() - t0
            fit = c.truth.copy(); fit[free] = res.x
            da = fit[:N] - c.truth[:N]
            dphi = fit[N:2 * N] - c.truth[N:2 * N]
            fits[spacing] = fit
            # analytic Hessian at the minimum (mipwa_nll_hessian).  The knot errors are strongly correlated (a_0 at the
            # threshold anchors the common scale weakly), so the closure check is the quadratic form
            # d^T H d of d = fit - truth, which should equal 2 (NLL(truth) - NLL(fit)) and follow chi^2(n_free).
            _, _, H = m.nll_hessian(fit)
            Hf = H[np.ix_(free, free)]
            dfree = (fit - c.truth)[free]
            sig = np.sqrt(np.diag(np.linalg.inv(Hf)))
            print(json.dumps({"probe": "grid-bias", "spacing_gev2": spacing, "grid_cells_inside": int(g12.size),
                              "n_ev": int(e12.numel()), "n_free": int(free.sum()), "fit_wall_s": fit_s,
                              "nll_grad_calls": calls[0], "ms_per_call_incl_minimiser": fit_s / max(calls[0], 1) * 1e3,
                              "converged": bool(res.success), "nll_fit_minus_truth": float(res.fun - nll_truth),
                              "median_abs_da": float(np.median(np.abs(da))), "rms_da": float(np.sqrt(np.mean(da ** 2))),
                              "median_abs_dphi": float(np.median(np.abs(dphi))), "rms_dphi": float(np.sqrt(np.mean(dphi ** 2))),
                              "d_phi1020_mag": float(fit[2 * N] - c.truth[2 * N]),
                              "chi2_quadratic_form": float(dfree @ Hf @ dfree), "two_delta_nll": float(2 * (nll_truth - res.fun)),
                              "median_sigma_a": float(np.median(sig[:N - 1])),
                              "hessian_positive_definite": bool(np.all(np.linalg.eigvalsh(Hf) > 0)),
                              "event_generation_s": gen_s}), flush=True)
        # the same sample in every fit, so the statistical scatter is common: the shift against the finest grid is
        # the bias the coarser normalisation grid causes (the paper's Fig. 2 observation)
        for spacing in (0.01, 0.004):
            d = fits[spacing] - fits[0.001]
            print(json.dumps({"probe": "grid-bias", "shift_against_spacing_0.001": spacing,
                              "rms_da": float(np.sqrt(np.mean(d[:N] ** 2))), "max_abs_da": float(np.max(np.abs(d[:N]))),
                              "rms_dphi": float(np.sqrt(np.mean(d[N:2 * N] ** 2))),
                              "max_abs_dphi": float(np.max(np.abs(d[N:2 * N])))}), flush=True)
        m.close()
    elif args.probe == "sweep4":
        # BASELINE.json configs[4]: K = 56 cached paths against the event count (default 1 M .. 100 M), 10 M-point Gram
        c = I.Config(4)
        sizes = [args.events] if args.events else [1_000_000, 2_000_000, 5_000_000, 10_000_000, 20_000_000,
                                                   50_000_000, 100_000_000]
        g12, g13 = I.phase_space_points(args.norm_points or 10_000_000, c.key(8))
        dg = [torch.from_numpy(a).cuda() for a in (g12, g13)]
        E12, E13 = I.phase_space_points(max(sizes), c.key(7), chunk=1 << 24)
        m = B.Mipwa(c.kin, c.knots, c.resonances)
        m.set_norm_points(dg[0], dg[1], None); m.enable_timing(True)
        for n in sizes:
            de = [torch.from_numpy(E12[:n]).cuda(), torch.from_numpy(E13[:n]).cuda()]
            m.set_events(de[0], de[1]); m.prepare()
            row = {"probe": "sweep4", "n_ev": n, "K": c.N + c.R}
            for name, path in (("dense", B.PATH_CACHED), ("compact", B.PATH_CACHED_COMPACT)):
                m.set_path(path)
                t0 = time.perf_counter(); m.nll(c.truth); setup = time.perf_counter() - t0
                k, v = timed(m, c.perturbed(1), calls=22, skip=2)
                byt = m.basis_bytes()
                row[name] = {"kernel_ms": k, "cache_GB": byt / 1e9, "GB_per_s": byt / k * 1e-6, "events_per_s": n / k * 1e3,
                             "evals_per_s": 1e3 / k, "first_call_s": setup, "nll": v}
            if n <= 20_000_000:
                m.set_path(B.PATH_RECOMPUTE)
                row["recompute_nll"] = m.nll(c.perturbed(1))
            print(json.dumps(row), flush=True)
            del de
            torch.cuda.empty_cache()
        m.close()
    elif args.probe == "latency":
        # wall clock per call (timing events off) and kernel time at the small configs and at the paper's scale
        for idx, n_ev, n_norm in ((0, None, None), (1, None, None), (2, 100_000, 1_000_000), (2, None, None),
                                  (5, None, None)):       # 5 = the paper's own toy (K+K+K-, 100 K events, 918^2 grid)
            c = I.Config(idx, n_ev=n_ev, n_norm=n_norm)
            e12, e13 = I.phase_space_points(c.n_ev, c.key(7), c.kin)
            g12, g13, w = c.norm_points()
            d = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (e12, e13, g12, g13, w)]
            m = B.Mipwa(c.kin, c.knots, c.resonances)
            m.set_events(d[0], d[1]); m.set_norm_points(d[2], d[3], d[4]); m.prepare()
            ps = [c.perturbed(t) for t in range(120)]
            row = {"probe": "latency", "config": idx, "n_ev": c.n_ev, "n_norm": int(g12.size)}
            for name, path, grad in (("recompute", B.PATH_RECOMPUTE, False), ("compact", B.PATH_CACHED_COMPACT, False),
                                     ("dense", B.PATH_CACHED, False), ("grad_recompute", B.PATH_RECOMPUTE, True),
                                     ("grad_compact", B.PATH_CACHED_COMPACT, True)):
                m.set_path(path)
                f = (lambda q: m.nll_grad(q)[0]) if grad else m.nll
                m.enable_timing(True)
                km = []
                for t in range(20):
                    f(ps[t]); km.append(m.last_kernel_ms())
                m.enable_timing(False)
                t0 = time.perf_counter()
                for t in range(100):
                    f(ps[20 + t])
                row[name] = {"wall_us": (time.perf_counter() - t0) / 100 * 1e6, "kernel_us": float(np.median(km[5:])) * 1e3}
            print(json.dumps(row), flush=True)
            m.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--events", type=int, default=None)
    ap.add_argument("--norm-points", type=int, default=None)
    ap.add_argument("--probe", default=None, choices=["resonances", "hybrid", "recompute-shape", "grid-bias", "sweep4", "latency"])
    args = ap.parse_args()
    if args.probe:
        return run_probe(args)
    args.warmup = max(args.warmup, 3)
    cfg = I.Config(args.config, n_ev=args.events, n_norm=args.norm_points)
    workload = {"workload": f"BASELINE.json configs[{args.config}]: {cfg.N} knots + "
                            + " + ".join(f"BW(m={r['mass']},G={r['width']},L={r['spin']}{',floating' if r['shape_floats'] else ''})"
                                         for r in cfg.resonances)
                            + f"; {cfg.n_ev} events + {cfg.norm_size} normalisation points per GPU; NLL value, full recompute",
                "n_knots": cfg.N, "n_resonances": cfg.R, "n_params": int(cfg.n_params)}
    if args.impl == "reference":
        run_reference(args, cfg, workload)
    else:
        run_ours(args, cfg, workload)


if __name__ == "__main__":
    main()
