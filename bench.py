#!/usr/bin/env python
"""bench.py -- throughput of the LSD window-verification hot path on B200.

A "step" is one pass of the whole hot path over one window of K draft steps:
draft rollout -> window-shared neighbour lists -> batched target forces -> transport map + first-reject scan ->
override/commit -> rollback.  `value` = atom-steps verified per second (K * N * steps * n_gpus / time);
committed ("accepted target-exact") MD steps/s is reported beside it.  One JSON line on stdout (rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference] [--no-side]

The line of the default run also carries `all_workloads` (the other BASELINE.json workloads, a few windows each, same
measurement code), `measured_peaks` (fp32 / fp64 FMA peaks measured by a kernel of the library, next to the driver's
MEASURED_PEAKS.json), a three-term roofline of the batched force evaluation (tensor, HBM, special-function unit) and a
labelled `acceptance_variant` (draft = target with the gap shrunk until Eq. 9 gives beta ~ 0.1), and `async_depth` (committed steps/s
with 0 / 1 / 3 speculative windows drafted ahead on the second stream, Alg. 2 on one device).

Multi-GPU (weak scaling): every rank runs an independent replica of the workload (its own seed); there is no
data-path collective.  --impl reference times the CPU oracle (oracle/, fp64, as it stands).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "batched force-eval atom-steps/s (whole verified window; accepted target-exact MD steps/s beside it)"
UNIT = "atom-steps/s"

# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel from one ncu capture of this
# command (per workload and arithmetic type; null where no capture is committed).  Not measured by this run: a run under a
# profiler is never a bench run; `roofline.traffic_source` names the committed capture the figure comes from.  The third field is
# the identity of the kernel the capture was taken on, as lsd_get_edge_launch_info reports it (kernel, network width, threads per
# block; None for the fp32 kernels, which have one instantiation per width): when the kernel that runs differs, the figure is
# stale and `traffic` is reported as null.
NCU_TRAFFIC = {("cfg5", "bf16"): (1.6515e9 + 0.1405e9, "profiles/r2_traffic.md (k_edge_rows<1,2>)", ("k_edge_rows", 128, 512)),
               ("cfg4", "bf16"): (0.2073e9 + 0.0250e9, "profiles/r2_traffic.md (k_edge_rows<1,2>)", ("k_edge_rows", 128, 512)),
               ("cfg4", "f32"): (0.2750e9 + 0.0565e9, "profiles/r2_traffic.md (k_edge<128,bwd>)", None),
               ("cfg3", "bf16"): (0.05723e9 + 0.00023e9, "profiles/r3_traffic_cfg3_bf16.md (k_edge_rows<64,1,1>)", ("k_edge_rows_narrow", 64, 512)),
               ("cfg3", "f32"): (0.0635e9 + 0.0002e9, "profiles/r2_traffic.md (k_edge<64,bwd>)", None)}


def traffic_for(name, dtype, running):
    """(traffic, source) for the roofline block; `running` = (kernel, width, threads) of the dominant kernel of this run or None."""
    tr = NCU_TRAFFIC.get((name, dtype))
    if tr is None:
        return None, None
    if tr[2] is not None and running is not None and tuple(tr[2]) != tuple(running):
        return None, f"stale: {tr[1]} was captured on {tr[2]}, this run launched {tuple(running)}"
    return tr[0], tr[1]


# the workloads of BASELINE.json with the arithmetic types it lists for them (north_star: "report throughput on the five synthetic
# workloads"): the default run times --workload in full and the others for a few windows each (`all_workloads`)
ALL_WORKLOADS = [("cfg1", None), ("cfg2", "fp32"), ("cfg3", "fp32"), ("cfg3", "bf16"), ("cfg4", "fp32"), ("cfg4", "bf16"), ("cfg5", "bf16")]
SIDE_STEPS = 8

# bounded oracle samples: same per-atom cost as the full workload, sized for ~10-30 s of CPU work
CPU_SAMPLES = {
    "cfg1": dict(kw={}, K=4, windows=4000),
    "cfg2": dict(kw={}, K=16, windows=150),
    "cfg3": dict(kw={"n_grid": 7}, K=4, windows=12),
    "cfg4": dict(kw={"n_atoms": 1000}, K=4, windows=4),
    "cfg5": dict(kw={"cells": (6, 6, 6)}, K=4, windows=4),
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16=d.get("bf16_tflops_sustained", d["bf16_tflops"]), bf16_burst=d["bf16_tflops"],
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm_gbs=6650.0, bf16=1400.0, bf16_burst=1590.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i", str(self.index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7), ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=sorted(reasons), samples=len(sm))


def cpu_baseline(name, steps=1):
    """The oracle as it stands, on the host cores, on a bounded sample of the workload."""
    import lsd_inputs as L
    import oracle
    s = CPU_SAMPLES[name]
    w = L.make_workload(name, **s["kw"])
    p0 = oracle.initial_momenta(w)
    oracle.lsd_window(w, w.q0, p0, 0, K=1, debug=False)                 # warm (build + page-in)
    q, p, n = w.q0, p0, 0
    atom_steps = committed = 0
    t0 = time.perf_counter()
    for _ in range(steps * s["windows"]):
        r = oracle.lsd_window(w, q, p, n, K=s["K"], debug=True)         # debug=True: all K target evaluations, like the batched GPU call
        q, p, n = r["q"], r["p"], n + r["n_commit"]
        atom_steps += s["K"] * w.n_atoms
        committed += r["n_commit"]
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return dict(value=atom_steps / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{name} scaled to {w.n_atoms} atoms ({s['kw'] or 'full size'}), {steps * s['windows']} window(s) of K={s['K']}, fp64, {dt:.1f} s",
                committed_md_steps_per_s=committed / dt, seconds=dt)


def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    per = []
    base = None
    for _ in range(args.warmup if args.warmup < 1 else 1):
        cpu_baseline(args.workload, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        base = cpu_baseline(args.workload, 1)
        per.append(base["value"])
    dt = time.perf_counter() - t0
    val = float(np.mean(per))
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / max(args.steps, 1), higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, note="CPU oracle (oracle/lsd_oracle.c) on a bounded sample; each step = one sample"),
                cpu_baseline=dict(value=val, unit=UNIT, cores=base["cores"], kind="oracle", sample=base["sample"]),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def reduce_over_ranks(ms, committed, device=None):
    """Multi-GPU aggregation (independent replicas, no data-path collective): the step time is the MAX over
    ranks, committed steps are SUMMED.  Works on any initialised process group (nccl on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(committed)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(committed)], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), float(c.item())


def replica_seed(base_seed, rank):
    """Every rank runs its own replica of the workload: same system, different noise stream."""
    return int(base_seed) + 1000 * int(rank)




def _sync_all(torch, world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


def measure_workload(env, name, precision, steps, warmup, full, ec=0, overlap=0):
    """One workload through the public C ABI.  env: dict(torch, L, P, rank, world, local, stream, flush, peaks, fma_peaks).
    full: also the serial baselines / adaptive lookahead blocks (headline workload only).  Returns the fields of a bench line."""
    torch, L, P = env["torch"], env["L"], env["P"]
    rank, world, local, stream, peaks = env["rank"], env["world"], env["local"], env["stream"], env["peaks"]
    w = L.make_workload(name)
    K, N = w.K, w.n_atoms
    prec = {"fp32": P.LSD_FP32, "bf16": P.LSD_BF16_TC, None: None}[precision]
    ctx = P.context_from_workload(w, precision=prec, seed=replica_seed(w.seed, rank))
    if ec:
        P.lsd_set_error_correction(ctx.h, True)
    tgt = w.target.mlip
    work_bytes = 0 if tgt is None else 4 * N * K * tgt.width * (5 + 2 * tgt.n_blocks)
    need_flush = work_bytes < 2 * 126e6
    skin = [float(w.skin)]

    def one_window():
        if overlap:
            P.lsd_run(ctx.h, K, K, overlap=True, stream=stream)
            return None
        try:
            return ctx.window(K, stream)
        except P.LsdError as e:                          # as lsd_run does: a skin violation / row overflow is answered by larger lists, never ignored
            if e.status not in (-6, -7):
                raise
            if e.status == -7:
                skin[0] *= 2.0
            P.lsd_set_skin(ctx.h, skin[0])
            return ctx.window(K, stream)

    def timed_pass():
        """`steps` timed windows, CUDA events on the launching stream around every window (L2 flush outside the events)."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for s in range(steps):
            if need_flush:
                with torch.cuda.stream(stream):
                    env["flush"].fill_(s & 0xFF)
            ev[s][0].record(stream)
            one_window()
            ev[s][1].record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev)

    for _ in range(warmup):
        one_window()
    torch.cuda.synchronize()
    st0 = P.lsd_get_stats(ctx.h)
    launches_before = P.lsd_launch_count(ctx.h)
    sampler = ClockSampler(local)
    _sync_all(torch, world)
    sampler.start()
    ms = timed_pass()                                   # the reported value: no per-kernel events, CUDA graphs replayed
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    launches = P.lsd_launch_count(ctx.h) - launches_before
    st1 = P.lsd_get_stats(ctx.h)
    committed = st1["committed_steps"] - st0["committed_steps"]
    windows = st1["windows"] - st0["windows"]            # == steps unless --overlap (lsd_run runs as many windows as it takes to commit K steps)
    # second, identically configured pass with the library's per-kernel CUDA events on (they bypass graph replay and cost
    # ~2 us per launch, which is why the value above is not taken from this pass): stage times, roofline
    P.lsd_profile(ctx.h, True)
    ms_prof = timed_pass()
    clocks = sampler.stop()
    prof = P.lsd_get_profile(ctx.h)
    P.lsd_profile(ctx.h, False)
    edges = P.lsd_get_edge_count(ctx.h, P.LSD_TARGET, 0, K) if tgt is not None else 0
    ms, committed_all = reduce_over_ranks(ms, committed, device="cuda")
    value = K * N * windows * world / (ms * 1e-3)
    out = dict(workload=name, n_atoms=N, window_K=K, ms_per_step=ms / steps, value=value, windows_timed=int(windows),
               committed_md_steps_per_s=committed_all / (ms * 1e-3), committed_per_window=committed_all / max(windows * world, 1),
               clocks=clocks, gpu_launches=int(launches), need_flush=need_flush, skin=skin[0])

    speedup = None
    if full:
        # ---- the serial baselines of the paper's speed-up definition: plain Langevin with the target alone and
        # with the draft alone, same kernels, same stream; c = t_draft / t_target (:155); synchronous-window prediction Eq. 21
        # (:559) without the bonus step (R3).  Context only: alpha and c are those of the synthetic models.
        def plain_rate(which):
            nst = K * max(1, min(steps, 8))
            P.lsd_plain_langevin(ctx.h, which, K, stream)                      # warm (graph capture on the second chunk)
            P.lsd_plain_langevin(ctx.h, which, K, stream)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            P.lsd_plain_langevin(ctx.h, which, nst, stream)
            b.record(stream)
            torch.cuda.synchronize()
            return nst / (a.elapsed_time(b) * 1e-3)
        st_all = P.lsd_get_stats(ctx.h)
        alpha = 1.0 - st_all["rejections"] / max(st_all["committed_steps"], 1)
        plain_t, plain_d = plain_rate(P.LSD_TARGET), plain_rate(P.LSD_DRAFT)
        cfrac = plain_t / plain_d
        pred = (K if alpha >= 1.0 else (1.0 - alpha ** K) / (1.0 - alpha)) / (K * cfrac + 1.0)
        committed_rate = committed_all / world / (ms * 1e-3)
        speedup = dict(plain_target_md_steps_per_s=plain_t, plain_draft_md_steps_per_s=plain_d, cost_fraction_c=cfrac, acceptance_alpha=alpha,
                       measured_speedup_vs_plain_target=committed_rate / plain_t, eq21_sync_prediction_K_target_instances=pred,
                       note="one B200 evaluates the K target calls as ONE batched call, not on K instances: Eq. 21 is the paper's multi-GPU model")
        # ---- adaptive lookahead (lsd_run with K = 0): committed steps/s when the window length is chosen by
        # measurement instead of being the configuration's K
        for key, ov in (("adaptive_K", False), ("adaptive_K_overlap", True)):     # without / with the speculative second-stream rollout
            P.lsd_run(ctx.h, 40 * K, 0, overlap=ov, stream=stream)          # exploration
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0 = P.lsd_get_stats(ctx.h)["committed_steps"]
            a0.record(stream)
            P.lsd_run(ctx.h, 20 * K, 0, overlap=ov, stream=stream)
            a1.record(stream)
            torch.cuda.synchronize()
            ad_rate = (P.lsd_get_stats(ctx.h)["committed_steps"] - c0) / (a0.elapsed_time(a1) * 1e-3)
            speedup[key] = dict(committed_md_steps_per_s=ad_rate, settled_K=P.lsd_get_adaptive_k(ctx.h), speedup_vs_plain_target=ad_rate / plain_t)
    out["speedup"] = speedup

    # ---- end-to-end through the C ABI with HOST buffers (pinned): upload x_n, run the window, read x_{n+commit} back
    qh = torch.empty((3, N), dtype=torch.float64).pin_memory()
    ph = torch.empty((3, N), dtype=torch.float64).pin_memory()
    step0 = P.lsd_get_state(ctx.h, qh.numpy(), ph.numpy())
    _sync_all(torch, world)
    t0 = time.perf_counter()
    for s in range(steps):
        P.lsd_set_state(ctx.h, qh.numpy(), ph.numpy(), step0)
        ctx.window(K, stream)
        step0 = P.lsd_get_state(ctx.h, qh.numpy(), ph.numpy())
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s, _ = reduce_over_ranks(e2e_s, 0, device="cuda")
    out["e2e"] = dict(value=K * N * steps * world / e2e_s, unit=UNIT, h2d_bytes_per_step=2 * 3 * N * 8, d2h_bytes_per_step=2 * 3 * N * 8 + 8,
                      ms_per_step=1e3 * e2e_s / steps)
    out["roofline"], out["dtype"] = build_roofline(env, w, name, precision, prec, ctx, prof, edges, steps, ms_prof)
    ctx.close()
    return out


def build_roofline(env, w, name, precision, prec, ctx, prof, edges, steps, ms_prof):
    """Roofline block of one workload from the profiled pass: dominant kernel against the peak of the unit
    north_star names for it, plus the three-term roofline of the whole batched force evaluation."""
    P, peaks = env["P"], env["peaks"]
    fp32_peak, fp64_peak = env["fma_peaks"]
    tgt = w.target.mlip
    K, N = w.K, w.n_atoms
    stage = {k: v["ms"] / steps for k, v in prof.items() if v["launches"]}
    if tgt is None:
        # cfg1: fp64 pair potentials only.  Dominant kernel class = k_prior (draft: K launches of one state, target: one launch of K states)
        pe = P.lsd_get_edge_count(ctx.h, P.LSD_TARGET, 1, K)
        flops = 2 * pe * 60.0                                              # ~60 fp64 flop per directed pair term; draft + target
        pr = prof["prior"]
        ach = flops * steps / (pr["ms"] * 1e-3) / 1e12 if pr["ms"] > 0 else 0.0
        return dict(bound="alu", achieved=ach, peak=fp64_peak, unit="TFLOP/s", frac=ach / fp64_peak, traffic=None, traffic_source=None,
                    kernel="k_prior (fp64 pair terms, draft + target launches of a window)", avg_launch_ms=pr["ms"] / max(pr["launches"], 1),
                    launches=pr["launches"], algorithmic_flops_per_window=flops, peak_note="fp64 FMA peak measured by lsd_measure_fma_peak in this run",
                    note="launch-latency-bound: 256 atom-steps per window; the fraction only shows how far from any throughput limit this size is",
                    share_of_step=pr["ms"] / ms_prof if ms_prof > 0 else None, profiled_ms_per_step=ms_prof / steps, stage_ms_per_step=stage), "f64"
    F, R, T = tgt.width, tgt.n_rbf, tgt.n_blocks
    eb = prof["mlip_edge_bwd"]
    flops_per_launch = edges * (2 * R * F + 2 * F * F + 6 * F)            # strict algorithmic count of the backward edge pass
    avg_ms = eb["ms"] / max(eb["launches"], 1)
    achieved = flops_per_launch / (avg_ms * 1e-3) / 1e12 if avg_ms > 0 else 0.0
    use_tc = (prec if prec is not None else (P.LSD_BF16_TC if w.precision == "bf16" else P.LSD_FP32)) == P.LSD_BF16_TC and P.lsd_tc_enabled(ctx.h)
    if use_tc:
        bound, peak, dtype = "tensor", peaks["bf16"], "bf16"
        peak_note = f"bf16 dense sustained, {peaks['source']}"
        info_b, info_f = P.lsd_get_edge_launch_info(True), P.lsd_get_edge_launch_info(False)
        kernel = f"{info_b['kernel']} (grid {info_b['grid']} x {info_b['threads']} threads, {info_b['atoms_per_chunk']} atoms per chunk)"
        fwd_kernel = info_f["kernel"]
        running = (info_b["kernel"], info_b["width"], info_b["threads"])
    else:
        bound, dtype, peak = "alu", "f32", fp32_peak
        peak_note = "fp32 FMA peak measured by lsd_measure_fma_peak in this run"
        kernel, fwd_kernel = f"k_edge<{F},bwd>", f"k_edge<{F},fwd>"
        running = None
    mlip_ms = prof["mlip_edge_bwd"]["ms"] + prof["mlip_edge_fwd"]["ms"] + prof["mlip_dense"]["ms"]
    a2_ms = mlip_ms / steps
    # three-term roofline of the batched target force evaluation (a2) per window: strict tensor / FMA flops, algorithmic
    # HBM bytes, special-function-unit operations the kernels issue (one tanh per edge, channel and pass; R ex2 per edge and pass)
    strict_flops = edges * T * (2 * R * F + 2 * F * F + 8 * F)
    hbm_bytes = 24.0 * N * K + 4.0 * edges * 2 * T + 4.0 * F * N * K * 6 * T
    mufu_ops = edges * T * 2.0 * (F + R)
    sm_hz = (env["peaks"]["sm_max_mhz"]) * 1e6
    t_tensor = strict_flops / (peak * 1e12) * 1e3
    t_hbm = hbm_bytes / (peaks["hbm_gbs"] * 1e9) * 1e3
    t_sfu = mufu_ops / (16.0 * 148.0 * sm_hz) * 1e3
    terms = {"tensor" if use_tc else "fma": t_tensor, "hbm": t_hbm, "sfu": t_sfu}
    traffic, traffic_source = traffic_for(name, dtype, running)
    roofline = dict(bound=bound, achieved=achieved, peak=peak, unit="TFLOP/s", frac=achieved / peak,
                    traffic=traffic, traffic_source=traffic_source,
                    kernel=kernel + " (MLIP edge backward: filter value + tangent, cfconv adjoints)", avg_launch_ms=avg_ms, launches=eb["launches"],
                    algorithmic_flops_per_launch=flops_per_launch, directed_edges_per_window=edges, peak_note=peak_note,
                    share_of_step=eb["ms"] / ms_prof if ms_prof > 0 else None, profiled_ms_per_step=ms_prof / steps,
                    a2_strict_tflops=steps * strict_flops / (mlip_ms * 1e-3) / 1e12 if mlip_ms > 0 else None,
                    a2_directed_tflops=steps * edges * T * (2 * (2 * R * F + 2 * F * F) + 8 * F) / (mlip_ms * 1e-3) / 1e12 if mlip_ms > 0 else None,
                    kernel_executed_tflops=edges * 2 * (2 * R * F + 2 * F * F) / (avg_ms * 1e-3) / 1e12 if avg_ms > 0 else None,
                    a2_three_term=dict(t_tensor_ms=t_tensor if use_tc else None, t_fma_ms=None if use_tc else t_tensor, t_hbm_ms=t_hbm, t_sfu_ms=t_sfu,
                                       measured_ms=a2_ms, frac_of_slowest_term=max(terms.values()) / a2_ms if a2_ms > 0 else None,
                                       slowest_term=max(terms, key=terms.get), sfu_ops_per_window=mufu_ops, hbm_bytes_per_window=hbm_bytes,
                                       note="strict flops / measured peak; algorithmic bytes / measured HBM copy bandwidth; MUFU ops the kernels issue "
                                            "(edges x blocks x 2 passes x (F tanh + R ex2)) / (16 per clk per SM x 148 SMs x max SM clock)"),
                    stage_ms_per_step=stage)
    if use_tc and F == 128:
        # the other two kernel families of the width-128 tensor-core path, from the same profiled pass
        rows = K * N
        chain_bytes = rows * (2048 * T + 1024 + 1536 + 2560 * (T - 1))          # algorithmic bytes per row of the chain kernels
        dense_ms, fwd_ms = prof["mlip_dense"]["ms"] / steps, prof["mlip_edge_fwd"]["ms"] / steps
        roofline["other_kernels"] = dict(
            atom_chain=dict(bound="hbm", achieved=chain_bytes / (dense_ms * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                            frac=chain_bytes / (dense_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], ms_per_step=dense_ms,
                            note="k_atom_tc128<*> incl. the embedding kernel; ncu: profiles/r1_atom_tc128_cfg5.md"),
            edge_forward=dict(bound="tensor", achieved=edges * T * (2 * R * F + 2 * F * F) / (fwd_ms * 1e-3) / 1e12, peak=peaks["bf16"], unit="TFLOP/s",
                              frac=edges * T * (2 * R * F + 2 * F * F) / (fwd_ms * 1e-3) / 1e12 / peaks["bf16"], ms_per_step=fwd_ms,
                              note=f"{fwd_kernel}, executed filter flops (the strict count shares the value with the backward)"))
    return roofline, dtype


def async_depth_block(env, cases=(("cfg1", None, 0), ("cfg1", None, 1), ("cfg2", "fp32", 1), ("cfg4", "bf16", 1)), depths=(0, 1, 3), slots=4, windows=24):
    """Labelled side block (SURVEY.md 8(f) rank 3; Alg. 2 on one device, PAPER.md:555-566 Eq. 21 vs Eq. 22, :568-618): committed steps/s of
    lsd_run at the configuration's K with 0, 1 and 3 speculative windows kept drafted ahead on the second stream (ring of `slots` window
    slots), on the workloads whose acceptance is high enough for a speculative rollout to survive (EC = error correction, Alg. 3)."""
    torch, L, P, stream = env["torch"], env["L"], env["P"], env["stream"]
    out = {}
    for name, precision, ec in cases:
        w = L.make_workload(name)
        K = w.K
        prec = {"fp32": P.LSD_FP32, "bf16": P.LSD_BF16_TC, None: None}[precision]
        ctx = P.context_from_workload(w, precision=prec)
        P.lsd_set_window_slots(ctx.h, slots)
        if ec:
            P.lsd_set_error_correction(ctx.h, True)
        res = dict(window_K=K, window_slots=slots, error_correction=bool(ec), committed_md_steps_per_s={})
        for d in depths:
            P.lsd_run(ctx.h, 4 * K, K, overlap=d, stream=stream)           # warm (graph capture of every slot)
            st0 = P.lsd_get_stats(ctx.h)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            P.lsd_run(ctx.h, windows * K, K, overlap=d, stream=stream)
            a1.record(stream)
            torch.cuda.synchronize()
            st1 = P.lsd_get_stats(ctx.h)
            nc = st1["committed_steps"] - st0["committed_steps"]
            res["committed_md_steps_per_s"][str(d)] = nc / (a0.elapsed_time(a1) * 1e-3)
            res["acceptance_alpha"] = 1.0 - (st1["rejections"] - st0["rejections"]) / max(nc, 1)
        ctx.close()
        out[name + ("" if precision is None else "_" + precision) + ("_ec" if ec else "")] = res
    return out


def acceptance_variant(env, name, precision, target_beta=0.1, windows=6):
    """Labelled side block (last paragraph): the same workload with the draft / target gap shrunk until Eq. 9
    (beta = erf(|delta| / sqrt 8)) gives beta ~ target_beta per step, so that 'accepted target-exact MD steps/s' and the
    speculative second-stream rollout measure something other than 1 / t_window.  The draft is the TARGET potential with its network's
    energy scale changed by a factor (1 + eps); delta is linear in eps, so one probe window fixes eps.  c = t_draft / t_target = 1 here."""
    import dataclasses
    from scipy.special import erfinv
    torch, L, P, stream = env["torch"], env["L"], env["P"], env["stream"]
    w = L.make_workload(name)
    if w.target.mlip is None:
        return None
    K = w.K
    prec = {"fp32": P.LSD_FP32, "bf16": P.LSD_BF16_TC, None: None}[precision]

    def variant(eps):
        m = dataclasses.replace(w.target.mlip, alpha=w.target.mlip.alpha * (1.0 + eps))
        return dataclasses.replace(w, draft=dataclasses.replace(w.target, mlip=m))
    want = float(erfinv(target_beta)) * np.sqrt(8.0)                       # |delta| that gives the target rejection probability
    eps = 1e-2
    ctx = P.context_from_workload(variant(eps), precision=prec)
    ctx.window(K, stream)
    s2 = float(np.sqrt(np.mean(ctx.debug("S2", K))))
    ctx.close()
    eps *= want / max(s2, 1e-300)
    res = dict(label="NOT a BASELINE.json workload: draft = target with the network's energy scale x (1 + eps)", eps=eps, target_beta=target_beta)
    ctx = P.context_from_workload(variant(eps), precision=prec)
    for key, ov in (("sync", False), ("overlap", True)):
        P.lsd_run(ctx.h, 2 * K, K, overlap=ov, stream=stream)             # warm (graph capture)
        st0 = P.lsd_get_stats(ctx.h)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        P.lsd_run(ctx.h, windows * K, K, overlap=ov, stream=stream)
        a1.record(stream)
        torch.cuda.synchronize()
        st1 = P.lsd_get_stats(ctx.h)
        nc, nw = st1["committed_steps"] - st0["committed_steps"], st1["windows"] - st0["windows"]
        res[key] = dict(committed_md_steps_per_s=nc / (a0.elapsed_time(a1) * 1e-3), committed_per_window=nc / max(nw, 1), windows=int(nw),
                        measured_beta=(st1["rejections"] - st0["rejections"]) / max(nc, 1),
                        predicted_beta=(st1["beta_sum"] - st0["beta_sum"]) / max(nc, 1))
    P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, K, stream); P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, K, stream)
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record(stream)
    P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, 2 * K, stream)
    a1.record(stream)
    torch.cuda.synchronize()
    res["plain_target_md_steps_per_s"] = 2 * K / (a0.elapsed_time(a1) * 1e-3)
    res["note"] = ("one GPU and c = 1: the batched verification costs about K target evaluations and the rollout K more, so the ratio to the plain target "
                   "stays below 1; the block shows the acceptance statistics (measured vs Eq. 9) and what the second-stream rollout buys when windows are accepted")
    ctx.close()
    return res


def sweep_workload(L, cells, tau_fs, eps):
    """fcc Cu of cells^3 unit cells at the paper's Fig. 4 conditions (T = 1500 K, dt = 1 fs, friction time scale tau = 1 / gamma,
    PAPER.md:208-212) with the cfg5 potentials; draft = target with the network's energy scale x (1 + eps) (force error eps F_NN:
    the same per-atom error scale at every N, which is what Eq. 11 assumes)."""
    import dataclasses
    w = L.make_workload("cfg5", cells=(cells, cells, cells))
    m = dataclasses.replace(w.target.mlip, alpha=w.target.mlip.alpha * (1.0 + eps))
    return dataclasses.replace(w, draft=dataclasses.replace(w.target, mlip=m), temperature_K=1500.0, dt_fs=1.0, friction_per_fs=1.0 / tau_fs)


def run_sweep(args):
    """the FORM of Fig. 4 (PAPER.md:185 Eq. 11, :208-212): mean rejection rate R(K)/K over a segment of `--sweep-steps`
    committed steps against N and tau, compared with erf(sqrt(N tau / (N0 tau0)) erfinv(beta0)) where beta0 is the measured rate at
    (N0 = 500, tau0 = 1 ps) -- the paper's fit of epsilon at that point -- with and without speculative error correction.
    N starts at 256: the library keeps a single minimum image, i.e. box >= 2 (r_c + skin) = 13 A (R10)."""
    import torch
    from scipy.special import erf, erfinv
    import lsd_inputs as L
    import paper_2606_02455_b200 as P
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    P.load_library()
    stream = torch.cuda.Stream()
    K, nsteps, beta0_target = 8, args.sweep_steps, 0.3
    # one probe window at (N0, tau0) fixes eps: delta is linear in eps (Eq. 8), beta = erf(|delta| / sqrt 8) (Eq. 9)
    eps = 1e-2
    ctx = P.context_from_workload(sweep_workload(L, 5, 1000.0, eps), k_max=K, precision=P.LSD_BF16_TC)
    ctx.window(K, stream)
    eps *= float(erfinv(beta0_target)) * np.sqrt(8.0) / float(np.mean(np.sqrt(ctx.debug("S2", K))))
    ctx.close()
    rows = []
    for tau in (1000.0, 100.0):
        for cells in (4, 5, 6, 7, 8, 10):
            w = sweep_workload(L, cells, tau, eps)
            row = dict(N=w.n_atoms, tau_fs=tau)
            for key, ec in (("no_ec", False), ("ec", True)):
                ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_BF16_TC)
                if ec:
                    P.lsd_set_error_correction(ctx.h, True)
                P.lsd_run(ctx.h, 5 * K, K, overlap=False, stream=stream)            # equilibrate the EC cache / warm
                s0 = P.lsd_get_stats(ctx.h)
                t0 = time.perf_counter()
                P.lsd_run(ctx.h, nsteps, K, overlap=False, stream=stream)
                dt = time.perf_counter() - t0
                s1 = P.lsd_get_stats(ctx.h)
                nc = s1["committed_steps"] - s0["committed_steps"]
                row[key] = dict(rejected=int(s1["rejections"] - s0["rejections"]), steps=int(nc), rate=(s1["rejections"] - s0["rejections"]) / nc,
                                eq9_mean_beta=(s1["beta_sum"] - s0["beta_sum"]) / nc, committed_md_steps_per_s=nc / dt)
                ctx.close()
            rows.append(row)
    b0 = next(r for r in rows if r["N"] == 500 and r["tau_fs"] == 1000.0)["no_ec"]["rate"]
    for r in rows:
        r["eq11_prediction"] = float(erf(np.sqrt(r["N"] * r["tau_fs"] / (500 * 1000.0)) * erfinv(b0)))
    print(json.dumps(dict(sweep="Fig. 4 form (Eq. 11)", T_K=1500.0, dt_fs=1.0, K=K, segment_steps=nsteps, eps=eps, fit_point=dict(N=500, tau_fs=1000.0, beta=b0),
                          draft="target with network energy scale x (1 + eps)", rows=rows)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default=None, choices=[None, "fp32", "bf16"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip all_workloads and the acceptance variant (kernel tuning runs)")
    ap.add_argument("--ec", type=int, default=0, help="1: speculative error correction (Alg. 3) on")
    ap.add_argument("--overlap", type=int, default=0, help="1: time lsd_run with the speculative second-stream rollout instead of explicit calls")
    ap.add_argument("--sweep", action="store_true", help="rejection rate against N and tau (form of Fig. 4 / Eq. 11) instead of the bench line")
    ap.add_argument("--sweep-steps", type=int, default=1000)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import lsd_inputs as L
    import paper_2606_02455_b200 as P

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    P.load_library()
    peaks = load_peaks()
    stream = torch.cuda.Stream()
    env = dict(torch=torch, L=L, P=P, rank=rank, world=world, local=local, stream=stream, peaks=peaks,
               flush=torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda"),     # > 126 MB L2
               fma_peaks=(P.lsd_measure_fma_peak(0, stream), P.lsd_measure_fma_peak(1, stream)))

    m = measure_workload(env, args.workload, args.precision, args.steps, args.warmup, full=True, ec=args.ec, overlap=args.overlap)

    side, variant, ring = None, None, None
    if not args.no_side and world == 1 and not args.ec and not args.overlap:
        # the other BASELINE.json workloads, a few windows each, through the same measurement code (the headline is listed again in short form)
        side = {}
        for name, precn in ALL_WORKLOADS:
            key = name + ("" if precn is None else "_" + precn)
            if name == args.workload and (precn or "") == (args.precision or ("bf16" if m["dtype"] == "bf16" else "fp32" if m["dtype"] == "f32" else "")):
                r = m
            else:
                r = measure_workload(env, name, precn, SIDE_STEPS * (5 if name in ("cfg1", "cfg2") else 1), 3, full=False)   # (0.1-0.5 ms windows: more of them)
            rf = r["roofline"]
            side[key] = dict(ms_per_step=r["ms_per_step"], value=r["value"], unit=UNIT, dtype=r["dtype"], committed_md_steps_per_s=r["committed_md_steps_per_s"],
                             committed_per_window=r["committed_per_window"], e2e_value=r["e2e"]["value"], gpu_launches=r["gpu_launches"],
                             roofline=dict(bound=rf["bound"], frac=rf["frac"], achieved=rf["achieved"], peak=rf["peak"], unit=rf["unit"], kernel=rf["kernel"],
                                           three_term=rf.get("a2_three_term")),
                             clocks=r["clocks"], steps=r["windows_timed"])
        # the labelled side blocks never take the headline line down with them: a failure is reported in their place
        def guarded(fn, *a):
            try:
                return fn(*a)
            except Exception as exc:                                  # noqa: BLE001
                return dict(error=f"{type(exc).__name__}: {exc}")
        variant = guarded(acceptance_variant, env, args.workload, args.precision)
        ring = guarded(async_depth_block, env)

    if rank == 0:
        N, K = m["n_atoms"], m["window_K"]
        ov_note = ("lsd_run with the speculative next-window rollout on a second stream" if args.overlap else
                   "explicit rollout -> verify -> transport -> rollback on one stream: with the synthetic draft of this workload the acceptance is ~0 for "
                   "N >= 1e3 (Eq. 9), so a speculative rollout is always discarded and only costs device time (speedup.adaptive_K_overlap vs adaptive_K); "
                   "the second stream is exercised where it can pay in `acceptance_variant`")
        line = dict(metric=METRIC, value=m["value"], unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=m["ms_per_step"],
                    higher_is_better=True, scaling="weak", vs_baseline=None, dtype=m["dtype"], data="synthetic",
                    config=dict(workload=args.workload, n_atoms=N, window_K=K, atoms_per_window=K * N, integrator="ABOBA (Eq. 2)",
                                l2="flushed between timed steps (256 MiB write)" if m["need_flush"] else "working set larger than L2",
                                overlap=bool(args.overlap), overlap_note=ov_note, error_correction=bool(args.ec), skin_A=m["skin"], replicas=world,
                                peaks=peaks["source"], windows_timed=m["windows_timed"]),
                    committed_md_steps_per_s=m["committed_md_steps_per_s"], committed_per_window=m["committed_per_window"],
                    clocks=m["clocks"], e2e=m["e2e"], gpu_launches=m["gpu_launches"], roofline=m["roofline"], speedup=m["speedup"],
                    measured_peaks=dict(fp32_fma_tflops=env["fma_peaks"][0], fp64_fma_tflops=env["fma_peaks"][1], how="lsd_measure_fma_peak (16 FMA chains per thread, "
                                        "CUDA events, best of 3) in this run", hbm_gbs=peaks["hbm_gbs"], bf16_tflops_sustained=peaks["bf16"], bf16_tflops_burst=peaks["bf16_burst"],
                                        hbm_bf16_source="MEASURED_PEAKS.json (driver)" if peaks["source"] == "measured" else "fallback of B200_PROFILING.md"))
        if side is not None:
            line["all_workloads"] = side
        if variant is not None:
            line["acceptance_variant"] = variant
        if ring is not None:
            line["async_depth"] = ring
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = {k: v for k, v in cpu_baseline(args.workload).items() if k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
