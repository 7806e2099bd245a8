#!/usr/bin/env python
"""bench.py -- exact INLA gradients/sec (f + grad_theta f) on B200, per BASELINE.json.

One "step" = one call of the whole hot path `inla_value_and_grad` (assemble -> fused forward sweeps ->
fused backward sweeps with selected inversion and trace contractions -> scalar assembly, on Q_c and Q_p)
on a synthetic BTA model.  Default workload: BASELINE.json configs[4] (largest single-GPU model), the one
north_star's FP64-fraction target is quoted on; `--config i` selects another.

  python bench.py --gpus N --steps K --warmup W            # our arm (N > 1: independent replicas, no collective)
  python bench.py --impl reference ...                      # the CPU oracle on a bounded sample (rank 0 only)

Every number in the JSON line is measured by this run, with two labelled exceptions: `roofline.traffic` (DRAM bytes
per launch of the dominant kernel) is read from the committed ncu extract named in `roofline.traffic_source` (null
when that file has no row for the kernel), and `vs_baseline` is null (the paper publishes no gradients/s).
"""
import argparse
import csv
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "exact INLA gradients/sec (f+grad_theta, FP64)"
UNIT = "gradients/s"
# Student t, two-sided 95 %, by degrees of freedom (mean and 95 % CI over >= 10 runs after warm-up)
T95 = {1: 12.706, 2: 4.303, 3: 3.182, 4: 2.776, 5: 2.571, 6: 2.447, 7: 2.365, 8: 2.306, 9: 2.262, 10: 2.228,
       11: 2.201, 12: 2.179, 13: 2.160, 14: 2.145, 15: 2.131, 19: 2.093, 24: 2.064, 29: 2.045}
# bounded oracle sample per config: the first nt_s time blocks (configs 0-1: the whole model)
ORACLE_NT = {0: 6, 1: 50, 2: 4, 3: 2, 4: 2, 5: 2, 6: 1}
# the reference arm repeats its sample K times: config 1 takes 10 of its 50 blocks there (the whole model is ~18 s)
REFERENCE_NT = {0: 6, 1: 10, 2: 4, 3: 2, 4: 2, 5: 2, 6: 1}


def f_alg(model):
    """Algorithmic flops of one gradient (DESIGN.md / SURVEY.md §8(d)): 14 nt b^3, symmetric outputs once."""
    return 14.0 * model.nt * float(model.b) ** 3


def mean_ci95(samples):
    x = np.asarray(samples, dtype=np.float64)
    n = x.size
    if n < 2:
        return float(x.mean()) if n else float("nan"), None
    dof = n - 1
    t = T95.get(dof) or T95[max(k for k in T95 if k <= dof)]
    return float(x.mean()), float(t * x.std(ddof=1) / math.sqrt(n))


def workload_name(idx, model):
    if idx >= 5:
        from workloads import EXTREME_NAMES
        return (f"extreme[{idx}] {EXTREME_NAMES[idx]} (SURVEY.md 8(f) NEXT-4, not a BASELINE config): g={model.g} "
                f"ns={model.ns} k={model.k} b={model.b} nt={model.nt} a={model.a} d={model.d} N={model.N}")
    return (f"configs[{idx}]: g={model.g} ns={model.ns} k={model.k} b={model.b} nt={model.nt} a={model.a} "
            f"d={model.d} N={model.N}")


def hbm_peak():
    """(GB/s, source): the driver-measured copy bandwidth, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(kernel_regex):
    """dram read+write bytes per launch of the dominant kernel from the committed `ncu --set full` extract."""
    import re
    path = os.path.join(ROOT, "profiles", "r02_gemm_full_raw.csv")
    if not os.path.exists(path):
        return None, None
    try:
        with open(path) as fh:
            for row in csv.DictReader(fh):
                if re.search(kernel_regex, row.get("kernel", "")):
                    return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), "profiles/r02_gemm_full_raw.csv"
    except Exception:
        pass
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(idx, nt_s):
    """The oracle, as it stands, on the first nt_s time blocks of the workload (m scaled with nt_s)."""
    from oracle import bta_oracle as O
    from workloads import CONFIGS, make_config
    full_model, mpv, _, _ = CONFIGS[idx]
    nt_s = min(nt_s, full_model.nt)
    model, obs, th = make_config(idx, nt=nt_s, m_per_var=max(1, mpv * nt_s // full_model.nt))
    t0 = time.perf_counter()
    O.value_and_grad(model, obs, th)
    dt = time.perf_counter() - t0
    est_full = dt * full_model.nt / nt_s          # work is linear in nt
    return dt, est_full, nt_s, model


def threads_used():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(n) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def sample_text(idx, nts, full_nt, dt):
    if nts >= full_nt:
        return f"oracle/bta_oracle.value_and_grad on the whole model (all {full_nt} time blocks), {dt:.2f} s per call"
    return (f"oracle/bta_oracle.value_and_grad on the first {nts} of {full_nt} time blocks (observations scaled "
            f"alike), {dt:.1f} s; time scaled by nt/{nts} (the work is linear in nt)")


def cpu_baseline(idx, model_nt):
    """The oracle timed on this box's host cores: a bounded sample (whole model at configs 0-1, where the
    single-thread time is taken too)."""
    dt, est, nts, _ = oracle_sample(idx, ORACLE_NT[idx])
    if idx <= 1:                                   # fast enough to repeat once: the better of two calls
        dt = min(dt, oracle_sample(idx, ORACLE_NT[idx])[0])
        est = dt * model_nt / nts
    out = {"value": 1.0 / est, "unit": UNIT, "cores": threads_used(), "kind": "oracle",
           "sample": sample_text(idx, nts, model_nt, dt)}
    if idx <= 1:
        try:
            from threadpoolctl import threadpool_limits
            with threadpool_limits(limits=1):
                d1 = oracle_sample(idx, ORACLE_NT[idx])[0]
            out["single_thread"] = {"value": 1.0 / d1, "unit": UNIT, "cores": 1}
        except Exception:
            pass
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from workloads import CONFIGS
    full_model = CONFIGS[args.config][0]
    nt_s = REFERENCE_NT[args.config]
    for _ in range(args.warmup if args.config < 2 else min(args.warmup, 1)):
        oracle_sample(args.config, nt_s)
    ts, dts = [], []
    for _ in range(args.steps):
        dt, est, nts, _ = oracle_sample(args.config, nt_s)
        ts.append(est)
        dts.append(dt)
    ms = 1e3 * float(np.mean(ts))
    val = 1e3 / ms
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, full_model)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads_used(), "kind": "oracle",
                             "sample": sample_text(args.config, nts, full_model.nt, float(np.mean(dts)))},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def kernel_breakdown(M, theta, peak_tf, hbm_gbs):
    """One extra step with both matrices on ONE stream (BTA_OPT_SERIAL) and every launch bracketed by CUDA events
    (include/bta_diag.h: bta_diag_ktime_*): exclusive per-class kernel times, the in-step rate of each class
    (algorithmic flops or bytes / summed launch durations) and exclusive stage times."""
    from paper_2605_06392_b200 import binding as B
    M.bta_set_option(B.OPT_SERIAL, 1)
    M.bta_set_option(B.OPT_GRAPH, 0)
    M.inla_value_and_grad(theta)                                   # warm-up in this mode
    B.ktime_begin()
    _, _, st = M.inla_value_and_grad(theta, stages=True)
    kt = B.ktime_end()
    M.bta_set_option(B.OPT_SERIAL, 0)
    M.bta_set_option(B.OPT_GRAPH, -1)
    tot = sum(v["ms"] for v in kt.values())
    table = {}
    for k, v in kt.items():
        if v["launches"] == 0:
            continue
        row = {"ms": v["ms"], "launches": v["launches"], "share_of_kernel_time": v["ms"] / tot if tot > 0 else None,
               "mean_launch_us": 1e3 * v["ms"] / v["launches"]}
        if k.startswith("gemm") or k == "leaf":
            row["alg_tflops"] = v["flop"] / (v["ms"] * 1e-3) / 1e12 if v["ms"] > 0 else None
            row["frac_of_dmma_peak"] = row["alg_tflops"] / peak_tf if row["alg_tflops"] else None
        elif k in ("skinny", "contract", "assemble"):
            row["alg_gbs"] = v["bytes"] / (v["ms"] * 1e-3) / 1e9 if v["ms"] > 0 else None
            row["frac_of_hbm_peak"] = row["alg_gbs"] / hbm_gbs if row["alg_gbs"] else None
        table[k] = row
    fwd = st["fwd_Qc"] + st["fwd_Qp"]
    bwd = st["bwd_Qc"] + st["bwd_Qp"]
    return kt, table, {"stage_ms_exclusive": st, "kernel_ms_total": tot,
                       "beta_bwd_over_fwd": bwd / fwd if fwd > 0 else None,
                       "note": "single stream, single chain per matrix (BTA_OPT_SERIAL), the two matrices' steps "
                               "interleaved: fwd_Qc and fwd_Qp both span the forward phase of BOTH matrices, likewise "
                               "bwd_*; phases do not overlap each other"}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2605_06392_b200 import BtaModel, fp64_peak
    from paper_2605_06392_b200.replicas import max_over_ranks, replica_thetas
    from workloads import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- this library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.nt is not None:
        from workloads import CONFIGS
        full_nt = CONFIGS[args.config][0].nt
        model, obs, th = make_config(args.config, nt=args.nt,
                                     m_per_var=max(1, CONFIGS[args.config][1] * args.nt // full_nt))
    else:
        model, obs, th = make_config(args.config)
    M = BtaModel.from_workload(model, obs, device=local)
    store_modes = {"factor": 0, "carry": 1, "host": 2}
    if args.store != "factor":
        M.bta_set_store_mode(store_modes[args.store])
    if args.partitions is not None:
        from paper_2605_06392_b200 import binding as B
        M.bta_set_option(B.OPT_PARTITIONS, args.partitions)
    ws_bytes = M.workspace_bytes()
    # one replica per GPU: each rank evaluates f, grad at its own theta (line-search / Hessian-stencil points)
    thetas = replica_thetas(th, rank, args.steps + args.warmup)

    peak_tf, _ = fp64_peak(0, 100000)
    dfma_tf, _ = fp64_peak(1, 100000)
    hbm_gbs, hbm_src = hbm_peak()

    for i in range(args.warmup):
        M.inla_value_and_grad(thetas[i])
    # ---- device-timed region: K steps between CUDA events on the launching stream ----
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    barrier()
    n0 = M.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_acc = {}
    step_ms = []
    e0.record()
    for i in range(args.steps):
        f, g, st = M.inla_value_and_grad(thetas[args.warmup + i], stages=True)
        step_ms.append(st.get("total", float("nan")))
        for k_, v in st.items():
            stage_acc[k_] = stage_acc.get(k_, 0.0) + v / args.steps
    e1.record()
    barrier()
    ms_dev = e0.elapsed_time(e1)
    launches = M.kernel_launches() - n0
    # ---- end-to-end region: the same call, host theta in (pinned staging inside the library), host f/grad
    #      out, wall clock around synchronised calls ----
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        M.inla_value_and_grad(thetas[args.warmup + i])
    torch.cuda.synchronize()
    ms_e2e = 1e3 * (time.perf_counter() - t0)
    clocks = sampler.stop()
    ms_dev, ms_e2e = max_over_ranks([ms_dev, ms_e2e], device="cuda")
    ms_step = ms_dev / args.steps
    value = world * 1e3 / ms_step
    e2e_val = world * 1e3 / (ms_e2e / args.steps)
    d = model.d
    mean_ms, ci_ms = mean_ci95(step_ms)
    step_tf = f_alg(model) / (ms_step * 1e-3) / 1e12
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, model), "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2 (blocks of both matrices: %.1f GB per replica)" % (ws_bytes / 1e9),
                       "workspace_bytes": ws_bytes,
                       "chains": "two-way elimination: up and down chains of Q_c and Q_p on four streams "
                                 "(+ priority lanes, pipelined forward steps)",
                       "store_mode": args.store, "partitions": args.partitions},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * d,
                    "d2h_bytes_per_step": 8 * (1 + d + 2 + 3 * d + model.k + 1) + 8},
            "gpu_launches": int(launches),
            "stage_ms": stage_acc,
            "stage_ms_note": "CUDA-event intervals per chain; the four chains overlap, so stages do not add up to "
                             "total (exclusive times: kernel_breakdown.stage_ms_exclusive)",
            "step_ms_samples": step_ms,
            "step_ms_mean_ci95": {"mean": mean_ms, "ci95_half_width": ci_ms, "n": len(step_ms),
                                  "note": "library-side CUDA events per call; Student t"},
            "fp64": {"alg_flop_per_gradient": f_alg(model),
                     "carry_rebuild_flop_per_gradient": (10.0 / 3.0) * model.nt * float(model.b) ** 3
                     if args.store != "factor" else 0.0, "achieved_tflops": step_tf,
                     "dmma_issue_peak_tflops": peak_tf, "dfma_issue_peak_tflops": dfma_tf}}
    # ---- in-step kernel breakdown: one extra serial step with every launch timed (never part of `value`)
    bd = None
    if not args.no_breakdown:
        kt, table, extra = kernel_breakdown(M, thetas[0], peak_tf, hbm_gbs)
        bd = {"classes": table, **extra}
        line["kernel_breakdown"] = bd
    # ---- the b x b x b product alone (isolated rate of the GEMM kernel; operands 3 b^2 8 B > L2 at the large configs)
    from paper_2605_06392_b200 import gemm as _gemm
    b = model.b
    ga = torch.randn(b, b, dtype=torch.float64, device="cuda")
    gb = torch.randn(b, b, dtype=torch.float64, device="cuda")
    gc = torch.empty(b, b, dtype=torch.float64, device="cuda")
    for _ in range(3):
        _gemm(0, ga, gb, gc)
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 10 if b >= 1024 else 200
    g0.record()
    for _ in range(reps):
        _gemm(0, ga, gb, gc)
    g1.record()
    torch.cuda.synchronize()
    gemm_ms = g0.elapsed_time(g1) / reps
    gemm_tf = 2.0 * float(b) ** 3 / (gemm_ms * 1e-3) / 1e12
    del ga, gb, gc
    peak_src = ("measured live: mma.sync.m8n8k4.f64 issue loop on all SMs (MEASURED_PEAKS.json has no FP64 entry; "
                "the nominal-ratio alternative, bf16_tflops x 40/2250, is lower)")
    # ---- roofline: the dominant kernel, measured IN the step (summed CUDA-event durations of its launches in the
    #      serial breakdown step, algorithmic flops of those launches)
    roof = {"bound": "tensor", "peak": peak_tf, "unit": "TFLOP/s", "peak_source": peak_src,
            "step": {"achieved": step_tf, "frac": step_tf / peak_tf,
                     "note": "algorithmic flops of one gradient (14 nt b^3) / ms_per_step: the whole hot path"},
            "isolated": {"achieved": gemm_tf, "frac": gemm_tf / peak_tf, "launch_ms": gemm_ms,
                         "note": "one b x b x b product alone, CUDA events"}}
    if bd:
        gem = {k: v for k, v in bd["classes"].items() if k.startswith("gemm")}
        dom = max(gem, key=lambda k: gem[k]["ms"]) if gem else None
        if dom:
            r = gem[dom]
            tile = {"gemm_128": "128x128", "gemm_64": "64x64", "gemm_32": "32x32"}[dom]
            traffic, tsrc = ncu_traffic(r"gemm_kernel<128" if dom == "gemm_128" else r"gemm_kernel<64")
            roof.update({"kernel": f"gemm_kernel, {tile} tiles (FP64 mma.sync m8n8k4 = DMMA.8x8x4)",
                         "achieved": r["alg_tflops"], "frac": r["frac_of_dmma_peak"],
                         "launches_per_step": r["launches"], "mean_launch_ms": r["ms"] / r["launches"],
                         "alg_flop_per_launch": kt[dom]["flop"] / r["launches"],
                         "share_of_step": r["share_of_kernel_time"],
                         "share_note": "share of the summed kernel time of the serial breakdown step",
                         "traffic": traffic, "traffic_source": tsrc})
    else:
        roof.update({"kernel": "whole step", "achieved": step_tf, "frac": step_tf / peak_tf, "traffic": None})
    line["roofline"] = roof
    line["roofline_step"] = {"bound": "tensor", "achieved": step_tf, "peak": peak_tf, "unit": "TFLOP/s",
                             "frac": step_tf / peak_tf}
    line["hbm_peak"] = {"gbs": hbm_gbs, "source": hbm_src}
    # ---- the paper's comparison: one exact gradient against a
    #      central finite-difference gradient = 2d+1 objective evaluations (inla_value), same kernels, same GPU
    if not args.no_fd:
        for _ in range(2):
            M.inla_value(thetas[0])
        nfd = min(args.steps, 5)
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record()
        for i in range(nfd):
            M.inla_value(thetas[args.warmup + i])
        v1.record()
        torch.cuda.synchronize()
        t_eval = v0.elapsed_time(v1) / nfd
        fwd_ph, bwd_ph = stage_acc.get("fwd_Qc", 0.0), stage_acc.get("bwd_Qc", 0.0)
        line["fd_compare"] = {"t_eval_ms": t_eval, "t_ad_ms": ms_step, "c_ad": ms_step / t_eval,
                              "fd_gradient_ms": (2 * d + 1) * t_eval,
                              "speedup_ad_vs_fd": (2 * d + 1) * t_eval / ms_step,
                              "beta_phases": (bwd_ph / fwd_ph) if fwd_ph > 0 else None,
                              "beta_serial": bd["beta_bwd_over_fwd"] if bd else None,
                              "beta_by_flops": 13.0 / 8.0,
                              "note": "FD gradient = (2d+1) x inla_value (Eq. 2); beta_phases = backward phase / forward "
                                      "phase of the timed step (all four chains run each phase together; null when the "
                                      "step is a graph replay), beta_serial = the same ratio in the serial breakdown "
                                      "step; paper: 4.2-7.9x per-gradient speedup, c_AD 2.3-3.9, beta 1.3-2.4 on GH200 "
                                      "(context only, BASELINE.md)"}
    # ---- storage policy a7: the same step in the other store mode (workspace and time side by side)
    if not args.no_store_compare and args.store == "factor" and args.partitions is None:
        M.bta_set_store_mode(1)
        wsc = M.workspace_bytes()
        for _ in range(2):
            M.inla_value_and_grad(thetas[0])
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ncarry = min(args.steps, 3)
        c0.record()
        for i in range(ncarry):
            M.inla_value_and_grad(thetas[args.warmup + i])
        c1.record()
        torch.cuda.synchronize()
        line["store_compare"] = {"factor": {"ms_per_step": ms_step, "workspace_bytes": ws_bytes},
                                 "carry": {"ms_per_step": c0.elapsed_time(c1) / ncarry, "workspace_bytes": wsc},
                                 "note": "carry mode rebuilds X_t, L_Bt in the backward sweep (+10/3 nt b^3 flops)"}
        M.bta_set_store_mode(0)
    if rank == 0 and not args.no_cpu_baseline and world == 1 and args.config <= 4 and args.nt is None:
        line["cpu_baseline"] = cpu_baseline(args.config, model.nt)
    M.close()
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fd", action="store_true", help="skip the finite-difference comparison (NEXT-1)")
    ap.add_argument("--no-breakdown", action="store_true", help="skip the serial per-kernel-class breakdown step")
    ap.add_argument("--no-store-compare", action="store_true", help="skip the carry-mode comparison")
    ap.add_argument("--store", default="factor", choices=["factor", "carry", "host"],
                    help="storage policy a7: keep the factor blocks (default), only the Schur carries, or the "
                         "carries staged in pinned host memory (PAPER.md:185)")
    ap.add_argument("--partitions", type=int, default=None,
                    help="time-domain partitions P per matrix inside the GPU (NEXT-3); default: the library's choice")
    ap.add_argument("--nt", type=int, default=None,
                    help="profiling aid: truncate the workload to its first NT time blocks (same kernels per block)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
