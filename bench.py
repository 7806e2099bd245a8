#!/usr/bin/env python
"""bench.py -- exact INLA gradients/sec (f + grad_theta f) on B200, per BASELINE.json.

One "step" = one call of the whole hot path `inla_value_and_grad` (assemble -> fused forward sweeps ->
fused backward sweeps with selected inversion and trace contractions -> scalar assembly, on Q_c and Q_p)
on a synthetic BTA model.  Default workload: BASELINE.json configs[4] (largest single-GPU model), the one
north_star's FP64-fraction target is quoted on; `--config i` selects another.

  python bench.py --gpus N --steps K --warmup W            # our arm (N > 1: independent replicas, no collective)
  python bench.py --impl reference ...                      # the CPU oracle on a bounded sample (rank 0 only)
"""
import argparse
import json
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


def f_alg(model):
    """Algorithmic flops of one gradient (DESIGN.md / SURVEY.md §8(d)): 14 nt b^3, symmetric outputs once."""
    return 14.0 * model.nt * float(model.b) ** 3


def workload_name(idx, model):
    if idx >= 5:
        from workloads import EXTREME_NAMES
        return (f"extreme[{idx}] {EXTREME_NAMES[idx]} (SURVEY.md 8(f) NEXT-4, not a BASELINE config): g={model.g} "
                f"ns={model.ns} k={model.k} b={model.b} nt={model.nt} a={model.a} d={model.d} N={model.N}")
    return (f"configs[{idx}]: g={model.g} ns={model.ns} k={model.k} b={model.b} nt={model.nt} a={model.a} "
            f"d={model.d} N={model.N}")


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


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from workloads import CONFIGS
    full_model = CONFIGS[args.config][0]
    nt_s = {0: 6, 1: 10, 2: 4, 3: 2, 4: 2, 5: 2, 6: 1}[args.config]
    for _ in range(args.warmup if args.config < 2 else min(args.warmup, 1)):
        oracle_sample(args.config, nt_s)
    ts = []
    for _ in range(args.steps):
        dt, est, nts, _ = oracle_sample(args.config, nt_s)
        ts.append(est)
    ms = 1e3 * float(np.mean(ts))
    val = 1e3 / ms
    sample = (f"oracle/bta_oracle.value_and_grad on the first {nts} of {full_model.nt} time blocks "
              f"(observations scaled alike); time scaled by nt/{nts} (work is linear in nt)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, full_model)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


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
    if args.store == "carry":
        M.bta_set_store_mode(1)
    ws_bytes = M.workspace_bytes()
    # one replica per GPU: each rank evaluates f, grad at its own theta (line-search / Hessian-stencil points)
    thetas = replica_thetas(th, rank, args.steps + args.warmup)

    peak_tf, _ = fp64_peak(0, 100000)
    dfma_tf, _ = fp64_peak(1, 100000)

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
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, model), "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2 (blocks of both matrices: %.1f GB per replica)" % (ws_bytes / 1e9),
                       "workspace_bytes": ws_bytes, "chains": "two-way elimination: up and down chains of Q_c and Q_p on four streams (+ priority lanes)", "store_mode": args.store},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * d,
                    "d2h_bytes_per_step": 8 * (1 + d + 2 + 3 * d + model.k + 1) + 8},
            "gpu_launches": int(launches),
            "stage_ms": stage_acc,
            "step_ms_samples": step_ms,
            "fp64": {"alg_flop_per_gradient": f_alg(model),
                     "carry_rebuild_flop_per_gradient": (10.0 / 3.0) * model.nt * float(model.b) ** 3
                     if args.store == "carry" else 0.0, "achieved_tflops": f_alg(model) / (ms_step * 1e-3) / 1e12,
                     "dmma_issue_peak_tflops": peak_tf, "dfma_issue_peak_tflops": dfma_tf}}
    # ---- roofline of the dominant kernel: the 128x128-tile DMMA GEMM (79 % of the serialised kernel time of a
    #      step, profiles/r01_launches_bench_nt5.md), timed live on a b x b x b product (operands 3 b^2 8 B > L2
    #      at the large configs), CUDA events on the launching stream.
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
    line["roofline"] = {"bound": "tensor", "kernel": "gemm_kernel (FP64 mma.sync m8n8k4 / DMMA.8x8x4), C = A B, b^3",
                        "achieved": gemm_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": gemm_tf / peak_tf,
                        "launch_ms": gemm_ms, "alg_flop_per_launch": 2.0 * float(b) ** 3,
                        "traffic": 0.940e9 if b == 4096 else None,
                        "traffic_note": "dram read+write bytes per launch at b=4096 from ncu --set full "
                                        "(profiles/r01_gemm_full.md); algorithmic bytes 3 b^2 8 = 4.03e8",
                        "share_of_step": 0.786,
                        "peak_source": "measured live: mma.sync.m8n8k4.f64 issue loop on all SMs (MEASURED_PEAKS.json "
                                       "has no FP64 entry; nominal-ratio alternative bf16_tflops x 40/2250 = "
                                       "29.1 TFLOP/s is lower)"}
    line["roofline_step"] = {"bound": "tensor", "achieved": line["fp64"]["achieved_tflops"], "peak": peak_tf,
                             "unit": "TFLOP/s", "frac": line["fp64"]["achieved_tflops"] / peak_tf,
                             "note": "algorithmic flops of one gradient (14 nt b^3) / step time"}
    # ---- the paper's comparison: one exact gradient against a
    #      central finite-difference gradient = 2d+1 objective evaluations (inla_value), same kernels, same GPU
    if not args.no_fd:
        for _ in range(2):
            M.inla_value(thetas[0])
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record()
        for i in range(args.steps):
            M.inla_value(thetas[args.warmup + i])
        v1.record()
        torch.cuda.synchronize()
        t_eval = v0.elapsed_time(v1) / args.steps
        fwd = stage_acc.get("fwd_Qc", 0.0) + stage_acc.get("fwd_Qp", 0.0)
        bwd = stage_acc.get("bwd_Qc", 0.0) + stage_acc.get("bwd_Qp", 0.0)
        line["fd_compare"] = {"t_eval_ms": t_eval, "t_ad_ms": ms_step, "c_ad": ms_step / t_eval,
                              "fd_gradient_ms": (2 * d + 1) * t_eval,
                              "speedup_ad_vs_fd": (2 * d + 1) * t_eval / ms_step,
                              "beta_bwd_over_fwd": (bwd / fwd) if fwd > 0 else None,
                              "note": "FD gradient = (2d+1) x inla_value (Eq. 2); paper reports 4.2-7.9x per-gradient "
                                      "speedup and c_AD 2.3-3.9 on GH200 (context only, BASELINE.md)"}
    if rank == 0 and not args.no_cpu_baseline and world == 1 and args.config <= 4:
        nt_s = {0: 6, 1: 10, 2: 4, 3: 2, 4: 2}[args.config]
        dt, est, nts, _ = oracle_sample(args.config, nt_s)
        line["cpu_baseline"] = {"value": 1.0 / est, "unit": UNIT, "cores": threads_used(), "kind": "oracle",
                                "sample": f"oracle on the first {nts} of {model.nt} time blocks ({dt:.1f} s), "
                                          f"scaled by nt/{nts}"}
    M.close()
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fd", action="store_true", help="skip the finite-difference comparison (NEXT-1)")
    ap.add_argument("--store", default="factor", choices=["factor", "carry"],
                    help="storage policy a7: keep the factor blocks (default) or only the Schur carries")
    ap.add_argument("--nt", type=int, default=None,
                    help="profiling aid: truncate the workload to its first NT time blocks (same kernels per block)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
