"""Diagnostic: SM-slot occupancy timeline of the GEMM CTAs during one gradient ("Where the forward
sweep loses time").  Not part of the hot path: it arms `bta_debug_cta_trace` (include/bta_diag.h), runs one
`inla_value_and_grad` and bins the per-CTA {start, end, SM id, tile} records.

    python -m paper_2605_06392_b200.diagnostics --config 2 [--nt N] [--slices 20]
"""
import argparse

import numpy as np


def timeline(cfg, nt=None, slices=20, cap=1 << 21):
    import torch
    from workloads import make_config
    from . import BtaModel
    from .binding import cta_trace_count, cta_trace_start
    model, obs, th = make_config(cfg, nt=nt)
    M = BtaModel.from_workload(model, obs, device=0)
    for _ in range(2):
        M.inla_value_and_grad(th)
    buf = torch.zeros(cap, 4, dtype=torch.int64, device="cuda")
    cta_trace_start(buf)
    _, _, st = M.inla_value_and_grad(th, stages=True)
    n = cta_trace_count()
    cta_trace_start(None)
    r = buf[:min(n, cap)].cpu().numpy()
    M.close()
    t0 = r[:, 0].min()
    b, e = (r[:, 0] - t0) / 1e6, (r[:, 1] - t0) / 1e6          # ms
    sm, tile, krange = r[:, 2] & 0xFFFF, (r[:, 2] >> 16) & 0xFFF, r[:, 3] & 0xFFFFFFFF
    # CTAs resident per SM for each tile class (gemm.cu: launch_gemm): 1 x 128x128, 3 x 64x64, 7 x 32x32
    slots = {128: 1.0, 64: 3.0, 32: 7.0}
    edges = np.linspace(0.0, float(e.max()), slices + 1)
    rows = []
    for i in range(slices):
        lo, hi = edges[i], edges[i + 1]
        frac = []
        for tl in (128, 64, 32):
            m = tile == tl
            ov = np.clip(np.minimum(e[m], hi) - np.maximum(b[m], lo), 0, None).sum() / slots[tl]
            frac.append(float(ov / ((hi - lo) * 148)))
        rows.append((float(lo), sum(frac), *frac))
    # SMs used by the step products of the forward sweeps (k-range above b/2: the recursion's products stay below)
    half = model.b // 2 + 128
    fw = (e < 0.35 * e.max()) & (krange >= half)
    return {"ctas_seen": int(n), "ctas_recorded": int(len(r)), "span_ms": float(e.max()), "stage_ms": st, "rows": rows,
            "forward_product_sms": int(len(np.unique(sm[fw]))), "sms_seen": int(len(np.unique(sm)))}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--nt", type=int, default=None)
    ap.add_argument("--slices", type=int, default=20)
    a = ap.parse_args()
    t = timeline(a.config, a.nt, a.slices)
    print(f"CTAs seen {t['ctas_seen']} (recorded {t['ctas_recorded']}), span of the recorded CTAs {t['span_ms']:.1f} ms")
    print("stage_ms", {k: round(v, 1) for k, v in t["stage_ms"].items()})
    print(f"SMs used by the forward sweeps' step products: {t['forward_product_sms']} of {t['sms_seen']}")
    print("slice start (ms) | SM slots busy | in 128x128 | 64x64 | 32x32 CTAs")
    for lo, tot, f128, f64, f32 in t["rows"]:
        print(f"{lo:9.1f} | {tot:.3f} | {f128:.3f} | {f64:.3f} | {f32:.3f}")


if __name__ == "__main__":
    main()
