"""N sweep of the X-engine (the x-axis of the paper's Fig. 4) and the five BASELINE.json
shapes: effective TOPS and achieved HBM GB/s per shape, device-timed with CUDA events.

    python sweep.py [--reps 20] [--csv out.csv] [--shape N,F,T] [--op corr|shift|gated]

Inputs are random bytes generated on the device (every byte is a legal sample pair; timing does not
depend on the values); correctness is the parity tests' job, not this script's.
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

# (label, N, F, T, accumulate): sweep shapes keep the input >= 256 MB for small N so GB/s means something
SHAPES = [
    ("sweep", 16, 256, 65536, 0), ("sweep", 32, 128, 65536, 0), ("sweep", 64, 64, 65536, 0),
    ("sweep", 128, 64, 32768, 0), ("sweep", 256, 32, 32768, 0), ("sweep", 512, 32, 16384, 0),
    ("sweep", 1024, 16, 16384, 0), ("sweep", 2048, 8, 16384, 0), ("sweep", 4096, 4, 8192, 0),
    ("sweep", 8192, 1, 8192, 0),
    ("cfg1", 16, 4, 1024, 0), ("cfg2", 256, 16, 16384, 0), ("cfg3", 2048, 8, 8192, 0),
    ("cfg4", 8192, 1, 4096, 0), ("cfg5 (one accumulate call)", 512, 64, 8192, 1),
]


def other_op(args):
    """Times corr_time_shift or corr_execute_gated on one shape (read + written bytes per second for the shift)."""
    import numpy as np
    import torch
    from paper_1503_06203_b200 import Plan, time_shift
    n, f, t = (int(v) for v in (args.shape or "2048,8,8192").split(","))
    dev = torch.device("cuda:0")
    a = torch.randint(0, 256, (t, f, n), dtype=torch.uint8, device=dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.op == "shift":
        # three lag patterns: every input its own lag, 16 inputs sharing a lag (a few cable lengths), a wide spread
        out = torch.empty_like(a)
        pats = {"independent +-16": torch.randint(-16, 17, (n,), dtype=torch.int32, device=dev),
                "shared by 16 inputs +-16": torch.randint(-16, 17, ((n + 15) // 16,), dtype=torch.int32, device=dev).repeat_interleave(16)[:n].contiguous(),
                "independent +-256": torch.randint(-256, 257, (n,), dtype=torch.int32, device=dev)}
        for name, lags in pats.items():
            e0.record()
            for _ in range(3):
                time_shift(a, lags, out=out)
            e1.record()
            torch.cuda.synchronize()
            for _ in range(min(400, int(8.0 / max(e0.elapsed_time(e1) / 3, 1e-3)))):   # 8 ms of warm-up, see main()
                time_shift(a, lags, out=out)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(args.reps):
                time_shift(a, lags, out=out)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.reps
            print(f"shift,{name},N={n},F={f},T={t},ms={ms:.4g},read+written_GBs={2 * a.numel() / (ms * 1e-3) / 1e9:.4g}")
        return
    else:
        plan = Plan(n, f, t)
        gate = ((np.arange(t) % 64) * 4 // 64).astype(np.int32)
        vis = plan.execute_gated(a, gate, 4)
        run = lambda: plan.execute_gated(a, gate, 4, vis=vis)
    for _ in range(20):    # 8 ms of warm-up, see main()
        run()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.reps):
        run()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.reps
    print(f"{args.op},N={n},F={f},T={t},ms={ms:.4g},stream_GBs={a.numel() / (ms * 1e-3) / 1e9:.4g}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--csv", default=None)
    ap.add_argument("--shape", default=None, help="N,F,T: time this one shape only (e.g. under ncu)")
    ap.add_argument("--op", default="corr", choices=["corr", "shift", "gated"],
                    help="with --shape: corr_execute (default), corr_time_shift (lags of +-16) or corr_execute_gated (4 gates)")
    args = ap.parse_args()
    if args.op != "corr":
        return other_op(args)
    shapes = SHAPES
    if args.shape:
        n, f, t = (int(v) for v in args.shape.split(","))
        shapes = [("shape", n, f, t, 0)]
    import torch
    from paper_1503_06203_b200 import Plan
    if not torch.cuda.is_available():
        sys.exit("sweep needs a CUDA device (there is no CPU path)")
    dev = torch.device("cuda:0")
    rows = []
    for label, N, F, T, acc in shapes:
        plan = Plan(N, F, T)
        nbuf = 2 if N * F * T >= (64 << 20) else 8
        ins = [torch.randint(0, 256, (T, F, N), dtype=torch.uint8, device=dev) for _ in range(nbuf)]
        vis = torch.zeros((F, plan.baselines, 2), dtype=torch.int32, device=dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        # warm-up: 3 calls, then as many as make 8 ms of work (after the allocations above the part has idled, and it
        # takes some 5 ms of load to get back to full speed: profiles/r02_tc3_ncu_summary.md)
        e0.record()
        for i in range(3):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        e1.record()
        torch.cuda.synchronize()
        for i in range(min(400, int(8.0 / max(e0.elapsed_time(e1) / 3, 1e-3)))):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        torch.cuda.synchronize()
        e0.record()
        for i in range(args.reps):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.reps
        ops = 8.0 * plan.baselines * F * T
        out_bytes = vis.numel() * 4 * (2 if acc else 1)
        gbs = (N * F * T + out_bytes) / (ms * 1e-3) / 1e9
        rows.append((label, N, F, T, plan.info["path"], plan.info["slices"], plan.info["units"], ms,
                     ops / (ms * 1e-3) / 1e12, gbs, F * T / (ms * 1e-3) / 1e6))
        plan.close()
        del ins, vis
        torch.cuda.empty_cache()
    # Mmatrices_per_s: correlation matrices (one channel, one time step) per second, the unit of the paper's
    # Fig. 4 upper panel (0.3318 M/s at N = 2048 on an R9 280X)
    hdr = ("shape", "N", "F", "T", "path", "slices", "units", "ms", "eff_TOPS", "HBM_GBs", "Mmatrices_per_s")
    lines = [",".join(hdr)] + [",".join(f"{v:.4g}" if isinstance(v, float) else str(v) for v in r) for r in rows]
    print("\n".join(lines))
    if args.csv:
        with open(args.csv, "w") as fh:
            fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
