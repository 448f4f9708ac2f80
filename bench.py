#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native X-engine (arXiv 1503.06203 hot path).

One "step" = one pass of the whole hot path (TMA fetch, unpack, tile schedule, tcgen05 int8 MMA,
epilogue: one corr_execute call) over one batch of synthetic input.  Workload at any N: cfg3 of
BASELINE.json (N=2048 inputs, F=8 channels, T=8192 samples, iid quantised Gaussians sigma 2.5),
one such batch per GPU (frequency channels are independent: F-sharding, no
collective, weak scaling).

Metric: effective correlation TOPS = 8 * N(N+1)/2 * F * T / seconds / 1e12  (8 ops per complex
multiply-accumulate over the unique baselines, Eq. 2 at :52).

Prints ONE JSON line (see the task contract): value (inputs resident in HBM), e2e (through
corr_execute_host with pinned HOST buffers, copies inside the timed region), roofline of the
dominant kernel, cpu_baseline (the oracle as it stands, on the host cores, on a bounded sample).

`--impl reference` times the CPU oracle instead (rank 0 only), on a bounded sample per step.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "effective correlation TOPS (8 ops/CMAC/baseline) at N=2048; % of int8 TC peak"
NOMINAL_INT8_TOPS = 4500.0  # dense int8 = 2x dense bf16 2250 (B200_PROFILING.md nominal table)
# roofline.traffic comes from a tracked ncu summary (profiles/), which records the kernel it was captured on and
# the SHA-256 of that kernel's sources at capture time; a stale record (sources changed since) reports null.
TRAFFIC_RECORD = ROOT / "profiles" / "tc_traffic.txt"
KERNEL_SOURCES = ("corr_tc3.cuh", "corr_tc5.cuh", "corr_tc.cuh", "corr_ptx.cuh", "corr_api.cu")

# the N sweep of the paper's Fig. 4 axis (inputs >= 256 MB for small N so that GB/s means something)
# and the five BASELINE.json shapes: (label, N, F, T, accumulate)
TABLE_SHAPES = [
    ("n16", 16, 256, 65536, 0), ("n32", 32, 128, 65536, 0), ("n64", 64, 64, 65536, 0), ("n128", 128, 64, 32768, 0),
    ("n256", 256, 32, 32768, 0), ("n512", 512, 32, 16384, 0), ("n1024", 1024, 16, 16384, 0),
    ("n2048", 2048, 8, 16384, 0), ("n4096", 4096, 4, 8192, 0), ("n8192", 8192, 1, 8192, 0),
    ("cfg1", 16, 4, 1024, 0), ("cfg2", 256, 16, 16384, 0), ("cfg3", 2048, 8, 8192, 0), ("cfg4", 8192, 1, 4096, 0),
    ("cfg5_one_accumulate_call", 512, 64, 8192, 1),
]


def kernel_source_sha():
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        h.update((ROOT / "paper_1503_06203_b200" / "csrc" / name).read_bytes())
    return h.hexdigest()


def recorded_traffic(kernel: str, workload: str):
    """dram bytes (read + write) per launch from profiles/tc_traffic.txt, or None if there is no record for this
    kernel and workload or the kernel sources have changed since the capture."""
    if not TRAFFIC_RECORD.exists():
        return None, "no record"
    rec = {}
    for ln in TRAFFIC_RECORD.read_text().splitlines():
        if "=" in ln and not ln.lstrip().startswith("#"):
            k, v = ln.split("=", 1)
            rec[k.strip()] = v.strip()
    if rec.get("kernel") != kernel or rec.get("workload") != workload:
        return None, "record is for another kernel/workload"
    if rec.get("source_sha256") != kernel_source_sha():
        return None, f"stale: kernel sources changed since the capture at commit {rec.get('commit', '?')}"
    try:
        return float(rec["dram_bytes_read"]) + float(rec["dram_bytes_write"]), f"ncu capture at commit {rec.get('commit', '?')}"
    except (KeyError, ValueError):
        return None, "malformed record"


def eff_ops(N: int, F: int, T: int) -> float:
    return 8.0 * (N * (N + 1) // 2) * F * T


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.t_begin = None    # samples before begin() (taken while the device warms up) are not reported
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                if self.t_begin is not None:
                    self.samples.append(mhz)
                    for k, bit in names.items():
                        if mask & bit:
                            self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self, recording: bool = True):
        """recording=False: the thread polls but keeps nothing until begin() (NVML start-up and the thread start stay
        out of the gap between the warm-up and the timed region: after some ten milliseconds of idling the part needs
        about fifteen 0.3 ms steps to get back to its full speed)."""
        if recording:
            self.t_begin = time.perf_counter()
        if self.nv is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def begin(self):
        self.t_begin = time.perf_counter()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


def oracle_sample_tops(N, F, T, seed):
    """Times oracle.level1 on an (N, F, T) iid sample; returns (TOPS, seconds, threads)."""
    import oracle
    import workloads
    packed = workloads.iid_gaussian(N, F, T, seed)
    t0 = time.perf_counter()
    oracle.level1(packed)
    dt = time.perf_counter() - t0
    return eff_ops(N, F, T) / dt / 1e12, dt, oracle.threads()


def config_table(corr, dev, peaks, reps=20):
    """ms, effective TOPS, GB/s and the fraction of the bounding roofline for every shape of TABLE_SHAPES.
    Inputs are random bytes made on the device (every byte is a legal sample; timing does not depend on values),
    two rotating buffers (eight for small inputs) so that successive calls do not find their input in L2."""
    import torch
    int8_peak = 2.0 * float(peaks["bf16_tflops"])
    hbm_peak = float(peaks["hbm_gbs"])
    out = {}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for label, N, F, T, acc in TABLE_SHAPES:
        plan = corr.Plan(N, F, T)
        nbuf = 2 if N * F * T >= (64 << 20) else 8
        ins = [torch.randint(0, 256, (T, F, N), dtype=torch.uint8, device=dev) for _ in range(nbuf)]
        vis = torch.zeros((F, plan.baselines, 2), dtype=torch.int32, device=dev)
        # warm-up: 3 calls, then as many as make 8 ms of work (after the allocations above the part has idled, and it
        # takes some 5 ms of load to get back to full speed)
        e0.record()
        for i in range(3):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        e1.record()
        torch.cuda.synchronize(dev)
        for i in range(min(400, int(8.0 / max(e0.elapsed_time(e1) / 3, 1e-3)))):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        torch.cuda.synchronize(dev)
        e0.record()
        for i in range(reps):
            plan.execute(ins[i % nbuf], vis, accumulate=bool(acc))
        e1.record()
        torch.cuda.synchronize(dev)
        ms = e0.elapsed_time(e1) / reps
        tops = eff_ops(N, F, T) / (ms * 1e-3) / 1e12
        gbs = (N * F * T + vis.numel() * 4 * (2 if acc else 1)) / (ms * 1e-3) / 1e9
        # 4 (N + 1) ops per input byte against the ridge int8_peak / hbm_peak: HBM-bound below it
        hbm_bound = 4.0 * (N + 1) < int8_peak * 1e12 / (hbm_peak * 1e9)
        row = {"N": N, "F": F, "T": T, "ms": round(ms, 5), "value": round(tops, 2), "gbs": round(gbs, 1),
               "path": plan.info["path"], "bound": "hbm" if hbm_bound else "tensor",
               "frac": round(gbs / hbm_peak if hbm_bound else tops / int8_peak, 4),
               "frac_of_nominal_4500": round(tops / NOMINAL_INT8_TOPS, 4)}
        if label == "cfg1":
            row["bound"] = "launch latency (64 KB of input)"
        out[label] = row
        plan.close()
        del ins, vis
        torch.cuda.empty_cache()
    return out


def run_reference(args, cfg):
    """The reference arm for this tier is the CPU oracle (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    Fs, Ts = 1, 1024  # bounded sample of the same workload per step: 1 channel, 1024 samples
    for _ in range(args.warmup):
        oracle_sample_tops(cfg.N, Fs, Ts, cfg.seed0)
    total, threads = 0.0, 1
    for _ in range(args.steps):
        _, dt, threads = oracle_sample_tops(cfg.N, Fs, Ts, cfg.seed0)  # times the oracle call only
        total += dt
    value = eff_ops(cfg.N, Fs, Ts) * args.steps / total / 1e12
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "TOPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8",
        "data": "synthetic",
        "config": {"workload": f"{args.config} N={cfg.N} F={cfg.F} T={cfg.T} ({cfg.kind} recipe of workloads/, DESIGN.md section 4)",
                   "sample_per_step": f"N={cfg.N}, F={Fs}, T={Ts}"},
        "cpu_baseline": {"value": value, "unit": "TOPS", "cores": threads, "kind": "oracle",
                         "sample": f"oracle.level1 on N={cfg.N}, F={Fs}, T={Ts} per step"},
        "e2e": {"value": value, "unit": "TOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg3", help="workload (BASELINE.json config name)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sustained-seconds", type=float, default=2.5,
                    help="length of the sustained leg on the same workload (N=1 only; 0 = skip)")
    ap.add_argument("--no-table", action="store_true", help="skip the per-config / N-sweep table (N=1 only)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    import workloads
    cfg = workloads.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import numpy as np
    import torch
    import torch.distributed as dist

    import __graft_entry__
    import paper_1503_06203_b200 as corr
    from paper_1503_06203_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        __graft_entry__.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    corr.load_library()  # fails loudly if the CUDA library is missing: no fallback

    N, F, T = cfg.N, cfg.F, cfg.T
    NBUF = 3  # rotate distinct inputs; each input (134 MB) + output (134 MB) already exceeds L2
    host_inputs = [workloads.generate(cfg, 0)]
    for k in range(1, NBUF):
        host_inputs.append(workloads.iid_gaussian(N, F, T, seed=cfg.seed0 + 100 * (rank + 1) + k)
                           if cfg.kind == "iid" else workloads.generate(cfg, k % cfg.calls))
    dev_inputs = [torch.from_numpy(h).to(dev) for h in host_inputs]
    plan = corr.Plan(N, F, T)
    vis = plan.new_vis(dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # the int8 ceiling of THIS device: a bare issue loop of the hot path's own tcgen05.mma.kind::i8 (~3 ms each).  Measured
    # before the timed region (it also brings the part out of its idle clocks, which W = 5 steps of 0.3 ms do not)
    sampler = ClockSampler(local_rank)
    sampler.start(recording=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    int8_measured = max(corr.corr_measure_int8_tops(20000), corr.corr_measure_int8_tops(20000))
    for i in range(args.warmup):
        plan.execute(dev_inputs[i % NBUF], vis)
    barrier()
    sampler.begin()
    e0.record(stream)
    for i in range(args.steps):
        plan.execute(dev_inputs[i % NBUF], vis)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms_total = shard.max_over_ranks(ms_total, dev)
    ms_per_step = ms_total / args.steps
    value = eff_ops(N, F, T) * world / (ms_per_step * 1e-3) / 1e12

    # ---- sustained leg: the same step back to back for >= 2 s (the headline above is a burst of a few ms, during
    #      which the part holds its boost clock; under sustained load it is power-capped)
    sustained = None
    if world == 1 and args.sustained_seconds > 0:
        n_sus = max(args.steps, int(args.sustained_seconds * 1e3 / ms_per_step))
        sampler_s = ClockSampler(local_rank)
        torch.cuda.synchronize(dev)
        sampler_s.start()
        e0.record(stream)
        for i in range(n_sus):
            plan.execute(dev_inputs[i % NBUF], vis)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        ms_sus = e0.elapsed_time(e1) / n_sus
        sustained = {"value": eff_ops(N, F, T) / (ms_sus * 1e-3) / 1e12, "unit": "TOPS", "steps": n_sus,
                     "ms_per_step": ms_sus, "seconds": ms_sus * n_sus * 1e-3, "clocks": sampler_s.stop()}

    # ---- per-config table: the five BASELINE.json shapes and the N sweep, same process, device-timed
    table = None
    if world == 1 and not args.no_table:
        table = config_table(corr, dev, measured_peaks()[0])

    # ---- e2e: host buffers through the library's host API, copies inside the timed region.  Streaming use
    #      (corr_submit_host per step, one corr_wait_host at the end): every step copies its 134 MB in from pinned
    #      host memory and its 134 MB result back out; successive steps overlap on the PCIe link.
    ph = [torch.from_numpy(h).pin_memory() for h in host_inputs[:2]]
    vhs = [torch.empty((F, plan.baselines, 2), dtype=torch.int32).pin_memory() for _ in range(2)]
    vh = vhs[0]
    plan.execute_host(ph[0], vhs[0])          # warm-up of both forms (plans, staging buffers, streams are created lazily)
    plan.submit_host(ph[1], vhs[1])
    plan.submit_host(ph[0], vhs[0])
    plan.wait_host()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        plan.submit_host(ph[i % 2], vhs[i % 2])
    plan.wait_host()
    torch.cuda.synchronize(dev)
    e2e_s = (time.perf_counter() - t0) / args.e2e_steps
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        plan.execute_host(ph[i % 2], vhs[i % 2])   # blocking variant: each call waits for its own result
    torch.cuda.synchronize(dev)
    e2e_blocking_s = (time.perf_counter() - t0) / args.e2e_steps
    e2e_s = shard.max_over_ranks(e2e_s, dev)
    e2e_value = eff_ops(N, F, T) * world / e2e_s / 1e12
    # ---- what the host link gives on this box (PAPER.md:129 lower panel is the paper's own I/O concern): one pinned
    #      copy of the step's input in, one of its output out, alone and both at once on two streams
    link = None
    if world == 1:
        s_a, s_b = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        d_in, d_out = torch.empty_like(dev_inputs[0]), vis
        def timed(h2d, d2h):
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            if h2d:
                with torch.cuda.stream(s_a):
                    d_in.copy_(ph[0], non_blocking=True)
            if d2h:
                with torch.cuda.stream(s_b):
                    vhs[1].copy_(d_out, non_blocking=True)
            torch.cuda.synchronize(dev)
            return time.perf_counter() - t0
        for _ in range(2):
            t_in, t_out, t_both = timed(True, False), timed(False, True), timed(True, True)
        b_in, b_out = float(N * F * T), float(vis.numel() * 4)
        link = {"h2d_gbs": b_in / t_in / 1e9, "d2h_gbs": b_out / t_out / 1e9,
                "both_at_once_ms": t_both * 1e3, "both_at_once_gbs_total": (b_in + b_out) / t_both / 1e9,
                "e2e_gbs_total": (b_in + b_out) / e2e_s / 1e9,
                "note": "one monolithic pinned copy per direction; e2e interleaves channel-group copies in both directions"}
    checksum = int(vh.numpy()[0, :8, 0].astype(np.int64).sum())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, peaks_kind = measured_peaks()
    int8_peak = 2.0 * float(peaks["bf16_tflops"])  # dense int8 : bf16 nominal ratio is 2 (4.5 / 2.25 PF)
    kernel_ms = ms_per_step  # one kernel launch per step; launch gaps are inside the figure
    achieved = eff_ops(N, F, T) / (kernel_ms * 1e-3) / 1e12
    path = plan.info["path"]
    if path == corr.PATH_TCGEN05:
        variant = os.environ.get("CORR_TC_VARIANT", "3")
        kernel = {"1": "corr_tc_kernel", "5": "corr_tc5_kernel"}.get(variant, "corr_tc3_kernel")
        traffic, traffic_source = recorded_traffic(kernel, args.config)
        roofline = {
            "bound": "tensor", "achieved": achieved, "peak": int8_peak, "unit": "TOP/s", "frac": achieved / int8_peak,
            "traffic": traffic, "traffic_source": traffic_source,
            "peak_source": f"2 x bf16_tflops burst of MEASURED_PEAKS.json ({peaks_kind}); int8:bf16 nominal ratio 2",
            "frac_of_nominal_4500": achieved / NOMINAL_INT8_TOPS,
            "int8_issue_loop_tops": int8_measured, "frac_of_int8_issue_loop": achieved / int8_measured,
            # the sustained leg against the sustained denominator (both power-capped); burst against burst is `frac`
            "frac_of_sustained": (sustained["value"] / (2.0 * float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])))
                                  if sustained else None),
            "kernel": kernel, "kernel_ms": kernel_ms,
            "algorithmic_ops_per_launch": eff_ops(N, F, T),
        }
    else:
        # small-N paths: one input byte per (sample, input) in, the (tiny) triangle out
        alg_bytes = float(N * F * T + vis.numel() * 4)
        gbs = alg_bytes / (kernel_ms * 1e-3) / 1e9
        roofline = {
            "bound": "hbm", "achieved": gbs, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
            "frac": gbs / float(peaks["hbm_gbs"]), "traffic": None,
            "peak_source": f"hbm_gbs of MEASURED_PEAKS.json ({peaks_kind})",
            "kernel": "corr_imma_kernel" if path == corr.PATH_IMMA else "corr_dp4a_kernel", "kernel_ms": kernel_ms,
            "algorithmic_bytes_per_launch": alg_bytes,
        }
    cpu_baseline = None
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        Fs = min(F, 4)
        v, dt, threads = oracle_sample_tops(N, Fs, T, cfg.seed0)
        cpu_baseline = {"value": v, "unit": "TOPS", "cores": threads, "kind": "oracle",
                        "sample": f"oracle.level1 on the first {Fs} of {F} channels of the workload shape "
                                  f"(N={N}, T={T}); {dt:.2f} s wall"}

    line = {
        "metric": METRIC, "value": value, "unit": "TOPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": {"workload": f"{args.config} N={N} F={F} T={T} ({cfg.kind} recipe of workloads/, DESIGN.md section 4), one batch per GPU",
                   "l2": f"{NBUF} rotating inputs of {N * F * T / 1e6:.0f} MB each + {vis.numel() * 4 / 1e6:.0f} MB output per step: larger than the 126 MB L2",
                   "path": plan.info},
        "pct_of_int8_peak": {"nominal_4500": 100 * value / world / NOMINAL_INT8_TOPS,
                             "measured_2x_bf16_burst": 100 * value / world / int8_peak},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "TOPS", "h2d_bytes_per_step": N * F * T,
                "d2h_bytes_per_step": vis.numel() * 4, "ms_per_step": e2e_s * 1e3, "checksum": checksum,
                "api": "corr_submit_host per step + corr_wait_host", "blocking_ms_per_step": e2e_blocking_s * 1e3,
                "blocking_value": eff_ops(N, F, T) * world / e2e_blocking_s / 1e12, "link": link},
        "gpu_launches": args.steps * plan.info["kernels"],
        "roofline": roofline,
        "sustained": sustained,
        "configs": table,
        "cpu_baseline": cpu_baseline,
        "paper_context": "5.6 effective TOPS on a 4.3 TOPS AMD R9 280X (PAPER.md:15); another machine",
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
