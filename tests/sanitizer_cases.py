"""Small shapes that reach every synchronisation mechanism of the CUDA path, for compute-sanitizer
(SURVEY section 4 tier 5): one tool per run, e.g.

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Every case is also compared with the CPU oracle (the script exits non-zero on a mismatch), so a sanitizer run is a
parity run too.  Not collected by pytest (no test_ prefix): the sanitizers slow the kernels down by 10-100x.

Where compute-sanitizer is not available (it is closed on the pool this was developed on, profiles/r02_sanitizer.md),
`python tests/sanitizer_cases.py --repeat 50` runs every case that many times with fresh seeds instead: a race in the
flag / barrier protocols shows up as a mismatch against the oracle or as a hang (run it under `timeout`).
"""
import os
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import numpy as np
import torch

import oracle
import paper_1503_06203_b200 as corr
import workloads


def run(name, packed, path, variant=None, accumulate=False, env=None):
    if variant:
        os.environ["CORR_TC_VARIANT"] = variant
    else:
        os.environ.pop("CORR_TC_VARIANT", None)
    for k in ("CORR_TCD_MAX_N", "CORR_TCD_SHARES"):
        os.environ.pop(k, None)
    os.environ.update(env or {})
    T, F, N = packed.shape
    want = oracle.level1(packed)
    with corr.Plan(N, F, T, path) as plan:
        dev = torch.from_numpy(packed).cuda()
        vis = plan.execute(dev)
        if accumulate:
            plan.execute(dev, vis, accumulate=True)
            want = 2 * want
        torch.cuda.synchronize()
        got = vis.cpu().numpy()
        info = dict(plan.info)
    ok = np.array_equal(got, want)
    print(f"{name}: N={N} F={F} T={T} units={info['units']} ctas={info['ctas']} {'bit-exact' if ok else 'MISMATCH'}", flush=True)
    return ok


def main():
    corr.load_library()
    oracle.build()
    repeat = int(sys.argv[sys.argv.index("--repeat") + 1]) if "--repeat" in sys.argv else 1
    ok = True
    for rep in range(repeat):
        ok &= cases(1000 * rep)
    sys.exit(0 if ok else 1)


def cases(s0):
    ok = True
    # corr_tc3_kernel: cut units (claim / stored flags, bulk reduce-add), whole units + early pieces, transposed tiles
    ok &= run("tc3 cut units", workloads.uniform_bytes(256, 2, 20000, seed=s0 + 1), corr.PATH_TCGEN05, "3", accumulate=True)
    ok &= run("tc3 transposed tiles, ragged N and T", workloads.uniform_bytes(400, 2, 777, seed=s0 + 2), corr.PATH_TCGEN05, "3")
    ok &= run("tc3 whole waves + tail pieces", workloads.uniform_bytes(1024, 5, 1024, seed=s0 + 3), corr.PATH_TCGEN05, "3")
    # corr_tc5_kernel: the same schedule, per-element sums through shared memory of both CTAs of the pair
    ok &= run("tc5 cut units", workloads.uniform_bytes(256, 2, 20000, seed=s0 + 4), corr.PATH_TCGEN05, "5", accumulate=True)
    ok &= run("tc5 transposed tiles, ragged N and T", workloads.uniform_bytes(400, 2, 777, seed=s0 + 5), corr.PATH_TCGEN05, "5")
    # corr_tcd_kernel: one CTA per channel's block (N <= 128), padded stream
    ok &= run("tcd one block per channel", workloads.uniform_bytes(100, 3, 3000, seed=s0 + 6), corr.PATH_TCGEN05, None)
    # ... equal shares (every segment added into a cleared output), two channels of 64 per tile, many segments per CTA
    ok &= run("tcd equal shares", workloads.uniform_bytes(128, 5, 9000, seed=s0 + 11), corr.PATH_TCGEN05, None,
              accumulate=True, env={"CORR_TCD_SHARES": "1"})
    ok &= run("tcd two channels per tile", workloads.uniform_bytes(64, 6, 5000, seed=s0 + 12), corr.PATH_AUTO, None,
              env={"CORR_TCD_SHARES": "1"})
    ok &= run("tcd many units per CTA", workloads.uniform_bytes(128, 600, 300, seed=s0 + 13), corr.PATH_TCGEN05, None,
              env={"CORR_TCD_SHARES": "0"})
    # corr_tcd_kernel<true>: off-diagonal blocks, the row image handed from one half of a block to the other (named
    # barriers 2 / 3), (ring position, unpack group) barriers of the double-stage ring
    ok &= run("tcd off-diagonal blocks, units", workloads.uniform_bytes(256, 70, 700, seed=s0 + 14), corr.PATH_TCGEN05, None,
              env={"CORR_TCD_MAX_N": "512", "CORR_TCD_SHARES": "0"})
    ok &= run("tcd off-diagonal blocks, shares", workloads.uniform_bytes(400, 3, 3000, seed=s0 + 15), corr.PATH_TCGEN05, None,
              accumulate=True, env={"CORR_TCD_MAX_N": "512", "CORR_TCD_SHARES": "1"})
    # corr_imma_kernel: several chunks per strip (shared-memory atomics, global atomics)
    ok &= run("imma several chunks", workloads.uniform_bytes(32, 9, 4099, seed=s0 + 7), corr.PATH_IMMA)
    ok &= run("dp4a", workloads.uniform_bytes(17, 3, 650, seed=s0 + 8), corr.PATH_DP4A)
    # time shift and gated correlation
    packed = workloads.uniform_bytes(144, 2, 1500, seed=s0 + 9)
    lags = np.random.default_rng(s0 + 9).integers(-40, 41, size=144).astype(np.int32)
    got = corr.time_shift(torch.from_numpy(packed).cuda(), torch.from_numpy(lags).cuda()).cpu().numpy()
    same = np.array_equal(got, oracle.time_shift(packed, lags))
    print(f"time shift: {'byte-exact' if same else 'MISMATCH'}", flush=True)
    ok &= same
    gate = (np.arange(1500) // 50 % 3).astype(np.int32) - (np.arange(1500) % 7 == 0)
    with corr.Plan(144, 2, 1500) as plan:
        got = plan.execute_gated(torch.from_numpy(packed).cuda(), gate, 3).cpu().numpy()
    same = np.array_equal(got, oracle.gated(packed, gate, 3))
    print(f"gated: {'bit-exact' if same else 'MISMATCH'}", flush=True)
    ok &= same
    return ok


if __name__ == "__main__":
    main()
