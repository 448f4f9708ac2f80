"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

Integer work, so the bar is exact equality (np.array_equal) everywhere; there is no tolerance.
Every input is seeded and synthetic (workloads/).  Nothing here reads /root/reference.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def corr():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import __graft_entry__
    __graft_entry__.build()
    import paper_1503_06203_b200 as c
    c.load_library()
    return c


def _run(corr, packed, path=0, accumulate_into=None, prefill=None):
    import torch
    T, F, N = packed.shape
    with corr.Plan(N, F, T, path) as plan:
        dev = torch.from_numpy(packed).cuda()
        if accumulate_into is not None:
            vis = torch.from_numpy(accumulate_into).cuda()
            plan.execute(dev, vis, accumulate=True)
        else:
            vis = plan.new_vis()
            if prefill is not None:
                vis.fill_(prefill)
            plan.execute(dev, vis, accumulate=False)
        torch.cuda.synchronize()
        return vis.cpu().numpy(), dict(plan.info)


# ------------------------------------------------------------------ tiny shapes, both paths
TINY_N = [1, 2, 3, 5, 15, 16, 17, 31, 32, 33, 64, 100, 127, 128, 129]
TINY_T = [1, 2, 3, 31, 32, 33, 63, 64, 65, 255, 256, 257]


@pytest.mark.parametrize("N", TINY_N)
def test_dp4a_tiny_shapes(corr, oracle, N):
    for F in (1, 3):
        for T in TINY_T:
            packed = workloads.uniform_bytes(N, F, T, seed=N * 7919 + F * 31 + T)
            got, info = _run(corr, packed, corr.PATH_DP4A, prefill=-559038737)
            assert info["path"] == corr.PATH_DP4A
            assert np.array_equal(got, oracle.level0(packed)), (N, F, T)


@pytest.mark.parametrize("N", [16, 32, 48, 112, 128, 144, 256, 272, 400])
def test_tcgen05_small_shapes(corr, oracle, N):
    for F in (1, 3):
        for T in (1, 31, 32, 33, 64, 65, 127, 128, 129, 200, 1000):
            packed = workloads.uniform_bytes(N, F, T, seed=N * 104729 + F * 31 + T)
            got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=-559038737)
            assert info["path"] == corr.PATH_TCGEN05
            assert np.array_equal(got, oracle.level1(packed)), (N, F, T)


@pytest.mark.parametrize("N", [16, 32, 48, 64])
def test_imma_small_n(corr, oracle, N):
    # warp-MMA path (whole channels per CTA): ragged T, F not a multiple of the channels per strip,
    # several time chunks (atomic accumulation), stale output, accumulate flag, extreme bytes
    for F in (1, 3, 9):
        for T in TINY_T + [1000, 4099]:
            packed = workloads.uniform_bytes(N, F, T, seed=N * 31337 + F * 31 + T)
            got, info = _run(corr, packed, corr.PATH_IMMA, prefill=-559038737)
            assert info["path"] == corr.PATH_IMMA
            assert np.array_equal(got, oracle.level1(packed)), (N, F, T)
    packed = workloads.iid_gaussian(N, 5, 70000, seed=N)          # several chunks per channel
    want = oracle.level1(packed)
    got, info = _run(corr, packed, corr.PATH_IMMA, prefill=123)
    assert info["slices"] > 1
    assert np.array_equal(got, want)
    again, _ = _run(corr, packed, corr.PATH_IMMA, accumulate_into=got.copy())
    assert np.array_equal(again, 2 * want)
    small = workloads.uniform_bytes(N, 2, 300, seed=7)             # one chunk: read-add-store
    w2 = oracle.level1(small)
    acc, info = _run(corr, small, corr.PATH_IMMA, accumulate_into=w2.copy())
    assert info["slices"] == 1 and np.array_equal(acc, 2 * w2)
    for byte in (0x00, 0xFF, 0x0F, 0xF0):
        packed = np.full((5000, 3, N), byte, np.uint8)
        got, _ = _run(corr, packed, corr.PATH_IMMA)
        assert np.array_equal(got, oracle.level1(packed)), (N, hex(byte))
    auto, info = _run(corr, small)   # AUTO picks this path for N = 16, 32, 48 (N = 64 with an even F: two channels per tcgen05 tile)
    assert info["path"] == (corr.PATH_TCGEN05 if N == 64 else corr.PATH_IMMA) and np.array_equal(auto, w2)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 15, 17, 31, 33, 47, 49, 63, 65, 100, 127, 129, 200, 255, 257, 1000])
def test_n_not_a_multiple_of_16(corr, oracle, N):
    # the TMA-fed paths read a copy of the stream padded to the next multiple of 16 inputs with stored zeros;
    # the output keeps the caller's N.  Automatic path, and both tensor-core paths forced where they apply.
    for F in (1, 3):
        for T in (1, 33, 257, 1000):
            packed = workloads.uniform_bytes(N, F, T, seed=N * 7 + F + T)
            want = oracle.level1(packed)
            got, info = _run(corr, packed, prefill=-559038737)
            assert info["path"] == (corr.PATH_IMMA if N <= 64 else corr.PATH_TCGEN05)
            assert np.array_equal(got, want), (N, F, T, info)
            both, _ = _run(corr, packed, accumulate_into=got.copy())
            assert np.array_equal(both, 2 * want), (N, F, T, "accumulate")
    packed = workloads.uniform_bytes(N, 2, 300, seed=N)
    got, _ = _run(corr, packed, corr.PATH_TCGEN05)                 # small N through the big-tile path too
    assert np.array_equal(got, oracle.level1(packed))
    # an input pointer that is not 16-byte aligned is fine when the stream is copied anyway
    import torch
    T, F = 100, 2
    packed = workloads.uniform_bytes(N, F, T, seed=1)
    with corr.Plan(N, F, T) as plan:
        buf = torch.zeros(packed.size + 64, dtype=torch.uint8, device="cuda")
        dev = buf[3:3 + packed.size].view(T, F, N)
        dev.copy_(torch.from_numpy(packed))
        vis = plan.execute(dev)
        torch.cuda.synchronize()
        assert np.array_equal(vis.cpu().numpy(), oracle.level1(packed))


def test_tcgen05_extreme_values(corr, oracle):
    # all samples -8-8i: largest products (16*-8 = -128 on both operands), Re = 128 T, Im = 0
    N, F, T = 256, 2, 4096
    packed = np.zeros((T, F, N), np.uint8)
    got, _ = _run(corr, packed, corr.PATH_TCGEN05)
    assert (got[..., 0] == 128 * T).all() and (got[..., 1] == 0).all()
    # alternating extreme pairs: x = -8-8i, y = -8+7i  ->  |Im| = 120 per sample
    packed[:, :, 1::2] = 0x0F
    got, _ = _run(corr, packed, corr.PATH_TCGEN05)
    assert np.array_equal(got, oracle.level1(packed))


def test_split_t_and_multi_wave(corr, oracle):
    # few tiles, long T  -> the plan splits T (atomic accumulation); many tiles -> several waves
    packed = workloads.iid_gaussian(256, 2, 20000, seed=77)   # 4 units on 74 CTA pairs: every unit is cut in many segments
    got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=123456)
    assert info["units"] < info["ctas"] // 2
    assert np.array_equal(got, oracle.level1(packed))
    packed = workloads.iid_gaussian(256, 1, 40000, seed=79)   # T > 32768: sliced for int32 headroom as well
    got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=-7)
    assert info["slices"] > 1
    assert np.array_equal(got, oracle.level1(packed))
    packed = workloads.iid_gaussian(1024, 8, 300, seed=78)
    got, info = _run(corr, packed, corr.PATH_TCGEN05)
    assert info["units"] > info["ctas"] // (2 if info["tile_x"] == 256 else 1)   # more than one wave
    assert np.array_equal(got, oracle.level1(packed))


@pytest.mark.parametrize("path_name", ["dp4a", "tcgen05"])
def test_accumulate_and_stale_output(corr, oracle, path_name):
    path = getattr(corr, "PATH_" + path_name.upper())
    N, F = (144, 2)
    a = workloads.uniform_bytes(N, F, 500, seed=1)
    b = workloads.uniform_bytes(N, F, 500, seed=2)
    want = oracle.level1(np.concatenate([a, b], axis=0))
    first, _ = _run(corr, a, path, prefill=-559038737)      # flag 0 ignores stale contents (P11)
    assert np.array_equal(first, oracle.level1(a))
    both, _ = _run(corr, b, path, accumulate_into=first.copy())  # flag 1 adds (P7)
    assert np.array_equal(both, want)
    garbage = np.full_like(want, -559038737)
    acc, _ = _run(corr, a, path, accumulate_into=garbage.copy())  # garbage + corr mod 2^32
    exp = (garbage.astype(np.int64) + oracle.level1(a).astype(np.int64) + 2**31) % 2**32 - 2**31
    assert np.array_equal(acc.astype(np.int64), exp)


def test_determinism(corr):
    packed = workloads.iid_gaussian(512, 3, 3000, seed=5)
    r1, _ = _run(corr, packed, corr.PATH_TCGEN05)
    r2, _ = _run(corr, packed, corr.PATH_TCGEN05)
    assert np.array_equal(r1, r2)
    r3, _ = _run(corr, packed, corr.PATH_DP4A)
    assert np.array_equal(r1, r3)
    packed = workloads.iid_gaussian(64, 7, 3000, seed=6)
    assert np.array_equal(_run(corr, packed, corr.PATH_IMMA)[0], _run(corr, packed, corr.PATH_DP4A)[0])
    assert np.array_equal(_run(corr, packed, corr.PATH_IMMA)[0], _run(corr, packed, corr.PATH_TCGEN05)[0])


@pytest.mark.parametrize("F", [2, 6, 16, 3, 5, 63])
def test_n64_two_channels_per_tile(corr, oracle, F):
    # N = 64, even F: AUTO runs corr_tcd_kernel (one CTA per 128-block) on the stream seen as [T][F/2][128] and writes the two
    # diagonal 64-blocks of each tile as channels 2f, 2f + 1; an odd F from 5 on as well (the last tile holds one channel
    # and zeros from beyond the row), a small odd F stays on the warp-MMA kernel.  Ragged T, split T,
    # stale output, accumulation, extreme bytes.
    for T in (1, 63, 300, 4099, 70000 if F == 2 else 1000):
        packed = workloads.uniform_bytes(64, F, T, seed=64 * F + T)
        want = oracle.level1(packed)
        got, info = _run(corr, packed, corr.PATH_AUTO, prefill=-559038737)
        assert info["path"] == (corr.PATH_TCGEN05 if (F % 2 == 0 or F >= 5) else corr.PATH_IMMA)
        assert np.array_equal(got, want), (F, T)
        again, _ = _run(corr, packed, corr.PATH_AUTO, accumulate_into=got.copy())
        assert np.array_equal(again, 2 * want), (F, T, "accumulate")
    for byte in (0x00, 0xFF):
        packed = np.full((2048, F, 64), byte, np.uint8)
        got, _ = _run(corr, packed, corr.PATH_AUTO)
        assert np.array_equal(got, oracle.level1(packed)), (F, hex(byte))


@pytest.mark.parametrize("shape", [(128, 3, 1000), (128, 1, 70000), (128, 310, 300), (112, 2, 257), (100, 5, 4099),
                                   (96, 2, 64), (17, 3, 900), (128, 2, 1), (65, 4, 33000)])
@pytest.mark.parametrize("shares", ["auto", "1", "0"])
def test_diagonal_block_kernel(corr, oracle, shape, shares, monkeypatch):
    # N <= 128 on the tcgen05 path is one 128-block per channel: corr_tcd_kernel (A operand in TMEM, two groups of
    # unpack warps, row images of the upper triangle sent as bulk copies).  Ragged N (also N % 16 != 0 through the padded
    # stream) and T, T split into slices of whole groups of 256 samples, more units than SMs, stale output, accumulation.
    # Both schedules: units (channel, T-slice) dealt round-robin, and equal shares of all groups of all channels added
    # into a cleared output (CORR_TCD_SHARES forces one; the plan chooses by a cost model otherwise)
    if shares != "auto":
        monkeypatch.setenv("CORR_TCD_SHARES", shares)
    N, F, T = shape
    packed = workloads.uniform_bytes(N, F, T, seed=N * 7 + F + T)
    want = oracle.level1(packed)
    got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=-559038737)
    assert info["path"] == corr.PATH_TCGEN05 and info["tiles_per_channel"] == 1
    assert np.array_equal(got, want), shape
    again, _ = _run(corr, packed, corr.PATH_TCGEN05, accumulate_into=got.copy())
    assert np.array_equal(again, 2 * want), (shape, "accumulate")
    if T >= 900:
        for byte in (0x00, 0xFF, 0x0F, 0xF0):                  # largest magnitudes everywhere
            packed = np.full((min(T, 5000), min(F, 3), N), byte, np.uint8)
            got, _ = _run(corr, packed, corr.PATH_TCGEN05)
            assert np.array_equal(got, oracle.level1(packed)), (shape, hex(byte))


@pytest.mark.parametrize("shape", [(100, 64, 3000), (100, 4, 777), (113, 16, 1000), (65, 16, 20000), (72, 2, 300), (97, 32, 257),
                                   (104, 6, 5000), (37, 16, 3000), (37, 128, 700), (50, 8, 20000), (20, 12, 1000), (10, 8, 300),
                                   (5, 16, 257), (3, 32, 1000), (1, 16, 100), (56, 6, 900), (24, 10, 4000)])
def test_unpadded_stream_through_aligned_windows(corr, oracle, shape, monkeypatch):
    # N % 16 != 0, N <= 113 and rows of a multiple of 16 bytes: corr_tcd_kernel reads the stream as it is, channel f through
    # the 128-byte window at column f N rounded down to 16 (its inputs are rows / columns (f N) % 16 ... of the tile; what the
    # window holds of the neighbouring channels is computed and dropped).  N <= 56: several whole channels per window, tile g
    # holds channels g c ... g c + c - 1, c = 113 // N (and AUTO takes this route instead of a padded copy + the warp-MMA
    # kernel).  Both schedules; a buffer that is not 16-byte aligned takes the padded copy instead (same bits), or is
    # refused when a window holds several channels
    import torch
    N, F, T = shape
    packed = workloads.uniform_bytes(N, F, T, seed=N + F + T)
    want = oracle.level1(packed)
    for shares in ("0", "1"):
        monkeypatch.setenv("CORR_TCD_SHARES", shares)
        for off in (0, 3):
            with corr.Plan(N, F, T, corr.PATH_AUTO if N < 64 else corr.PATH_TCGEN05) as plan:
                assert plan.info["kernels"] == 1 and plan.info["path"] == corr.PATH_TCGEN05
                raw = torch.full((packed.size + 64,), 0x88, dtype=torch.uint8, device="cuda")
                dev = raw[off:off + packed.size].view(T, F, N)
                dev.copy_(torch.from_numpy(packed))
                vis = plan.new_vis()
                vis.fill_(-559038737)
                if off and N <= 56:
                    with pytest.raises(corr.CorrError, match="16-byte aligned"):
                        plan.execute(dev, vis)
                    continue
                plan.execute(dev, vis)
                torch.cuda.synchronize()
                assert np.array_equal(vis.cpu().numpy(), want), (shape, shares, off)
                plan.execute(dev, vis, accumulate=True)
                torch.cuda.synchronize()
                assert np.array_equal(vis.cpu().numpy(), 2 * want), (shape, shares, off, "accumulate")


@pytest.mark.parametrize("shares", ["0", "1"])
@pytest.mark.parametrize("shape", [(256, 3, 20000), (256, 40, 300), (272, 3, 777), (400, 1, 300), (512, 2, 257), (130, 5, 64),
                                   (200, 2, 5000), (192, 1, 1)])
def test_diagonal_block_kernel_with_off_diagonal_blocks(corr, oracle, shape, shares, monkeypatch):
    # corr_tcd_kernel<true>: several 128-blocks per channel (automatic for 128 < N <= 256 with long segments; here
    # CORR_TCD_MAX_N lets it take every shape): off-diagonal blocks load two packed blocks per stage and write all
    # 128 x 128 baselines, the row image is used by the two halves of a block in turn.  Ragged N (also N % 16 != 0) and T,
    # both schedules, stale output, accumulation
    monkeypatch.setenv("CORR_TCD_MAX_N", "512")
    monkeypatch.setenv("CORR_TCD_SHARES", shares)
    N, F, T = shape
    packed = workloads.uniform_bytes(N, F, T, seed=N * 5 + F + T)
    want = oracle.level1(packed)
    got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=-559038737)
    nb = (N + 127) // 128
    assert info["tiles_per_channel"] == nb * (nb + 1) // 2 and info["tile_x"] == 128
    assert np.array_equal(got, want), shape
    again, _ = _run(corr, packed, corr.PATH_TCGEN05, accumulate_into=got.copy())
    assert np.array_equal(again, 2 * want), (shape, "accumulate")


@pytest.mark.parametrize("variant", ["1", "3", "5"])
def test_every_tcgen05_kernel_variant(corr, oracle, variant, monkeypatch):
    # CORR_TC_VARIANT forces the kernel at plan creation: 1 single-CTA tiles with both operands in shared memory (round 1's kernel; N <= 128 runs corr_tcd_kernel unless this forces it), 3 CTA pair
    # with the A operand in TMEM (automatic above), 5 three products per complex MAC on the stored bytes with
    # fused per-element sums (offset route, Eq. 3).  Same bits from all of them, including ragged N (also
    # N % 16 != 0 through the padded stream), split T, cut units and accumulation.
    monkeypatch.setenv("CORR_TC_VARIANT", variant)
    for (N, F, T, seed) in [(272, 3, 1000, 11), (1024, 2, 333, 12), (256, 1, 40000, 13), (2048, 1, 640, 14), (100, 3, 500, 15),
                            (400, 2, 777, 16), (512, 4, 8192, 17)]:
        packed = workloads.uniform_bytes(N, F, T, seed=seed)
        want = oracle.level1(packed)
        got, info = _run(corr, packed, corr.PATH_TCGEN05, prefill=-559038737)
        assert np.array_equal(got, want), (variant, N, F, T)
        again, _ = _run(corr, packed, corr.PATH_TCGEN05, accumulate_into=got.copy())
        assert np.array_equal(again, 2 * want), (variant, N, F, T, "accumulate")
    # extreme values: all samples -8-8i (largest magnitudes everywhere) and the 0xFF byte (+7+7i)
    for byte in (0x00, 0xFF, 0x0F, 0xF0):
        packed = np.full((4096, 2, 256), byte, np.uint8)
        got, _ = _run(corr, packed, corr.PATH_TCGEN05)
        assert np.array_equal(got, oracle.level1(packed)), (variant, hex(byte))


def _fuzz_cases(seed, count):
    rng = np.random.default_rng(seed)
    for _ in range(count):
        kind = rng.integers(0, 4)
        if kind == 0:
            N = int(rng.choice([16, 32, 64]))                      # warp-MMA path
        elif kind == 1:
            N = int(rng.integers(1, 200))                          # dp4a path (or tcgen05 when N % 16 == 0, N >= 96)
        else:
            N = 16 * int(rng.integers(6, 90))                      # tcgen05 path: odd / even block counts, ragged blocks
        F = int(rng.integers(1, 6))
        T = int(rng.choice([1, 63, 64, 255, 256, 257, 1000, 3000, 5000])) + int(rng.integers(0, 3))
        if N > 700:
            T = min(T, 1100)
        yield N, F, T, bool(rng.integers(0, 2)), int(rng.integers(0, 1 << 30))


def test_fuzz_shapes(corr, oracle):
    # random shapes through the automatic path choice, overwrite then (sometimes) accumulate, stale output
    for N, F, T, acc, seed in _fuzz_cases(20240607, 40):
        packed = workloads.uniform_bytes(N, F, T, seed=seed)
        want = oracle.level1(packed)
        got, info = _run(corr, packed, prefill=-559038737)
        assert np.array_equal(got, want), (N, F, T, info)
        if acc:
            both, _ = _run(corr, packed, accumulate_into=got.copy())
            assert np.array_equal(both, 2 * want), (N, F, T, info, "accumulate")


def test_cuda_graph_replay(corr, oracle):
    # corr_execute only enqueues (kernels + memsets), so it can be captured; a replayed launch carries the
    # same call counter, which the schedule's flags must survive (the last CTA clears them)
    import torch
    for (N, F, T) in [(256, 2, 20000), (1024, 3, 700), (64, 5, 70000)]:   # cut units / whole waves + tail / chunked atomics
        packed = workloads.iid_gaussian(N, F, T, seed=N + F)
        want = oracle.level1(packed)
        with corr.Plan(N, F, T) as plan:
            dev = torch.from_numpy(packed).cuda()
            vis = plan.new_vis()
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                plan.execute(dev, vis, stream=side)          # warm-up outside the graph (tensor map, attributes)
                side.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    plan.execute(dev, vis, stream=side)
            for rep in range(3):
                vis.fill_(-559038737)
                g.replay()
                torch.cuda.synchronize()
                assert np.array_equal(vis.cpu().numpy(), want), (N, F, T, rep)


def test_execute_host(corr, oracle):
    import torch
    packed = workloads.iid_gaussian(160, 2, 700, seed=9)
    T, F, N = packed.shape
    with corr.Plan(N, F, T) as plan:
        ph = torch.from_numpy(packed).pin_memory()
        vh = torch.empty((F, plan.baselines, 2), dtype=torch.int32).pin_memory()
        plan.execute_host(ph, vh, accumulate=False)
        want = oracle.level1(packed)
        assert np.array_equal(vh.numpy(), want)
        plan.execute_host(ph, vh, accumulate=True)
        assert np.array_equal(vh.numpy(), 2 * want)


def test_execute_host_pipelined(corr, oracle):
    # >= 32 MB of transfers and F > 1: corr_execute_host pipelines copy-in | kernels | copy-out over channel groups
    import torch
    packed = workloads.iid_gaussian(1024, 6, 5500, seed=21)
    T, F, N = packed.shape
    want = oracle.level1(packed)
    with corr.Plan(N, F, T) as plan:
        ph = torch.from_numpy(packed).pin_memory()
        vh = torch.full((F, plan.baselines, 2), -559038737, dtype=torch.int32).pin_memory()
        plan.execute_host(ph, vh, accumulate=False)
        assert np.array_equal(vh.numpy(), want)
        plan.execute_host(ph, vh, accumulate=True)
        assert np.array_equal(vh.numpy(), 2 * want)
        pageable = np.empty_like(want)                     # pageable host memory works too (just slower)
        plan.execute_host(packed, pageable, accumulate=False)
        assert np.array_equal(pageable, want)


@pytest.mark.parametrize("shape", [(1024, 6, 5500), (160, 2, 700)])   # pipelined over channel groups / small single-stream path
def test_submit_host_streaming(corr, oracle, shape):
    # several calls in flight: distinct inputs and outputs, then an accumulating chain through one host buffer
    import torch
    N, F, T = shape
    ins = [workloads.iid_gaussian(N, F, T, seed=30 + k) for k in range(3)]
    wants = [oracle.level1(a) for a in ins]
    with corr.Plan(N, F, T) as plan:
        ph = [torch.from_numpy(a).pin_memory() for a in ins]
        vh = [torch.full((F, plan.baselines, 2), -1, dtype=torch.int32).pin_memory() for _ in ins]
        for k in range(3):
            plan.submit_host(ph[k], vh[k])
        plan.wait_host()
        for k in range(3):
            assert np.array_equal(vh[k].numpy(), wants[k]), (shape, k)
        acc = torch.zeros((F, plan.baselines, 2), dtype=torch.int32).pin_memory()
        for k in range(3):
            plan.submit_host(ph[k], acc, accumulate=True)
        plan.wait_host()
        assert np.array_equal(acc.numpy(), wants[0] + wants[1] + wants[2]), shape
        plan.execute_host(ph[0], acc)                    # the blocking call still works after streaming ones
        assert np.array_equal(acc.numpy(), wants[0])
        plan.submit_host(ph[1], acc, accumulate=True)    # ... and the two forms chain through one host buffer
        plan.execute_host(ph[2], acc, accumulate=True)
        assert np.array_equal(acc.numpy(), wants[0] + wants[1] + wants[2])
        for k in range(5):                               # more calls in flight than device images
            plan.submit_host(ph[k % 3], vh[k % 3])
        plan.wait_host()
        for k in range(3):
            assert np.array_equal(vh[k].numpy(), wants[k]), (shape, k, "second round")


def test_int32_headroom_edge(corr):
    # pin P10: the largest T the ABI takes, every sample -8-8i: Re = 128 * (2^24 - 1) =
    # 2 147 483 520 on every baseline, Im = 0, no wrap (closed form, PAPER.md:41-44 with constant input)
    import torch
    N, F, T = 16, 1, (1 << 24) - 1
    with corr.Plan(N, F, T) as plan:
        dev = torch.zeros((T, F, N), dtype=torch.uint8, device="cuda")
        vis = plan.execute(dev)
        torch.cuda.synchronize()
        got = vis.cpu().numpy()
    assert (got[..., 0] == 2147483520).all() and (got[..., 1] == 0).all()
    # the same length through the tcgen05 path (sliced for accumulator headroom), fewer samples to keep it short
    N, T = 128, 100000
    packed = np.zeros((T, 1, N), np.uint8)
    got, info = _run(corr, packed, corr.PATH_TCGEN05)
    assert info["slices"] > 1
    assert (got[..., 0] == 128 * T).all() and (got[..., 1] == 0).all()


def test_imma_ring_barriers_under_repetition(corr):
    # regression: with one barrier per ring position (six positions, four K-split groups) a group waited for the same
    # parity on every visit and, when TMA loads completed out of order, took another group's phase for its own: launch
    # failures in about half of such loops, at this size, after the pad copy.  300 calls, then the same bits as the
    # tcgen05 path
    import torch
    N, F, T = 24, 128, 65536
    dev = torch.randint(0, 256, (T, F, N), dtype=torch.uint8, device="cuda")
    with corr.Plan(N, F, T, corr.PATH_IMMA) as plan, corr.Plan(N, F, T, corr.PATH_TCGEN05) as ref:
        vis = plan.new_vis()
        for _ in range(300):
            plan.execute(dev, vis)
        want = ref.execute(dev)
        torch.cuda.synchronize()
        assert torch.equal(vis, want)


@pytest.mark.parametrize("N,F", [(16, 2368), (32, 592), (48, 296), (64, 296)])
def test_imma_headroom_when_the_strips_fill_the_gpu(corr, N, F):
    # The warp-MMA path accumulates 256 * sum (x16 planes) per time chunk, so a chunk must stay below 65536
    # samples whatever the wave-fill heuristic would like: F is chosen so that ONE chunk per strip already fills
    # whole waves (148 or 296 CTAs), T = 70000 of the byte 0x00 (-8-8i) would then wrap an int32 accumulator
    # (256 * 128 * 70000 > 2^31).  Closed form (pin P2): Re = 128 T, Im = 0 on every baseline.
    import torch
    T = 70000
    with corr.Plan(N, F, T, corr.PATH_IMMA) as plan:   # (AUTO takes N = 64 with an even F to the tcgen05 tiles)
        assert plan.info["path"] == corr.PATH_IMMA
        assert plan.info["slices"] >= 2, plan.info
        dev = torch.zeros((T, F, N), dtype=torch.uint8, device="cuda")
        vis = plan.new_vis()
        vis.fill_(-559038737)
        plan.execute(dev, vis)
        torch.cuda.synchronize()
        assert bool((vis[..., 0] == 128 * T).all()) and bool((vis[..., 1] == 0).all())
        dev.fill_(0xFF)                                   # +7+7i: Re = 98 T
        plan.execute(dev, vis, accumulate=True)
        torch.cuda.synchronize()
        assert bool((vis[..., 0] == (128 + 98) * T).all()) and bool((vis[..., 1] == 0).all())


def test_concurrent_plans_with_cut_units(corr, oracle):
    # Two plans whose units are all cut into pieces (4 and 6 units on 74 CTA pairs), run at the same time on two
    # streams, and again while an unrelated long kernel holds part of the GPU: the pieces of a cut unit order
    # their store through a claim flag that only ever waits for a CTA that is already running, so this must
    # finish (it would hang if a piece waited for a CTA that is not resident) and be bit-exact.
    import torch
    shapes = [(256, 2, 20000, 301), (384, 1, 12000, 302)]
    packs = [workloads.iid_gaussian(N, F, T, seed=sd) for (N, F, T, sd) in shapes]
    wants = [oracle.level1(pk) for pk in packs]
    plans = [corr.Plan(N, F, T, corr.PATH_TCGEN05) for (N, F, T, _) in shapes]
    try:
        devs = [torch.from_numpy(pk).cuda() for pk in packs]
        viss = [pl.new_vis() for pl in plans]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        busy = torch.cuda.Stream()
        a = torch.randn(4096, 4096, device="cuda")
        torch.cuda.synchronize()
        for rep in range(6):
            for v in viss:
                v.fill_(-559038737)
            torch.cuda.synchronize()
            if rep >= 3:
                with torch.cuda.stream(busy):
                    for _ in range(4):
                        a = torch.tanh(a) * 1.0001        # elementwise kernels with many small CTAs
            for k in range(4):
                for pl, d, v, st in zip(plans, devs, viss, streams):
                    pl.execute(d, v, stream=st)
            torch.cuda.synchronize()
            for v, w, sh in zip(viss, wants, shapes):
                assert np.array_equal(v.cpu().numpy(), w), (sh, rep)
    finally:
        for pl in plans:
            pl.close()


@pytest.mark.parametrize("case", [(272, 3, 700, "TCGEN05"), (2048, 1, 300, "TCGEN05"), (400, 2, 520, "TCGEN05"),
                                  (16, 9, 3000, "IMMA"), (64, 3, 1300, "IMMA"), (100, 2, 300, "DP4A"), (17, 3, 65, "DP4A")])
def test_no_write_outside_the_output(corr, oracle, case):
    # guard words on both sides of vis (and of the device input): every kernel, store / add / atomic modes,
    # tiles and rows that hang over N, ragged T
    import torch
    N, F, T, path = case
    packed = workloads.uniform_bytes(N, F, T, seed=N * 3 + T)
    want = oracle.level1(packed)
    G = 256   # guard ints (1 KB keeps vis 16-byte aligned)
    for variant in (("1", "3", "5") if path == "TCGEN05" else ("3",)):
        import os
        os.environ["CORR_TC_VARIANT"] = variant
        try:
            with corr.Plan(N, F, T, getattr(corr, "PATH_" + path)) as plan:
                buf = torch.full((2 * G + plan.vis_elems,), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
                vis = buf[G:G + plan.vis_elems].view(F, plan.baselines, 2)
                inbuf = torch.full((2048 + packed.size,), 0x88, dtype=torch.uint8, device="cuda")
                dev = inbuf[1024:1024 + packed.size].view(T, F, N)
                dev.copy_(torch.from_numpy(packed))
                plan.execute(dev, vis)
                plan.execute(dev, vis, accumulate=True)
                torch.cuda.synchronize()
                assert np.array_equal(vis.cpu().numpy(), 2 * want), (case, variant)
                assert (buf[:G] == 0x5A5A5A5A).all() and (buf[G + plan.vis_elems:] == 0x5A5A5A5A).all(), (case, variant)
                assert (inbuf[:1024] == 0x88).all() and (inbuf[1024 + packed.size:] == 0x88).all()
        finally:
            os.environ.pop("CORR_TC_VARIANT", None)


@pytest.mark.parametrize("case", [(128, 3, 700, "1"), (100, 2, 520, "0"), (64, 4, 900, "1"), (127, 5, 3000, "1"), (256, 5, 1300, "0"),
                                  (272, 3, 700, "1"), (250, 2, 9000, "1")])
def test_no_write_outside_the_output_tcd(corr, oracle, case, monkeypatch):
    # the same guard words around vis and the input for corr_tcd_kernel: one block per channel, two channels per tile,
    # several blocks per channel (rows and columns that hang over N), both schedules, store then add
    import torch
    N, F, T, shares = case
    monkeypatch.setenv("CORR_TCD_MAX_N", "512")
    monkeypatch.setenv("CORR_TCD_SHARES", shares)
    packed = workloads.uniform_bytes(N, F, T, seed=N * 3 + T)
    want = oracle.level1(packed)
    G = 256
    with corr.Plan(N, F, T, corr.PATH_AUTO if N == 64 else corr.PATH_TCGEN05) as plan:
        assert plan.info["path"] == corr.PATH_TCGEN05 and plan.info["tile_x"] == 128
        buf = torch.full((2 * G + plan.vis_elems,), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        vis = buf[G:G + plan.vis_elems].view(F, plan.baselines, 2)
        inbuf = torch.full((2048 + packed.size,), 0x88, dtype=torch.uint8, device="cuda")
        dev = inbuf[1024:1024 + packed.size].view(T, F, N)
        dev.copy_(torch.from_numpy(packed))
        plan.execute(dev, vis)
        plan.execute(dev, vis, accumulate=True)
        torch.cuda.synchronize()
        assert np.array_equal(vis.cpu().numpy(), 2 * want), case
        assert (buf[:G] == 0x5A5A5A5A).all() and (buf[G + plan.vis_elems:] == 0x5A5A5A5A).all(), case
        assert (inbuf[:1024] == 0x88).all() and (inbuf[1024 + packed.size:] == 0x88).all()


def test_int8_issue_loop_measurement(corr):
    # measurement aid: a bare tcgen05.mma.kind::i8 issue loop; on a B200 it lands between the power-capped and the
    # boost-clock ceiling (8192 MAC/clk/SM x 148 SMs x 2 ops at 1.3 .. 1.97 GHz)
    tops = corr.corr_measure_int8_tops(5000)
    assert 2500.0 < tops < 5000.0, tops


def test_invalid_arguments(corr):
    for bad in [(0, 1, 1), (16, 0, 1), (16, 1, 0), (16, 1, 1 << 24)]:
        with pytest.raises(corr.CorrError):
            corr.corr_plan_create(*bad)
    with pytest.raises(corr.CorrError):
        corr.corr_plan_create(65, 1, 64, corr.PATH_IMMA)       # warp-MMA path: N <= 64
    with pytest.raises(corr.CorrError):
        corr.corr_plan_create(80, 1, 64, corr.PATH_IMMA)       # warp-MMA path: N <= 64 only


# ------------------------------------------------------------------ the five BASELINE.json configs
def _config_case(corr, oracle, name, path=0):
    import torch
    cfg = workloads.CONFIGS[name]
    with corr.Plan(cfg.N, cfg.F, cfg.T, path) as plan:
        vis = plan.new_vis()
        vis.fill_(-1)
        want = None
        for call in range(cfg.calls):
            packed = workloads.generate(cfg, call)
            plan.execute(torch.from_numpy(packed).cuda(), vis, accumulate=(call > 0))
            torch.cuda.synchronize()
            want = oracle.level1(packed, accumulate_into=want) if want is not None else oracle.level1(packed)
        got = vis.cpu().numpy()
    assert got.shape == (cfg.F, cfg.baselines, 2)
    assert np.array_equal(got, want), f"{name}: {(got != want).sum()} mismatches"


@pytest.mark.parametrize("shape", [(20000, 1, 300), (40000, 2, 64)])
def test_very_large_n_sampled(corr, oracle, shape):
    # sizes the oracle cannot finish whole (0.8 and 3.2 G complex MACs per sample, up to 1.6 G baselines): sampled
    # baselines one by one (oracle.pair) at the corners, around the edges of the 128-blocks and at random; every
    # baseline written (none left at the fill value, which no sum can reach); the diagonal against the power sums
    import torch
    N, F, T = shape
    rng = np.random.default_rng(N)
    packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
    fill = -2 ** 31
    with corr.Plan(N, F, T) as plan:
        vis = plan.new_vis()
        vis.fill_(fill)
        plan.execute(torch.from_numpy(packed).cuda(), vis)
        torch.cuda.synchronize()
        assert int((vis == fill).sum().item()) == 0
        xs, ys = list(rng.integers(0, N, 300)), list(rng.integers(0, N, 300))
        for e in (0, 1, 127, 128, 129, N - 129, N - 128, N - 2, N - 1):
            for g in (0, 127, 128, N - 1):
                xs.append(e)
                ys.append(g)
        for f in range(F):
            idx = [oracle.baseline_index(N, int(min(x, y)), int(max(x, y))) for x, y in zip(xs, ys)]
            got = vis[f, torch.tensor(idx, device="cuda")].cpu().numpy()
            for (x, y), g in zip(zip(xs, ys), got):
                assert tuple(g) == tuple(oracle.pair(packed, f, int(min(x, y)), int(max(x, y)))), (f, x, y)
        re, im = (packed >> 4).astype(np.int64) - 8, (packed & 15).astype(np.int64) - 8
        power = (re * re + im * im).sum(axis=0)                                  # [F][N]
        diag = torch.tensor([oracle.baseline_index(N, x, x) for x in range(N)], device="cuda")
        got = vis[:, diag].cpu().numpy()
        assert np.array_equal(got[..., 0], power) and not got[..., 1].any()


def test_cfg1(corr, oracle):
    _config_case(corr, oracle, "cfg1")


def test_cfg2(corr, oracle):
    _config_case(corr, oracle, "cfg2")


def test_cfg3(corr, oracle):
    _config_case(corr, oracle, "cfg3")


def test_cfg4(corr, oracle):
    _config_case(corr, oracle, "cfg4")


def test_cfg5(corr, oracle):
    _config_case(corr, oracle, "cfg5")


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5"])
def test_configs_on_the_three_product_kernel(corr, oracle, name, monkeypatch):
    # the BASELINE.json shapes through corr_tc5_kernel (three products per complex MAC, fused per-element sums):
    # cfg1 is 16 inputs padded into one 128-block, cfg2 runs only cut units, cfg5 accumulates over eight calls
    monkeypatch.setenv("CORR_TC_VARIANT", "5")
    _config_case(corr, oracle, name, corr.PATH_TCGEN05)


def test_cfg5_memset_then_eight_accumulates(corr, oracle):
    # reading 10: memset + 8 x flag 1 must give the same bits as flag 0 then 7 x flag 1
    import torch
    cfg = workloads.CONFIGS["cfg5"]
    T = 512   # reduced length per call: this checks the flag semantics, not throughput
    with corr.Plan(cfg.N, cfg.F, T) as plan:
        vis_a = plan.new_vis()
        vis_b = torch.zeros_like(vis_a)
        want = None
        for call in range(cfg.calls):
            packed = workloads.generate(cfg, call, T=T)
            dev = torch.from_numpy(packed).cuda()
            plan.execute(dev, vis_a, accumulate=(call > 0))
            plan.execute(dev, vis_b, accumulate=True)
            want = oracle.level1(packed, accumulate_into=want) if want is not None else oracle.level1(packed)
        torch.cuda.synchronize()
        assert np.array_equal(vis_a.cpu().numpy(), want)
        assert np.array_equal(vis_b.cpu().numpy(), want)
