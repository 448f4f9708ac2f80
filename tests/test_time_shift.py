"""SURVEY section 8(f) item 4, the pre-correlation time shift: oracle pins (CPU) and
byte-exact parity of corr_time_shift against the oracle (GPU)."""
import numpy as np
import pytest

import workloads


# ------------------------------------------------------------------ oracle pins (no GPU)
def test_shift_definition_brute_force(oracle):
    rng = np.random.default_rng(5)
    for (T, F, N) in [(1, 1, 1), (7, 2, 3), (20, 1, 5), (33, 3, 4)]:
        packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
        lags = rng.integers(-T - 2, T + 3, N)
        got = oracle.time_shift(packed, lags)
        for t in range(T):
            for f in range(F):
                for n in range(N):
                    s = t - int(lags[n])
                    want = packed[s, f, n] if 0 <= s < T else 0x88
                    assert got[t, f, n] == want


def test_shift_zero_lag_is_identity_and_inverse_restores_interior(oracle):
    packed = workloads.uniform_bytes(6, 2, 50, seed=3)
    assert np.array_equal(oracle.time_shift(packed, np.zeros(6, int)), packed)
    d = np.array([0, 1, 5, 9, 2, 7])
    back = oracle.time_shift(oracle.time_shift(packed, d), -d)
    for n in range(6):
        assert np.array_equal(back[:50 - d[n], :, n], packed[:50 - d[n], :, n])
        assert (back[50 - d[n]:, :, n] == 0x88).all()       # what left the block is gone: stored zero


def test_shift_aligns_a_delayed_copy(oracle):
    # element 1 carries element 0's signal d samples late (a longer cable); delaying
    # element 0 by d makes the two streams identical, so their visibility becomes real and equal to
    # the power of the overlap; shifted-in samples are 0 + 0i and add nothing (Eq. 1)
    T, d = 400, 13
    base = workloads.iid_gaussian(1, 1, T, seed=11)[:, 0, 0]
    packed = np.full((T, 1, 2), 0x88, np.uint8)
    packed[:, 0, 0] = base
    packed[d:, 0, 1] = base[:T - d]
    raw = oracle.level0(packed)
    fixed = oracle.level0(oracle.time_shift(packed, [d, 0]))
    re = (base[:T - d] >> 4).astype(int) - 8
    im = (base[:T - d] & 15).astype(int) - 8
    power = int((re * re + im * im).sum())
    b01 = oracle.baseline_index(2, 0, 1)
    assert tuple(fixed[0, b01]) == (power, 0)
    assert tuple(fixed[0, oracle.baseline_index(2, 1, 1)]) == (power, 0)
    assert tuple(raw[0, b01]) != (power, 0)                  # without the shift the pair decorrelates


# ------------------------------------------------------------------ GPU parity (byte-exact)
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


def _gpu_shift(corr, packed, lags):
    import torch
    out = corr.time_shift(torch.from_numpy(packed).cuda(), torch.from_numpy(np.asarray(lags, np.int32)).cuda())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.gpu
def test_time_shift_parity(corr, oracle):
    rng = np.random.default_rng(17)
    shapes = [(1, 1, 1), (300, 2, 16), (257, 3, 48), (1000, 2, 272), (513, 1, 2048), (700, 2, 100), (50, 3, 5),
              (900, 4, 100), (400, 16, 37)]      # the last two: N % 16 != 0 with rows of a multiple of 16 bytes
    for (T, F, N) in shapes:
        packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
        for spread in (0, 3, 200, 1500, 5000):              # 1500+: wider than the staged window -> general path
            lags = rng.integers(-spread, spread + 1, N)
            assert np.array_equal(_gpu_shift(corr, packed, lags), oracle.time_shift(packed, lags)), (T, F, N, spread)
    packed = rng.integers(0, 256, (64, 1, 32), dtype=np.uint8)
    lags = np.array([64, -64, 63, -63, 10 ** 9, -10 ** 9] + [0] * 26)   # |lag| >= T empties the element
    assert np.array_equal(_gpu_shift(corr, packed, lags), oracle.time_shift(packed, lags))


@pytest.mark.gpu
def test_time_shift_long_stream_mixed_spreads(corr, oracle):
    # every group of 128 inputs takes its own route through the kernel (windows of one and of two time blocks, the
    # 16-byte-wide window, byte by byte), over enough tiles per CTA to wrap the ring of rows several times
    rng = np.random.default_rng(29)
    T, F, N = 40000, 2, 5 * 128 + 48
    packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
    lags = np.zeros(N, np.int64)
    lags[0:128] = rng.integers(-8, 9, 128)
    lags[128:256] = 1000 + rng.integers(-90, 91, 128)        # a common offset costs nothing: only the spread counts
    lags[256:384] = rng.integers(-450, 451, 128)
    lags[384:512] = rng.integers(-1900, 1901, 128)
    lags[512:640] = rng.integers(-30000, 30001, 128)
    lags[640:] = -7
    assert np.array_equal(_gpu_shift(corr, packed, lags), oracle.time_shift(packed, lags))


@pytest.mark.gpu
def test_time_shift_many_tiles_per_cta(corr, oracle):
    # one group of inputs, one channel: every CTA walks two dozen tiles whose windows (128 + 32 rows) fill the ring of
    # rows exactly, so the ring wraps at its last row
    rng = np.random.default_rng(31)
    T, F, N = 128 * 148 * 24 + 77, 1, 128
    packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
    lags = rng.integers(-16, 17, N)
    lags[5], lags[77] = -16, 16
    assert np.array_equal(_gpu_shift(corr, packed, lags), oracle.time_shift(packed, lags))


@pytest.mark.gpu
def test_time_shift_then_correlate(corr, oracle):
    # the two kernels chained on the device give what the oracle gives for the same chain
    import torch
    packed = workloads.iid_gaussian(256, 2, 3000, seed=23)
    lags = np.random.default_rng(1).integers(-40, 41, 256)
    want = oracle.level1(oracle.time_shift(packed, lags))
    dev = corr.time_shift(torch.from_numpy(packed).cuda(), torch.from_numpy(lags.astype(np.int32)).cuda())
    with corr.Plan(256, 2, 3000) as plan:
        vis = plan.execute(dev)
        torch.cuda.synchronize()
        assert np.array_equal(vis.cpu().numpy(), want)


@pytest.mark.gpu
def test_time_shift_rejects_bad_arguments(corr):
    import torch
    a = torch.zeros((8, 1, 16), dtype=torch.uint8, device="cuda")
    lags = torch.zeros(16, dtype=torch.int32, device="cuda")
    with pytest.raises(corr.CorrError):
        corr.time_shift(a, lags, out=a)                      # not in place
    with pytest.raises(ValueError):
        corr.time_shift(a, lags[:8])
