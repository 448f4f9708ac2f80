"""SURVEY section 8(f) item 3, gated correlation: oracle pins (CPU) and bit-exact parity of
corr_execute_gated against the oracle (GPU)."""
import numpy as np
import pytest

import workloads


def _gate_pattern(T, G, period, seed):
    """Periodic gates (a pulsar / switched calibration source): phase bins of `period` samples, a few
    samples in no gate, deterministic."""
    rng = np.random.default_rng(seed)
    gate = ((np.arange(T) % period) * G // period).astype(np.int32)
    gate[rng.random(T) < 0.05] = -1
    return gate


# ------------------------------------------------------------------ oracle pins (no GPU)
def test_gated_brute_force(oracle):
    rng = np.random.default_rng(2)
    T, F, N, G = 37, 2, 3, 3
    packed = rng.integers(0, 256, (T, F, N), dtype=np.uint8)
    gate = rng.integers(-1, G, T)
    got = oracle.gated(packed, gate, G)
    for g in range(G):
        for f in range(F):
            for x in range(N):
                for y in range(x, N):
                    re = im = 0
                    for t in range(T):
                        if gate[t] != g:
                            continue
                        xr, xi = (int(packed[t, f, x]) >> 4) - 8, (int(packed[t, f, x]) & 15) - 8
                        yr, yi = (int(packed[t, f, y]) >> 4) - 8, (int(packed[t, f, y]) & 15) - 8
                        re += xr * yr + xi * yi          # Eq. 1
                        im += xi * yr - xr * yi
                    assert tuple(got[g, f, oracle.baseline_index(N, x, y)]) == (re, im)


def test_gates_partition_the_ungated_sum(oracle):
    packed = workloads.uniform_bytes(9, 2, 500, seed=4)
    gate = _gate_pattern(500, 4, 37, seed=1)
    g = oracle.gated(packed, gate, 4)
    used = oracle.level1(np.ascontiguousarray(packed[gate >= 0]))
    assert np.array_equal(g.sum(axis=0), used)                       # additivity over disjoint sample sets
    assert np.array_equal(oracle.gated(packed, np.zeros(500, int), 1)[0], oracle.level1(packed))   # one gate = ungated
    empty = oracle.gated(packed, np.full(500, -1), 2)
    assert not empty.any()


def test_gated_closed_form(oracle):
    # constant input a + ib: gate g holds T_g (a^2 + b^2) on every baseline, zero imaginary part
    T, G = 300, 3
    gate = _gate_pattern(T, G, 50, seed=9)
    for byte, a, b in [(0x00, -8, -8), (0xFF, 7, 7), (0xB6, 3, -2)]:
        got = oracle.gated(np.full((T, 1, 4), byte, np.uint8), gate, G)
        for g in range(G):
            tg = int((gate == g).sum())
            assert (got[g, ..., 0] == tg * (a * a + b * b)).all() and (got[g, ..., 1] == 0).all()


# ------------------------------------------------------------------ GPU parity (bit-exact)
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


@pytest.mark.gpu
@pytest.mark.parametrize("per_gate", [False, True])
@pytest.mark.parametrize("shape", [(16, 5, 3000), (64, 3, 2500), (100, 2, 900), (272, 2, 2000), (1024, 1, 1500)])
def test_gated_parity(corr, oracle, shape, per_gate, monkeypatch):
    # gates of about the same length share one pass (the gates as extra channels); per_gate forces one pass per gate
    import torch
    if per_gate:
        monkeypatch.setenv("CORR_GATED_PER_GATE", "1")
    N, F, T = shape
    packed = workloads.iid_gaussian(N, F, T, seed=N + T)
    dev = torch.from_numpy(packed).cuda()
    with corr.Plan(N, F, T) as plan:
        for G, period in [(1, 7), (4, 64), (3, 1000)]:
            gate = _gate_pattern(T, G, period, seed=G)
            want = oracle.gated(packed, gate, G)
            vis = plan.execute_gated(dev, gate, G)
            torch.cuda.synchronize()
            assert np.array_equal(vis.cpu().numpy(), want), (shape, G, period)
            plan.execute_gated(dev, gate, G, vis=vis, accumulate=True)      # flag 1 adds, gate by gate
            torch.cuda.synchronize()
            assert np.array_equal(vis.cpu().numpy(), 2 * want), (shape, G, period, "accumulate")
        # a gate with no sample: zeroed when overwriting, left alone when accumulating
        gate = np.zeros(T, np.int32)
        gate[::3] = 2
        vis = torch.full((3, F, plan.baselines, 2), 77, dtype=torch.int32, device="cuda")
        plan.execute_gated(dev, gate, 3, vis=vis)
        torch.cuda.synchronize()
        got = vis.cpu().numpy()
        assert np.array_equal(got, oracle.gated(packed, gate, 3)) and not got[1].any()
        vis.fill_(5)
        plan.execute_gated(dev, gate, 3, vis=vis, accumulate=True)
        torch.cuda.synchronize()
        assert (vis.cpu().numpy()[1] == 5).all()


@pytest.mark.gpu
def test_gated_rejects_bad_gate(corr):
    import torch
    with corr.Plan(32, 1, 64) as plan:
        dev = torch.zeros((64, 1, 32), dtype=torch.uint8, device="cuda")
        with pytest.raises(corr.CorrError):
            plan.execute_gated(dev, np.full(64, 2), 2)        # gate index == G
        with pytest.raises(ValueError):
            plan.execute_gated(dev, np.zeros(10), 2)
