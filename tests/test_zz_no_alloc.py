"""corr_execute_noalloc (include/corr.h): the small-N pass without a plan and without any allocation -- its one piece of
scratch memory, the padded copy of the stream, is a static device array inside the library.  Checked against the
existing path (a plan + corr_execute) bit for bit: integer work, no tolerance, as everywhere in tests/.

This file is named to be collected last (the suite runs with pytest -x); it depends on no other test and passes in a
fresh process as well as after the others."""
import numpy as np
import pytest

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


def _existing_path(corr, dev, accumulate_into=None):
    import torch
    T, F, N = dev.shape
    with corr.Plan(N, F, T) as plan:
        vis = plan.new_vis() if accumulate_into is None else accumulate_into.clone()
        plan.execute(dev, vis, accumulate=accumulate_into is not None)
        torch.cuda.synchronize()
        return vis


def test_two_calls_in_a_row_match_the_existing_path(corr):
    import torch
    rng = np.random.default_rng(41)
    # (N, F, T): the first call leaves 720 KB of its padded stream in the scratch array, the second one (smaller, other
    # padding) must not see any of it; then a T long enough to be split into chunks (atomic adds into a cleared
    # output), a shape that needs no padding at all, and N = 64 - 1
    shapes = [(37, 5, 3000), (20, 3, 1201), (50, 2, 70000), (32, 4, 2500), (63, 2, 900), (5, 7, 333)]
    prev = None
    for (N, F, T) in shapes:
        dev = torch.from_numpy(rng.integers(0, 256, (T, F, N), dtype=np.uint8)).cuda()
        want = _existing_path(corr, dev)
        vis = torch.full_like(want, -559038737)              # flag 0 overwrites whatever the buffer held
        corr.execute_noalloc(dev, vis)
        torch.cuda.synchronize()
        assert torch.equal(vis, want), (N, F, T)
        # the same buffers again, accumulating: twice the sums, bit for bit what the existing path adds
        want2 = _existing_path(corr, dev, accumulate_into=want)
        corr.execute_noalloc(dev, vis, accumulate=True)
        torch.cuda.synchronize()
        assert torch.equal(vis, want2), (N, F, T, "accumulate")
        prev = (N, F, T)
    assert prev is not None


def test_back_to_back_calls_without_a_sync_in_between(corr):
    # two calls enqueued one after the other on one stream share the scratch array in stream order
    import torch
    rng = np.random.default_rng(43)
    a = torch.from_numpy(rng.integers(0, 256, (4000, 6, 44), dtype=np.uint8)).cuda()
    b = torch.from_numpy(rng.integers(0, 256, (2500, 9, 17), dtype=np.uint8)).cuda()
    want_a, want_b = _existing_path(corr, a), _existing_path(corr, b)
    vis_a, vis_b = torch.zeros_like(want_a), torch.zeros_like(want_b)
    for rep in range(3):
        vis_a.fill_(rep + 1)
        vis_b.fill_(-rep - 1)
        corr.execute_noalloc(a, vis_a)
        corr.execute_noalloc(b, vis_b)
        torch.cuda.synchronize()
        assert torch.equal(vis_a, want_a) and torch.equal(vis_b, want_b), rep


def test_allocates_nothing_so_it_can_be_captured(corr):
    # a cudaMalloc under stream capture fails and invalidates the capture: two calls captured into one graph, replayed
    import torch
    rng = np.random.default_rng(47)
    a = torch.from_numpy(rng.integers(0, 256, (3000, 4, 37), dtype=np.uint8)).cuda()
    b = torch.from_numpy(rng.integers(0, 256, (40000, 2, 24), dtype=np.uint8)).cuda()     # split T: memset + atomics
    want_a, want_b = _existing_path(corr, a), _existing_path(corr, b)
    vis_a, vis_b = torch.zeros_like(want_a), torch.zeros_like(want_b)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        corr.execute_noalloc(a, vis_a, stream=side)          # the first call on a device does the one-time set-up
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            corr.execute_noalloc(a, vis_a, stream=side)
            corr.execute_noalloc(b, vis_b, stream=side)
    for rep in range(2):
        vis_a.fill_(7)
        vis_b.fill_(9)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(vis_a, want_a) and torch.equal(vis_b, want_b), rep


def test_rejects_what_does_not_fit(corr):
    import torch
    # padded stream 16384 * 64 * 48 = 48 MiB > the 32 MiB scratch array
    N, F, T = 37, 64, 16384
    assert T * F * 48 > corr.NOALLOC_MAX_BYTES
    dev = torch.zeros((T, F, N), dtype=torch.uint8, device="cuda")
    vis = torch.zeros((F, N * (N + 1) // 2, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(corr.CorrError, match="exceeds the static scratch"):
        corr.execute_noalloc(dev, vis)
    # the same shape without padding needs no scratch and is served
    dev48 = torch.full((2048, 2, 48), 0x88, dtype=torch.uint8, device="cuda")    # 0x88 = the sample 0 + 0i
    vis48 = torch.ones((2, 48 * 49 // 2, 2), dtype=torch.int32, device="cuda")
    corr.execute_noalloc(dev48, vis48)
    torch.cuda.synchronize()
    assert not vis48.any()
    # larger N belongs to the plans
    dev65 = torch.zeros((64, 1, 65), dtype=torch.uint8, device="cuda")
    vis65 = torch.zeros((1, 65 * 66 // 2, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(corr.CorrError):
        corr.execute_noalloc(dev65, vis65)
    with pytest.raises(ValueError):
        corr.execute_noalloc(dev48, vis65)
