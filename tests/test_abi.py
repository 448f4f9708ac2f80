"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/corr.h
declares, its pure-host helpers agree with the paper's constants, and it fails loudly (no CPU
fallback) when there is no sm_100 device.  No compute calls here."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def corr():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1503_06203_b200 as c
    c.load_library()
    return c


def test_exports_every_declared_symbol(corr):
    header = (ROOT / "include" / "corr.h").read_text()
    declared = set(re.findall(r"\b(corr_[a-z0-9_]+)\s*\(", header))
    from paper_1503_06203_b200 import binding
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    lib = ctypes.CDLL(str(corr.lib_path()))
    for name in declared:
        assert hasattr(lib, name), name


def test_baseline_index_and_tile_count(corr, oracle):
    for N in (1, 2, 5, 16, 129):
        k = 0
        for x in range(N):
            for y in range(x, N):
                assert corr.baseline_index(N, x, y) == k == oracle.baseline_index(N, x, y)
                k += 1
    with pytest.raises(ValueError):
        corr.baseline_index(4, 2, 1)
    assert corr.count_tiles(256, 32, 32) == 36          # Fig. 1
    assert corr.count_tiles(2048, 128, 128) == 136
    assert corr.count_tiles(8192, 128, 128) == 2080
    assert corr.count_tiles(100, 64, 64) == 3
    assert corr.count_tiles(2048, 256, 128) == 72       # rectangular (CTA-pair) tiles


def test_no_cpu_fallback(corr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(corr.CorrError):
        corr.corr_plan_create(16, 4, 1024)


def test_product_and_oracle_share_nothing():
    for path in (ROOT / "paper_1503_06203_b200").rglob("*"):
        if path.suffix in {".py", ".cu", ".cuh", ".h"}:
            assert "oracle" not in path.read_text().lower(), path
    for path in (ROOT / "include").rglob("*.h"):
        assert "oracle" not in path.read_text().lower(), path
    for path in (ROOT / "oracle").rglob("*"):
        if path.suffix in {".py", ".c", ".h"}:
            text = path.read_text()
            assert "import paper_1503_06203_b200" not in text and "#include \"../paper" not in text, path
            assert "corr.h" not in text, path
