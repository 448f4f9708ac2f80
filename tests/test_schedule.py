"""Host logic of step S3 (no GPU): the CTA-pair tile table and the tail of the schedule (corr_schedule_pairs, the same
code corr_plan_create runs).  PAPER.md:64-72 fixes what has to be covered (every block on or above the diagonal, once);
how the work is dealt to CTAs is this build's."""
import pytest

import paper_1503_06203_b200 as corr

SHAPES = [(2048, 8, 8192), (256, 16, 16384), (512, 64, 8192), (8192, 1, 4096), (272, 3, 1000), (400, 2, 777),
          (1024, 5, 1024), (129, 1, 1), (2048, 1, 640), (640, 7, 70000), (3000, 3, 300), (256, 2, 20000)]


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__
    __graft_entry__.build()
    corr.load_library()
    return corr


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("pairs", [74, 66, 1, 7])
def test_every_group_of_every_unit_is_computed_exactly_once(lib, shape, pairs):
    N, F, T = shape
    info, pieces = lib.schedule_pairs(N, F, T, pairs)
    units, used = info["units"], info["pairs_used"]
    assert units == F * info["tiles_per_channel"] * info["slices"] and 1 <= used <= pairs

    def length(u):
        return info["groups_last"] if u % info["slices"] == info["slices"] - 1 else info["groups_full"]

    covered = {}
    waves = units // used
    assert waves == info["waves"]
    for p in range(used):                       # whole waves: unit = pair + k * pairs
        for k in range(waves):
            covered.setdefault(p + k * used, []).append((0, length(p + k * used)))
    for p, plist in enumerate(pieces):
        assert len(plist) <= 4
        for (u, first, cnt, early) in plist:
            assert waves * used <= u < units and first >= 0 and cnt >= 1 and first + cnt <= length(u)
            # early pieces: only the first piece of a unit that is really cut, and only when there are whole waves
            if early:
                assert first == 0 and cnt < length(u) and waves > 0
            covered.setdefault(u, []).append((first, cnt))
    assert sorted(covered) == list(range(units))
    for u, runs in covered.items():
        runs.sort()
        pos = 0
        for first, cnt in runs:
            assert first == pos, (u, runs)
            pos += cnt
        assert pos == length(u), (u, runs)
        # a cut unit has exactly one piece that starts it (the one that may be early)
    # balance: no pair carries more than the mean tail load plus one piece's worth of slack
    loads = [sum(c for (_, _, c, _) in pl) + 3 * len(pl) for pl in pieces]
    tail = sum(length(u) for u in range(waves * used, units))
    if tail:
        assert max(loads) <= tail / used + 3 * 4 + 2, (max(loads), tail / used)


def test_tile_table_counts():
    # pair tiles per channel: nb^2/4 + nb/4 rounded up as the pairing of left-over blocks allows
    want = {128: 1, 256: 2, 384: 3, 512: 5, 1024: 18, 2048: 68, 4096: 264, 8192: 1040}
    for N, tiles in want.items():
        info, _ = corr.schedule_pairs(N, 1, 256, 74)
        assert info["tiles_per_channel"] == tiles, (N, info)
    info, _ = corr.schedule_pairs(2048, 1, 256, 74)
    assert info["transposed_tiles"] == 4          # 8 left-over blocks (0, j), j even, paired two by two
    info, _ = corr.schedule_pairs(256, 1, 256, 74)
    assert info["transposed_tiles"] == 1          # block (0, 0) alone: next to an idle CTA


def test_t_slices_keep_the_int32_headroom():
    info, _ = corr.schedule_pairs(256, 1, 16777215, 74)
    assert info["slices"] == 512 and info["groups_full"] * 256 <= 32768


def test_invalid_schedule_arguments():
    with pytest.raises(corr.CorrError):
        corr.schedule_pairs(0, 1, 1, 74)
    with pytest.raises(corr.CorrError):
        corr.schedule_pairs(128, 1, 1, 0)
