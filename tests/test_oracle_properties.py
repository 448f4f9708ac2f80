"""Property tests of the oracle (hypothesis): the algebraic facts Eq. 1 implies, on random small
streams.  They pin the oracle to the mathematics, not to itself: each property relates outputs for DIFFERENT
inputs, so a dropped term, a wrong sign or a transposed index breaks at least one of them."""
import numpy as np
from hypothesis import given, settings, strategies as st

MAXEX = 40


@st.composite
def streams(draw, max_n=9, max_f=3, max_t=24):
    N = draw(st.integers(1, max_n)); F = draw(st.integers(1, max_f)); T = draw(st.integers(1, max_t))
    seed = draw(st.integers(0, 2 ** 31 - 1))
    return np.random.default_rng(seed).integers(0, 256, (T, F, N), dtype=np.uint8)


def _decode(packed):
    return (packed >> 4).astype(np.int64) - 8, (packed & 15).astype(np.int64) - 8


def _encode(re, im):
    return (((re + 8) << 4) | (im + 8)).astype(np.uint8)


@settings(max_examples=MAXEX, deadline=None)
@given(streams())
def test_matches_complex_outer_product(oracle, packed):
    # the definition with numpy complex arithmetic (exact: all integers far below 2^53)
    re, im = _decode(packed)
    z = re + 1j * im                                   # [T][F][N]
    A = np.einsum("tfx,tfy->fxy", z, np.conj(z))
    T, F, N = packed.shape
    got = oracle.level1(packed)
    for f in range(F):
        for x in range(N):
            for y in range(x, N):
                b = oracle.baseline_index(N, x, y)
                assert got[f, b, 0] == round(A[f, x, y].real) and got[f, b, 1] == round(A[f, x, y].imag)


@settings(max_examples=MAXEX, deadline=None)
@given(streams(), st.integers(0, 2 ** 31 - 1))
def test_time_order_does_not_matter_and_sums_split(oracle, packed, seed):
    rng = np.random.default_rng(seed)
    perm = rng.permutation(packed.shape[0])
    assert np.array_equal(oracle.level1(np.ascontiguousarray(packed[perm])), oracle.level1(packed))
    k = int(rng.integers(0, packed.shape[0] + 1))
    parts = [p for p in (packed[:k], packed[k:]) if p.shape[0]]
    total = sum(oracle.level1(np.ascontiguousarray(p)).astype(np.int64) for p in parts)
    assert np.array_equal(total, oracle.level1(packed))


@settings(max_examples=MAXEX, deadline=None)
@given(streams())
def test_conjugating_every_input_negates_the_imaginary_parts(oracle, packed):
    re, im = _decode(packed)
    im = np.clip(im, -7, 7)                            # -(-8) is not a 4-bit value
    a = oracle.level1(_encode(re, im))
    b = oracle.level1(_encode(re, -im))
    assert np.array_equal(a[..., 0], b[..., 0]) and np.array_equal(a[..., 1], -b[..., 1])


@settings(max_examples=MAXEX, deadline=None)
@given(streams(), st.integers(0, 2 ** 31 - 1))
def test_swapping_two_inputs_permutes_and_conjugates(oracle, packed, seed):
    T, F, N = packed.shape
    if N < 2:
        return
    rng = np.random.default_rng(seed)
    i, j = sorted(rng.choice(N, 2, replace=False))
    sw = packed.copy()
    sw[:, :, [i, j]] = sw[:, :, [j, i]]
    a, b = oracle.level1(packed), oracle.level1(sw)
    idx = lambda x, y: oracle.baseline_index(N, x, y)
    pi = {i: j, j: i}
    for x in range(N):
        for y in range(x, N):
            u, v = pi.get(x, x), pi.get(y, y)           # where the pair came from
            if u <= v:
                assert np.array_equal(b[:, idx(x, y)], a[:, idx(u, v)])
            else:                                       # order flipped: Hermitian partner
                assert np.array_equal(b[:, idx(x, y), 0], a[:, idx(v, u), 0])
                assert np.array_equal(b[:, idx(x, y), 1], -a[:, idx(v, u), 1])


@settings(max_examples=MAXEX, deadline=None)
@given(streams())
def test_channels_are_independent(oracle, packed):
    T, F, N = packed.shape
    full = oracle.level1(packed)
    for f in range(F):
        assert np.array_equal(oracle.level1(np.ascontiguousarray(packed[:, f:f + 1, :]))[0], full[f])
