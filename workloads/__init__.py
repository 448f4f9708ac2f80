"""Seeded synthetic F-engine streams for the X-engine hot path of arXiv 1503.06203.

This module is the ONE thing the oracle-side tests and the CUDA-side tests share.
It holds none of the method's arithmetic: it only draws samples, quantises them to
the paper's 4-bit range and packs them in the paper's stream format.

Stream format (PAPER.md:76 SIII, Fig. 2): time-major, then frequency,
then the N input elements; one byte per complex sample, Re and Im each stored in
excess-8 ("offset-encoded") form.  Nibble order is not stated in the paper's text;
BASELINE.json fixes it: stored byte = ((Re+8) << 4) | (Im+8).

The paper measured on live CHIME data, which is not public; the five configs of
BASELINE.json stand in for it (shapes: N=256 Pathfinder PAPER.md:29, N=2048 full
CHIME PAPER.md:113, N=8192 largest tested PAPER.md:29).  Recipes are restated in
DESIGN.md "Input recipe".
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

SIGMA = 2.5  # BASELINE.json: "round(Normal(0,2.5)) clipped to [-8,7]"


@dataclass(frozen=True)
class Config:
    """One BASELINE.json workload. `calls` successive corr_execute calls of T samples each."""
    name: str
    N: int
    F: int
    T: int          # samples per call
    calls: int
    kind: str       # "iid" | "source" | "saturated"
    seed0: int      # seed of call 0; call c uses seed0 + c

    @property
    def baselines(self) -> int:
        return self.N * (self.N + 1) // 2

    @property
    def input_bytes(self) -> int:
        return self.T * self.F * self.N

    @property
    def vis_elems(self) -> int:
        return self.F * self.baselines * 2


# seed(cfg i, call c) = 1000*(i-1) + c  (cfg 1 gets seed 0 as BASELINE.json requires)
CONFIGS = {
    "cfg1": Config("cfg1", N=16, F=4, T=1024, calls=1, kind="iid", seed0=0),
    "cfg2": Config("cfg2", N=256, F=16, T=16384, calls=1, kind="source", seed0=1000),
    "cfg3": Config("cfg3", N=2048, F=8, T=8192, calls=1, kind="iid", seed0=2000),
    "cfg4": Config("cfg4", N=8192, F=1, T=4096, calls=1, kind="iid", seed0=3000),
    "cfg5": Config("cfg5", N=512, F=64, T=8192, calls=8, kind="saturated", seed0=4000),
}


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def quantise(v: np.ndarray) -> np.ndarray:
    """q(v) = clip(rint(v), -8, 7) as int8 (the 4-bit range of PAPER.md:76)."""
    return np.clip(np.rint(v), -8, 7).astype(np.int8)


def pack(re: np.ndarray, im: np.ndarray) -> np.ndarray:
    """int8 Re, Im in [-8,7] -> one uint8 per sample: ((Re+8)<<4) | (Im+8)."""
    re = np.asarray(re)
    im = np.asarray(im)
    if re.shape != im.shape:
        raise ValueError("re/im shape mismatch")
    if re.size and (re.min() < -8 or re.max() > 7 or im.min() < -8 or im.max() > 7):
        raise ValueError("sample outside the 4-bit range [-8,7]")
    hi = (re.astype(np.int16) + 8).astype(np.uint8)
    lo = (im.astype(np.int16) + 8).astype(np.uint8)
    return ((hi << 4) | lo).astype(np.uint8)


def _t_chunks(T: int, per_t_elems: int, budget_elems: int = 1 << 25):
    step = max(1, budget_elems // max(1, per_t_elems))
    t0 = 0
    while t0 < T:
        t1 = min(T, t0 + step)
        yield t0, t1
        t0 = t1


def iid_gaussian(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """cfg 1/3/4: Re, Im iid round(Normal(0, 2.5)) clipped to [-8,7].  Returns uint8 [T][F][N].

    Drawn as 2.5*standard_normal((T,F,N,2), float32), Re = [...,0], Im = [...,1]; generated in
    T-chunks from one generator so the stream equals the single big draw.
    """
    rng = _rng(seed)
    out = np.empty((T, F, N), dtype=np.uint8)
    for t0, t1 in _t_chunks(T, F * N * 2):
        g = rng.standard_normal((t1 - t0, F, N, 2), dtype=np.float32) * np.float32(SIGMA)
        out[t0:t1] = pack(quantise(g[..., 0]), quantise(g[..., 1]))
    return out


def common_source(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """cfg 2: per channel a common complex source s_t ~ CN(0,1) seen through gains g_n ~ CN(0,1),
    plus noise CN(0,1); v = 2.5*(g*s + w); quantised.  CN(0,1) = (a+ib)/sqrt(2), a,b ~ N(0,1).
    Draw order: gains [F][N], then per T-chunk: source [t][F], noise [t][F][N].
    """
    rng = _rng(seed)
    inv = np.float32(1.0 / np.sqrt(2.0))

    def cn(shape):
        z = rng.standard_normal(shape + (2,), dtype=np.float32) * inv
        return z[..., 0] + 1j * z[..., 1]

    g = cn((F, N)).astype(np.complex64)
    out = np.empty((T, F, N), dtype=np.uint8)
    for t0, t1 in _t_chunks(T, F * N * 4):
        s = cn((t1 - t0, F)).astype(np.complex64)
        w = cn((t1 - t0, F, N)).astype(np.complex64)
        v = np.float32(SIGMA) * (g[None, :, :] * s[:, :, None] + w)
        out[t0:t1] = pack(quantise(v.real), quantise(v.imag))
    return out


def saturated_mix(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """cfg 5: even-numbered elements saturated (Re and Im each independently -8 or +7, p = 1/2),
    odd-numbered elements uniform integers on [-8,7]."""
    rng = _rng(seed)
    out = np.empty((T, F, N), dtype=np.uint8)
    even = (np.arange(N) % 2 == 0)
    for t0, t1 in _t_chunks(T, F * N * 4):
        shape = (t1 - t0, F, N)
        sat = np.where(rng.integers(0, 2, size=shape + (2,), dtype=np.int8) == 0, -8, 7).astype(np.int8)
        uni = rng.integers(-8, 8, size=shape + (2,), dtype=np.int8)
        re = np.where(even[None, None, :], sat[..., 0], uni[..., 0])
        im = np.where(even[None, None, :], sat[..., 1], uni[..., 1])
        out[t0:t1] = pack(re, im)
    return out


def uniform_bytes(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """Every byte value equally likely (all 256 (Re,Im) pairs, including -8): the brute-force
    test input for tiny shapes."""
    return _rng(seed).integers(0, 256, size=(T, F, N), dtype=np.uint8)


def generate(cfg: Config, call: int = 0, T: int | None = None) -> np.ndarray:
    """Packed stream [T][F][N] for call `call` of `cfg` (optionally only the first T samples)."""
    if not 0 <= call < cfg.calls:
        raise ValueError("call index out of range")
    T = cfg.T if T is None else T
    seed = cfg.seed0 + call
    if cfg.kind == "iid":
        full = iid_gaussian(cfg.N, cfg.F, T, seed)
    elif cfg.kind == "source":
        full = common_source(cfg.N, cfg.F, T, seed)
    elif cfg.kind == "saturated":
        full = saturated_mix(cfg.N, cfg.F, T, seed)
    else:
        raise ValueError(cfg.kind)
    return full


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
