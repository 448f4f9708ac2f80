"""CPU oracle for the X-engine hot path of arXiv 1503.06203 -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_1503_06203_b200/ (the CUDA product) and
neither imports the other.  The arithmetic lives in corr_oracle.c (plain C, gcc); this file
only compiles it and marshals numpy arrays.

    level0(packed, accumulate_into=None)   definition loop, PAPER.md:41-50 (Eq. 1 summed over t)
    level1(packed, accumulate_into=None)   planar + OpenMP version of the same loops
    pair(packed, f, x, y)                  one ordered pair, any order (Hermitian pin)
    eq3_route(packed)                      stored-nibble products + Eq. 3 offsets
    baseline_index(N, x, y)                b(x,y) = x*N - x(x-1)/2 + (y-x)
    time_shift(packed, lags)               per-element integer time shift, PAPER.md:125-131 (numpy)
    gated(packed, gate, G)                 one matrix per gate of time samples
"""
from __future__ import annotations

import ctypes
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "corr_oracle.c"
_LIB = _HERE / "libcorr_oracle.so"

# Portable AVX2 baseline, not -march=native: the .so built in the CPU container also runs on
# the GPU box's host cores.
_CFLAGS = ["-O3", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> Path:
    """Compile corr_oracle.c -> libcorr_oracle.so (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", *_CFLAGS, str(_SRC), "-o", str(_LIB)]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        u8p = ctypes.POINTER(ctypes.c_uint8)
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        ci = ctypes.c_int
        lib.corr_oracle_level0.argtypes = [u8p, ci, ci, ci, i32p, ci]
        lib.corr_oracle_level0.restype = ci
        lib.corr_oracle_level1.argtypes = [u8p, ci, ci, ci, i32p, ci]
        lib.corr_oracle_level1.restype = ci
        lib.corr_oracle_eq3_route.argtypes = [u8p, ci, ci, ci, i32p]
        lib.corr_oracle_eq3_route.restype = ci
        lib.corr_oracle_pair.argtypes = [u8p, ci, ci, ci, ci, ci, ci, i64p, i64p]
        lib.corr_oracle_pair.restype = ci
        lib.corr_oracle_baseline_index.argtypes = [ci, ci, ci]
        lib.corr_oracle_baseline_index.restype = ctypes.c_size_t
        lib.corr_oracle_threads.argtypes = []
        lib.corr_oracle_threads.restype = ci
        _lib = lib
    return _lib


def _check_packed(packed: np.ndarray):
    if packed.dtype != np.uint8 or packed.ndim != 3:
        raise ValueError("packed must be uint8 [T][F][N]")
    packed = np.ascontiguousarray(packed)
    T, F, N = packed.shape
    return packed, N, F, T


def _run(fn, packed, accumulate_into):
    packed, N, F, T = _check_packed(packed)
    B = N * (N + 1) // 2
    if accumulate_into is None:
        vis = np.empty((F, B, 2), dtype=np.int32)
        acc = 0
    else:
        vis = accumulate_into
        if vis.dtype != np.int32 or vis.shape != (F, B, 2) or not vis.flags.c_contiguous:
            raise ValueError("accumulate_into must be C-contiguous int32 [F][B][2]")
        acc = 1
    rc = fn(packed.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), N, F, T,
            vis.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), acc)
    if rc != 0:
        raise RuntimeError(f"oracle error code {rc}")
    return vis


def level0(packed: np.ndarray, accumulate_into: np.ndarray | None = None) -> np.ndarray:
    """vis[F][N(N+1)/2][2] int32 by the definition loop (single thread; tiny shapes)."""
    return _run(_load().corr_oracle_level0, packed, accumulate_into)


def level1(packed: np.ndarray, accumulate_into: np.ndarray | None = None) -> np.ndarray:
    """Same result through planar int8 + OpenMP over (f, x); the large-config oracle."""
    return _run(_load().corr_oracle_level1, packed, accumulate_into)


def eq3_route(packed: np.ndarray) -> np.ndarray:
    packed, N, F, T = _check_packed(packed)
    vis = np.empty((F, N * (N + 1) // 2, 2), dtype=np.int32)
    rc = _load().corr_oracle_eq3_route(packed.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), N, F, T,
                                       vis.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)))
    if rc != 0:
        raise RuntimeError(f"oracle error code {rc}")
    return vis


def pair(packed: np.ndarray, f: int, x: int, y: int) -> tuple[int, int]:
    """(Re, Im) of sum_t X_t[x] conj(X_t[y]) for ANY ordered pair (x, y)."""
    packed, N, F, T = _check_packed(packed)
    re = ctypes.c_int64()
    im = ctypes.c_int64()
    rc = _load().corr_oracle_pair(packed.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), N, F, T,
                                  f, x, y, ctypes.byref(re), ctypes.byref(im))
    if rc != 0:
        raise RuntimeError(f"oracle error code {rc}")
    return int(re.value), int(im.value)


def baseline_index(N: int, x: int, y: int) -> int:
    if not 0 <= x <= y < N:
        raise ValueError("need 0 <= x <= y < N")
    return int(_load().corr_oracle_baseline_index(N, x, y))


def threads() -> int:
    """OpenMP threads level1 will use (bench.py reports this as cpu_baseline.cores)."""
    return int(_load().corr_oracle_threads())


def time_shift(packed: np.ndarray, lags) -> np.ndarray:
    """The paper's pre-correlation time shift, written out as its definition:
    out[t][f][n] = packed[t - lags[n]][f][n] if 0 <= t - lags[n] < T else 0x88 (the stored form of 0 + 0i).
    Plain numpy, one input element at a time."""
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    T, F, N = packed.shape
    lags = np.asarray(lags, dtype=np.int64)
    if lags.shape != (N,):
        raise ValueError("lags must have N entries")
    out = np.full_like(packed, 0x88)
    for n in range(N):
        d = int(lags[n])
        if d >= T or d <= -T:
            continue
        if d >= 0:
            out[d:, :, n] = packed[:T - d, :, n]
        else:
            out[:T + d, :, n] = packed[-d:, :, n]
    return out


def gated(packed: np.ndarray, gate, G: int) -> np.ndarray:
    """Gated correlation: vis[g] = Eq. 1 summed over the samples t with gate[t] == g
    (gate -1 = in no gate).  The definition written out: select the samples of a gate, then the same
    level-1 loops; a gate without samples is all zero.  Returns int32 [G][F][B][2]."""
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    T, F, N = packed.shape
    gate = np.asarray(gate)
    if gate.shape != (T,) or gate.min(initial=0) < -1 or gate.max(initial=-1) >= G:
        raise ValueError("gate must have T entries in [-1, G)")
    out = np.zeros((G, F, N * (N + 1) // 2, 2), np.int32)
    for g in range(G):
        sel = packed[gate == g]
        if sel.shape[0]:
            out[g] = level1(np.ascontiguousarray(sel))
    return out
