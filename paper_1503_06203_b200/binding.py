"""ctypes binding of include/corr.h.  Same names as the C ABI; argument marshalling only."""
from __future__ import annotations

import ctypes
from pathlib import Path

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "libcorr_b200.so"

PATH_AUTO, PATH_DP4A, PATH_TCGEN05, PATH_IMMA = 0, 1, 2, 3

# every symbol include/corr.h declares (tests check the library exports all of them)
SYMBOLS = ("corr_plan_create", "corr_plan_create_ex", "corr_execute", "corr_execute_host",
           "corr_plan_destroy", "corr_last_error", "corr_input_bytes", "corr_vis_elems",
           "corr_baseline_index", "corr_plan_info", "corr_count_tiles", "corr_schedule_pairs", "corr_time_shift", "corr_execute_gated", "corr_measure_int8_tops", "corr_submit_host", "corr_wait_host", "corr_execute_noalloc")


class CorrError(RuntimeError):
    pass


_lib = None


def lib_path() -> Path:
    return _LIB_PATH


def load_library():
    """dlopen libcorr_b200.so.  Fails loudly if it has not been built (python -m
    paper_1503_06203_b200.build or __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise CorrError(f"{_LIB_PATH} not built; run __graft_entry__.build() - there is no fallback path")
        lib = ctypes.CDLL(str(_LIB_PATH))
        vp, ci, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
        lib.corr_plan_create.argtypes = [ci, ci, ci]
        lib.corr_plan_create.restype = vp
        lib.corr_plan_create_ex.argtypes = [ci, ci, ci, ci]
        lib.corr_plan_create_ex.restype = vp
        lib.corr_execute.argtypes = [vp, vp, vp, ci, vp]
        lib.corr_execute.restype = ci
        lib.corr_execute_host.argtypes = [vp, vp, vp, ci, vp]
        lib.corr_execute_host.restype = ci
        lib.corr_submit_host.argtypes = [vp, vp, vp, ci, vp]
        lib.corr_submit_host.restype = ci
        lib.corr_wait_host.argtypes = [vp]
        lib.corr_wait_host.restype = ci
        lib.corr_plan_destroy.argtypes = [vp]
        lib.corr_plan_destroy.restype = None
        lib.corr_last_error.argtypes = []
        lib.corr_last_error.restype = ctypes.c_char_p
        lib.corr_input_bytes.argtypes = [vp]
        lib.corr_input_bytes.restype = sz
        lib.corr_vis_elems.argtypes = [vp]
        lib.corr_vis_elems.restype = sz
        lib.corr_baseline_index.argtypes = [ci, ci, ci]
        lib.corr_baseline_index.restype = sz
        lib.corr_plan_info.argtypes = [vp, ctypes.POINTER(ci * 8)]
        lib.corr_plan_info.restype = ci
        lib.corr_count_tiles.argtypes = [ci, ci, ci]
        lib.corr_count_tiles.restype = ci
        lib.corr_schedule_pairs.argtypes = [ci, ci, ci, ci, ctypes.POINTER(ci * 8), vp]
        lib.corr_schedule_pairs.restype = ci
        lib.corr_execute_gated.argtypes = [vp, vp, vp, ci, vp, ci, vp]
        lib.corr_execute_gated.restype = ci
        lib.corr_measure_int8_tops.argtypes = [ci, ctypes.POINTER(ctypes.c_double)]
        lib.corr_measure_int8_tops.restype = ci
        lib.corr_time_shift.argtypes = [ci, ci, ci, vp, vp, vp, vp]
        lib.corr_time_shift.restype = ci
        lib.corr_execute_noalloc.argtypes = [ci, ci, ci, vp, vp, ci, vp]
        lib.corr_execute_noalloc.restype = ci
        _lib = lib
    return _lib


def _err() -> str:
    return load_library().corr_last_error().decode(errors="replace")


# ------------------------------------------------------------------ C-ABI names, 1:1
def corr_plan_create(N: int, F: int, T: int, path: int = PATH_AUTO) -> int:
    lib = load_library()
    h = lib.corr_plan_create(N, F, T) if path == PATH_AUTO else lib.corr_plan_create_ex(N, F, T, path)
    if not h:
        raise CorrError(_err())
    return h


def corr_execute(plan: int, packed_dev_ptr: int, vis_dev_ptr: int, accumulate_flag: int, stream: int) -> None:
    rc = load_library().corr_execute(plan, packed_dev_ptr, vis_dev_ptr, int(bool(accumulate_flag)), stream)
    if rc != 0:
        raise CorrError(f"corr_execute -> {rc}: {_err()}")


def corr_execute_host(plan: int, packed_host_ptr: int, vis_host_ptr: int, accumulate_flag: int, stream: int) -> None:
    rc = load_library().corr_execute_host(plan, packed_host_ptr, vis_host_ptr, int(bool(accumulate_flag)), stream)
    if rc != 0:
        raise CorrError(f"corr_execute_host -> {rc}: {_err()}")


def corr_execute_gated(plan: int, packed_dev_ptr: int, gate_host_ptr: int, G: int, vis_dev_ptr: int,
                       accumulate_flag: int, stream: int) -> None:
    rc = load_library().corr_execute_gated(plan, packed_dev_ptr, gate_host_ptr, G, vis_dev_ptr,
                                           int(bool(accumulate_flag)), stream)
    if rc != 0:
        raise CorrError(f"corr_execute_gated -> {rc}: {_err()}")


def corr_measure_int8_tops(iters: int = 20000) -> float:
    """Dense int8 TOPS of a bare tcgen05.mma.kind::i8 issue loop on the current device (synchronises)."""
    out = ctypes.c_double(0.0)
    rc = load_library().corr_measure_int8_tops(iters, ctypes.byref(out))
    if rc != 0:
        raise CorrError(f"corr_measure_int8_tops -> {rc}: {_err()}")
    return out.value


def corr_time_shift(N: int, F: int, T: int, packed_in_ptr: int, lags_ptr: int, packed_out_ptr: int, stream: int) -> None:
    rc = load_library().corr_time_shift(N, F, T, packed_in_ptr, lags_ptr, packed_out_ptr, stream)
    if rc != 0:
        raise CorrError(f"corr_time_shift -> {rc}: {_err()}")


def time_shift(packed, lags, out=None, stream=None):
    """packed: uint8 CUDA tensor [T][F][N]; lags: int32 CUDA tensor [N].  Returns the shifted stream
    (a new tensor unless `out` is given).  Enqueues only."""
    import torch
    if not packed.is_cuda or packed.dtype != torch.uint8 or not packed.is_contiguous() or packed.dim() != 3:
        raise ValueError("packed must be a contiguous uint8 CUDA tensor [T][F][N]")
    T, F, N = packed.shape
    if not lags.is_cuda or lags.dtype != torch.int32 or lags.numel() != N or not lags.is_contiguous():
        raise ValueError("lags must be a contiguous int32 CUDA tensor of N elements")
    if out is None:
        out = torch.empty_like(packed)
    s = torch.cuda.current_stream(packed.device) if stream is None else stream
    corr_time_shift(N, F, T, packed.data_ptr(), lags.data_ptr(), out.data_ptr(), s.cuda_stream)
    return out


NOALLOC_MAX_BYTES = 32 << 20   # CORR_NOALLOC_MAX_BYTES of include/corr.h


def corr_execute_noalloc(N: int, F: int, T: int, packed_dev_ptr: int, vis_dev_ptr: int, accumulate_flag: int, stream: int) -> None:
    rc = load_library().corr_execute_noalloc(N, F, T, packed_dev_ptr, vis_dev_ptr, int(bool(accumulate_flag)), stream)
    if rc != 0:
        raise CorrError(f"corr_execute_noalloc -> {rc}: {_err()}")


def execute_noalloc(packed, vis, accumulate=False, stream=None):
    """packed: uint8 CUDA tensor [T][F][N], N <= 64; vis: int32 CUDA tensor [F][N(N+1)/2][2] (the caller allocates it:
    this call allocates nothing, see corr_execute_noalloc in include/corr.h).  Enqueues only; returns vis."""
    import torch
    if not packed.is_cuda or packed.dtype != torch.uint8 or not packed.is_contiguous() or packed.dim() != 3:
        raise ValueError("packed must be a contiguous uint8 CUDA tensor [T][F][N]")
    T, F, N = packed.shape
    if (not vis.is_cuda or vis.dtype != torch.int32 or not vis.is_contiguous()
            or tuple(vis.shape) != (F, N * (N + 1) // 2, 2)):
        raise ValueError("vis must be a contiguous int32 CUDA tensor [F][N(N+1)/2][2]")
    s = torch.cuda.current_stream(packed.device) if stream is None else stream
    corr_execute_noalloc(N, F, T, packed.data_ptr(), vis.data_ptr(), accumulate, s.cuda_stream)
    return vis


def corr_submit_host(plan: int, packed_host_ptr: int, vis_host_ptr: int, accumulate_flag: int, stream: int) -> None:
    rc = load_library().corr_submit_host(plan, packed_host_ptr, vis_host_ptr, int(bool(accumulate_flag)), stream)
    if rc != 0:
        raise CorrError(f"corr_submit_host -> {rc}: {_err()}")


def corr_wait_host(plan: int) -> None:
    rc = load_library().corr_wait_host(plan)
    if rc != 0:
        raise CorrError(f"corr_wait_host -> {rc}: {_err()}")


def corr_plan_destroy(plan: int) -> None:
    load_library().corr_plan_destroy(plan)


def baseline_index(N: int, x: int, y: int) -> int:
    v = load_library().corr_baseline_index(N, x, y)
    if v == ctypes.c_size_t(-1).value:
        raise ValueError("need 0 <= x <= y < N")
    return int(v)


def count_tiles(N: int, tile_x: int, tile_y: int) -> int:
    return int(load_library().corr_count_tiles(N, tile_x, tile_y))


def schedule_pairs(N: int, F: int, T: int, pairs: int):
    """corr_schedule_pairs: (info dict, pieces) with pieces[pair] = list of (unit, first group, groups, early)."""
    lib = load_library()
    info = (ctypes.c_int * 8)()
    buf = (ctypes.c_int * (16 * pairs))()
    rc = lib.corr_schedule_pairs(N, F, T, pairs, ctypes.byref(info), ctypes.cast(buf, ctypes.c_void_p))
    if rc != 0:
        raise CorrError(f"corr_schedule_pairs -> {rc}: {_err()}")
    keys = ("tiles_per_channel", "slices", "units", "groups_full", "groups_last", "pairs_used", "waves", "transposed_tiles")
    d = dict(zip(keys, (int(v) for v in info)))
    pieces = [[tuple(buf[16 * p + 4 * k + j] for j in range(4)) for k in range(4) if buf[16 * p + 4 * k + 2] > 0]
              for p in range(d["pairs_used"])]
    return d, pieces


# ------------------------------------------------------------------ convenience wrapper
class Plan:
    """corr_plan with torch tensors as device buffers (torch: allocation + streams only)."""

    def __init__(self, N: int, F: int, T: int, path: int = PATH_AUTO):
        self.N, self.F, self.T = N, F, T
        self._h = corr_plan_create(N, F, T, path)
        lib = load_library()
        self.input_bytes = int(lib.corr_input_bytes(self._h))
        self.vis_elems = int(lib.corr_vis_elems(self._h))
        arr = (ctypes.c_int * 8)()
        if lib.corr_plan_info(self._h, ctypes.byref(arr)) != 0:
            raise CorrError(_err())
        keys = ("path", "tile_x", "tile_y", "tiles_per_channel", "slices", "units", "ctas", "kernels")
        self.info = dict(zip(keys, list(arr)))

    @property
    def baselines(self) -> int:
        return self.N * (self.N + 1) // 2

    def new_vis(self, device="cuda"):
        import torch
        return torch.empty((self.F, self.baselines, 2), dtype=torch.int32, device=device)

    def execute(self, packed, vis=None, accumulate: bool = False, stream=None):
        """packed: uint8 CUDA tensor [T][F][N]; vis: int32 CUDA tensor [F][B][2] (allocated if None).
        Enqueues on `stream` (default: torch's current stream); does not synchronise."""
        import torch
        if not packed.is_cuda or packed.dtype != torch.uint8 or not packed.is_contiguous():
            raise ValueError("packed must be a contiguous uint8 CUDA tensor")
        if packed.numel() != self.input_bytes:
            raise ValueError(f"packed has {packed.numel()} bytes, plan expects {self.input_bytes}")
        if vis is None:
            if accumulate:
                raise ValueError("accumulate=True needs an existing vis tensor")
            vis = self.new_vis(packed.device)
        if not vis.is_cuda or vis.dtype != torch.int32 or not vis.is_contiguous() or vis.numel() != self.vis_elems:
            raise ValueError("vis must be a contiguous int32 CUDA tensor of F*B*2 elements")
        s = torch.cuda.current_stream(packed.device) if stream is None else stream
        corr_execute(self._h, packed.data_ptr(), vis.data_ptr(), int(accumulate), s.cuda_stream)
        return vis

    def execute_gated(self, packed, gate, G: int, vis=None, accumulate: bool = False, stream=None):
        """packed: uint8 CUDA tensor [T][F][N]; gate: T integers in [-1, G) (numpy array or list, host);
        vis: int32 CUDA tensor [G][F][B][2] (allocated if None).  Enqueues; does not synchronise."""
        import numpy as np
        import torch
        if not packed.is_cuda or packed.dtype != torch.uint8 or not packed.is_contiguous() or packed.numel() != self.input_bytes:
            raise ValueError("packed must be a contiguous uint8 CUDA tensor of T*F*N bytes")
        gate = np.ascontiguousarray(gate, dtype=np.int32)
        if gate.shape != (self.T,):
            raise ValueError("gate must have T entries")
        if vis is None:
            if accumulate:
                raise ValueError("accumulate=True needs an existing vis tensor")
            vis = torch.empty((G, self.F, self.baselines, 2), dtype=torch.int32, device=packed.device)
        if not vis.is_cuda or vis.dtype != torch.int32 or not vis.is_contiguous() or vis.numel() != G * self.vis_elems:
            raise ValueError("vis must be a contiguous int32 CUDA tensor of G*F*B*2 elements")
        s = torch.cuda.current_stream(packed.device) if stream is None else stream
        corr_execute_gated(self._h, packed.data_ptr(), gate.ctypes.data, G, vis.data_ptr(), int(accumulate), s.cuda_stream)
        return vis

    def execute_host(self, packed_host, vis_host, accumulate: bool = False, stream=None):
        """packed_host / vis_host: CPU torch tensors (pinned for async copies) or numpy arrays."""
        import torch
        s = torch.cuda.current_stream() if stream is None else stream

        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data

        corr_execute_host(self._h, ptr(packed_host), ptr(vis_host), int(accumulate), s.cuda_stream)
        return vis_host

    def submit_host(self, packed_host, vis_host, accumulate: bool = False, stream=None):
        """execute_host without the final wait: keep both buffers alive and untouched until wait_host()."""
        import torch
        s = torch.cuda.current_stream() if stream is None else stream

        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data

        corr_submit_host(self._h, ptr(packed_host), ptr(vis_host), int(accumulate), s.cuda_stream)
        return vis_host

    def wait_host(self):
        corr_wait_host(self._h)

    def close(self):
        if getattr(self, "_h", None):
            corr_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
