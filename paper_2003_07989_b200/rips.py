"""Thin ctypes binding of include/rips.h (argument marshalling only; every step runs in the CUDA kernels).

Same names as the C ABI.  PyTorch is used for device memory (views of the library's arrays are
copied into torch tensors) and for the stream.  There is no CPU fallback: if librips_b200.so is
missing or no CUDA device is usable, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librips_b200.so")
_lib = None

RIPS_OK, RIPS_EINVAL, RIPS_EOVERFLOW, RIPS_ENOMEM, RIPS_ECUDA = 0, -1, -2, -3, -4

# every symbol include/rips.h declares (checked by tests/test_abi.py against the header)
SYMBOLS = [
    "rips_workspace_bytes", "rips_init", "rips_set_mode", "rips_compute", "rips_dim0", "rips_stage1", "rips_stage2", "rips_reduce", "rips_import_pivots",
    "rips_barcodes", "rips_filtration", "rips_apparent_pairs", "rips_nonapparent", "rips_pivots",
    "rips_pivot_lookup", "rips_stats", "rips_timings", "rips_device_bytes", "rips_workspace_in_use", "rips_kernel_launches",
    "rips_sort_u64", "rips_sort_u64_static", "rips_strerror", "rips_last_error", "rips_last_required_bytes", "rips_free",
]


class RipsStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in (
        "n_candidates", "n_removed_by_diameter", "n_cleared", "n_columns", "n_apparent", "n_nonapparent",
        "n_reduced_pivots", "n_essential", "n_additions", "n_bars", "n_slots", "n_regular", "n_reduce_serial",
        "n_reduce_displaced", "reduce_arena_bytes")] + [(k, C.c_int32) for k in (
        "key_bits", "index_bits", "sort_passes", "pair_sort_passes")]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class RipsTimings(C.Structure):
    _fields_ = [(k, C.c_float) for k in (
        "clear_bitmap_ms", "enumerate_ms", "sort_hist_ms", "sort_pass_ms", "apparent_ms", "pair_hist_ms",
        "pair_sort_ms", "stage1_ms", "stage2_ms", "dim0_ms", "reduce_device_ms", "reduce_host_ms", "reduce_xfer_ms")]

    def as_dict(self):
        return {k: float(getattr(self, k)) for k, _ in self._fields_}


class RipsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        l = lib()
        msg = l.rips_strerror(code).decode()
        detail = l.rips_last_error().decode()
        super().__init__(f"{where}: {msg} ({code})" + (f": {detail}" if detail else ""))


def lib():
    """Load librips_b200.so (built by paper_2003_07989_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2003_07989_b200.build` "
                               "(the CUDA extension is required; there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int
        pp = C.POINTER(C.c_void_p)
        pi64 = C.POINTER(C.c_int64)
        l.rips_workspace_bytes.argtypes = [i64, i32, pi64]
        l.rips_init.argtypes = [pp, vp, i64, i32, C.c_float, vp, i64, vp]
        for f in ("rips_compute", "rips_dim0"):
            getattr(l, f).argtypes = [vp]
        for f in ("rips_stage1", "rips_stage2", "rips_reduce", "rips_set_mode"):
            getattr(l, f).argtypes = [vp, i32]
        for f in ("rips_barcodes",):
            getattr(l, f).argtypes = [vp, i32, pp, pi64]
        for f in ("rips_filtration", "rips_apparent_pairs", "rips_nonapparent", "rips_pivots"):
            getattr(l, f).argtypes = [vp, i32, pp, pp, pi64]
        l.rips_import_pivots.argtypes = [vp, i32, vp, vp, i64]
        l.rips_pivot_lookup.argtypes = [vp, i32, vp, i64, vp]
        l.rips_stats.argtypes = [vp, i32, C.POINTER(RipsStats)]
        l.rips_timings.argtypes = [vp, i32, C.POINTER(RipsTimings)]
        l.rips_device_bytes.argtypes = [vp, pi64]
        l.rips_kernel_launches.argtypes = [vp, pi64]
        l.rips_workspace_in_use.argtypes = [vp, pi64, pi64]
        l.rips_last_required_bytes.argtypes = []
        l.rips_last_required_bytes.restype = C.c_int64
        l.rips_sort_u64.argtypes = [vp, vp, i64, i32, i32, vp]
        l.rips_sort_u64_static.argtypes = [vp, vp, i64, i32, i32, vp]
        l.rips_strerror.argtypes = [i32]
        l.rips_strerror.restype = C.c_char_p
        l.rips_last_error.argtypes = []
        l.rips_last_error.restype = C.c_char_p
        l.rips_free.argtypes = [vp]
        l.rips_free.restype = None
        _lib = l
    return _lib


def use_library(path=None):
    """Load another build of the same C ABI (the stress build of build.build_stress); None = the product library."""
    global _lib, LIB_PATH
    _lib = None
    LIB_PATH = path or os.path.join(_HERE, "librips_b200.so")
    return lib()


def _check(code, where):
    if code != RIPS_OK:
        raise RipsError(code, where)


def _torch():
    import torch
    return torch


class _DevView:
    """__cuda_array_interface__ wrapper of a raw device pointer (zero-copy view for torch.as_tensor)."""

    def __init__(self, ptr, count, typestr):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2}


def _dev_to_torch(ptr, count, dtype_name):
    """Copy `count` elements at device pointer `ptr` (owned by the library) into a fresh torch CUDA tensor."""
    torch = _torch()
    dt, ts = {"f32": (torch.float32, "<f4"), "i64": (torch.int64, "<i8")}[dtype_name]
    if not count:
        return torch.empty(0, dtype=dt, device="cuda")
    return torch.as_tensor(_DevView(ptr, count, ts), device="cuda").clone()


def rips_workspace_bytes(n, dim_max):
    b = C.c_int64()
    _check(lib().rips_workspace_bytes(n, dim_max, C.byref(b)), "rips_workspace_bytes")
    return b.value


def rips_last_required_bytes():
    return int(lib().rips_last_required_bytes())


def rips_sort_u64(keys, lo_bit, hi_bit):
    """In-place stable sort of a torch int64 CUDA tensor (read as uint64) on bits [lo_bit, hi_bit)."""
    torch = _torch()
    assert keys.is_cuda and keys.dtype == torch.int64 and keys.is_contiguous()
    tmp = torch.empty_like(keys)
    st = torch.cuda.current_stream().cuda_stream
    _check(lib().rips_sort_u64(keys.data_ptr(), tmp.data_ptr(), keys.numel(), lo_bit, hi_bit, st), "rips_sort_u64")
    return keys


def rips_sort_u64_static(keys, tmp, lo_bit, hi_bit):
    """rips_sort_u64 without any allocation: the sort's scratch is a static array inside the library (at most 2^22
    records), `tmp` is the caller's ping-pong buffer.  Enqueued on torch's current stream; calls must not overlap."""
    torch = _torch()
    assert keys.is_cuda and keys.dtype == torch.int64 and keys.is_contiguous()
    assert tmp.is_cuda and tmp.dtype == torch.int64 and tmp.is_contiguous() and tmp.numel() >= keys.numel()
    st = torch.cuda.current_stream().cuda_stream
    _check(lib().rips_sort_u64_static(keys.data_ptr(), tmp.data_ptr(), keys.numel(), lo_bit, hi_bit, st), "rips_sort_u64_static")
    return keys


class Rips:
    """One context = one distance matrix.  Methods mirror the C entry points (rips_<method>)."""

    def __init__(self, dist_lower, n, dim_max, threshold=float("inf"), stream=None, workspace=None):
        """workspace: None = the library allocates its own; an int = that many bytes of torch device memory; a torch
        uint8 CUDA tensor = that memory (it must outlive the context, which keeps a reference)."""
        torch = _torch()
        l = lib()
        self._h = C.c_void_p()
        self.n, self.dim_max, self.threshold = int(n), int(dim_max), float(threshold)
        if hasattr(dist_lower, "is_cuda"):
            assert dist_lower.dtype == torch.float32 and dist_lower.is_contiguous()
            ptr, self._keep = dist_lower.data_ptr(), dist_lower
        else:
            arr = np.ascontiguousarray(dist_lower, dtype=np.float32)
            ptr, self._keep = arr.ctypes.data, arr
        assert self._keep.size == n * (n - 1) // 2 if not hasattr(self._keep, "numel") else self._keep.numel() == n * (n - 1) // 2
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream().cuda_stream
        if isinstance(workspace, int):
            workspace = torch.empty(workspace, dtype=torch.uint8, device="cuda")
        self._workspace = workspace
        wptr, wbytes = (workspace.data_ptr(), workspace.numel()) if workspace is not None else (None, 0)
        _check(l.rips_init(C.byref(self._h), ptr if n > 1 else None, n, dim_max, threshold, wptr, wbytes, stream or None),
               "rips_init")

    # -- life cycle
    def free(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().rips_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.free()

    # -- compute
    def set_mode(self, mode):
        """0 = auto, 1 = dense, 2 = sparse (RIPS_MODE_*); before the first stage 1."""
        _check(lib().rips_set_mode(self._h, {"auto": 0, "dense": 1, "sparse": 2}.get(mode, mode)), "rips_set_mode")
        return self

    def compute(self):
        _check(lib().rips_compute(self._h), "rips_compute")
        return self

    def dim0(self):
        _check(lib().rips_dim0(self._h), "rips_dim0")

    def stage1(self, d):
        _check(lib().rips_stage1(self._h, d), "rips_stage1")

    def stage2(self, d):
        _check(lib().rips_stage2(self._h, d), "rips_stage2")

    def reduce(self, d):
        _check(lib().rips_reduce(self._h, d), "rips_reduce")

    def import_pivots(self, d, t, s):
        """Install pivots found elsewhere (host arrays, ascending by t) as dimension d's non-apparent pivots."""
        t = np.ascontiguousarray(t, dtype=np.uint64)
        s = np.ascontiguousarray(s, dtype=np.uint64)
        assert t.size == s.size
        _check(lib().rips_import_pivots(self._h, d, t.ctypes.data if t.size else None,
                                        s.ctypes.data if s.size else None, t.size), "rips_import_pivots")

    # -- results
    def barcodes(self, d):
        p, k = C.c_void_p(), C.c_int64()
        _check(lib().rips_barcodes(self._h, d, C.byref(p), C.byref(k)), "rips_barcodes")
        if k.value == 0:
            return np.zeros((0, 2), dtype=np.float32)
        buf = (C.c_float * (2 * k.value)).from_address(p.value)
        return np.frombuffer(buf, dtype=np.float32).reshape(-1, 2).copy()

    def _two(self, fn, d, first):
        a, b, k = C.c_void_p(), C.c_void_p(), C.c_int64()
        _check(getattr(lib(), fn)(self._h, d, C.byref(a), C.byref(b), C.byref(k)), fn)
        return _dev_to_torch(a.value, k.value, first), _dev_to_torch(b.value, k.value, "i64")

    def filtration(self, d):
        """(diam float32[len], cidx int64[len]) torch CUDA tensors, coboundary order."""
        return self._two("rips_filtration", d, "f32")

    def apparent_pairs(self, d):
        return self._two("rips_apparent_pairs", d, "i64")

    def nonapparent(self, d):
        return self._two("rips_nonapparent", d, "f32")

    def pivots(self, d):
        return self._two("rips_pivots", d, "i64")

    def pivot_lookup(self, d, t_query):
        torch = _torch()
        q = torch.as_tensor(np.asarray(t_query, dtype=np.int64), device="cuda").contiguous()
        out = torch.empty_like(q)
        _check(lib().rips_pivot_lookup(self._h, d, q.data_ptr(), q.numel(), out.data_ptr()), "rips_pivot_lookup")
        return out

    def stats(self, d):
        s = RipsStats()
        _check(lib().rips_stats(self._h, d, C.byref(s)), "rips_stats")
        return s.as_dict()

    def timings(self, d):
        t = RipsTimings()
        _check(lib().rips_timings(self._h, d, C.byref(t)), "rips_timings")
        return t.as_dict()

    def device_bytes(self):
        b = C.c_int64()
        _check(lib().rips_device_bytes(self._h, C.byref(b)), "rips_device_bytes")
        return b.value

    def workspace_in_use(self):
        """(bytes handed out now, peak)"""
        a, b = C.c_int64(), C.c_int64()
        _check(lib().rips_workspace_in_use(self._h, C.byref(a), C.byref(b)), "rips_workspace_in_use")
        return a.value, b.value

    def kernel_launches(self):
        b = C.c_int64()
        _check(lib().rips_kernel_launches(self._h, C.byref(b)), "rips_kernel_launches")
        return b.value
