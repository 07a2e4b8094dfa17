"""ctypes front end of the C oracle (oracle/rips_oracle.c) and the per-dimension driver.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg.  It does not import the product package and the product
never imports it.

The driver `barcodes()` follows the paper's per-dimension pipeline (Fig. 3(b)):
dimension 0 by union-find, then for d = 1..dim_max: filtration construction with
clearing (Alg. 7-8), apparent pairs (Alg. 3), reduction of the remaining columns (Alg. 2); the
pivots of dimension d are the clearing set of dimension d+1.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from math import inf

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rips_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

u64p = C.POINTER(C.c_uint64)
f32p = C.POINTER(C.c_float)
i64p = C.POINTER(C.c_int64)


def build(force: bool = False) -> str:
    """Compile oracle/rips_oracle.c with gcc (plain C, OpenMP over independent simplices)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_binomial.restype = C.c_uint64
        _lib.oracle_binomial.argtypes = [C.c_int, C.c_int]
        _lib.oracle_encode.restype = C.c_uint64
        _lib.oracle_diameter.restype = C.c_float
        _lib.oracle_diameter.argtypes = [C.c_void_p, C.c_uint64, C.c_int, C.c_int]
        _lib.oracle_decode.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_void_p]
        _lib.oracle_free.argtypes = [C.c_void_p]
        _lib.oracle_stage1.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_int64,
                                       C.c_uint64, C.c_uint64, C.c_int, C.POINTER(f32p), C.POINTER(u64p),
                                       i64p, i64p]
        _lib.oracle_stage2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int64,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.oracle_dim0.argtypes = [C.c_void_p, C.c_int, C.c_float, C.POINTER(u64p), C.POINTER(u64p),
                                     C.POINTER(f32p), i64p, i64p]
        _lib.oracle_reduce.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_int64,
                                       C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(u64p), C.POINTER(u64p),
                                       i64p, C.POINTER(u64p), i64p, i64p]
        _lib.oracle_reduce_explicit.argtypes = _lib.oracle_reduce.argtypes
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(t: int) -> None:
    """OpenMP threads of stage 1 / stage 2 (bench.py's cpu_baseline reports all cores and one thread)."""
    lib().oracle_set_threads(int(t))


def _take(ptr, count, dtype):
    """Copy a malloc'ed C array into numpy and free it."""
    if count:
        arr = np.ctypeslib.as_array(ptr, shape=(count,)).astype(dtype, copy=True)
    else:
        arr = np.zeros(0, dtype=dtype)
    lib().oracle_free(ptr)
    return arr


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _u64(a):
    return np.ascontiguousarray(a, dtype=np.uint64)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a.size else None


def binomial(n: int, k: int) -> int:
    return int(lib().oracle_binomial(n, k))


def decode(idx: int, m: int, n: int):
    out = np.zeros(m, dtype=np.int32)
    lib().oracle_decode(idx, m, n, out.ctypes.data_as(C.c_void_p))
    return [int(x) for x in out]


def encode(verts_decreasing, n: int) -> int:
    v = np.ascontiguousarray(verts_decreasing, dtype=np.int32)
    return int(lib().oracle_encode(v.ctypes.data_as(C.c_void_p), len(v), n))


def diameter(dist, idx: int, m: int, n: int) -> float:
    dist = _f32(dist)
    return float(lib().oracle_diameter(_ptr(dist), idx, m, n))


def stage1(dist, n, d, threshold=inf, cleared=(), idx_lo=0, idx_hi=None, sort=True):
    """Algorithms 7-8.  Returns (diam float32[len], cidx uint64[len], counts dict)."""
    dist = _f32(dist)
    cleared = _u64(np.sort(np.asarray(cleared, dtype=np.uint64)))
    if idx_hi is None:
        idx_hi = binomial(n, d + 1)
    pd, pc, ln = f32p(), u64p(), C.c_int64()
    counts = (C.c_int64 * 3)()
    lib().oracle_stage1(_ptr(dist), n, d, threshold, _ptr(cleared), cleared.size, idx_lo, idx_hi,
                        1 if sort else 0, C.byref(pd), C.byref(pc), C.byref(ln), counts)
    k = ln.value
    return (_take(pd, k, np.float32), _take(pc, k, np.uint64),
            {"kept": counts[0], "removed_by_diameter": counts[1], "cleared": counts[2]})


def stage2(dist, n, d, diam, cidx, want_visits=False):
    """Algorithm 3 per column.  Returns dict with
       flag  uint8[len]   1 iff the column is apparent
       app_t, app_s       the apparent pairs (cidx(t), cidx(s)) ascending by t
       non_diam, non_cidx the non-apparent columns in the order given
       visits             cofacets evaluated per column (if asked)"""
    dist, diam, cidx = _f32(dist), _f32(diam), _u64(cidx)
    ln = diam.size
    flag = np.zeros(ln, dtype=np.uint8)
    t = np.zeros(ln, dtype=np.uint64)
    visits = np.zeros(ln, dtype=np.int32) if want_visits else None
    lib().oracle_stage2(_ptr(dist), n, d, _ptr(diam), _ptr(cidx), ln, _ptr(flag), _ptr(t),
                        _ptr(visits) if want_visits else None)
    app = flag == 1
    order = np.argsort(t[app], kind="stable")
    out = {"flag": flag, "app_t": t[app][order], "app_s": cidx[app][order],
           "non_diam": diam[~app], "non_cidx": cidx[~app]}
    if want_visits:
        out["visits"] = visits
    return out


def dim0(dist, n, threshold=inf):
    """Union-find.  Returns dict: t (edge cidx, ascending), s (birth vertex of the dying class),
    death (edge diameter), n_components."""
    dist = _f32(dist)
    pt, ps, pd = u64p(), u64p(), f32p()
    npairs, ncomp = C.c_int64(), C.c_int64()
    lib().oracle_dim0(_ptr(dist), n, threshold, C.byref(pt), C.byref(ps), C.byref(pd), C.byref(npairs),
                      C.byref(ncomp))
    k = npairs.value
    return {"t": _take(pt, k, np.uint64), "s": _take(ps, k, np.uint64), "death": _take(pd, k, np.float32),
            "n_components": ncomp.value}


def reduce_columns(dist, n, d, threshold, col_cidx, known_t=(), known_s=(), explicit=False):
    """The reduction over the given columns (coboundary order).  Returns dict: t, s (pivots in processing
    order), essential (cidx of zero columns), additions.  explicit=False: implicit columns, working column a
    heap (oracle_reduce); explicit=True: Algorithm 1 on the explicit coboundary matrix, working column a bit
    array over all rows (oracle_reduce_explicit) -- the same pairs, for inputs whose reduced columns fill in."""
    dist, col_cidx = _f32(dist), _u64(col_cidx)
    known_t, known_s = _u64(known_t), _u64(known_s)
    pt, ps, pe = u64p(), u64p(), u64p()
    npiv, ness, adds = C.c_int64(), C.c_int64(), C.c_int64()
    fn = lib().oracle_reduce_explicit if explicit else lib().oracle_reduce
    fn(_ptr(dist), n, d, threshold, _ptr(col_cidx), col_cidx.size, _ptr(known_t),
                        _ptr(known_s), known_t.size, C.byref(pt), C.byref(ps), C.byref(npiv), C.byref(pe),
                        C.byref(ness), C.byref(adds))
    # the three arrays were allocated with ncols entries each; copy the used prefix
    t = _take(pt, npiv.value, np.uint64)
    s = _take(ps, npiv.value, np.uint64)
    e = _take(pe, ness.value, np.uint64)
    return {"t": t, "s": s, "essential": e, "additions": adds.value}


def barcodes(dist, n, dim_max, threshold=inf, use_apparent=True, explicit=False):
    """The whole pipeline.  Returns dict d -> dict with every exposed array:

      d = 0:  pivot_t, pivot_s (ascending t), bars
      d >= 1: filt_diam, filt_cidx (coboundary order), counts, app_t, app_s, non_diam, non_cidx,
              red_t, red_s (pivots found by the reduction, processing order), essential,
              pivot_t, pivot_s (A_d united with the reduced pivots, ascending t), bars, additions

    bars: float32 array [k,2] in column order of the birth simplex (reading R13), zero-length
    bars dropped (R11), death = +inf for essential classes (R12).
    use_apparent=False reduces ALL uncleared columns (apparent pairs are then only reported, so that
    "apparent pairs are persistence pairs", is a real test)."""
    dist = _f32(dist)
    out = {}
    z = dim0(dist, n, threshold)
    bars0 = [(0.0, float(x)) for x in z["death"] if x > 0] + [(0.0, inf)] * z["n_components"]
    out[0] = {"pivot_t": z["t"], "pivot_s": z["s"], "bars": np.array(bars0, dtype=np.float32).reshape(-1, 2),
              "n_components": z["n_components"]}
    cleared = z["t"]
    for d in range(1, dim_max + 1):
        fd, fc, counts = stage1(dist, n, d, threshold, cleared)
        s2 = stage2(dist, n, d, fd, fc)
        if use_apparent:
            red = reduce_columns(dist, n, d, threshold, s2["non_cidx"], s2["app_t"], s2["app_s"], explicit)
            all_t = np.concatenate([s2["app_t"], red["t"]])
            all_s = np.concatenate([s2["app_s"], red["s"]])
        else:
            red = reduce_columns(dist, n, d, threshold, fc, explicit=explicit)
            all_t, all_s = red["t"], red["s"]
        order = np.argsort(all_t, kind="stable")
        piv_t, piv_s = all_t[order], all_s[order]
        # bars in column order of the birth simplex
        diam_of = dict(zip((int(c) for c in fc), (float(x) for x in fd))) if fc.size < 2_000_000 else None
        events = []
        m = d + 2
        for t, s in zip(red["t"], red["s"]):
            b = diam_of[int(s)] if diam_of is not None else diameter(dist, int(s), d + 1, n)
            dd = diameter(dist, int(t), m, n)
            if dd != b:
                events.append((int(s), b, dd))
        for s in red["essential"]:
            b = diam_of[int(s)] if diam_of is not None else diameter(dist, int(s), d + 1, n)
            events.append((int(s), b, inf))
        # column order = (diam desc, cidx asc)
        events.sort(key=lambda e: (-e[1], e[0]))
        bars = np.array([(e[1], e[2]) for e in events], dtype=np.float32).reshape(-1, 2)
        out[d] = {"filt_diam": fd, "filt_cidx": fc, "counts": counts,
                  "app_t": s2["app_t"], "app_s": s2["app_s"], "non_diam": s2["non_diam"],
                  "non_cidx": s2["non_cidx"], "red_t": red["t"], "red_s": red["s"],
                  "essential": red["essential"], "pivot_t": piv_t, "pivot_s": piv_s, "bars": bars,
                  "additions": red["additions"]}
        cleared = piv_t
    return out
