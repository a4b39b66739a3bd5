"""ctypes front end of the CPU oracle (oracle/oracle.cpp) — TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs
may import this package. It imports nothing from ``paper_1405_2915_b200``; the product never imports
it. See oracle.cpp's header for the definitions, readings and pins.

Two builds of the same source: ``liboracle.so`` (single thread, the parity oracle) and
``liboracle_omp.so`` (``-fopenmp``: the same loops over independent outputs run in parallel; Reduce
and Scan stay sequential). ``use_openmp(True)`` selects the latter for the long full-size runs.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIBS = {False: os.path.join(_HERE, "liboracle.so"), True: os.path.join(_HERE, "liboracle_omp.so")}

FN_ADD, FN_MULT, FN_MAX, FN_SAXPY = 0, 1, 2, 3
EDGE_CONSTANT, EDGE_DUPLICATE, EDGE_CYCLIC = 0, 1, 2
SCAN_INCLUSIVE, SCAN_EXCLUSIVE = 0, 1
AXIS_ROW, AXIS_COL = 0, 1


def build(force: bool = False) -> None:
    """Compile both builds of the oracle with g++ (building the checker is not using it)."""
    for omp, path in _LIBS.items():
        if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
            continue
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-o", path, _SRC]
        if omp:
            cmd.insert(1, "-fopenmp")
        subprocess.run(cmd, check=True)


_loaded: dict[bool, C.CDLL] = {}
_omp = False


def use_openmp(flag: bool) -> None:
    global _omp
    _omp = bool(flag)


def threads() -> int:
    """Threads the stencil/Map loops of the selected build use."""
    return (os.cpu_count() or 1) if _omp else 1


_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")


def _lib() -> C.CDLL:
    if _omp not in _loaded:
        build()
        L = C.CDLL(_LIBS[_omp])
        vp, sz, dbl, i = C.c_void_p, C.c_size_t, C.c_double, C.c_int
        L.oracle_map_f32.argtypes = [i, dbl, _f32p, vp, sz, _f64p]
        L.oracle_map_i32.argtypes = [i, C.c_int32, _i32p, vp, sz, _i32p]
        L.oracle_map3_f32.argtypes = [_f32p, _f32p, _f32p, sz, _f64p]
        L.oracle_map3_i32.argtypes = [_i32p, _i32p, _i32p, sz, _i32p]
        L.oracle_reduce_f32.argtypes = [i, _f32p, sz, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_reduce_i32.argtypes = [i, _i32p, sz, C.POINTER(C.c_int32), C.POINTER(C.c_int64)]
        L.oracle_reduce_rows_f32.argtypes = [i, _f32p, sz, sz, _f64p, _f64p]
        L.oracle_reduce_rows_i32.argtypes = [i, _i32p, sz, sz, _i32p]
        L.oracle_mapreduce_f32.argtypes = [i, i, dbl, _f32p, vp, sz, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_mapreduce_i32.argtypes = [i, i, C.c_int32, _i32p, vp, sz, C.POINTER(C.c_int32)]
        L.oracle_scan_i32.argtypes = [i, i, C.c_int32, _i32p, sz, _i32p]
        L.oracle_scan_f32.argtypes = [i, i, dbl, _f32p, sz, _f64p, _f64p]
        L.oracle_mapoverlap_1d_f32.argtypes = [_f32p, i, i, dbl, _f32p, sz, sz, sz, _f64p, _f64p]
        L.oracle_mapoverlap_1d_matrix_f32.argtypes = [_f32p, i, i, dbl, i, _f32p, sz, sz, _f64p, _f64p]
        L.oracle_mapoverlap_1d_matrix_f64.argtypes = [_f32p, i, i, dbl, i, _f64p, sz, sz, _f64p, _f64p]
        L.oracle_mapoverlap_2d_f32.argtypes = [_f32p, i, i, i, dbl, _f32p, sz, sz, sz, sz, _f64p, _f64p]
        L.oracle_map_f64.argtypes = [i, dbl, _f64p, vp, sz, _f64p]
        L.oracle_map3_f64.argtypes = [_f64p, _f64p, _f64p, sz, _f64p]
        L.oracle_mapreduce_f64.argtypes = [i, i, dbl, _f64p, vp, sz, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_mapreduce_f64.restype = i
        L.oracle_scan_f64.argtypes = [i, i, dbl, _f64p, sz, _f64p, _f64p]
        L.oracle_mapoverlap_1d_matrix_f64w.argtypes = [_f64p, i, i, dbl, i, _f64p, sz, sz, _f64p, _f64p]
        L.oracle_mapoverlap_2d_f64w.argtypes = [_f64p, i, i, i, dbl, _f64p, sz, sz, _f64p, _f64p]
        L.oracle_mapoverlap_1d_i32.argtypes = [_i32p, i, i, C.c_int32, _i32p, sz, sz, sz, _i32p]
        L.oracle_mapoverlap_1d_matrix_i32.argtypes = [_i32p, i, i, C.c_int32, i, _i32p, sz, sz, _i32p]
        L.oracle_mapoverlap_2d_i32.argtypes = [_i32p, i, i, i, C.c_int32, _i32p, sz, sz, _i32p]
        for name in ("oracle_reduce_f32", "oracle_reduce_i32", "oracle_mapreduce_f32", "oracle_mapreduce_i32",
                     "oracle_reduce_rows_f32", "oracle_reduce_rows_i32"):
            getattr(L, name).restype = i
        _loaded[_omp] = L
    return _loaded[_omp]


def _opt(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


# ---------------------------------------------------------------- Map
def map_f32(fn: int, c: float, in0, in1=None) -> np.ndarray:
    in0 = _c(in0, np.float32)
    in1 = None if in1 is None else _c(in1, np.float32)
    out = np.empty(in0.size, np.float64)
    _lib().oracle_map_f32(fn, float(c), in0, _opt(in1), in0.size, out)
    return out


def map_i32(fn: int, c: int, in0, in1=None) -> np.ndarray:
    in0 = _c(in0, np.int32)
    in1 = None if in1 is None else _c(in1, np.int32)
    out = np.empty(in0.size, np.int32)
    _lib().oracle_map_i32(fn, int(c), in0, _opt(in1), in0.size, out)
    return out


def map3_muladd_f32(in0, in1, in2) -> np.ndarray:
    """Three-vector Map, MULADD: in0 * in1 + in2 in fp64."""
    a, b, c = _c(in0, np.float32), _c(in1, np.float32), _c(in2, np.float32)
    out = np.empty(a.size, np.float64)
    _lib().oracle_map3_f32(a, b, c, a.size, out)
    return out


def map3_muladd_i32(in0, in1, in2) -> np.ndarray:
    a, b, c = _c(in0, np.int32), _c(in1, np.int32), _c(in2, np.int32)
    out = np.empty(a.size, np.int32)
    _lib().oracle_map3_i32(a, b, c, a.size, out)
    return out


# ---------------------------------------------------------------- Reduce / MapReduce
def reduce_f32(op: int, x):
    """-> (fp64 result, sum |x|)."""
    x = _c(x, np.float32)
    r, a = C.c_double(), C.c_double()
    if _lib().oracle_reduce_f32(op, x, x.size, C.byref(r), C.byref(a)) != 0:
        raise ValueError("reduce of an empty vector")
    return r.value, a.value


def reduce_i32(op: int, x):
    """-> (int32 result wrapped mod 2^32, exact int64 sum)."""
    x = _c(x, np.int32)
    r, e = C.c_int32(), C.c_int64()
    if _lib().oracle_reduce_i32(op, x, x.size, C.byref(r), C.byref(e)) != 0:
        raise ValueError("reduce of an empty vector")
    return r.value, e.value


def reduce_rows_f32(op: int, X):
    """Row-wise Reduce of a matrix -> (fp64 results[rows], sum |x| per row)."""
    X = _c(X, np.float32)
    rows, cols = X.shape
    r, a = np.empty(rows, np.float64), np.empty(rows, np.float64)
    if _lib().oracle_reduce_rows_f32(op, X.reshape(-1), rows, cols, r, a) != 0:
        raise ValueError("reduce of empty rows")
    return r, a


def reduce_rows_i32(op: int, X) -> np.ndarray:
    X = _c(X, np.int32)
    rows, cols = X.shape
    r = np.empty(rows, np.int32)
    if _lib().oracle_reduce_rows_i32(op, X.reshape(-1), rows, cols, r) != 0:
        raise ValueError("reduce of empty rows")
    return r


def mapreduce_f32(map_f: int, red_op: int, c: float, in0, in1=None):
    in0 = _c(in0, np.float32)
    in1 = None if in1 is None else _c(in1, np.float32)
    r, a = C.c_double(), C.c_double()
    if _lib().oracle_mapreduce_f32(map_f, red_op, float(c), in0, _opt(in1), in0.size, C.byref(r), C.byref(a)) != 0:
        raise ValueError("mapreduce of empty vectors")
    return r.value, a.value


def mapreduce_i32(map_f: int, red_op: int, c: int, in0, in1=None) -> int:
    in0 = _c(in0, np.int32)
    in1 = None if in1 is None else _c(in1, np.int32)
    r = C.c_int32()
    if _lib().oracle_mapreduce_i32(map_f, red_op, int(c), in0, _opt(in1), in0.size, C.byref(r)) != 0:
        raise ValueError("mapreduce of empty vectors")
    return r.value


# ---------------------------------------------------------------- Scan
def scan_i32(op: int, mode: int, init: int, x) -> np.ndarray:
    x = _c(x, np.int32)
    out = np.empty(x.size, np.int32)
    _lib().oracle_scan_i32(op, mode, int(init), x, x.size, out)
    return out


def scan_f32(op: int, mode: int, init: float, x):
    """-> (fp64 out, abs-prefix denominators)."""
    x = _c(x, np.float32)
    out = np.empty(x.size, np.float64)
    ab = np.empty(x.size, np.float64)
    _lib().oracle_scan_f32(op, mode, float(init), x, x.size, out, ab)
    return out, ab


# ---------------------------------------------------------------- MapOverlap
def mapoverlap_1d(w, r: int, edge: int, pad: float, x, i0: int = 0, i1: int | None = None):
    """-> (fp64 out[i0:i1], sum_k |w_k x~_{i+k}|)."""
    w = _c(w, np.float32)
    x = _c(x, np.float32)
    assert w.size == 2 * r + 1
    i1 = x.size if i1 is None else i1
    out = np.empty(i1 - i0, np.float64)
    ab = np.empty(i1 - i0, np.float64)
    _lib().oracle_mapoverlap_1d_f32(w, r, edge, float(pad), x, x.size, i0, i1, out, ab)
    return out, ab


def mapoverlap_1d_matrix(w, r: int, edge: int, pad: float, axis: int, X):
    """X: 2-D array, fp32 or fp64 (fp64 input keeps a separable pair's intermediate in fp64)."""
    w = _c(w, np.float32)
    assert w.size == 2 * r + 1 and X.ndim == 2
    rows, cols = X.shape
    out = np.empty((rows, cols), np.float64)
    ab = np.empty((rows, cols), np.float64)
    if X.dtype == np.float64:
        _lib().oracle_mapoverlap_1d_matrix_f64(w, r, edge, float(pad), axis, _c(X, np.float64), rows, cols, out, ab)
    else:
        _lib().oracle_mapoverlap_1d_matrix_f32(w, r, edge, float(pad), axis, _c(X, np.float32), rows, cols, out, ab)
    return out, ab


def mapoverlap_2d(W, ry: int, rx: int, edge: int, pad: float, X, row0: int = 0, row1: int | None = None):
    W = _c(W, np.float32).reshape(-1)
    X = _c(X, np.float32)
    assert W.size == (2 * ry + 1) * (2 * rx + 1) and X.ndim == 2
    rows, cols = X.shape
    row1 = rows if row1 is None else row1
    out = np.empty((row1 - row0, cols), np.float64)
    ab = np.empty((row1 - row0, cols), np.float64)
    _lib().oracle_mapoverlap_2d_f32(W, ry, rx, edge, float(pad), X, rows, cols, row0, row1, out, ab)
    return out, ab


# ---------------------------------------------------------------- int32 MapOverlap (wraps modulo 2^32)
def mapoverlap_1d_i32(w, r: int, edge: int, pad: int, x, i0: int = 0, i1: int | None = None) -> np.ndarray:
    w = _c(w, np.int32)
    x = _c(x, np.int32)
    assert w.size == 2 * r + 1
    i1 = x.size if i1 is None else i1
    out = np.empty(i1 - i0, np.int32)
    _lib().oracle_mapoverlap_1d_i32(w, r, edge, int(pad), x, x.size, i0, i1, out)
    return out


def mapoverlap_1d_matrix_i32(w, r: int, edge: int, pad: int, axis: int, X) -> np.ndarray:
    w = _c(w, np.int32)
    X = _c(X, np.int32)
    assert w.size == 2 * r + 1 and X.ndim == 2
    rows, cols = X.shape
    out = np.empty((rows, cols), np.int32)
    _lib().oracle_mapoverlap_1d_matrix_i32(w, r, edge, int(pad), axis, X.reshape(-1), rows, cols, out.reshape(-1))
    return out


def mapoverlap_2d_i32(W, ry: int, rx: int, edge: int, pad: int, X) -> np.ndarray:
    W = _c(W, np.int32).reshape(-1)
    X = _c(X, np.int32)
    assert W.size == (2 * ry + 1) * (2 * rx + 1) and X.ndim == 2
    rows, cols = X.shape
    out = np.empty((rows, cols), np.int32)
    _lib().oracle_mapoverlap_2d_i32(W, ry, rx, edge, int(pad), X.reshape(-1), rows, cols, out.reshape(-1))
    return out


# ---------------------------------------------------------------- fp64 elements (binary128 arithmetic, rounded once)
def map_f64(fn: int, c: float, in0, in1=None) -> np.ndarray:
    in0 = _c(in0, np.float64)
    in1 = None if in1 is None else _c(in1, np.float64)
    out = np.empty(in0.size, np.float64)
    _lib().oracle_map_f64(fn, float(c), in0, _opt(in1), in0.size, out)
    return out


def map3_muladd_f64(in0, in1, in2) -> np.ndarray:
    a, b, c = _c(in0, np.float64), _c(in1, np.float64), _c(in2, np.float64)
    out = np.empty(a.size, np.float64)
    _lib().oracle_map3_f64(a, b, c, a.size, out)
    return out


def reduce_f64(op: int, x):
    """-> (result rounded to fp64, sum |x|)."""
    return mapreduce_f64(-1, op, 0.0, x, None)


def mapreduce_f64(map_f: int, red_op: int, c: float, in0, in1=None):
    in0 = _c(in0, np.float64)
    in1 = None if in1 is None else _c(in1, np.float64)
    r, a = C.c_double(), C.c_double()
    if _lib().oracle_mapreduce_f64(map_f, red_op, float(c), in0, _opt(in1), in0.size, C.byref(r), C.byref(a)) != 0:
        raise ValueError("reduce of an empty vector")
    return r.value, a.value


def scan_f64(op: int, mode: int, init: float, x):
    x = _c(x, np.float64)
    out, ab = np.empty(x.size, np.float64), np.empty(x.size, np.float64)
    _lib().oracle_scan_f64(op, mode, float(init), x, x.size, out, ab)
    return out, ab


def mapoverlap_1d_f64(w, r: int, edge: int, pad: float, x):
    out, ab = mapoverlap_1d_matrix_f64(w, r, edge, pad, AXIS_ROW, _c(x, np.float64).reshape(1, -1))
    return out.reshape(-1), ab.reshape(-1)


def mapoverlap_1d_matrix_f64(w, r: int, edge: int, pad: float, axis: int, X):
    w, X = _c(w, np.float64), _c(X, np.float64)
    assert w.size == 2 * r + 1 and X.ndim == 2
    rows, cols = X.shape
    out, ab = np.empty((rows, cols), np.float64), np.empty((rows, cols), np.float64)
    _lib().oracle_mapoverlap_1d_matrix_f64w(w, r, edge, float(pad), axis, X.reshape(-1), rows, cols, out.reshape(-1), ab.reshape(-1))
    return out, ab


def mapoverlap_2d_f64(W, ry: int, rx: int, edge: int, pad: float, X):
    W, X = _c(W, np.float64).reshape(-1), _c(X, np.float64)
    assert W.size == (2 * ry + 1) * (2 * rx + 1) and X.ndim == 2
    rows, cols = X.shape
    out, ab = np.empty((rows, cols), np.float64), np.empty((rows, cols), np.float64)
    _lib().oracle_mapoverlap_2d_f64w(W, ry, rx, edge, float(pad), X.reshape(-1), rows, cols, out.reshape(-1), ab.reshape(-1))
    return out, ab
