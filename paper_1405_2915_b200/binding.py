"""Thin ctypes binding of libskel.so (include/skel.h). Argument marshalling only: every step of
the skeleton path runs in the library's CUDA kernels. There is no CPU fallback; importing this
module fails loudly when the library has not been built (``python -m paper_1405_2915_b200.build`` or
``__graft_entry__.build()``).

The module-level ``skel_*`` functions are the C entry points with their argtypes set. The small
classes below (Context, Vector, Matrix) only own handles and convert numpy arrays / torch
tensors to pointers. PyTorch supplies the CUDA stream and the caching allocator, nothing else.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libskel.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: the CUDA library has not been built. Run __graft_entry__.build() "
        "(nvcc, sm_100a). There is no CPU fallback.")
lib = C.CDLL(LIB_PATH)

# ---- enums (include/skel.h) --------------------------------------------------------------------
OK, ERR_INVALID_ARG, ERR_SIZE_MISMATCH, ERR_DTYPE, ERR_UNSUPPORTED, ERR_EMPTY, ERR_ALIAS, ERR_UNINIT, \
    ERR_OOM, ERR_CUDA, ERR_BUSY, ERR_IO = range(12)
STATUS_NAMES = ["OK", "INVALID_ARG", "SIZE_MISMATCH", "DTYPE", "UNSUPPORTED", "EMPTY", "ALIAS", "UNINIT", "OOM",
                "CUDA", "BUSY", "IO"]
F32, I32, F64 = 0, 1, 2
FN_ADD, FN_MULT, FN_MAX, FN_SAXPY, FN_WSTENCIL, FN_MULADD = 0, 1, 2, 3, 4, 5
EDGE_CONSTANT, EDGE_DUPLICATE, EDGE_CYCLIC = 0, 1, 2
SCAN_INCLUSIVE, SCAN_EXCLUSIVE = 0, 1
AXIS_ROW, AXIS_COL = 0, 1
READ, WRITE, READWRITE = 0, 1, 2
LAZY, EAGER = 0, 1
SK_MAP, SK_REDUCE, SK_MAPREDUCE, SK_SCAN, SK_OVERLAP1D, SK_OVERLAP1D_COL, SK_OVERLAP2D, SK_SEPARABLE, SK_REDUCE_ROWS, SK_COUNT = range(10)
ST_UNINIT, ST_HOST, ST_DEVICE, ST_SHARED = 0, 1, 2, 3

_NP = {F32: np.float32, I32: np.int32, F64: np.float64}
_CT = {F32: C.c_float, I32: C.c_int32, F64: C.c_double}
_FROM_NP = {np.dtype(np.float32): F32, np.dtype(np.int32): I32, np.dtype(np.float64): F64}


class SkelInstance(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("skeleton", "fn", "fn2", "dtype", "r0", "r1", "edge", "mode")]


class SkelStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("h2d_bytes", "h2d_count", "d2h_bytes", "d2h_count", "h2d_elided",
                                           "d2h_elided", "scalar_d2h_count", "launches", "fused_launches",
                                           "fused_calls")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_vp, _sz, _i, _d = C.c_void_p, C.c_size_t, C.c_int, C.c_double
_pp = C.POINTER(C.c_void_p)
_SIGS = {
    "skel_abi_version": ([], _i),
    "skel_ctx_create": ([_vp, ALLOC_FN, FREE_FN, _vp, _pp], _i),
    "skel_ctx_destroy": ([_vp], _i),
    "skel_ctx_sync": ([_vp], _i),
    "skel_ctx_set_coherence": ([_vp, _i], _i),
    "skel_probe_fma_peak": ([_vp, _i, C.POINTER(C.c_double)], _i),
    "skel_probe_fma_with_loads": ([_vp, _i, _i, C.POINTER(C.c_double)], _i),
    "skel_ctx_set_fusion": ([_vp, _i], _i),
    "skel_ctx_set_l2_reuse": ([_vp, _i], _i),
    "skel_ctx_flush": ([_vp], _i),
    "skel_last_error": ([_vp], C.c_char_p),
    "skel_vector_create": ([_vp, _i, _sz, _pp], _i),
    "skel_vector_create_from": ([_vp, _i, _sz, _vp, _pp], _i),
    "skel_vector_adopt_device": ([_vp, _i, _sz, _vp, _pp], _i),
    "skel_vector_destroy": ([_vp], _i),
    "skel_vector_size": ([_vp, C.POINTER(_sz)], _i),
    "skel_vector_host_acquire": ([_vp, _i, _pp], _i),
    "skel_vector_prefetch_host": ([_vp], _i),
    "skel_matrix_prefetch_host": ([_vp], _i),
    "skel_vector_host_acquire_range": ([_vp, _i, _sz, _sz, _pp], _i),
    "skel_matrix_host_acquire_rows": ([_vp, _i, _sz, _sz, _pp], _i),
    "skel_ranges_add": ([C.POINTER(C.c_uint64), C.POINTER(C.c_size_t), _sz, C.c_uint64, C.c_uint64], _i),
    "skel_vector_host_release": ([_vp], _i),
    "skel_vector_device_ptr": ([_vp, _pp, C.POINTER(_i)], _i),
    "skel_vector_state": ([_vp, C.POINTER(_i)], _i),
    "skel_matrix_create": ([_vp, _i, _sz, _sz, _pp], _i),
    "skel_matrix_create_from": ([_vp, _i, _sz, _sz, _vp, _pp], _i),
    "skel_matrix_adopt_device": ([_vp, _i, _sz, _sz, _vp, _pp], _i),
    "skel_matrix_destroy": ([_vp], _i),
    "skel_matrix_shape": ([_vp, C.POINTER(_sz), C.POINTER(_sz)], _i),
    "skel_matrix_host_acquire": ([_vp, _i, _pp], _i),
    "skel_matrix_host_release": ([_vp], _i),
    "skel_matrix_as_vector": ([_vp, _pp], _i),
    "skel_map": ([_vp, _i, _d, _vp, _vp, _vp], _i),
    "skel_reduce": ([_vp, _i, _vp, _vp], _i),
    "skel_reduce_to": ([_vp, _i, _vp, _vp, _sz], _i),
    "skel_mapreduce": ([_vp, _i, _i, _d, _vp, _vp, _vp], _i),
    "skel_mapreduce_to": ([_vp, _i, _i, _d, _vp, _vp, _vp, _sz], _i),
    "skel_map3": ([_vp, _i, _vp, _vp, _vp, _vp], _i),
    "skel_reduce_rows": ([_vp, _i, _vp, _vp], _i),
    "skel_reduce_async": ([_vp, _i, _vp, _pp], _i),
    "skel_mapreduce_async": ([_vp, _i, _i, _d, _vp, _vp, _pp], _i),
    "skel_future_wait": ([_vp, _vp], _i),
    "skel_future_ready": ([_vp, C.POINTER(_i)], _i),
    "skel_future_destroy": ([_vp], _i),
    "skel_mapoverlap_1d": ([_vp, _vp, _i, _i, _d, _vp, _vp], _i),
    "skel_mapoverlap_1d_matrix": ([_vp, _vp, _i, _i, _d, _i, _vp, _vp], _i),
    "skel_mapoverlap_2d": ([_vp, _vp, _i, _i, _i, _d, _vp, _vp], _i),
    "skel_mapoverlap_1d_f64": ([_vp, _vp, _i, _i, _d, _vp, _vp], _i),
    "skel_mapoverlap_1d_matrix_f64": ([_vp, _vp, _i, _i, _d, _i, _vp, _vp], _i),
    "skel_mapoverlap_2d_f64": ([_vp, _vp, _i, _i, _i, _d, _vp, _vp], _i),
    "skel_mapoverlap_1d_i32": ([_vp, _vp, _i, _i, C.c_int32, _vp, _vp], _i),
    "skel_mapoverlap_1d_matrix_i32": ([_vp, _vp, _i, _i, C.c_int32, _i, _vp, _vp], _i),
    "skel_mapoverlap_2d_i32": ([_vp, _vp, _i, _i, _i, C.c_int32, _vp, _vp], _i),
    "skel_mapoverlap_separable": ([_vp, _vp, _i, _vp, _i, _i, _d, _vp, _vp], _i),
    "skel_scan": ([_vp, _i, _i, _d, _vp, _vp], _i),
    "skel_variant_count": ([_i], _i),
    "skel_variant_name": ([_i, _i], C.c_char_p),
    "skel_tune_instance": ([_vp, C.POINTER(SkelInstance), _i, _i, _sz, _i], _i),
    "skel_plan_save": ([_vp, C.c_char_p], _i),
    "skel_plan_load": ([_vp, C.c_char_p], _i),
    "skel_plan_clear": ([_vp], _i),
    "skel_plan_lookup": ([_vp, C.POINTER(SkelInstance), _sz, C.POINTER(_i)], _i),
    "skel_plan_set": ([_vp, C.POINTER(SkelInstance), _sz, _i], _i),
    "skel_plan_explain": ([_vp, C.POINTER(SkelInstance), _sz, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i)], _i),
    "skel_replay_begin": ([_vp], _i),
    "skel_replay_end": ([_vp, C.POINTER(_i)], _i),
    "skel_replay_run": ([_vp, _i, _i, C.POINTER(_d), C.POINTER(_d)], _i),
    "skel_tune_table": ([_vp, C.POINTER(C.c_float), _sz, C.POINTER(_sz)], _i),
    "skel_force_variant": ([_vp, _i, _i], _i),
    "skel_last_variant": ([_vp, C.POINTER(_i), C.POINTER(_i)], _i),
    "skel_get_stats": ([_vp, C.POINTER(SkelStats)], _i),
    "skel_reset_stats": ([_vp], _i),
    "skel_coherence_step": ([_i, _i, _i, _i, C.POINTER(_i), C.POINTER(_i)], _i),
    "skel_reduce_f32_noalloc": ([_i, _vp, _sz, _vp, _vp], _i),
    "skel_noalloc_max_elements": ([], _sz),
    "skel_noalloc_scratch_bytes": ([], _sz),
    "skel_noalloc_last_error": ([], C.c_char_p),
}
EXPORTS = sorted(_SIGS)
for _name, (_args, _res) in _SIGS.items():
    _f = getattr(lib, _name)  # AttributeError here = the library does not export a declared symbol
    _f.argtypes = _args
    _f.restype = _res
    globals()[_name] = _f


class SkelError(RuntimeError):
    def __init__(self, status: int, msg: str = ""):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__(f"SKEL_ERR_{name}: {msg}")


def coherence_step(state: int, actor: int, access: int, mode: int = LAZY):
    """Pure protocol function. -> (status, new_state, transfer_mask)."""
    ns, tr = C.c_int(), C.c_int()
    st = lib.skel_coherence_step(state, actor, access, mode, C.byref(ns), C.byref(tr))
    return st, ns.value, tr.value


def reduce_f32_noalloc(op: int, device_in: int, n: int, device_result: int, stream: int = 0) -> None:
    """skel_reduce_f32_noalloc: Reduce of n floats at DEVICE address `device_in` into the float at DEVICE address
    `device_result`, asynchronous on `stream` (a cudaStream_t as an integer), scratch in a static device array:
    no allocation, no context. n <= noalloc_max_elements()."""
    st = lib.skel_reduce_f32_noalloc(op, device_in, n, device_result, stream)
    if st != OK:
        raise SkelError(st, (lib.skel_noalloc_last_error() or b"").decode())


def noalloc_max_elements() -> int:
    return int(lib.skel_noalloc_max_elements())


def variant_names(skeleton: int) -> list[str]:
    return [lib.skel_variant_name(skeleton, v).decode() for v in range(lib.skel_variant_count(skeleton))]


class Future:
    """skel_future: the scalar of a skel_reduce_async / skel_mapreduce_async call (marshalling only)."""

    def __init__(self, ctx: "Context", h, dtype: int):
        self.ctx, self.h, self.dtype = ctx, h, dtype

    def wait(self):
        res = _CT[self.dtype]()
        self.ctx.check(lib.skel_future_wait(self.h, C.byref(res)))
        return res.value

    def ready(self) -> bool:
        r = C.c_int()
        self.ctx.check(lib.skel_future_ready(self.h, C.byref(r)))
        return bool(r.value)

    def destroy(self):
        if self.h:
            self.ctx.check(lib.skel_future_destroy(self.h))
            self.h = None

    def result(self):
        """wait + destroy"""
        v = self.wait()
        self.destroy()
        return v


class Context:
    """Owns a skel_ctx. `stream`: an int cudaStream_t (default: torch's current stream).
    `torch_allocator`: route container device memory through torch's caching allocator."""

    def __init__(self, stream: int | None = None, torch_allocator: bool = True, lazy_cuda: bool = False):
        self._alloc_cb = ALLOC_FN()
        self._free_cb = FREE_FN()
        if stream is None and not lazy_cuda:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        if torch_allocator and not lazy_cuda:
            import torch
            dev = torch.cuda.current_device()

            def _alloc(nbytes, strm, _user):
                try:
                    return torch.cuda.caching_allocator_alloc(nbytes, dev, strm or 0)
                except Exception:  # OOM -> NULL, reported as SKEL_ERR_OOM
                    return None

            def _free(ptr, _user):
                torch.cuda.caching_allocator_delete(ptr)

            self._alloc_cb = ALLOC_FN(_alloc)
            self._free_cb = FREE_FN(_free)
        h = C.c_void_p()
        st = lib.skel_ctx_create(C.c_void_p(stream or 0), self._alloc_cb, self._free_cb, None, C.byref(h))
        if st != OK:
            raise SkelError(st, "skel_ctx_create")
        self.h = h
        self.stream = stream or 0

    def check(self, st: int):
        if st != OK:
            raise SkelError(st, lib.skel_last_error(self.h).decode())

    def close(self):
        if self.h:
            self.check(lib.skel_ctx_destroy(self.h))
            self.h = None

    def sync(self):
        self.check(lib.skel_ctx_sync(self.h))

    def set_coherence(self, mode: int):
        self.check(lib.skel_ctx_set_coherence(self.h, mode))

    def probe_fma_with_loads(self, lds128_per_iter: int, reps: int = 5) -> float:
        """FMAs per second of an FFMA2 stream with `lds128_per_iter` LDS.128 per 144 FMA-pipe cycles."""
        out = C.c_double(0.0)
        self.check(lib.skel_probe_fma_with_loads(self.h, lds128_per_iter, reps, C.byref(out)))
        return out.value

    def probe_fma_peak(self, reps: int = 5) -> float:
        """FP32 FMAs per second of the device (register-only FFMA kernel)."""
        out = C.c_double(0.0)
        self.check(lib.skel_probe_fma_peak(self.h, reps, C.byref(out)))
        return out.value

    def set_l2_reuse(self, enable: bool):
        self.check(lib.skel_ctx_set_l2_reuse(self.h, 1 if enable else 0))

    def set_fusion(self, enable: bool):
        self.check(lib.skel_ctx_set_fusion(self.h, 1 if enable else 0))

    def flush(self):
        self.check(lib.skel_ctx_flush(self.h))

    def stats(self) -> dict:
        s = SkelStats()
        self.check(lib.skel_get_stats(self.h, C.byref(s)))
        return s.as_dict()

    def reset_stats(self):
        self.check(lib.skel_reset_stats(self.h))

    def force_variant(self, skeleton: int, variant: int):
        self.check(lib.skel_force_variant(self.h, skeleton, variant))

    def last_variant(self):
        a, b = C.c_int(), C.c_int()
        self.check(lib.skel_last_variant(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    # ---- containers
    def vector(self, n: int, dtype: int = F32) -> "Vector":
        h = C.c_void_p()
        self.check(lib.skel_vector_create(self.h, dtype, n, C.byref(h)))
        return Vector(self, h, dtype, n)

    def vector_from(self, arr: np.ndarray) -> "Vector":
        arr = np.ascontiguousarray(arr)
        dtype = _FROM_NP[arr.dtype]
        h = C.c_void_p()
        self.check(lib.skel_vector_create_from(self.h, dtype, arr.size, arr.ctypes.data_as(C.c_void_p), C.byref(h)))
        return Vector(self, h, dtype, arr.size)

    def vector_adopt(self, tensor) -> "Vector":
        """Wrap a contiguous 1-D torch CUDA tensor (float32 / int32); keeps a reference to it."""
        import torch
        assert tensor.is_cuda and tensor.is_contiguous()
        dtype = {torch.float32: F32, torch.int32: I32, torch.float64: F64}[tensor.dtype]
        h = C.c_void_p()
        self.check(lib.skel_vector_adopt_device(self.h, dtype, tensor.numel(), C.c_void_p(tensor.data_ptr()), C.byref(h)))
        v = Vector(self, h, dtype, tensor.numel())
        v._keep = tensor
        return v

    def matrix(self, rows: int, cols: int, dtype: int = F32) -> "Matrix":
        h = C.c_void_p()
        self.check(lib.skel_matrix_create(self.h, dtype, rows, cols, C.byref(h)))
        return Matrix(self, h, dtype, rows, cols)

    def matrix_from(self, arr: np.ndarray) -> "Matrix":
        arr = np.ascontiguousarray(arr)
        assert arr.ndim == 2
        dtype = _FROM_NP[arr.dtype]
        h = C.c_void_p()
        self.check(lib.skel_matrix_create_from(self.h, dtype, arr.shape[0], arr.shape[1], arr.ctypes.data_as(C.c_void_p), C.byref(h)))
        return Matrix(self, h, dtype, arr.shape[0], arr.shape[1])

    def matrix_adopt(self, tensor) -> "Matrix":
        import torch
        assert tensor.is_cuda and tensor.is_contiguous() and tensor.dim() == 2
        dtype = {torch.float32: F32, torch.int32: I32, torch.float64: F64}[tensor.dtype]
        h = C.c_void_p()
        self.check(lib.skel_matrix_adopt_device(self.h, dtype, tensor.shape[0], tensor.shape[1], C.c_void_p(tensor.data_ptr()), C.byref(h)))
        m = Matrix(self, h, dtype, tensor.shape[0], tensor.shape[1])
        m._keep = tensor
        return m

    # ---- skeletons (same names and argument order as the C entry points)
    def map(self, f: int, c: float, in0: "Vector", in1: "Vector | None", out: "Vector"):
        self.check(lib.skel_map(self.h, f, c, in0.h, in1.h if in1 is not None else None, out.h))

    def map3(self, f: int, in0: "Vector", in1: "Vector", in2: "Vector", out: "Vector"):
        self.check(lib.skel_map3(self.h, f, in0.h, in1.h, in2.h, out.h))

    def reduce(self, op: int, x: "Vector"):
        res = _CT[x.dtype]()
        self.check(lib.skel_reduce(self.h, op, x.h, C.byref(res)))
        return res.value

    def reduce_to(self, op: int, x: "Vector", out: "Vector", out_index: int = 0):
        self.check(lib.skel_reduce_to(self.h, op, x.h, out.h, out_index))

    def mapreduce(self, map_f: int, red_op: int, c: float, in0: "Vector", in1: "Vector | None"):
        res = _CT[in0.dtype]()
        self.check(lib.skel_mapreduce(self.h, map_f, red_op, c, in0.h, in1.h if in1 is not None else None, C.byref(res)))
        return res.value

    def mapreduce_to(self, map_f: int, red_op: int, c: float, in0, in1, out: "Vector", out_index: int = 0):
        self.check(lib.skel_mapreduce_to(self.h, map_f, red_op, c, in0.h, in1.h if in1 is not None else None, out.h, out_index))

    def reduce_async(self, op: int, x: "Vector") -> "Future":
        h = C.c_void_p()
        self.check(lib.skel_reduce_async(self.h, op, x.h, C.byref(h)))
        return Future(self, h, x.dtype)

    def mapreduce_async(self, map_f: int, red_op: int, c: float, in0: "Vector", in1: "Vector | None") -> "Future":
        h = C.c_void_p()
        self.check(lib.skel_mapreduce_async(self.h, map_f, red_op, c, in0.h, in1.h if in1 is not None else None, C.byref(h)))
        return Future(self, h, in0.dtype)

    def reduce_rows(self, op: int, x: "Matrix", out: "Vector"):
        self.check(lib.skel_reduce_rows(self.h, op, x.h, out.h))

    def mapoverlap_1d(self, w, r: int, edge: int, pad: float, x: "Vector", out: "Vector"):
        w = np.ascontiguousarray(w, np.float32)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, x.h, out.h))

    def mapoverlap_1d_matrix(self, w, r: int, edge: int, pad: float, axis: int, x: "Matrix", out: "Matrix"):
        w = np.ascontiguousarray(w, np.float32)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d_matrix(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, axis, x.h, out.h))

    def mapoverlap_2d(self, W, ry: int, rx: int, edge: int, pad: float, x: "Matrix", out: "Matrix"):
        W = np.ascontiguousarray(W, np.float32)
        assert W.size == (2 * ry + 1) * (2 * rx + 1)
        self.check(lib.skel_mapoverlap_2d(self.h, W.ctypes.data_as(C.c_void_p), ry, rx, edge, pad, x.h, out.h))

    def mapoverlap_1d_f64(self, w, r: int, edge: int, pad: float, x: "Vector", out: "Vector"):
        w = np.ascontiguousarray(w, np.float64)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d_f64(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, x.h, out.h))

    def mapoverlap_1d_matrix_f64(self, w, r: int, edge: int, pad: float, axis: int, x: "Matrix", out: "Matrix"):
        w = np.ascontiguousarray(w, np.float64)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d_matrix_f64(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, axis, x.h, out.h))

    def mapoverlap_2d_f64(self, W, ry: int, rx: int, edge: int, pad: float, x: "Matrix", out: "Matrix"):
        W = np.ascontiguousarray(W, np.float64)
        assert W.size == (2 * ry + 1) * (2 * rx + 1)
        self.check(lib.skel_mapoverlap_2d_f64(self.h, W.ctypes.data_as(C.c_void_p), ry, rx, edge, pad, x.h, out.h))

    def mapoverlap_1d_i32(self, w, r: int, edge: int, pad: int, x: "Vector", out: "Vector"):
        w = np.ascontiguousarray(w, np.int32)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d_i32(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, x.h, out.h))

    def mapoverlap_1d_matrix_i32(self, w, r: int, edge: int, pad: int, axis: int, x: "Matrix", out: "Matrix"):
        w = np.ascontiguousarray(w, np.int32)
        assert w.size == 2 * r + 1
        self.check(lib.skel_mapoverlap_1d_matrix_i32(self.h, w.ctypes.data_as(C.c_void_p), r, edge, pad, axis, x.h, out.h))

    def mapoverlap_2d_i32(self, W, ry: int, rx: int, edge: int, pad: int, x: "Matrix", out: "Matrix"):
        W = np.ascontiguousarray(W, np.int32)
        assert W.size == (2 * ry + 1) * (2 * rx + 1)
        self.check(lib.skel_mapoverlap_2d_i32(self.h, W.ctypes.data_as(C.c_void_p), ry, rx, edge, pad, x.h, out.h))

    def mapoverlap_separable(self, w_row, r_row: int, w_col, r_col: int, edge: int, pad: float, x: "Matrix", out: "Matrix"):
        wr, wc = np.ascontiguousarray(w_row, np.float32), np.ascontiguousarray(w_col, np.float32)
        assert wr.size == 2 * r_row + 1 and wc.size == 2 * r_col + 1
        self.check(lib.skel_mapoverlap_separable(self.h, wr.ctypes.data_as(C.c_void_p), r_row, wc.ctypes.data_as(C.c_void_p),
                                                 r_col, edge, pad, x.h, out.h))

    def scan(self, op: int, mode: int, init: float, x: "Vector", out: "Vector"):
        self.check(lib.skel_scan(self.h, op, mode, init, x.h, out.h))

    # ---- selector
    def tune(self, inst: SkelInstance, log2_lo: int, log2_hi: int, cols: int = 0, reps: int = 5) -> np.ndarray:
        """-> timing table [log2 size, variant] in microseconds (NaN = not applicable)."""
        self.check(lib.skel_tune_instance(self.h, C.byref(inst), log2_lo, log2_hi, cols, reps))
        cnt = C.c_size_t()
        self.check(lib.skel_tune_table(self.h, None, 0, C.byref(cnt)))
        buf = (C.c_float * cnt.value)()
        self.check(lib.skel_tune_table(self.h, buf, cnt.value, C.byref(cnt)))
        nv = lib.skel_variant_count(inst.skeleton)
        return np.array(buf, np.float32).reshape(-1, nv)

    def plan_lookup(self, inst: SkelInstance, n: int) -> int:
        v = C.c_int()
        self.check(lib.skel_plan_lookup(self.h, C.byref(inst), n, C.byref(v)))
        return v.value

    def replay_begin(self):
        self.check(lib.skel_replay_begin(self.h))

    def replay_end(self) -> int:
        n = C.c_int()
        self.check(lib.skel_replay_end(self.h, C.byref(n)))
        return n.value

    def replay_run(self, raw: bool, reps: int):
        """-> (host enqueue microseconds, device microseconds) per pass over the recorded calls"""
        h, d = C.c_double(), C.c_double()
        self.check(lib.skel_replay_run(self.h, 1 if raw else 0, reps, C.byref(h), C.byref(d)))
        return h.value, d.value

    def plan_explain(self, inst: SkelInstance, n: int):
        """-> (variant, exact key tuned?, variant comes from the plan (not the preference list)?)"""
        v, ex, fp = C.c_int(), C.c_int(), C.c_int()
        self.check(lib.skel_plan_explain(self.h, C.byref(inst), n, C.byref(v), C.byref(ex), C.byref(fp)))
        return v.value, bool(ex.value), bool(fp.value)

    def plan_set(self, inst: SkelInstance, n_min: int, variant: int):
        self.check(lib.skel_plan_set(self.h, C.byref(inst), n_min, variant))

    def plan_save(self, path: str):
        self.check(lib.skel_plan_save(self.h, path.encode()))

    def plan_load(self, path: str):
        self.check(lib.skel_plan_load(self.h, path.encode()))

    def plan_clear(self):
        self.check(lib.skel_plan_clear(self.h))


class _Container:
    _acquire = _release = _destroy = _prefetch = None

    def __init__(self, ctx: Context, h, dtype: int, shape):
        self.ctx, self.h, self.dtype, self.shape = ctx, h, dtype, shape
        self._keep = None

    @property
    def size(self) -> int:
        return int(np.prod(self.shape))

    def host_view(self, mode: int) -> np.ndarray:
        """Acquire host access; returns a numpy view of the library's pinned buffer. Call release()."""
        p = C.c_void_p()
        self.ctx.check(self._acquire(self.h, mode, C.byref(p)))
        if self.size == 0:
            return np.empty(self.shape, _NP[self.dtype])
        buf = (C.c_byte * (self.size * np.dtype(_NP[self.dtype]).itemsize)).from_address(p.value)
        return np.frombuffer(buf, dtype=_NP[self.dtype]).reshape(self.shape)

    def release(self):
        self.ctx.check(self._release(self.h))

    def prefetch_host(self):
        """Start an asynchronous download on the context's copy stream (skel_*_prefetch_host)."""
        self.ctx.check(self._prefetch(self.h))

    def _range_view(self, fn, mode: int, a: int, b: int, count: int, shape) -> np.ndarray:
        p = C.c_void_p()
        self.ctx.check(fn(self.h, mode, a, b, C.byref(p)))
        buf = (C.c_byte * (count * np.dtype(_NP[self.dtype]).itemsize)).from_address(p.value)
        return np.frombuffer(buf, dtype=_NP[self.dtype]).reshape(shape)

    def read_range(self, offset: int, count: int) -> np.ndarray:
        """Copy of elements offset .. offset+count-1 (flattened index); downloads only that range if needed."""
        v = self.host_view_range(READ, offset, count)
        try:
            return v.copy()
        finally:
            self.release()

    def write_range(self, offset: int, arr: np.ndarray):
        """Overwrite elements from `offset` on; a valid device copy stays valid and gets just this range uploaded."""
        a = np.ascontiguousarray(arr, _NP[self.dtype]).reshape(-1)
        v = self.host_view_range(WRITE, offset, a.size)
        try:
            v[...] = a
        finally:
            self.release()

    def numpy(self) -> np.ndarray:
        """Copy of the contents (downloads if only the device copy is valid)."""
        v = self.host_view(READ)
        try:
            return v.copy()
        finally:
            self.release()

    def write(self, arr: np.ndarray):
        v = self.host_view(WRITE)
        try:
            v[...] = np.asarray(arr, _NP[self.dtype]).reshape(self.shape)
        finally:
            self.release()

    def destroy(self):
        if self.h:
            self.ctx.check(self._destroy(self.h))
            self.h = None
            self._keep = None


def ranges_add(ranges: list[tuple[int, int]], begin: int, end: int) -> list[tuple[int, int]]:
    """The library's range-list merge as a pure function (no GPU)."""
    cap = len(ranges) + 1
    buf = (C.c_uint64 * (2 * cap))(*[x for r in ranges for x in r])
    cnt = C.c_size_t(len(ranges))
    st = lib.skel_ranges_add(buf, C.byref(cnt), cap, begin, end)
    if st != OK:
        raise SkelError(st)
    return [(int(buf[2 * k]), int(buf[2 * k + 1])) for k in range(cnt.value)]


class Vector(_Container):
    _acquire = staticmethod(lib.skel_vector_host_acquire)
    _prefetch = staticmethod(lib.skel_vector_prefetch_host)
    _release = staticmethod(lib.skel_vector_host_release)
    _destroy = staticmethod(lib.skel_vector_destroy)

    def __init__(self, ctx, h, dtype, n):
        super().__init__(ctx, h, dtype, (n,))

    def state(self) -> int:
        s = C.c_int()
        self.ctx.check(lib.skel_vector_state(self.h, C.byref(s)))
        return s.value

    def host_view_range(self, mode: int, offset: int, count: int) -> np.ndarray:
        """Range-granular host access (skel_vector_host_acquire_range). Call release()."""
        return self._range_view(lib.skel_vector_host_acquire_range, mode, offset, count, count, (count,))

    def device_ptr(self):
        p, valid = C.c_void_p(), C.c_int()
        self.ctx.check(lib.skel_vector_device_ptr(self.h, C.byref(p), C.byref(valid)))
        return p.value, bool(valid.value)


class Matrix(_Container):
    _acquire = staticmethod(lib.skel_matrix_host_acquire)
    _prefetch = staticmethod(lib.skel_matrix_prefetch_host)
    _release = staticmethod(lib.skel_matrix_host_release)
    _destroy = staticmethod(lib.skel_matrix_destroy)

    def __init__(self, ctx, h, dtype, rows, cols):
        super().__init__(ctx, h, dtype, (rows, cols))

    def host_view_range(self, mode: int, offset: int, count: int) -> np.ndarray:
        """Whole rows only: offset and count must be multiples of cols."""
        cols = self.shape[1]
        assert offset % cols == 0 and count % cols == 0
        return self._range_view(lib.skel_matrix_host_acquire_rows, mode, offset // cols, count // cols, count,
                                (count // cols, cols))

    def as_vector(self) -> Vector:
        h = C.c_void_p()
        self.ctx.check(lib.skel_matrix_as_vector(self.h, C.byref(h)))
        return Vector(self.ctx, h, self.dtype, self.size)
