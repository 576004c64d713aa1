"""Thin ctypes binding of ``libttc.so`` (include/ttc.h): the same calls with the same names.

Argument marshalling only -- every step of the path (validation, canonicalisation, candidate
generation, tuning, the kernels) runs inside the library.  PyTorch appears only as the owner of
device memory and streams: tensors are passed as ``data_ptr()`` and the current stream as its
raw ``cudaStream_t``.  There is no CPU fallback: without the library the import fails, without
a CUDA device ``ttc_execute`` returns ``TTC_ERR_CUDA``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

TTC_MAX_RANK = 16
TTC_F32, TTC_F64, TTC_C64, TTC_C128 = 0, 1, 2, 3
TTC_OK = 0
STATUS_NAMES = ["TTC_OK", "TTC_ERR_INVALID_ARG", "TTC_ERR_NOT_PERMUTATION", "TTC_ERR_BAD_LD",
                "TTC_ERR_UNSUPPORTED", "TTC_ERR_ALLOC", "TTC_ERR_CUDA", "TTC_ERR_MISALIGNED", "TTC_ERR_SCRATCH_LIMIT"]
TTC_ERR_SCRATCH_LIMIT = 8
TTC_STATIC_SCRATCH_BYTES = 8 << 20
KERNEL_NAMES = {0: "none", 1: "copy", 2: "tile", 3: "gather", 4: "wide", 5: "tma", 6: "tensormap", 7: "skew"}
NP_DTYPE = {TTC_F32: np.float32, TTC_F64: np.float64, TTC_C64: np.complex64, TTC_C128: np.complex128}

EXPORTS = ["ttc_plan", "ttc_plan_mixed", "ttc_plan_strided", "ttc_plan_dtype_a", "ttc_execute", "ttc_execute_batched", "ttc_execute_host", "ttc_execute_host_static", "ttc_destroy", "ttc_last_error",
           "ttc_status_string", "ttc_plan_info", "ttc_plan_num_candidates", "ttc_plan_candidate",
           "ttc_plan_candidate_features", "ttc_plan_specialize", "ttc_plan_select", "ttc_plan_tune", "ttc_canonicalize", "ttc_launch_count",
           "ttc_debug_fastdiv", "ttc_debug_specialize_compile", "ttc_version", "ttc_release_host_staging"]


class ttc_info(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("rank", ctypes.c_int), ("canon_rank", ctypes.c_int),
                ("canon_extent", ctypes.c_int64 * TTC_MAX_RANK),
                ("canon_stride_a", ctypes.c_int64 * TTC_MAX_RANK),
                ("canon_stride_b", ctypes.c_int64 * TTC_MAX_RANK),
                ("numel", ctypes.c_int64), ("span_a", ctypes.c_int64), ("span_b", ctypes.c_int64),
                ("tuned", ctypes.c_int), ("n_candidates", ctypes.c_int * 2),
                ("chosen", ctypes.c_int * 2), ("chosen_us", ctypes.c_float * 2),
                ("tune_errors", ctypes.c_int), ("plan_ms", ctypes.c_float), ("tune_ms", ctypes.c_float),
                ("specialized", ctypes.c_int * 2), ("spec_us", ctypes.c_float * 2), ("generic_us", ctypes.c_float * 2)]


class ttc_candidate_info(ctypes.Structure):
    _fields_ = [("kernel", ctypes.c_int), ("vec_a", ctypes.c_int), ("vec_b", ctypes.c_int),
                ("tile_u", ctypes.c_int), ("tile_w", ctypes.c_int), ("n_u", ctypes.c_int),
                ("n_w", ctypes.c_int), ("threads", ctypes.c_int), ("smem_bytes", ctypes.c_int),
                ("loop_order", ctypes.c_int), ("sched", ctypes.c_int), ("flags", ctypes.c_int), ("grid", ctypes.c_int), ("est_cost", ctypes.c_float),
                ("tuned_us", ctypes.c_float), ("n_tiles", ctypes.c_int64),
                ("tile_ext", ctypes.c_int * TTC_MAX_RANK)]


def _load() -> ctypes.CDLL:
    # always through build(): its mtime check makes this cheap and a stale library can never
    # survive a source edit.  Raises if nvcc is missing and the library is out of date: there is no other path.
    path = _build.build()
    lib = ctypes.CDLL(path)
    i64p = ctypes.POINTER(ctypes.c_int64)
    i32p = ctypes.POINTER(ctypes.c_int)
    vp = ctypes.c_void_p
    lib.ttc_plan.restype = vp
    lib.ttc_plan.argtypes = [ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p]
    lib.ttc_plan_mixed.restype = vp
    lib.ttc_plan_mixed.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p]
    lib.ttc_plan_strided.restype = vp
    lib.ttc_plan_strided.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p]
    lib.ttc_plan_dtype_a.restype = ctypes.c_int
    lib.ttc_plan_dtype_a.argtypes = [vp]
    lib.ttc_execute.restype = ctypes.c_int
    lib.ttc_execute.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.ttc_execute_batched.restype = ctypes.c_int
    lib.ttc_execute_batched.argtypes = [vp, vp, ctypes.POINTER(vp), vp, ctypes.POINTER(vp), ctypes.c_int, vp]
    lib.ttc_execute_host.restype = ctypes.c_int
    lib.ttc_execute_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.ttc_execute_host_static.restype = ctypes.c_int
    lib.ttc_execute_host_static.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.ttc_destroy.restype = ctypes.c_int
    lib.ttc_destroy.argtypes = [vp]
    lib.ttc_last_error.restype = ctypes.c_int
    lib.ttc_status_string.restype = ctypes.c_char_p
    lib.ttc_status_string.argtypes = [ctypes.c_int]
    lib.ttc_plan_info.restype = ctypes.c_int
    lib.ttc_plan_info.argtypes = [vp, ctypes.POINTER(ttc_info)]
    lib.ttc_plan_num_candidates.restype = ctypes.c_int
    lib.ttc_plan_num_candidates.argtypes = [vp, ctypes.c_int]
    lib.ttc_plan_candidate.restype = ctypes.c_int
    lib.ttc_plan_candidate.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ttc_candidate_info)]
    lib.ttc_plan_candidate_features.restype = ctypes.c_int
    lib.ttc_plan_candidate_features.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_float)]
    lib.ttc_plan_specialize.restype = ctypes.c_int
    lib.ttc_plan_specialize.argtypes = [vp]
    lib.ttc_plan_select.restype = ctypes.c_int
    lib.ttc_plan_select.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    lib.ttc_plan_tune.restype = ctypes.c_int
    lib.ttc_plan_tune.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    lib.ttc_canonicalize.restype = ctypes.c_int
    lib.ttc_canonicalize.argtypes = [ctypes.c_int, i64p, i32p, i64p, i64p, i64p, i64p, i64p]
    lib.ttc_launch_count.restype = ctypes.c_int64
    lib.ttc_debug_fastdiv.restype = ctypes.c_uint32
    lib.ttc_debug_fastdiv.argtypes = [ctypes.c_uint32, ctypes.c_uint32]
    lib.ttc_version.restype = ctypes.c_char_p
    lib.ttc_debug_specialize_compile.restype = ctypes.c_int64
    lib.ttc_debug_specialize_compile.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_char_p, ctypes.c_int]
    lib.ttc_release_host_staging.restype = ctypes.c_int
    return lib


lib = _load()


class TTCError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__("%s: %s" % (where, name))


def _i64(seq: Optional[Sequence[int]]):
    if seq is None:
        return None
    return (ctypes.c_int64 * len(seq))(*[int(x) for x in seq])


def _i32(seq: Sequence[int]):
    return (ctypes.c_int * len(seq))(*[int(x) for x in seq])


def _ptr(x) -> int:
    """Address of a torch tensor, a numpy array or a raw integer address."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError("expected a tensor, an ndarray or an address, got %r" % type(x))


def _stream(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream) if torch.cuda.is_available() else 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


# ------------------------------------------------------------------------- the C calls, by name
def ttc_plan(dtype: int, N: int, sizes, perm, lda=None, ldb=None) -> int:
    h = lib.ttc_plan(int(dtype), int(N), _i64(sizes), _i32(perm) if perm is not None else None,
                     _i64(lda), _i64(ldb))
    if not h:
        raise TTCError(lib.ttc_last_error(), "ttc_plan")
    return h


def ttc_plan_mixed(dtype_a: int, dtype_b: int, N: int, sizes, perm, lda=None, ldb=None) -> int:
    """Mixed-precision plan: A of ``dtype_a``, B (and alpha, beta) of ``dtype_b``."""
    h = lib.ttc_plan_mixed(int(dtype_a), int(dtype_b), int(N), _i64(sizes), _i32(perm) if perm is not None else None,
                           _i64(lda), _i64(ldb))
    if not h:
        raise TTCError(lib.ttc_last_error(), "ttc_plan_mixed")
    return h


def ttc_plan_strided(dtype_a: int, dtype_b: int, N: int, sizes, perm, stride_a, stride_b) -> int:
    """Plan from explicit element strides (stride_a per A-index, stride_b per B-position)."""
    h = lib.ttc_plan_strided(int(dtype_a), int(dtype_b), int(N), _i64(sizes), _i32(perm) if perm is not None else None,
                             _i64(stride_a), _i64(stride_b))
    if not h:
        raise TTCError(lib.ttc_last_error(), "ttc_plan_strided")
    return h


def ttc_plan_dtype_a(plan: int) -> int:
    return int(lib.ttc_plan_dtype_a(plan))


_plan_dtype = {}     # plan handle -> numpy dtype of its scalars (marshalling cache)


def _scalar_dtype(plan: int):
    dt = _plan_dtype.get(plan)
    if dt is None:
        dt = _plan_dtype[plan] = NP_DTYPE[ttc_plan_info(plan).dtype]
    return dt


def ttc_execute(plan: int, alpha, A, beta, B, stream=None) -> None:
    npdt = _scalar_dtype(plan)
    a = np.array([alpha], dtype=npdt)
    b = np.array([beta], dtype=npdt)
    rc = lib.ttc_execute(plan, a.ctypes.data, _ptr(A), b.ctypes.data, _ptr(B), _stream(stream))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_execute")


def ttc_execute_batched(plan: int, alpha, A_list, beta, B_list, stream=None) -> None:
    """One launch (per 64 pairs) for a list of tensor pairs that share ``plan``."""
    npdt = _scalar_dtype(plan)
    a = np.array([alpha], dtype=npdt)
    b = np.array([beta], dtype=npdt)
    n = len(A_list)
    if len(B_list) != n:
        raise ValueError("A_list and B_list differ in length")
    pa = (ctypes.c_void_p * max(n, 1))(*[_ptr(x) for x in A_list])
    pb = (ctypes.c_void_p * max(n, 1))(*[_ptr(x) for x in B_list])
    rc = lib.ttc_execute_batched(plan, a.ctypes.data, pa, b.ctypes.data, pb, n, _stream(stream))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_execute_batched")


def ttc_execute_host(plan: int, alpha, A_host, beta, B_host, stream=None) -> None:
    npdt = _scalar_dtype(plan)
    a = np.array([alpha], dtype=npdt)
    b = np.array([beta], dtype=npdt)
    rc = lib.ttc_execute_host(plan, a.ctypes.data, _ptr(A_host), b.ctypes.data, _ptr(B_host), _stream(stream))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_execute_host")


def ttc_execute_host_static(plan: int, alpha, A_host, beta, B_host, stream=None) -> None:
    """ttc_execute_host staged through the library's file-scope device array: no device allocation; tensors
    beyond TTC_STATIC_SCRATCH_BYTES raise TTCError(TTC_ERR_SCRATCH_LIMIT)."""
    npdt = _scalar_dtype(plan)
    a = np.array([alpha], dtype=npdt)
    b = np.array([beta], dtype=npdt)
    rc = lib.ttc_execute_host_static(plan, a.ctypes.data, _ptr(A_host), b.ctypes.data, _ptr(B_host), _stream(stream))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_execute_host_static")


def ttc_destroy(plan: int) -> None:
    _plan_dtype.pop(plan, None)
    lib.ttc_destroy(plan)


def ttc_plan_info(plan: int) -> ttc_info:
    out = ttc_info()
    rc = lib.ttc_plan_info(plan, ctypes.byref(out))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_plan_info")
    return out


def ttc_plan_num_candidates(plan: int, which: int) -> int:
    return int(lib.ttc_plan_num_candidates(plan, which))


def ttc_plan_candidate(plan: int, which: int, index: int) -> ttc_candidate_info:
    out = ttc_candidate_info()
    rc = lib.ttc_plan_candidate(plan, which, index, ctypes.byref(out))
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_plan_candidate")
    return out


def ttc_plan_candidate_features(plan: int, which: int, index: int):
    out = (ctypes.c_float * 16)()
    rc = lib.ttc_plan_candidate_features(plan, which, index, out)
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_plan_candidate_features")
    return [float(x) for x in out]


def ttc_plan_specialize(plan: int) -> int:
    """NVRTC size-specialised twins of the plan's winners; returns the status (TTC_ERR_UNSUPPORTED = 4 when
    libnvrtc is missing or no winner is specialisable: the plan keeps its generic kernels)."""
    return int(lib.ttc_plan_specialize(plan))


def ttc_plan_select(plan: int, which: int, index: int) -> None:
    rc = lib.ttc_plan_select(plan, which, index)
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_plan_select")


def ttc_plan_tune(plan: int, top_k: int = 0, reps: int = 3) -> None:
    rc = lib.ttc_plan_tune(plan, top_k, reps)
    if rc != TTC_OK:
        raise TTCError(rc, "ttc_plan_tune")


def ttc_canonicalize(sizes, perm, lda=None, ldb=None):
    """Stage 1 alone: list of (extent, stride in A, stride in B), ascending stride in A."""
    n = len(sizes)
    e = (ctypes.c_int64 * TTC_MAX_RANK)()
    sa = (ctypes.c_int64 * TTC_MAX_RANK)()
    sb = (ctypes.c_int64 * TTC_MAX_RANK)()
    r = lib.ttc_canonicalize(n, _i64(sizes), _i32(perm), _i64(lda), _i64(ldb), e, sa, sb)
    if r < 0:
        raise TTCError(lib.ttc_last_error(), "ttc_canonicalize")
    return [(int(e[i]), int(sa[i]), int(sb[i])) for i in range(r)]


def ttc_launch_count() -> int:
    return int(lib.ttc_launch_count())


def ttc_debug_specialize_compile(plan: int, which: int, index: int):
    """(cubin bytes or negative code, compiler log) of the NVRTC-specialised source of one candidate (host only)."""
    buf = ctypes.create_string_buffer(8192)
    n = int(lib.ttc_debug_specialize_compile(plan, which, index, buf, len(buf)))
    return n, buf.value.decode(errors="replace")


def ttc_version() -> str:
    return lib.ttc_version().decode()


def ttc_release_host_staging() -> None:
    lib.ttc_release_host_staging()


def describe_candidate(c: ttc_candidate_info, rank: int) -> str:
    ext = "x".join(str(c.tile_ext[i]) for i in range(rank))
    return "%s%s tile=%s vec=%d/%d run=%d/%d loop=%s sched=%s smem=%d grid=%d cost=%.2f us=%.1f" % (
        KERNEL_NAMES.get(c.kernel, "?"), ("+stag" if c.flags & 1 else "") + ("+shift" if c.flags & 4 else ""), ext, c.vec_a, c.vec_b, c.tile_u, c.tile_w,
        "ABab"[c.loop_order], ("static", "dynamic", "atomic")[c.sched], c.smem_bytes, c.grid, c.est_cost, c.tuned_us)
