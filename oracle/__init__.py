"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes access to the plain-C oracle (``ttc_oracle.c``: Eq. 1 of PAPER.md:39 as one odometer
loop) and to the paper's OpenMP reference loop (``ttc_ref_omp.c``).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package.  It imports nothing from the product package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libttc_oracle.so")
_SOURCES = [os.path.join(_HERE, "ttc_oracle.c"), os.path.join(_HERE, "ttc_ref_omp.c")]
# -ffp-contract=off: one rounding per operation (reading A7); never -ffast-math.
# No -march=native: the oracle is "as it stands, never tuned".
_CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    newest = max(os.path.getmtime(s) for s in _SOURCES)
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < newest:
        tmp = _LIB_PATH + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *_CFLAGS, "-o", tmp, *_SOURCES])
        os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64p = ctypes.POINTER(ctypes.c_int64)
        i32p = ctypes.POINTER(ctypes.c_int)
        for name in ("ttc_oracle_transpose", "ttc_ref_omp_transpose"):
            fn = getattr(lib, name)
            fn.restype = ctypes.c_int
            fn.argtypes = [ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p,
                           ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.ttc_oracle_transpose_mixed.restype = ctypes.c_int
        lib.ttc_oracle_transpose_mixed.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p,
                                                   ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.ttc_oracle_transpose_strided.restype = ctypes.c_int
        lib.ttc_oracle_transpose_strided.argtypes = [ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p,
                                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.ttc_oracle_offsets.restype = ctypes.c_int
        lib.ttc_oracle_offsets.argtypes = [ctypes.c_int, i64p, i32p, i64p, i64p, i64p, i64p, i64p]
        lib.ttc_ref_omp_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


_NP = {0: np.float32, 1: np.float64, 2: np.complex64, 3: np.complex128}


def _i64(seq: Optional[Sequence[int]]):
    if seq is None:
        return None
    return (ctypes.c_int64 * len(seq))(*[int(x) for x in seq])


def _call(fn, dtype: int, sizes, perm, lda, ldb, alpha, A: np.ndarray, beta, B: np.ndarray) -> None:
    npdt = _NP[dtype]
    if A.dtype != npdt or B.dtype != npdt:
        raise TypeError("A/B dtype does not match dtype code %d" % dtype)
    if not (A.flags.c_contiguous and B.flags.c_contiguous and B.flags.writeable):
        raise ValueError("A and B must be flat contiguous buffers, B writeable")
    n = len(sizes)
    a = np.array([alpha], dtype=npdt)
    b = np.array([beta], dtype=npdt)
    rc = fn(dtype, n, _i64(sizes), (ctypes.c_int * n)(*[int(p) for p in perm]), _i64(lda), _i64(ldb),
            a.ctypes.data_as(ctypes.c_void_p), A.ctypes.data_as(ctypes.c_void_p),
            b.ctypes.data_as(ctypes.c_void_p), B.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError("oracle rejected its arguments (code %d)" % rc)


def transpose(dtype: int, sizes, perm, lda, ldb, alpha, A: np.ndarray, beta, B: np.ndarray) -> None:
    """In-place update of the flat buffer ``B`` by Eq. 1.  Single thread."""
    _call(_load().ttc_oracle_transpose, dtype, sizes, perm, lda, ldb, alpha, A, beta, B)


def transpose_mixed(dtype_a: int, dtype_b: int, sizes, perm, lda, ldb, alpha, A: np.ndarray, beta,
                    B: np.ndarray) -> None:
    """Mixed-precision Eq. 1 (reading M1): A of ``dtype_a`` is converted to B's
    ``dtype_b`` and the update is evaluated in B's precision.  ``alpha``/``beta`` are of ``dtype_b``."""
    if A.dtype != _NP[dtype_a] or B.dtype != _NP[dtype_b]:
        raise TypeError("A/B dtype does not match the dtype codes")
    if not (A.flags.c_contiguous and B.flags.c_contiguous and B.flags.writeable):
        raise ValueError("A and B must be flat contiguous buffers, B writeable")
    n = len(sizes)
    a = np.array([alpha], dtype=_NP[dtype_b])
    b = np.array([beta], dtype=_NP[dtype_b])
    rc = _load().ttc_oracle_transpose_mixed(
        dtype_a, dtype_b, n, _i64(sizes), (ctypes.c_int * n)(*[int(p) for p in perm]), _i64(lda), _i64(ldb),
        a.ctypes.data_as(ctypes.c_void_p), A.ctypes.data_as(ctypes.c_void_p),
        b.ctypes.data_as(ctypes.c_void_p), B.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError("oracle rejected its arguments (code %d)" % rc)


def transpose_strided(dtype: int, sizes, perm, stride_a, stride_b, alpha, A: np.ndarray, beta, B: np.ndarray) -> None:
    """Eq. 1 on tensors given by explicit element strides: ``stride_a[k]`` of A's index k, ``stride_b[k]`` of
    B's position k (optional extension).  The oracle of ``ttc_plan_strided``."""
    _call(_load().ttc_oracle_transpose_strided, dtype, sizes, perm, stride_a, stride_b, alpha, A, beta, B)


def transpose_batched(dtype: int, sizes, perm, lda, ldb, alpha, A_list, beta, B_list) -> None:
    """Eq. 1 for a list of independent tensor pairs that share sizes, permutation and leading dimensions
    (the packing of many GEMM blocks): BY DEFINITION the single-pair operation applied
    to each pair in turn.  The oracle of ``ttc_execute_batched``."""
    if len(A_list) != len(B_list):
        raise ValueError("A_list and B_list differ in length")
    for A, B in zip(A_list, B_list):
        transpose(dtype, sizes, perm, lda, ldb, alpha, A, beta, B)


def ref_omp_transpose(dtype: int, sizes, perm, lda, ldb, alpha, A: np.ndarray, beta, B: np.ndarray) -> None:
    """The paper's OpenMP reference loop nest, all host cores."""
    _call(_load().ttc_ref_omp_transpose, dtype, sizes, perm, lda, ldb, alpha, A, beta, B)


def ref_omp_threads() -> int:
    return int(_load().ttc_ref_omp_threads())


# ------------------------------------------------------------------ the timed CPU baseline
# BASELINE.md section 3 item 2 / SURVEY.md 8(d): the paper's reference loop nest built with
# ``-O3 -march=native -fopenmp`` (Table 2's compiler flags), all host cores.
# -march=native binds the object to the CPU it was compiled on, so it is compiled on the box that
# runs it, into a file named after that CPU's flags.  -ffp-contract=off keeps the separate
# roundings (reading A7), so the result can still be compared with the oracle bit for bit; it
# does not slow a bandwidth-bound loop.
_NATIVE_CFLAGS = ["-O3", "-march=native", "-fopenmp", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared"]
_native = None


def _cpu_tag() -> str:
    import hashlib
    try:
        with open("/proc/cpuinfo") as fh:
            flags = next((ln for ln in fh if ln.startswith("flags")), "")
    except OSError:
        flags = ""
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


def _load_native():
    global _native
    if _native is None:
        path = os.path.join(_HERE, "libttc_ref_omp_native.%s.so" % _cpu_tag())
        src = _SOURCES[1]
        if not os.path.exists(path) or os.path.getmtime(path) < os.path.getmtime(src):
            tmp = path + ".tmp.%d" % os.getpid()
            subprocess.check_call(["gcc", *_NATIVE_CFLAGS, "-o", tmp, src])
            os.replace(tmp, path)
        lib = ctypes.CDLL(path)
        i64p = ctypes.POINTER(ctypes.c_int64)
        i32p = ctypes.POINTER(ctypes.c_int)
        lib.ttc_ref_omp_transpose.restype = ctypes.c_int
        lib.ttc_ref_omp_transpose.argtypes = [ctypes.c_int, ctypes.c_int, i64p, i32p, i64p, i64p,
                                              ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.ttc_ref_omp_parallel_copy.restype = None
        lib.ttc_ref_omp_parallel_copy.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64]
        lib.ttc_ref_omp_threads.restype = ctypes.c_int
        _native = lib
    return _native


NATIVE_FLAGS = "gcc " + " ".join(_NATIVE_CFLAGS)


def ref_omp_native_transpose(dtype: int, sizes, perm, lda, ldb, alpha, A: np.ndarray, beta, B: np.ndarray) -> None:
    """The same loop nest as :func:`ref_omp_transpose`, built with ``NATIVE_FLAGS`` on this machine."""
    _call(_load_native().ttc_ref_omp_transpose, dtype, sizes, perm, lda, ldb, alpha, A, beta, B)


def ref_omp_native_threads() -> int:
    return int(_load_native().ttc_ref_omp_threads())


def first_touch_copy(src: np.ndarray) -> np.ndarray:
    """A copy of ``src`` whose pages are first touched by the OpenMP threads."""
    dst = np.empty_like(src)
    _load_native().ttc_ref_omp_parallel_copy(dst.ctypes.data_as(ctypes.c_void_p), src.ctypes.data_as(ctypes.c_void_p),
                                             int(src.nbytes))
    return dst


def first_touch_zeros(like: np.ndarray) -> np.ndarray:
    dst = np.empty_like(like)
    _load_native().ttc_ref_omp_parallel_copy(dst.ctypes.data_as(ctypes.c_void_p), None, int(like.nbytes))
    return dst


def offsets(sizes, perm, lda, ldb, index):
    """(offA, offB) in elements of the logical element with A multi-index ``index``."""
    n = len(sizes)
    oa = ctypes.c_int64()
    ob = ctypes.c_int64()
    rc = _load().ttc_oracle_offsets(n, _i64(sizes), (ctypes.c_int * n)(*[int(p) for p in perm]),
                                    _i64(lda), _i64(ldb), _i64(index), ctypes.byref(oa), ctypes.byref(ob))
    if rc != 0:
        raise ValueError("oracle rejected its arguments (code %d)" % rc)
    return int(oa.value), int(ob.value)
