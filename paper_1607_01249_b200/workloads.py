"""Seeded synthetic inputs and the BASELINE.json workload table.

This module is shared by the tests, ``bench.py`` and ``__graft_entry__.smoke()``.
It holds NONE of the method's arithmetic (no alpha/beta maths, no permutation,
no offset formula): it only draws counter-based pseudo-random values and lets
numpy place them inside a (possibly ld-padded) Fortran-order buffer.  Neither
the oracle nor the CUDA path is imported here.

Value recipe:
``r(c) = mix(seed * 0x9E3779B97F4A7C15 + c)`` in uint64 wrap-around arithmetic
with ``mix`` the public-domain SplitMix64 finaliser; fp32 takes the top 24 bits
``k`` and maps them to ``k / 2**23 - 1`` in [-1, 1) (exact in fp32), fp64 takes
the top 53 bits and maps them to ``k / 2**52 - 1`` (exact in fp64); the complex
element with logical linear index L uses counters 2L (re) and 2L+1 (im).  The
counter of a real element is its logical linear index L (column-major over the
*logical* sizes), so values do not depend on the padding.  All padding is a
quiet NaN, which the method must never read into B (Fig. 2).

The paper's own 57-case benchmark is only referenced by URL; the
five BASELINE.json configs below stand in for it (2-D..6-D after merging,
~200 MB, column-major, arbitrary permutation, ld-padded packing as in Fig. 3).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np

SEED_A = 160701249
SEED_B = 160701250

# dtype codes of include/ttc.h (s, d, c, z of PAPER.md:75)
F32, F64, C64, C128 = 0, 1, 2, 3
NP_DTYPE = {F32: np.float32, F64: np.float64, C64: np.complex64, C128: np.complex128}
DTYPE_NAME = {F32: "f32", F64: "f64", C64: "c64", C128: "c128"}
ELEM_SIZE = {F32: 4, F64: 8, C64: 8, C128: 16}

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, counters: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser applied to ``seed * GOLDEN + counter`` (uint64 wrap)."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) * _GOLDEN + counters.astype(np.uint64)
        z ^= z >> np.uint64(30)
        z *= _M1
        z ^= z >> np.uint64(27)
        z *= _M2
        z ^= z >> np.uint64(31)
    return z


def _uniform_real(seed: int, counters: np.ndarray, real_dtype) -> np.ndarray:
    r = splitmix64(seed, counters)
    if real_dtype == np.float32:
        k = (r >> np.uint64(40)).astype(np.int64)          # top 24 bits
        return (k.astype(np.float64) / 2.0**23 - 1.0).astype(np.float32)
    k = (r >> np.uint64(11)).astype(np.int64)              # top 53 bits
    # k / 2**52 - 1 is exact in fp64: k < 2**53 and the result is a multiple of 2**-52 in [-1, 1)
    return (k - (1 << 52)).astype(np.float64) / 2.0**52


def uniform_values(seed: int, n: int, dtype_code: int, chunk: int = 1 << 24) -> np.ndarray:
    """``n`` logical elements, element L drawn from counter L (2L, 2L+1 for complex)."""
    npdt = NP_DTYPE[dtype_code]
    out = np.empty(n, dtype=npdt)
    real = np.float32 if dtype_code in (F32, C64) else np.float64
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        c = np.arange(lo, hi, dtype=np.uint64)
        if dtype_code in (C64, C128):
            re = _uniform_real(seed, c * np.uint64(2), real)
            im = _uniform_real(seed, c * np.uint64(2) + np.uint64(1), real)
            out[lo:hi] = re + 1j * im
        else:
            out[lo:hi] = _uniform_real(seed, c, real)
    return out


def padded_extents(sizes: Sequence[int], ld: Optional[Sequence[int]]) -> Tuple[int, ...]:
    """Extents of the enclosing buffer: ld for every index but the last, whose
    leading dimension does not affect addressing (the buffer ends with the tensor)."""
    if ld is None:
        return tuple(int(s) for s in sizes)
    n = len(sizes)
    return tuple(int(ld[k]) if k < n - 1 else int(sizes[k]) for k in range(n))


def embed(values: np.ndarray, sizes: Sequence[int], ld: Optional[Sequence[int]],
          fill=np.nan) -> np.ndarray:
    """Place ``values`` (logical column-major order) in a flat buffer whose enclosing
    Fortran-order extents are ``ld``; everything else is ``fill``.  numpy does the
    addressing (Fortran-order slicing)."""
    ext = padded_extents(sizes, ld)
    if any(s == 0 for s in sizes):
        return np.full(int(np.prod(ext, dtype=np.int64)), fill, dtype=values.dtype)
    buf = np.full(ext, fill, dtype=values.dtype, order="F")
    buf[tuple(slice(0, int(s)) for s in sizes)] = values.reshape(tuple(int(s) for s in sizes), order="F")
    return buf.reshape(-1, order="F")


def extract(buf: np.ndarray, sizes: Sequence[int], ld: Optional[Sequence[int]]) -> np.ndarray:
    """Inverse of :func:`embed`: logical elements of a padded flat buffer, column-major."""
    ext = padded_extents(sizes, ld)
    nd = buf.reshape(ext, order="F")
    return np.ascontiguousarray(nd[tuple(slice(0, int(s)) for s in sizes)].reshape(-1, order="F"))


@dataclass(frozen=True)
class Workload:
    """One transposition problem in the paper's notation (Table 1)."""
    name: str
    dtype: int
    sizes: Tuple[int, ...]            # extents of A's indices i_0..i_{N-1}
    perm: Tuple[int, ...]             # perm[k] = A-index at position k of B
    alpha: complex = 1.0
    beta: complex = 0.0
    lda: Optional[Tuple[int, ...]] = None
    ldb: Optional[Tuple[int, ...]] = None
    note: str = ""

    @property
    def n(self) -> int:
        return len(self.sizes)

    @property
    def sizes_b(self) -> Tuple[int, ...]:
        return tuple(self.sizes[p] for p in self.perm)

    @property
    def numel(self) -> int:
        out = 1
        for s in self.sizes:
            out *= int(s)
        return out

    @property
    def elem_size(self) -> int:
        return ELEM_SIZE[self.dtype]

    @property
    def beta_nonzero(self) -> bool:
        return complex(self.beta) != 0

    @property
    def algorithmic_bytes(self) -> int:
        """Eq. 2 of the paper generalised: (2 | 3) * |A| * sizeof."""
        return (3 if self.beta_nonzero else 2) * self.numel * self.elem_size

    def scalar(self, x) -> np.ndarray:
        """alpha / beta as one host scalar of the tensor's dtype (complex = 2 reals)."""
        return np.array([x], dtype=NP_DTYPE[self.dtype])

    def make_a(self, seed: int = SEED_A) -> np.ndarray:
        return embed(uniform_values(seed, self.numel, self.dtype), self.sizes, self.lda)

    def make_b(self, seed: int = SEED_B, init: str = "auto") -> np.ndarray:
        """Initial B.  ``auto``: uniform from ``seed`` if beta != 0 else zeros;
        ``nan``: logical elements NaN (proves beta = 0 never reads B).  Padding is NaN."""
        szb = self.sizes_b
        if init == "auto":
            init = "uniform" if self.beta_nonzero else "zeros"
        if init == "uniform":
            vals = uniform_values(seed, self.numel, self.dtype)
        elif init == "zeros":
            vals = np.zeros(self.numel, dtype=NP_DTYPE[self.dtype])
        elif init == "nan":
            vals = np.full(self.numel, np.nan, dtype=NP_DTYPE[self.dtype])
        else:
            raise ValueError(init)
        return embed(vals, szb, self.ldb)


def config1() -> Workload:
    return Workload("c1_f32_3d", F32, (160, 144, 128), (2, 0, 1), 1.0, 0.0,
                    note="BASELINE.json configs[0]")


def config2_perms() -> Tuple[Tuple[int, ...], ...]:
    return tuple(p for p in itertools.permutations(range(4)) if p != (0, 1, 2, 3))


def config2(perm: Sequence[int]) -> Workload:
    perm = tuple(int(p) for p in perm)
    return Workload("c2_f64_4d_" + "".join(map(str, perm)), F64, (96, 72, 64, 56), perm, 1.0, 0.0,
                    note="BASELINE.json configs[1]")


def config2_all() -> Tuple[Workload, ...]:
    return tuple(config2(p) for p in config2_perms())


def config3() -> Workload:
    return Workload("c3_f32_6d", F32, (24, 20, 16, 24, 20, 16), (5, 2, 0, 4, 1, 3), 1.5, 0.5,
                    note="BASELINE.json configs[2]")


def config4() -> Workload:
    # 6144 x 4096 matrix in a buffer with lda = 6208, viewed as (mr=8, 768, 4096):
    # lda = (8, 776, .) gives element strides (1, 8, 6208)  (Fig. 3)
    return Workload("c4_f64_pack", F64, (8, 768, 4096), (0, 2, 1), 1.0, 0.0, lda=(8, 776, 4096),
                    note="BASELINE.json configs[3]")


def config5() -> Workload:
    return Workload("c5_c64_5d", C64, (7, 96, 5, 80, 64), (4, 2, 0, 3, 1), 0.5 - 0.25j, 0.0,
                    note="BASELINE.json configs[4]")


def baseline_configs() -> Tuple[Workload, ...]:
    return (config1(),) + config2_all() + (config3(), config4(), config5())
