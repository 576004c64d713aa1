"""Pins for the mixed-precision oracle (``ttc_oracle_transpose_mixed``).

The paper fixes only that A and B may have different data types (``--dataType=sd``: A single,
B double).  Reading M1 (oracle header): A's element is converted to B's type, then
Eq. 1 runs in B's precision.  The pins below check that reading against what mathematics and a
library routine fix, never against the oracle itself or the CUDA path:

  MP1  index-encoding closed form (as P1): integers are exact in both precisions;
  MP2  IEEE-754 convertFormat values known in closed form (ties-to-even, overflow, subnormals);
  MP3  special case that reduces to the pinned homogeneous oracle: convert A with numpy's
       ``astype`` (library routine) first, then the same-type Eq. 1 must give the same bits;
  MP4  exact small-integer axpby with Python's own complex arithmetic (signs/operands of A9);
  MP5  the precision of the arithmetic: a value where "evaluate in double, round once" and
       "convert, then evaluate in float" differ, expected value derived by hand;
  MP6  padding untouched / never read, beta = 0 never reads B; rejected type pairs.
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_1607_01249_b200 import workloads as wl

NP = wl.NP_DTYPE
PAIRS = ((wl.F32, wl.F64), (wl.F64, wl.F32), (wl.C64, wl.C128), (wl.C128, wl.C64))   # sd, ds, cz, zc


def sizes_b(sizes, perm):
    return tuple(sizes[p] for p in perm)


def run(da, db, sizes, perm, lda, ldb, alpha, beta, a_vals, b_vals=None, b_fill=np.nan):
    A = wl.embed(a_vals.astype(NP[da]), sizes, lda)
    szb = sizes_b(sizes, perm)
    if b_vals is None:
        b_vals = np.full(int(np.prod(sizes, dtype=np.int64)), b_fill, dtype=NP[db])
    B = wl.embed(b_vals.astype(NP[db]), szb, ldb)
    oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, alpha, A, beta, B)
    return B, wl.extract(B, szb, ldb)


@pytest.mark.parametrize("da,db", PAIRS[:2])
@pytest.mark.parametrize("sizes,perm", [((5, 3, 4), (2, 0, 1)), ((4, 3, 2, 5), (3, 1, 0, 2)),
                                        ((2, 3, 4, 3, 2), (4, 2, 0, 3, 1))])
@pytest.mark.parametrize("padded", [False, True])
def test_mp1_index_encoding(da, db, sizes, perm, padded):
    """alpha=1, beta=0: A holds L(i) (exact in fp32 and fp64); B decoded from
    its own offsets must hold L of the A-index Pi places there; padding stays NaN."""
    rng = np.random.default_rng(2)
    n = len(sizes)
    szb = sizes_b(sizes, perm)
    lda = tuple(int(e + rng.integers(0, 4)) for e in sizes) if padded else None
    ldb = tuple(int(e + rng.integers(0, 4)) for e in szb) if padded else None
    numel = int(np.prod(sizes))
    B, _ = run(da, db, sizes, perm, lda, ldb, 1.0, 0.0, np.arange(numel, dtype=np.float64), b_fill=-1.0)
    assert B.dtype == NP[db]
    ext_b = wl.padded_extents(szb, ldb)
    j = np.unravel_index(np.arange(B.size), ext_b, order="F")
    logical = np.ones(B.size, dtype=bool)
    L = np.zeros(B.size, dtype=np.int64)
    for k in range(n):
        logical &= j[k] < szb[k]
        L += j[k].astype(np.int64) * int(np.prod(sizes[:perm[k]], dtype=np.int64))
    assert np.array_equal(B[logical], L[logical].astype(NP[db]))
    assert np.isnan(B[~logical]).all()


def test_mp2_narrowing_is_round_to_nearest_even():
    """d -> s is ONE IEEE-754 round-to-nearest-even (reading M1).  Hand-derived cases around
    1.0 (fp32 spacing 2^-23): a tie goes to the even neighbour, anything above the tie goes up;
    values beyond FLT_MAX's rounding boundary overflow to inf; 2^-150 is a tie between 0 and the
    smallest subnormal 2^-149 and goes to 0 (even); 1.5*2^-149 is a tie that goes to 2^-148."""
    cases = [
        (1.0 + 2.0 ** -24, 1.0),                               # tie, 1.0 has even mantissa
        (1.0 + 2.0 ** -24 + 2.0 ** -50, 1.0 + 2.0 ** -23),     # just above the tie
        (1.0 + 3 * 2.0 ** -24, 1.0 + 2.0 ** -22),              # tie between odd and even: to even
        (1.0 - 2.0 ** -25, 1.0),                               # tie below 1 (spacing 2^-24): to even
        (-(1.0 + 2.0 ** -24 + 2.0 ** -50), -(1.0 + 2.0 ** -23)),
        (3.5e38, np.inf), (-3.5e38, -np.inf),
        (2.0 ** -150, 0.0), (2.0 ** -150 + 2.0 ** -200, 2.0 ** -149), (1.5 * 2.0 ** -149, 2.0 ** -148),
        (0.1, float.fromhex("0x1.99999ap-4")),                 # the textbook fp32 value of 0.1
    ]
    a = np.array([c[0] for c in cases], dtype=np.float64)
    want = np.array([c[1] for c in cases], dtype=np.float32)
    _, got = run(wl.F64, wl.F32, (len(cases),), (0,), None, None, 1.0, 0.0, a)
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
    # complex narrows component-wise (finite cases only: the textbook product has 0 * inf = NaN)
    z = (a[:4] + 1j * a[1:5]).astype(np.complex128)
    _, gz = run(wl.C128, wl.C64, (4,), (0,), None, None, 1.0, 0.0, z)
    assert np.array_equal(gz.real.view(np.uint32), want[:4].view(np.uint32))
    assert np.array_equal(gz.imag.view(np.uint32), want[1:5].view(np.uint32))


def test_mp2_widening_is_exact():
    """s -> d is exact for every finite fp32 (24-bit significands fit in 53 bits): the double holds
    the same rational number, checked through Python's exact ``float.hex`` of both."""
    bits = np.array([0x00000001, 0x007FFFFF, 0x00800000, 0x3F800001, 0x7F7FFFFF, 0x80000001, 0xBF99999A, 0x33D6BF95],
                    dtype=np.uint32)
    a = bits.view(np.float32)
    _, got = run(wl.F32, wl.F64, (bits.size,), (0,), None, None, 1.0, 0.0, a)
    assert got.dtype == np.float64
    for x, y in zip(a, got):
        assert float(x).hex() == float(y).hex()   # float(np.float32) is exact by IEEE widening in C as well
        assert np.float32(y) == x


@pytest.mark.parametrize("da,db", PAIRS)
@pytest.mark.parametrize("beta_nz", [False, True])
def test_mp3_reduces_to_same_type_oracle_after_library_conversion(da, db, beta_nz):
    """M1 stated with a library routine: mixed(A) == same-type Eq. 1 applied to ``A.astype(B's type)``
    (numpy's cast is IEEE convertFormat), bit for bit, for general alpha/beta and padded tensors.
    The same-type oracle is pinned by tests/test_oracle_pins.py."""
    sizes, perm = (6, 5, 4, 3), (2, 0, 3, 1)
    lda, ldb = (8, 5, 6, 3), (4, 9, 3, 6)
    szb = sizes_b(sizes, perm)
    n = int(np.prod(sizes))
    a = wl.uniform_values(wl.SEED_A, n, da)
    if da in (wl.F64, wl.C128):       # make the narrowing inexact for almost every element
        a = a * NP[da](1.0 + 2.0 ** -30)
    b0 = wl.uniform_values(wl.SEED_B, n, db)
    cplx = db >= 2
    alpha = (0.75 - 1.25j) if cplx else 1.7
    beta = ((0.3 + 0.6j) if cplx else -0.45) if beta_nz else 0.0
    A = wl.embed(a, sizes, lda)
    B1 = wl.embed(b0, szb, ldb)
    B2 = B1.copy()
    oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, alpha, A, beta, B1)
    oracle.transpose(db, sizes, perm, lda, ldb, alpha, np.ascontiguousarray(A.astype(NP[db])), beta, B2)
    assert np.array_equal(B1.view(np.uint8), B2.view(np.uint8))


@pytest.mark.parametrize("da,db", PAIRS)
def test_mp4_exact_small_integer_axpby(da, db):
    """Small integers: conversion, products and sums are exact in every precision, so Python's
    complex arithmetic gives the expected B (pins operands and signs of the complex product)."""
    sizes, perm = (4, 3, 5), (1, 2, 0)
    n = int(np.prod(sizes))
    rng = np.random.default_rng(5)
    cplx = db >= 2
    mk = lambda: rng.integers(-8, 9, size=n) + (1j * rng.integers(-8, 9, size=n) if cplx else 0)
    a, b = mk(), mk()
    alpha, beta = ((2 - 3j, -1 + 2j) if cplx else (3.0, -2.0))
    _, got = run(da, db, sizes, perm, None, None, alpha, beta, np.asarray(a), np.asarray(b))
    # expected: logical element L of A lands at the position Pi gives it; compute per element
    La = np.arange(n).reshape(sizes, order="F")
    want = np.empty(n, dtype=np.complex128)
    szb = sizes_b(sizes, perm)
    for idx in itertools.product(*[range(s) for s in sizes]):
        jb = tuple(idx[p] for p in perm)
        lb = int(np.ravel_multi_index(jb, szb, order="F"))
        want[lb] = alpha * complex(a[La[idx]]) + beta * complex(b[lb])
    want = want if cplx else want.real
    assert np.array_equal(got, want.astype(NP[db]))


def test_mp5_arithmetic_runs_in_b_precision():
    """ds, alpha = 3, a = 1 + 2^-24 + 2^-50 (hand-derived).  M1: float(a) = 1 + 2^-23 (above the tie), then
    3 * (1 + 2^-23) = 3 + 3*2^-23 is a tie in fp32 spacing 2^-22 at [2,4) -> even: 3 + 2^-21.
    "Evaluate in double, round once" would give round(3 + 3*2^-24 + ...) = 3 + 2^-22.  The two differ,
    so this value tells the readings apart."""
    a = np.array([1.0 + 2.0 ** -24 + 2.0 ** -50], dtype=np.float64)
    _, got = run(wl.F64, wl.F32, (1,), (0,), None, None, 3.0, 0.0, a)
    assert got[0] == np.float32(3.0 + 2.0 ** -21)
    assert got[0] != np.float32(3.0 + 2.0 ** -22)
    # sd: the product is rounded in double, not in float: 0.1f * 3 in double keeps bits a float product loses
    a32 = np.array([0.1], dtype=np.float32)
    _, g2 = run(wl.F32, wl.F64, (1,), (0,), None, None, 3.0, 0.0, a32)
    assert g2[0] == 3.0 * float(a32[0]) and g2[0] != float(np.float32(3.0) * a32[0])


@pytest.mark.parametrize("da,db", PAIRS)
def test_mp6_padding_and_beta_zero(da, db):
    """A's padding (NaN) never reaches B, B's padding keeps its bit pattern, and beta = 0 never
    reads B (NaN-filled B comes out finite): north_star, reading A5."""
    sizes, perm = (5, 4, 3), (2, 0, 1)
    lda, ldb = (7, 4, 5), (3, 8, 4)
    szb = sizes_b(sizes, perm)
    n = int(np.prod(sizes))
    a = wl.uniform_values(wl.SEED_A, n, da)
    A = wl.embed(a, sizes, lda)
    nb = int(np.prod(wl.padded_extents(szb, ldb)))
    B = np.frombuffer(np.full(nb * np.dtype(NP[db]).itemsize, 0xFF, dtype=np.uint8).tobytes(), dtype=NP[db]).copy()
    before = B.copy()
    oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, 1.0, A, 0.0, B)
    got = wl.extract(B, szb, ldb)
    assert np.isfinite(got.view(np.float32 if db in (wl.F32, wl.C64) else np.float64)).all()
    mask = wl.embed(np.zeros(n, dtype=NP[db]), szb, ldb, fill=1.0).real.astype(bool)
    assert np.array_equal(B.view(np.uint8).reshape(nb, -1)[mask], before.view(np.uint8).reshape(nb, -1)[mask])
    # the permuted values themselves: position check through numpy's transpose (library routine, P9)
    want = a.astype(NP[db]).reshape(sizes, order="F").transpose(perm).reshape(-1, order="F")
    assert np.array_equal(got, want)


@pytest.mark.parametrize("da,db", [(wl.F32, wl.C64), (wl.C64, wl.F32), (wl.F64, wl.C128), (wl.F32, wl.C128),
                                   (wl.C64, wl.F64)])
def test_mp6_real_complex_pairs_are_rejected(da, db):
    """PAPER.md:75 lists s, d, c, z and the mixed pairs sd, ds, cz, zc only."""
    A = np.zeros(4, dtype=NP[da])
    B = np.zeros(4, dtype=NP[db])
    with pytest.raises(ValueError):
        oracle.transpose_mixed(da, db, (4,), (0,), None, None, 1.0, A, 0.0, B)
