"""``-m gpu`` parity tests of the mixed-precision path (ttc_plan_mixed) against the
mixed-precision oracle (reading M1: convert A to B's type, evaluate Eq. 1 in B's precision).

The kernels convert with cvt.rn (the C cast of the oracle) and round every product and sum
separately, so the bar is bit-exact in every case, beta != 0 included.
"""
import itertools

import numpy as np
import pytest
import torch

import oracle
from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import GUARD, bits, to_dev

pytestmark = pytest.mark.gpu

NP = wl.NP_DTYPE
PAIRS = ((wl.F32, wl.F64), (wl.F64, wl.F32), (wl.C64, wl.C128), (wl.C128, wl.C64))   # sd, ds, cz, zc


def scalars(db, beta_nz):
    if db >= 2:
        return (0.75 - 1.25j, (0.5 + 0.375j) if beta_nz else 0.0)
    return (1.7, -0.45 if beta_nz else 0.0)


def make_inputs(da, db, sizes, perm, lda, ldb, beta_nz, b_init="auto"):
    n = int(np.prod(sizes, dtype=np.int64))
    szb = tuple(sizes[p] for p in perm)
    A = wl.embed(wl.uniform_values(wl.SEED_A, n, da), sizes, lda)
    if b_init == "auto":
        b_init = "uniform" if beta_nz else "zeros"
    vals = {"uniform": lambda: wl.uniform_values(wl.SEED_B, n, db),
            "zeros": lambda: np.zeros(n, dtype=NP[db]),
            "nan": lambda: np.full(n, np.nan, dtype=NP[db])}[b_init]()
    return A, wl.embed(vals, szb, ldb)


def check(da, db, sizes, perm, lda=None, ldb=None, beta_nz=False, plan=None, candidate=None, b_init="auto",
          misalign_a=0, misalign_b=0):
    alpha, beta = scalars(db, beta_nz)
    A, B0 = make_inputs(da, db, sizes, perm, lda, ldb, beta_nz, b_init)
    want = B0.copy()
    oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, alpha, A, beta, want)
    own = plan is None
    if own:
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    which = 1 if beta_nz else 0
    try:
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, candidate)
        ga, gb = np.array(-77.25, dtype=A.dtype), np.array(-77.25, dtype=B0.dtype)
        a_whole, a_dev = to_dev(A, ga, misalign_a)
        b_whole, b_dev = to_dev(B0, gb, misalign_b)
        ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
        torch.cuda.synchronize()
        out = b_whole.cpu().numpy()
        lo = GUARD + misalign_b
        assert np.all(out[:lo] == gb) and np.all(out[lo + B0.size:] == gb), "guard band of B written"
        a_after = a_whole.cpu().numpy()
        assert np.array_equal(bits(a_after[GUARD + misalign_a:GUARD + misalign_a + A.size]), bits(A)), "A modified"
        got = out[lo:lo + B0.size]
    finally:
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, -1)
        if own:
            ttc.ttc_destroy(plan)
    if not np.array_equal(bits(got), bits(want)):
        bad = np.nonzero((bits(got).reshape(got.size, -1) != bits(want).reshape(want.size, -1)).any(axis=1))[0]
        raise AssertionError("pair (%d,%d) %s %s cand=%s: %d of %d elements differ, first at %d: got %r want %r" % (
            da, db, sizes, perm, candidate, bad.size, got.size, bad[0], got[bad[0]], want[bad[0]]))


# ------------------------------------------------------------------ small: every candidate
@pytest.mark.parametrize("da,db", PAIRS)
@pytest.mark.parametrize("beta_nz", [False, True])
@pytest.mark.parametrize("sizes,perm,lda,ldb", [
    ((37, 29), (1, 0), None, None),                                  # 2-D, ragged everywhere
    ((64, 48), (1, 0), (72, 48), (56, 64)),                          # 2-D, padded
    ((20, 6, 18), (2, 1, 0), None, None),                            # 3-D reversal
    ((8, 16, 16), (2, 1, 0), (32, 32, 32), None),                    # Fig. 2
    ((8, 12, 40), (0, 2, 1), (8, 14, 40), None),                     # Fig. 3 shape: packing
    ((16, 9, 7, 5), (0, 3, 1, 2), None, None),                       # copy class
    ((6, 5, 4, 6, 5, 4), (5, 2, 0, 4, 1, 3), None, None),            # c3 shape, tiny
    ((7, 12, 5, 6, 8), (4, 2, 0, 3, 1), None, None),                 # c5 shape, tiny
    ((3, 1, 5, 1, 4), (4, 3, 2, 1, 0), (4, 2, 5, 3, 4), (5, 1, 6, 2, 3)),   # extent-1 + ld
])
def test_every_candidate_small(da, db, beta_nz, sizes, perm, lda, ldb):
    plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    try:
        which = 1 if beta_nz else 0
        n = ttc.ttc_plan_num_candidates(plan, which)
        assert n >= 1
        for i in range(n):
            check(da, db, sizes, perm, lda, ldb, beta_nz, plan=plan, candidate=i)
        check(da, db, sizes, perm, lda, ldb, beta_nz, plan=plan)     # the tuned winner
    finally:
        ttc.ttc_destroy(plan)


@pytest.mark.parametrize("da,db", PAIRS[:2])
def test_all_permutations_tiny(da, db):
    """All permutations for N <= 4 with extents from {1,2,3,5,7} and random ld >= size."""
    rng = np.random.default_rng(17)
    for n in (1, 2, 3, 4):
        for perm in itertools.permutations(range(n)):
            sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 5, 7], size=n))
            szb = tuple(sizes[p] for p in perm)
            lda = tuple(int(s + rng.integers(0, 3)) for s in sizes)
            ldb = tuple(int(s + rng.integers(0, 3)) for s in szb)
            for beta_nz in (False, True):
                check(da, db, sizes, perm, lda, ldb, beta_nz)


# ------------------------------------------------------------------ several tiles and a ragged tail
@pytest.mark.parametrize("da,db", PAIRS)
@pytest.mark.parametrize("sizes,perm", [
    ((300, 130), (1, 0)), ((96, 72, 40), (2, 0, 1)), ((50, 33, 21, 9), (3, 1, 0, 2)), ((96, 40, 56), (0, 2, 1)),
])
def test_mid_size_candidates(da, db, sizes, perm):
    """Sizes of several macro-tiles with remainders; every 5th candidate beyond the first 8."""
    for beta_nz in (False, True):
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm)
        try:
            n = ttc.ttc_plan_num_candidates(plan, 1 if beta_nz else 0)
            for i in range(n):
                if i >= 8 and i % 5:
                    continue
                check(da, db, sizes, perm, None, None, beta_nz, plan=plan, candidate=i)
            check(da, db, sizes, perm, None, None, beta_nz, plan=plan)
        finally:
            ttc.ttc_destroy(plan)


# ------------------------------------------------------------------ ring kernel (class tma) with conversion
@pytest.mark.parametrize("da,db", PAIRS)
@pytest.mark.parametrize("sizes,perm,lda,ldb", [
    ((128, 72, 20), (2, 1, 0), None, None),                          # whole tiles
    ((132, 50, 9), (1, 2, 0), None, None),                           # remainder tiles
    ((8, 40, 36), (0, 2, 1), (8, 44, 36), None),                     # packing shape: short rows joined into bulk rows
    ((24, 10, 8, 12), (3, 1, 0, 2), (24, 12, 8, 12), (12, 10, 28, 8)),   # leading dimensions on both sides
])
def test_ring_candidates_mixed(da, db, sizes, perm, lda, ldb):
    """Every ring-kernel candidate of a mixed plan: the bulk copies land A's bytes, the consumer warps
    convert (reading M1) while they store.  Bit-exact, beta = 0 and beta != 0."""
    seen = 0
    for beta_nz in (False, True):
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
        try:
            which = 1 if beta_nz else 0
            for i in range(ttc.ttc_plan_num_candidates(plan, which)):
                if ttc.ttc_plan_candidate(plan, which, i).kernel == 5:
                    check(da, db, sizes, perm, lda, ldb, beta_nz, plan=plan, candidate=i)
                    seen += 1
        finally:
            ttc.ttc_destroy(plan)
    assert seen > 0, "no ring candidate generated"


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("da,db", PAIRS)
def test_beta_zero_never_reads_b_and_misaligned_pointers_fall_back(da, db):
    sizes, perm = (64, 24, 10), (2, 0, 1)
    check(da, db, sizes, perm, b_init="nan")
    for ma, mb in ((1, 0), (0, 1), (1, 1)):
        check(da, db, sizes, perm, beta_nz=True, misalign_a=ma, misalign_b=mb)


def test_empty_mixed_tensor_is_noop():
    plan = ttc.ttc_plan_mixed(wl.F32, wl.F64, 3, (4, 0, 3), (2, 0, 1))
    ttc.ttc_execute(plan, 1.0, 0, 0.0, 0)
    ttc.ttc_destroy(plan)


# ------------------------------------------------------------------ full size (the shapes bench.py --detail times)
@pytest.mark.parametrize("da,db,perm,beta_nz", [
    (wl.F32, wl.F64, (1, 0, 3, 2), False), (wl.F64, wl.F32, (3, 2, 1, 0), False),
    (wl.F32, wl.F64, (0, 2, 1, 3), True), (wl.F64, wl.F32, (2, 0, 3, 1), True),
    (wl.C64, wl.C128, (3, 0, 2, 1), False), (wl.C128, wl.C64, (1, 3, 0, 2), True),
])
def test_full_size_config2_shape(da, db, perm, beta_nz):
    """configs[1]'s tensor (96x72x64x56, 24.8 M elements) with mixed types, tuned winner, whole tensor."""
    check(da, db, wl.config2(perm).sizes, perm, beta_nz=beta_nz)


@pytest.mark.parametrize("da,db", PAIRS[:2])
def test_packing_config4_shape_mixed(da, db):
    """BLAS-style A-panel packing with conversion ("level 3 BLAS routines can be extended to
    mixed-precision"): configs[3]'s shape, NaN padding rows must never reach B."""
    w = wl.config4()
    check(da, db, w.sizes, w.perm, w.lda, w.ldb)


@pytest.mark.parametrize("da,db", PAIRS[:2])
def test_execute_host_mixed(da, db):
    """ttc_execute_host with A and B of different element sizes (slab pipeline and plain staging)."""
    for sizes, perm in (((96, 72, 64, 16), (2, 0, 3, 1)), ((40, 30, 20), (1, 2, 0))):
        for beta_nz in (False, True):
            alpha, beta = scalars(db, beta_nz)
            A, B0 = make_inputs(da, db, sizes, perm, None, None, beta_nz)
            want = B0.copy()
            oracle.transpose_mixed(da, db, sizes, perm, None, None, alpha, A, beta, want)
            plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm)
            try:
                ah = torch.from_numpy(A).pin_memory()
                bh = torch.from_numpy(B0.copy()).pin_memory()
                ttc.ttc_execute_host(plan, alpha, ah, beta, bh)
                assert np.array_equal(bits(bh.numpy()), bits(want))
            finally:
                ttc.ttc_destroy(plan)
