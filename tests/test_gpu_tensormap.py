"""``-m gpu``: the tensor-map kernel class (TTC_KERNEL_TENSORMAP = 6: cp.async.bulk.tensor box loads and stores,
swizzled shared-memory boxes, in-register micro-tiles; north_star K2, SURVEY.md 8(d) "TMA feasibility") against
the oracle, bit for bit: every tensor-map candidate of every shape below, every element type, beta on and off.
The shapes cover: boxes that stick out of the tensor on every side (loads fill zeros, stores clip), padded A
and B, 2-D .. 7-D, the copy class (shared leading index: flavour 1, incl. the store-what-was-loaded path for
real alpha == 1, beta == 0), several boxes per tile, and tensors a map cannot express (no such candidate)."""
import numpy as np
import pytest
import torch

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import check_bit_exact

pytestmark = pytest.mark.gpu

ALL_DTYPES = (wl.F32, wl.F64, wl.C64, wl.C128)


def scalars(dtype, beta_nz):
    if dtype >= 2:
        return (0.75 - 1.25j, (0.5 + 0.375j) if beta_nz else 0.0)
    return (1.5, 0.5 if beta_nz else 0.0)


def tensormap_candidates(plan, which):
    return [i for i in range(ttc.ttc_plan_num_candidates(plan, which))
            if ttc.ttc_plan_candidate(plan, which, i).kernel == 6]


# sizes in units of 4 elements keep every stride a multiple of 16 bytes for all four element types
SHAPES = [
    ("t2d", (96, 80), (1, 0), None, None),
    ("t2d_ragged", (100, 52), (1, 0), None, None),                       # edge boxes on both sides
    ("t3d", (64, 24, 48), (2, 1, 0), None, None),
    ("t3d_ragged_padded", (100, 36, 44), (1, 2, 0), (104, 40, 44), (36, 48, 100)),
    ("t3d_half_rows", (40, 20, 24), (2, 1, 0), None, None),                # 64-byte rows: 40 and 24 fp64 / c64 without padding
    ("t4d", (36, 8, 12, 20), (3, 1, 0, 2), None, None),
    ("t5d", (20, 4, 12, 8, 16), (4, 2, 0, 3, 1), None, None),
    ("copy3d", (48, 12, 20), (0, 2, 1), None, None),                     # flavour 1
    ("copy3d_padded", (44, 9, 10), (0, 2, 1), (48, 9, 10), (52, 12, 9)),
    ("copy_long_rows", (1200, 6, 10), (0, 2, 1), None, None),            # rows longer than one box
    # A's rows are not a multiple of 16 bytes long inside a padded leading dimension that is (B's are: see ODD_B_ROWS)
    ("t3d_odd_a_rows_padded", (33, 9, 20), (2, 0, 1), (36, 12, 20), (20, 36, 9)),
]

# B's rows are not a multiple of 16 bytes long, inside leading dimensions that are: a tensor-map STORE clips at the edge of
# the tensor in whole 16-byte granules only and would overwrite the padding -- no tensor-map candidate (16-byte elements: fine)
ODD_B_ROWS = [
    ("t3d_odd_rows_padded", (33, 9, 21), (2, 0, 1), (36, 12, 21), (24, 36, 9)),
    ("copy_odd_rows_padded", (3, 5, 7), (0, 2, 1), (4, 8, 7), (8, 8, 5)),
    ("t2d_tiny_padded", (5, 3), (1, 0), (8, 3), (4, 5)),
]


@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("shape", ODD_B_ROWS, ids=[s[0] for s in ODD_B_ROWS])
def test_no_tensormap_store_into_rows_that_end_inside_a_granule(dtype, shape):
    name, sizes, perm, lda, ldb = shape
    for beta_nz in (False, True):
        alpha, beta = scalars(dtype, beta_nz)
        w = wl.Workload(name, dtype, sizes, perm, alpha, beta, lda=lda, ldb=ldb)
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        try:
            cands = tensormap_candidates(plan, 1 if beta_nz else 0)
            if dtype == wl.C128:
                for i in cands:
                    check_bit_exact(w, plan=plan, candidate=i)
            else:
                assert not cands
            check_bit_exact(w, plan=plan)            # whatever the plan chose: padding (NaN guards) intact
        finally:
            ttc.ttc_destroy(plan)


@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("beta_nz", [False, True])
@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_every_tensormap_candidate(dtype, beta_nz, shape):
    name, sizes, perm, lda, ldb = shape
    alpha, beta = scalars(dtype, beta_nz)
    w = wl.Workload(name, dtype, sizes, perm, alpha, beta, lda=lda, ldb=ldb)
    plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
    try:
        which = 1 if beta_nz else 0
        cands = tensormap_candidates(plan, which)
        assert cands, "no tensor-map candidate for %s dtype %d" % (name, dtype)
        for i in cands:
            c = ttc.ttc_plan_candidate(plan, which, i)
            assert c.flags & 2 and c.vec_a == c.vec_b
            check_bit_exact(w, plan=plan, candidate=i)
    finally:
        ttc.ttc_destroy(plan)


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64])
def test_copy_class_alpha_one_stores_what_it_loaded(dtype):
    """Real alpha == 1, beta == 0, shared leading index: no thread touches the data (complex types still compute)."""
    for sizes, perm, lda, ldb in (((48, 12, 20), (0, 2, 1), None, None), ((44, 9, 10), (0, 2, 1), (48, 9, 10), (52, 12, 9))):
        w = wl.Workload("copy1", dtype, sizes, perm, 1.0, 0.0, lda=lda, ldb=ldb)
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        try:
            cands = tensormap_candidates(plan, 0)
            assert cands
            for i in cands:
                check_bit_exact(w, plan=plan, candidate=i)
        finally:
            ttc.ttc_destroy(plan)


@pytest.mark.parametrize("sched", ["static", "atomic"])
def test_tensormap_work_distributions(sched, monkeypatch):
    monkeypatch.setenv("TTC_SCHED", sched)
    monkeypatch.setenv("TTC_TUNE", "0")
    for beta_nz in (False, True):
        alpha, beta = scalars(wl.F64, beta_nz)
        # many more tiles than resident CTAs: every CTA loops, the ring of stages wraps several times
        w = wl.Workload("many", wl.F64, (320, 48, 160), (2, 1, 0), alpha, beta)
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
        try:
            cands = tensormap_candidates(plan, 1 if beta_nz else 0)
            assert cands
            for i in cands[:4]:
                c = ttc.ttc_plan_candidate(plan, 1 if beta_nz else 0, i)
                assert c.sched == (0 if sched == "static" else 2)
                check_bit_exact(w, plan=plan, candidate=i)
        finally:
            ttc.ttc_destroy(plan)


def test_no_tensormap_candidate_where_a_map_cannot_express_the_tensor(monkeypatch):
    monkeypatch.setenv("TTC_TUNE", "0")
    cases = [
        (wl.F32, wl.F32, (1023, 2301), (1, 0)),              # strides of 4092 / 9204 bytes: not multiples of 16
        (wl.F64, wl.F64, (33, 9, 21), (2, 0, 1)),            # odd fp64 extents: 8-byte-aligned strides only
        (wl.F64, wl.F64, (7, 96, 40), (2, 1, 0)),            # rows of 7 fp64 (configs[4]'s A side)
        (wl.F32, wl.F64, (64, 64), (1, 0)),                  # mixed precision
        (wl.F64, wl.F64, (8, 4, 4, 4, 4, 4, 4), (6, 5, 4, 3, 2, 1, 0)),     # 7-D, 4 elements along B's leading index
    ]
    for da, db, sizes, perm in cases:
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm)
        try:
            for which in (0, 1):
                assert not tensormap_candidates(plan, which), (sizes, perm)
        finally:
            ttc.ttc_destroy(plan)


# More than 5 canonical indices: flavour 2 (ttc_tmap.h) folds every index beyond the plane into one map dimension.
HIGH_RANK = [
    ("r6", (20, 4, 6, 8, 6, 20), (5, 2, 0, 4, 1, 3)),
    ("r6_ragged", (36, 4, 3, 8, 5, 44), (5, 2, 0, 4, 1, 3)),
    ("r7", (16, 4, 2, 4, 3, 2, 24), (6, 2, 0, 4, 1, 5, 3)),
]


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64])
@pytest.mark.parametrize("beta_nz", [False, True])
@pytest.mark.parametrize("shape", HIGH_RANK, ids=[s[0] for s in HIGH_RANK])
def test_every_high_rank_tensormap_candidate(dtype, beta_nz, shape):
    name, sizes, perm = shape
    alpha, beta = scalars(dtype, beta_nz)
    w = wl.Workload(name, dtype, sizes, perm, alpha, beta)
    plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
    try:
        assert ttc.ttc_plan_info(plan).canon_rank == len(sizes)
        which = 1 if beta_nz else 0
        cands = tensormap_candidates(plan, which)
        assert cands, "no tensor-map candidate for %s dtype %d" % (name, dtype)
        for i in cands:
            check_bit_exact(w, plan=plan, candidate=i)
    finally:
        ttc.ttc_destroy(plan)


@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_random_small_padded_shapes_every_tensormap_candidate(dtype):
    """Seeded random small tensors (rank 2..5, extents 1..20, leading dimensions padded to 16-byte multiples along the
    first index and arbitrarily along the others, extent-1 indices, tiles far larger than the tensor): every tensor-map
    candidate a plan offers, and the plan's own choice, against the oracle with NaN guards in every padding element."""
    rng = np.random.default_rng(1607 + dtype)
    g = 16 // wl.ELEM_SIZE[dtype]
    checked = 0
    for case in range(36):
        n = int(rng.integers(2, 6))
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5, 7, 8, 12, 16, 20], size=n))
        perm = tuple(int(x) for x in rng.permutation(n))
        szb = tuple(sizes[p] for p in perm)

        def padded(sz):
            ld = [int(x + rng.integers(0, 3)) for x in sz]
            ld[0] = -(-int(sz[0] + rng.integers(0, 2 * g)) // g) * g          # rows start on 16-byte boundaries
            return tuple(ld)
        lda, ldb = padded(sizes), padded(szb)
        for beta_nz in (False, True):
            alpha, beta = scalars(dtype, beta_nz)
            w = wl.Workload("rnd%d" % case, dtype, sizes, perm, alpha, beta, lda=lda, ldb=ldb)
            plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
            try:
                for i in tensormap_candidates(plan, 1 if beta_nz else 0):
                    check_bit_exact(w, plan=plan, candidate=i)
                    checked += 1
                check_bit_exact(w, plan=plan)
            finally:
                ttc.ttc_destroy(plan)
    assert checked >= 20, checked


def test_tensormap_candidate_with_misaligned_pointers_falls_back():
    """The maps need 16-byte aligned base addresses: a forced tensor-map candidate is replaced for other pointers."""
    w = wl.Workload("mis", wl.F32, (96, 80), (1, 0), 1.5, 0.5)
    plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
    try:
        cands = tensormap_candidates(plan, 1)
        assert cands
        check_bit_exact(w, plan=plan, candidate=cands[0], misalign_a=1, misalign_b=1)
        check_bit_exact(w, plan=plan, candidate=cands[0], misalign_a=0, misalign_b=2)
    finally:
        ttc.ttc_destroy(plan)


def test_tensormap_full_size_configs():
    """configs[1] (96 x 72 x 64 x 56 fp64, beta != 0) in two permutations and configs[3]-like packing, full size:
    sampled elements against the definition (the oracle's formula for one element, evaluated in numpy fp64)."""
    rng = np.random.default_rng(7)
    for sizes, perm, alpha, beta in (((96, 72, 64, 56), (3, 2, 1, 0), 1.5, 0.5), ((96, 72, 64, 56), (0, 3, 1, 2), 1.0, 0.0),
                                     ((96, 72, 64, 56), (1, 0, 3, 2), 1.5, 0.5)):
        n = int(np.prod(sizes))
        A = wl.uniform_values(wl.SEED_A, n, wl.F64)
        B0 = wl.uniform_values(wl.SEED_B, n, wl.F64)
        plan = ttc.ttc_plan(wl.F64, len(sizes), sizes, perm)
        try:
            which = 1 if beta else 0
            cands = tensormap_candidates(plan, which)
            assert cands
            szb = [sizes[p] for p in perm]
            idx_b = [rng.integers(0, s, size=4096) for s in szb]
            off_b = np.zeros(4096, dtype=np.int64)
            off_a = np.zeros(4096, dtype=np.int64)
            sb = 1
            stride_a = np.cumprod([1] + list(sizes[:-1]))
            for k, s in enumerate(szb):
                off_b += idx_b[k] * sb
                off_a += idx_b[k] * stride_a[perm[k]]
                sb *= s
            a_dev = torch.from_numpy(A).cuda()
            for i in cands[:3]:
                ttc.ttc_plan_select(plan, which, i)
                b_dev = torch.from_numpy(B0).cuda()
                ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
                torch.cuda.synchronize()
                got = b_dev.cpu().numpy()
                want = alpha * A[off_a] + (beta * B0[off_b] if beta else 0.0)
                assert np.array_equal(got[off_b], want), (sizes, perm, i)
                # invariant that holds at any size: beta == 0 -> B is a permutation of alpha * A
                if not beta:
                    assert np.array_equal(np.sort(got), np.sort(alpha * A))
        finally:
            ttc.ttc_destroy(plan)
