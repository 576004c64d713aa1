"""Host logic of the tensor-map candidate class (csrc/plan.cpp add_tmap / add_tmapu), no GPU: where a <= 5-D
CUtensorMap can express both tensors (north_star K2 "where the strides allow"; SURVEY.md 8(d) "TMA feasibility") the
plan offers such candidates, elsewhere it must not -- the two hardware rules found on B200 (a box
must start on a 16-byte boundary; a store clips in whole 16-byte granules) are planner conditions, checked here."""
import pytest

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

ES = wl.ELEM_SIZE


def tmap(plan, which=0):
    out = []
    for i in range(ttc.ttc_plan_num_candidates(plan, which)):
        c = ttc.ttc_plan_candidate(plan, which, i)
        if c.kernel == 6:
            out.append(c)
    return out


@pytest.fixture(autouse=True)
def no_tuning(monkeypatch):
    monkeypatch.setenv("TTC_TUNE", "0")


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64, wl.C128])
def test_transposing_candidates_have_128_or_64_byte_planes(dtype):
    plan = ttc.ttc_plan(dtype, 4, (96, 72, 64, 56), (3, 2, 1, 0))
    try:
        info = ttc.ttc_plan_info(plan)
        for which in (0, 1):
            cs = tmap(plan, which)
            assert 4 <= len(cs) <= 40
            for c in cs:
                assert c.flags & 2 and c.vec_a == c.vec_b == 16 // ES[dtype]
                # canonical index 0 leads A, index 3 leads B: tile extents there are 1, 2 or 4 planes of 128 / es (or 64 / es)
                for k in (0, info.canon_rank - 1):
                    assert c.tile_ext[k] * ES[dtype] % 64 == 0 and c.tile_ext[k] * ES[dtype] <= 8 * 128
                assert c.n_tiles >= 1 and c.est_cost > 1.0
    finally:
        ttc.ttc_destroy(plan)


def test_all_23_permutations_of_config1_qualify():
    for w in wl.baseline_configs():
        if not w.name.startswith("c2"):
            continue
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        try:
            assert tmap(plan, 0) and tmap(plan, 1), w.name
        finally:
            ttc.ttc_destroy(plan)


@pytest.mark.parametrize("da,db,sizes,perm,lda,ldb,why", [
    (wl.F32, wl.F32, (1023, 2301), (1, 0), None, None, "strides of 4092 / 9204 bytes"),
    (wl.F64, wl.F64, (33, 9, 21), (2, 0, 1), None, None, "8-byte aligned strides only"),
    (wl.C64, wl.C64, (7, 96, 5, 80, 64), (4, 2, 0, 3, 1), None, None, "configs[4]: 56-byte stride in A"),
    (wl.F32, wl.F64, (64, 64), (1, 0), None, None, "mixed precision"),
    (wl.F64, wl.F32, (64, 64), (1, 0), None, None, "mixed precision"),
    (wl.F32, wl.F32, (5, 3), (1, 0), (8, 3), (4, 5), "B's rows are 12 bytes inside a pitch of 16: a store would clip at 16"),
    (wl.F64, wl.F64, (33, 9, 21), (2, 0, 1), (36, 12, 21), (24, 36, 9), "B's rows are 168 bytes: not whole granules"),
    (wl.F64, wl.F64, (3, 5, 7), (0, 2, 1), (4, 8, 7), (8, 8, 5), "copy class, rows of 24 bytes"),
])
def test_no_candidate_where_the_hardware_rules_forbid_it(da, db, sizes, perm, lda, ldb, why):
    plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    try:
        assert not tmap(plan, 0) and not tmap(plan, 1), why
        assert ttc.ttc_plan_num_candidates(plan, 0) >= 1            # the other classes still serve it
    finally:
        ttc.ttc_destroy(plan)


def test_rank_above_5_uses_the_folded_flavour_and_16_byte_elements_do_not():
    sizes, perm = (20, 4, 6, 8, 6, 20), (5, 2, 0, 4, 1, 3)
    for dtype, expect in ((wl.F32, True), (wl.F64, True), (wl.C64, True), (wl.C128, False)):
        plan = ttc.ttc_plan(dtype, 6, sizes, perm)
        try:
            assert ttc.ttc_plan_info(plan).canon_rank == 6
            assert bool(tmap(plan, 0)) == expect, dtype
        finally:
            ttc.ttc_destroy(plan)


def test_variants_switch_removes_the_class(monkeypatch):
    monkeypatch.setenv("TTC_VARIANTS", "3")
    plan = ttc.ttc_plan(wl.F64, 3, (64, 24, 48), (2, 1, 0))
    try:
        assert not tmap(plan, 0) and not tmap(plan, 1)
    finally:
        ttc.ttc_destroy(plan)


def test_padded_a_rows_are_fine_and_copy_class_gets_its_flavour():
    # A's rows end inside a granule (33 fp64 = 264 bytes in a pitch of 288): loads may, stores may not
    plan = ttc.ttc_plan(wl.F64, 3, (33, 9, 20), (2, 0, 1), (36, 12, 20), (20, 36, 9))
    try:
        assert tmap(plan, 0)
    finally:
        ttc.ttc_destroy(plan)
    plan = ttc.ttc_plan(wl.F64, 3, (8, 768, 4096), (0, 2, 1), (8, 776, 4096), None)       # configs[3]
    try:
        cs = tmap(plan, 0)
        assert cs and all(c.tile_ext[0] == 8 for c in cs)
    finally:
        ttc.ttc_destroy(plan)


def skew(plan, which=0):
    return [ttc.ttc_plan_candidate(plan, which, i) for i in range(ttc.ttc_plan_num_candidates(plan, which))
            if ttc.ttc_plan_candidate(plan, which, i).kernel == 7]


def test_skew_candidates_only_where_no_tensor_map_fits(monkeypatch):
    """The skew kernel (csrc/ttc_skew.cuh) is for what tensor maps cannot take: rows that are not 16-byte aligned.  By
    default only its direct-out variants (flag 8) are offered, the out-tile variants with TTC_VARIANTS bit 4."""
    plan = ttc.ttc_plan(wl.F32, 2, (1023, 2301), (1, 0))
    try:
        for which in (0, 1):
            cs = skew(plan, which)
            assert cs and all(c.flags & 8 for c in cs) and not tmap(plan, which)
            for c in cs:
                assert c.tile_ext[0] in (32, 64, 128, 256) and c.tile_ext[1] in (32, 64, 128)
    finally:
        ttc.ttc_destroy(plan)
    for dtype, sizes, perm in ((wl.F64, (96, 72, 64, 56), (3, 2, 1, 0)), (wl.C128, (37, 45), (1, 0)), (wl.F32, (48, 13, 21), (0, 2, 1)),
                               (wl.F32, (1023, 7), (1, 0))):
        plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm)
        try:
            assert not skew(plan, 0) and not skew(plan, 1), (sizes, perm)
        finally:
            ttc.ttc_destroy(plan)
    monkeypatch.setenv("TTC_VARIANTS", "31")
    plan = ttc.ttc_plan(wl.F64, 2, (137, 145), (1, 0))          # single-index runs: the out-tile variants exist as well
    try:
        assert {c.flags & 8 for c in skew(plan, 1)} == {0, 8}
    finally:
        ttc.ttc_destroy(plan)
    monkeypatch.setenv("TTC_VARIANTS", "7")
    plan = ttc.ttc_plan(wl.F32, 2, (1023, 2301), (1, 0))
    try:
        assert not skew(plan, 0)
    finally:
        ttc.ttc_destroy(plan)
