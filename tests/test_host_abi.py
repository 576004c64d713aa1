"""CPU-only tests of the host side of libttc.so: the library loads and exports every symbol
include/ttc.h declares, argument validation, the canonicaliser (stage 1),
the fast-divmod constants and the candidate generator (stages 2-3).
No kernel is launched here."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "ttc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ttc_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    syms = header_symbols()
    assert "ttc_plan" in syms and "ttc_execute" in syms and "ttc_destroy" in syms
    for s in syms:
        assert hasattr(ttc.lib, s), "libttc.so does not export %s" % s
    assert sorted(ttc.EXPORTS) == syms
    assert "sm_100a" in ttc.ttc_version()


def test_versions_agree():
    """Package __version__ and ttc_version() name the same release."""
    import paper_1607_01249_b200 as pkg
    major_minor = ".".join(pkg.__version__.split(".")[:2])
    assert ("ttc-b200 %s " % major_minor) in ttc.ttc_version()


def test_struct_layouts_match_header():
    """The ctypes mirrors must have the C sizes (int64 alignment included)."""
    assert ctypes.sizeof(ttc.ttc_info) == 4 * 4 + 3 * 16 * 8 + 3 * 8 + 4 + 2 * 4 + 2 * 4 + 2 * 4 + 3 * 4 + 6 * 4
    assert ctypes.sizeof(ttc.ttc_candidate_info) % 8 == 0


@pytest.mark.parametrize("args,status", [
    (dict(dtype=9, sizes=(2, 2), perm=(0, 1)), "INVALID_ARG"),
    (dict(dtype=0, sizes=(2, 2), perm=(0, 0)), "NOT_PERMUTATION"),
    (dict(dtype=0, sizes=(2, 2), perm=(0, 2)), "NOT_PERMUTATION"),
    (dict(dtype=0, sizes=(2, -1), perm=(0, 1)), "INVALID_ARG"),
    (dict(dtype=0, sizes=(4, 3), perm=(1, 0), lda=(3, 3)), "BAD_LD"),
    (dict(dtype=0, sizes=(4, 3), perm=(1, 0), ldb=(4, 4)), "BAD_LD"),      # ldb[0] pairs with sizes[perm[0]]=3? no: 4>=3 ok, ldb[1]=4>=4
    (dict(dtype=0, sizes=(2 ** 40, 2 ** 40), perm=(1, 0)), "UNSUPPORTED"),
])
def test_plan_argument_errors(args, status):
    if args.get("ldb") == (4, 4):
        args = dict(args, ldb=(2, 4))     # ldb[0] = 2 < sizes[perm[0]] = 3
    with pytest.raises(ttc.TTCError) as ei:
        ttc.ttc_plan(args["dtype"], len(args["sizes"]), args["sizes"], args["perm"],
                     args.get("lda"), args.get("ldb"))
    assert ttc.STATUS_NAMES[ei.value.status] == "TTC_ERR_" + status


def test_rank_limits():
    with pytest.raises(ttc.TTCError):
        ttc.ttc_plan(0, 17, (1,) * 17, tuple(range(17)))
    p = ttc.ttc_plan(0, 16, (2,) * 16, tuple(reversed(range(16))))
    assert ttc.ttc_plan_info(p).canon_rank == 16
    ttc.ttc_destroy(p)


# --------------------------------------------------------------------- canonicaliser
def test_merge_example_of_the_paper():
    """Pi(i0,i1,i2) = (i1,i2,i0) is the 2-D transposition with size(i1)*size(i2)."""
    assert ttc.ttc_canonicalize((5, 3, 4), (1, 2, 0)) == [(5, 1, 12), (12, 5, 1)]
    # config 1: (2,0,1) fuses (i0,i1): 2-D transpose of (23040, 128)
    assert ttc.ttc_canonicalize((160, 144, 128), (2, 0, 1)) == [(23040, 1, 128), (128, 23040, 1)]


def test_identity_collapses_to_one_index():
    assert ttc.ttc_canonicalize((4, 5, 6), (0, 1, 2)) == [(120, 1, 1)]


def test_padding_blocks_merging():
    """fn 5: merging needs ld(i_m) = size(i_m), in A and in B (reading A11)."""
    assert len(ttc.ttc_canonicalize((4, 5, 6), (0, 1, 2), lda=(4, 7, 6))) == 2
    assert len(ttc.ttc_canonicalize((4, 5, 6), (0, 1, 2), ldb=(5, 5, 6))) == 3 - 1
    assert ttc.ttc_canonicalize((4, 5, 6), (0, 1, 2), lda=(4, 7, 6)) == [(20, 1, 1), (6, 28, 20)]


def test_extent_one_indices_are_dropped_but_keep_their_stride_effect():
    """Reading A12: an extent-1 index with ld > 1 still multiplies later strides."""
    got = ttc.ttc_canonicalize((3, 1, 5), (2, 1, 0), lda=(4, 2, 5), ldb=(5, 3, 3))
    assert got == [(3, 1, 15), (5, 8, 1)]
    assert ttc.ttc_canonicalize((1, 1, 1), (2, 0, 1)) == [(1, 1, 1)]
    assert ttc.ttc_canonicalize((3, 0, 2), (2, 0, 1)) == []


def test_config_canonical_forms_match_survey_table():
    """c4 and c5 canonical (e, sA, sB) triples; c2 rank histogram 3/9/11."""
    w = wl.config4()
    assert ttc.ttc_canonicalize(w.sizes, w.perm, w.lda) == [(8, 1, 1), (768, 8, 32768), (4096, 6208, 8)]
    w = wl.config5()
    assert ttc.ttc_canonicalize(w.sizes, w.perm) == [
        (7, 1, 320), (96, 7, 179200), (5, 672, 64), (80, 3360, 2240), (64, 268800, 1)]
    ranks = [len(ttc.ttc_canonicalize(c.sizes, c.perm)) for c in wl.config2_all()]
    assert (ranks.count(2), ranks.count(3), ranks.count(4)) == (3, 9, 11)
    assert len(ttc.ttc_canonicalize(wl.config3().sizes, wl.config3().perm)) == 6


def test_canonical_form_preserves_the_offset_map():
    """The canonical triples enumerate exactly the same (offA, offB) pairs as the definition
    (checked against numpy index arithmetic, not against the oracle)."""
    rng = np.random.default_rng(7)
    for _ in range(40):
        n = int(rng.integers(1, 6))
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5], size=n))
        perm = tuple(int(x) for x in rng.permutation(n))
        szb = tuple(sizes[p] for p in perm)
        lda = tuple(int(s + rng.integers(0, 2)) for s in sizes)
        ldb = tuple(int(s + rng.integers(0, 2)) for s in szb)
        sA = np.cumprod((1,) + lda[:-1])
        tB = np.cumprod((1,) + ldb[:-1])
        idx = np.indices(sizes).reshape(n, -1)
        offA = (idx * sA[:, None]).sum(0)
        offB = sum(idx[perm[k]] * tB[k] for k in range(n))
        want = set(zip(offA.tolist(), offB.tolist()))
        can = ttc.ttc_canonicalize(sizes, perm, lda, ldb)
        cidx = np.indices([c[0] for c in can]).reshape(len(can), -1)
        ca = sum(cidx[i] * can[i][1] for i in range(len(can)))
        cb = sum(cidx[i] * can[i][2] for i in range(len(can)))
        assert set(zip(ca.tolist(), cb.tolist())) == want
        assert all(c[0] > 1 for c in can) or len(can) == 1


# --------------------------------------------------------------------- fast divmod
def test_fastdiv_is_exact():
    rng = np.random.default_rng(5)
    ds = [1, 2, 3, 5, 7, 24, 56, 96, 672, 4608, 65535, 65537, 2 ** 30 - 1, 2 ** 31 - 1] + \
        [int(x) for x in rng.integers(1, 2 ** 31, 40)]
    for d in ds:
        ns = [0, 1, d - 1, d, d + 1, 2 * d - 1, 2 ** 31 - 1] + [int(x) for x in rng.integers(0, 2 ** 31, 50)]
        for n in ns:
            if 0 <= n < 2 ** 31:
                assert ttc.lib.ttc_debug_fastdiv(n, d) == n // d, (n, d)


# --------------------------------------------------------------------- candidate generator
def test_candidates_exist_for_every_config_and_are_ranked():
    for w in wl.baseline_configs():
        p = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        try:
            info = ttc.ttc_plan_info(p)
            assert info.numel == w.numel
            for which in (0, 1):
                n = ttc.ttc_plan_num_candidates(p, which)
                assert 1 <= n <= 400                     # bounded list (default 200; ours 400)
                cs = [ttc.ttc_plan_candidate(p, which, i) for i in range(n)]
                costs = [c.est_cost for c in cs]
                assert costs == sorted(costs)
                # an always-valid scalar fallback exists
                assert any(c.kernel == 1 and c.vec_a == 1 for c in cs)
                for c in cs:
                    assert c.smem_bytes <= 227 * 1024
        finally:
            ttc.ttc_destroy(p)


def test_copy_class_configs_rank_a_vector_copy_first():
    """stride-1-unchanged cases are whole-column copies."""
    for perm in [(0, 1, 3, 2), (0, 2, 1, 3), (0, 3, 2, 1)]:
        w = wl.config2(perm)
        p = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
        c = ttc.ttc_plan_candidate(p, 0, 0)
        assert c.vec_a * 8 == 16 and c.vec_b * 8 == 16
        ttc.ttc_destroy(p)


# --------------------------------------------------------------------- mixed precision
MIXED_PAIRS = ((0, 1), (1, 0), (2, 3), (3, 2))     # sd, ds, cz, zc


@pytest.mark.parametrize("da,db", MIXED_PAIRS)
def test_mixed_plan_reports_both_types_and_has_ring_candidates(da, db):
    """ttc_plan_mixed: dtype of the plan is B's, ttc_plan_dtype_a gives A's; vectors are at most 16
    bytes of each side's own type; the ring kernel is a candidate with 16-byte bulk rows of A's type
    only (its tile holds A's bytes, the consumers convert)."""
    w = wl.config2((2, 0, 3, 1))
    p = ttc.ttc_plan_mixed(da, db, w.n, w.sizes, w.perm)
    try:
        info = ttc.ttc_plan_info(p)
        assert info.dtype == db and ttc.ttc_plan_dtype_a(p) == da
        assert info.numel == w.numel
        for which in (0, 1):
            n = ttc.ttc_plan_num_candidates(p, which)
            cs = [ttc.ttc_plan_candidate(p, which, i) for i in range(n)]
            assert any(c.kernel == 1 and c.vec_a == 1 for c in cs)          # scalar fallback
            assert any(c.kernel in (2, 3, 4) for c in cs)                   # tiled transposes
            ring = [c for c in cs if c.kernel == 5]
            assert ring and all(c.vec_a * wl.ELEM_SIZE[da] == 16 for c in ring)   # bulk rows only
            assert all(c.vec_a * wl.ELEM_SIZE[da] <= 16 and c.vec_b * wl.ELEM_SIZE[db] <= 16 for c in cs)
            if wl.ELEM_SIZE[da] < 16 and wl.ELEM_SIZE[db] < 16:   # 16-byte vectors on both sides exist
                assert any(c.vec_a * wl.ELEM_SIZE[da] == 16 and c.vec_b * wl.ELEM_SIZE[db] == 16 for c in cs)
    finally:
        ttc.ttc_destroy(p)


def test_mixed_plan_of_equal_types_is_the_plain_plan():
    w = wl.config1()
    p = ttc.ttc_plan_mixed(w.dtype, w.dtype, w.n, w.sizes, w.perm)
    q = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
    try:
        assert ttc.ttc_plan_dtype_a(p) == ttc.ttc_plan_dtype_a(q) == w.dtype
        assert ttc.ttc_plan_num_candidates(p, 0) == ttc.ttc_plan_num_candidates(q, 0)
    finally:
        ttc.ttc_destroy(p)
        ttc.ttc_destroy(q)


@pytest.mark.parametrize("da,db", [(0, 2), (2, 0), (1, 3), (0, 3), (2, 1)])
def test_real_complex_pairs_are_unsupported(da, db):
    with pytest.raises(ttc.TTCError) as ei:
        ttc.ttc_plan_mixed(da, db, 2, (4, 4), (1, 0))
    assert ttc.STATUS_NAMES[ei.value.status] == "TTC_ERR_UNSUPPORTED"
    with pytest.raises(ttc.TTCError) as ei:
        ttc.ttc_plan_mixed(7, 0, 2, (4, 4), (1, 0))
    assert ttc.STATUS_NAMES[ei.value.status] == "TTC_ERR_INVALID_ARG"


def test_plan_strided_canonical_form_and_errors():
    """ttc_plan_strided (SURVEY.md 8(b) optional extension): same canonical form as the leading-dimension call
    where both can describe the tensors; configs[3] by its raw outer stride; rejected layouts."""
    p1 = ttc.ttc_plan(ttc.TTC_F64, 3, (8, 768, 4096), (0, 2, 1), (8, 776, 4096), None)
    p2 = ttc.ttc_plan_strided(ttc.TTC_F64, ttc.TTC_F64, 3, (8, 768, 4096), (0, 2, 1), (1, 8, 6208), (1, 8, 8 * 4096))
    i1, i2 = ttc.ttc_plan_info(p1), ttc.ttc_plan_info(p2)
    assert i1.canon_rank == i2.canon_rank == 3
    for k in range(3):
        assert (i1.canon_extent[k], i1.canon_stride_a[k], i1.canon_stride_b[k]) == \
               (i2.canon_extent[k], i2.canon_stride_a[k], i2.canon_stride_b[k])
    assert (i1.span_a, i1.span_b) == (i2.span_a, i2.span_b)
    ttc.ttc_destroy(p1)
    ttc.ttc_destroy(p2)
    # an outer stride that no leading dimension can express (6209 is not a multiple of 8); A indices out of order
    p = ttc.ttc_plan_strided(ttc.TTC_F32, ttc.TTC_F32, 3, (8, 4, 5), (0, 2, 1), (1, 8, 6209), (1, 8, 40))
    assert ttc.ttc_plan_info(p).canon_stride_a[2] == 6209
    ttc.ttc_destroy(p)
    p = ttc.ttc_plan_strided(ttc.TTC_F32, ttc.TTC_F32, 2, (6, 4), (1, 0), (5, 1), (1, 4))     # A is row-major: a pure copy
    info = ttc.ttc_plan_info(p)
    assert info.canon_rank == 2 and info.canon_stride_a[0] == 1 and info.canon_extent[0] == 4
    ttc.ttc_destroy(p)
    for sa, sb in (((1, 3), (1, 6)),        # A overlaps itself: stride 3 < extent 6
                   ((1, 6), (1, 3)),        # B would be written twice
                   ((0, 6), (1, 4)), ((1, 6), (1, -4))):
        with pytest.raises(ttc.TTCError) as ei:
            ttc.ttc_plan_strided(ttc.TTC_F32, ttc.TTC_F32, 2, (6, 4), (1, 0), sa, sb)
        assert ei.value.status == 3          # TTC_ERR_BAD_LD
    with pytest.raises(ttc.TTCError) as ei:
        ttc.ttc_plan_strided(ttc.TTC_F32, ttc.TTC_C64, 2, (6, 4), (1, 0), (1, 6), (1, 4))
    assert ei.value.status == 4              # TTC_ERR_UNSUPPORTED: not one of the paper's type pairs


def test_specialised_source_compiles_with_nvrtc():
    """the size-specialised twin of a ring-kernel candidate -- the library's own device
    source with the candidate's parameter block as a constexpr object -- compiles with NVRTC for sm_100a (no
    device needed).  One candidate per flavour (plain, staggered, shifted rows, peeled) of three shapes."""
    import ctypes.util
    try:
        ctypes.CDLL("libnvrtc.so.12")
    except OSError:
        if not os.path.exists("/usr/local/cuda/lib64/libnvrtc.so"):
            pytest.skip("libnvrtc not installed: ttc_plan_specialize reports TTC_ERR_UNSUPPORTED and plans stay generic")
    compiled = 0
    for w in (wl.config2((1, 0, 2, 3)), wl.Workload("odd", wl.F32, (131, 9, 67), (2, 0, 1), 1.5, 0.5), wl.config5()):
        p = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        try:
            which = 1 if w.beta_nonzero else 0
            seen = set()
            for i in range(ttc.ttc_plan_num_candidates(p, which)):
                c = ttc.ttc_plan_candidate(p, which, i)
                key = (c.kernel, c.flags, c.vec_b > 1)
                if key in seen:
                    continue
                seen.add(key)
                n, log = ttc.ttc_debug_specialize_compile(p, which, i)
                if c.kernel in (1, 5):
                    assert n > 1000, log
                    compiled += 1
                else:
                    assert n == -2          # only ring- and direct-kernel candidates have a twin
        finally:
            ttc.ttc_destroy(p)
    assert compiled >= 5
