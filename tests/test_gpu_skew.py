"""``-m gpu``: the skew kernel class (TTC_KERNEL_SKEW = 7, csrc/ttc_skew.cuh) against the oracle, bit for bit: tensors
whose rows are NOT 16-byte aligned (odd extents of 4- and 8-byte elements) move with 1-D bulk copies in both
directions -- the aligned superset of every row in, the aligned body of every row out, heads and tails element-wise.
Guards (NaN) around and inside every padded tensor catch a store that reaches past its row; pointers that are only
element-aligned add one more skew; tiny tensors put every row at the end of the tensor (element-wise fallback).
Two variants: consumers that store to B themselves (coalesced element stores; offered by default) and an out-tile with bulk
stores (correct but 2x slower on B200: offered only with TTC_VARIANTS bit 4, which these tests set)."""
import numpy as np
import pytest
import torch

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import check_bit_exact

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def offer_skew_candidates(monkeypatch):
    monkeypatch.setenv("TTC_VARIANTS", "31")          # bit 4: the out-tile variants too (not offered by default)


def scalars(dtype, beta_nz):
    if dtype >= 2:
        return (0.75 - 1.25j, (0.5 + 0.375j) if beta_nz else 0.0)
    return (1.5, 0.5 if beta_nz else 0.0)


def skew_candidates(plan, which):
    return [i for i in range(ttc.ttc_plan_num_candidates(plan, which))
            if ttc.ttc_plan_candidate(plan, which, i).kernel == 7]


SHAPES = [
    ("s2d", (1023, 301), (1, 0), None, None),
    ("s2d_small", (37, 45), (1, 0), None, None),                        # every row within 16 bytes of a tensor end somewhere
    ("s2d_b_only", (100, 53), (1, 0), None, None),                      # A's rows are aligned for fp32, B's are not
    ("s2d_padded", (67, 131), (1, 0), (70, 131), (133, 67)),
    ("s3d", (37, 21, 45), (2, 1, 0), None, None),
    ("s3d_padded", (33, 9, 21), (2, 0, 1), (35, 9, 21), (23, 33, 10)),
    ("s4d", (19, 6, 10, 35), (3, 1, 0, 2), None, None),
    ("s5d", (21, 3, 5, 4, 17), (4, 2, 0, 3, 1), None, None),
    ("s2d_wide", (300, 257), (1, 0), None, None),                       # several tiles in both directions, ragged tails
    # short leading extents: the tile's b-range runs over B's two leading indices (15 x 27 contiguous in B), ...
    ("s5d_b_run", (63, 27, 10, 15, 4), (3, 1, 0, 4, 2), None, None),
    # ... its a-range over A's two leading indices (11 x 37 contiguous in A), b-range over 14 x 8
    ("s5d_ab_runs", (11, 37, 8, 9, 14), (4, 2, 1, 3, 0), None, None),
    ("s4d_runs_of_three", (5, 7, 3, 9, 5, 3), (5, 4, 3, 2, 1, 0), None, None),
    ("s4d_padded_no_runs", (21, 19, 5, 17), (3, 1, 0, 2), (22, 19, 5, 17), (18, 19, 21, 5)),
]


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64])
@pytest.mark.parametrize("beta_nz", [False, True])
@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_every_skew_candidate(dtype, beta_nz, shape):
    name, sizes, perm, lda, ldb = shape
    alpha, beta = scalars(dtype, beta_nz)
    w = wl.Workload(name, dtype, sizes, perm, alpha, beta, lda=lda, ldb=ldb)
    plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
    try:
        which = 1 if beta_nz else 0
        cands = skew_candidates(plan, which)
        assert cands, "no skew candidate for %s dtype %d" % (name, dtype)
        flavours = {ttc.ttc_plan_candidate(plan, which, i).flags & 8 for i in cands}
        assert 8 in flavours, flavours                                   # direct-out always; out-tile variants for single-index runs
        for i in cands:
            check_bit_exact(w, plan=plan, candidate=i)
        for flag in sorted(flavours):
            first = [i for i in cands if ttc.ttc_plan_candidate(plan, which, i).flags & 8 == flag][0]
            for ma, mb in ((1, 0), (0, 1), (3, 2)):                      # element-aligned pointers: one more skew
                if dtype != wl.F32:
                    ma, mb = ma % 2, mb % 2
                check_bit_exact(w, plan=plan, candidate=first, misalign_a=ma, misalign_b=mb)
    finally:
        ttc.ttc_destroy(plan)


@pytest.mark.parametrize("sched", ["static", "atomic"])
def test_skew_work_distributions(sched, monkeypatch):
    monkeypatch.setenv("TTC_SCHED", sched)
    monkeypatch.setenv("TTC_TUNE", "0")
    for beta_nz in (False, True):
        alpha, beta = scalars(wl.F32, beta_nz)
        w = wl.Workload("many", wl.F32, (1501, 1203), (1, 0), alpha, beta)     # many more tiles than resident CTAs
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
        try:
            cands = skew_candidates(plan, 1 if beta_nz else 0)
            assert cands
            for i in cands[:3]:
                assert ttc.ttc_plan_candidate(plan, 1 if beta_nz else 0, i).sched == (0 if sched == "static" else 2)
                check_bit_exact(w, plan=plan, candidate=i)
        finally:
            ttc.ttc_destroy(plan)


def test_no_skew_candidate_for_aligned_or_mixed_tensors(monkeypatch):
    monkeypatch.setenv("TTC_TUNE", "0")
    for da, db, sizes, perm in ((wl.F64, wl.F64, (96, 72, 64, 56), (3, 2, 1, 0)), (wl.F32, wl.F64, (1023, 301), (1, 0)),
                                (wl.C128, wl.C128, (37, 45), (1, 0)), (wl.F32, wl.F32, (48, 13, 21), (0, 2, 1))):
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm)
        try:
            assert not skew_candidates(plan, 0) and not skew_candidates(plan, 1), (sizes, perm)
        finally:
            ttc.ttc_destroy(plan)


def test_skew_full_size_unaligned_fp32():
    """The shape of the sweep's outliers (2-D fp32, odd extents, ~115 MB), beta on and off: sampled elements against the
    definition, corners included, and for beta == 0 B as a permutation of alpha * A."""
    sizes, perm = (5119, 5633), (1, 0)
    n = sizes[0] * sizes[1]
    A = wl.uniform_values(wl.SEED_A, n, wl.F32)
    B0 = wl.uniform_values(wl.SEED_B, n, wl.F32)
    rng = np.random.default_rng(11)
    i0 = np.concatenate([rng.integers(0, sizes[0], size=8192), [0, sizes[0] - 1, 0, sizes[0] - 1]])
    i1 = np.concatenate([rng.integers(0, sizes[1], size=8192), [0, 0, sizes[1] - 1, sizes[1] - 1]])
    off_a, off_b = i0 + sizes[0] * i1, i1 + sizes[1] * i0
    plan = ttc.ttc_plan(wl.F32, 2, sizes, perm)
    try:
        a_dev = torch.from_numpy(A).cuda()
        for alpha, beta in ((1.5, 0.5), (2.0, 0.0)):
            which = 1 if beta else 0
            cands = skew_candidates(plan, which)
            assert cands
            for i in cands[:3]:
                ttc.ttc_plan_select(plan, which, i)
                b_dev = torch.from_numpy(B0).cuda()
                ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
                torch.cuda.synchronize()
                got = b_dev.cpu().numpy()
                want = np.float32(alpha) * A[off_a]
                if beta:
                    want = want + np.float32(beta) * B0[off_b]
                assert np.array_equal(got[off_b], want), i
                if not beta:
                    assert np.array_equal(np.sort(got), np.sort(np.float32(alpha) * A))
            ttc.ttc_plan_select(plan, which, -1)
    finally:
        ttc.ttc_destroy(plan)
