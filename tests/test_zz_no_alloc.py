"""``-m gpu``: ``ttc_execute_host_static`` (include/ttc.h) -- the allocation-free variant of ``ttc_execute_host``
that stages A and B inside the library's file-scope ``__device__`` array -- against the existing paths
(``ttc_execute_host`` on host buffers and ``ttc_execute`` on device buffers), bit for bit (the tolerance the
parity tests use), on calls IN A ROW that share the array: different shapes, element types, beta == 0 with a
padded B (stale bytes of the previous call must not leak into B's padding or elements) and a candidate forced to
the atomic work distribution, whose counter lives in the array's first 256 bytes.  Collected last on purpose
(file name): the array and the module that holds it are loaded only here.
"""
import os

import numpy as np
import pytest
import torch

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import bits

pytestmark = pytest.mark.gpu

# (dtype_a, dtype_b, sizes, perm, lda, ldb, alpha, beta)
CASES = [
    (wl.F32, wl.F32, (96, 40, 64), (2, 1, 0), None, None, 1.5, 0.5),
    (wl.F64, wl.F64, (33, 9, 21), (2, 0, 1), (35, 9, 21), (24, 36, 9), -0.75, 0.0),     # beta == 0, B padded
    (wl.F32, wl.F32, (131, 67), (1, 0), None, None, 1.0, 0.0),                          # smaller than the call before
    (wl.C64, wl.C64, (20, 12, 10, 6), (3, 1, 0, 2), None, None, 0.5 - 0.25j, 0.25 + 1j),
    (wl.F64, wl.F32, (48, 50, 30), (1, 2, 0), None, None, 1.25, -0.5),                  # ds: narrowing pair
    (wl.F32, wl.F32, (96, 40, 64), (2, 1, 0), None, None, 1.5, 0.5),                    # the first one again
]


def buffers(da, db, sizes, perm, lda, ldb, k):
    n = int(np.prod(sizes))
    szb = tuple(sizes[p] for p in perm)
    A = wl.embed(wl.uniform_values(wl.SEED_A + k, n, da), sizes, lda)
    B = wl.embed(wl.uniform_values(wl.SEED_B + k, n, db), szb, ldb)
    return A, B


def existing_paths(plan, alpha, A, beta, B0):
    """B after ttc_execute_host and after ttc_execute: the two existing paths (they agree bit for bit)."""
    b_host = B0.copy()
    ttc.ttc_execute_host(plan, alpha, A, beta, b_host)
    b_dev = torch.from_numpy(B0.copy()).cuda()
    ttc.ttc_execute(plan, alpha, torch.from_numpy(A).cuda(), beta, b_dev)
    torch.cuda.synchronize()
    assert np.array_equal(bits(b_host), bits(b_dev.cpu().numpy()))
    return b_host


def test_static_scratch_matches_the_existing_paths_call_after_call():
    plans = [ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb) for da, db, sizes, perm, lda, ldb, _, _ in CASES]
    try:
        for rnd in range(2):                      # every case twice, back to back, on fresh inputs
            for k, (case, plan) in enumerate(zip(CASES, plans)):
                da, db, sizes, perm, lda, ldb, alpha, beta = case
                A, B0 = buffers(da, db, sizes, perm, lda, ldb, 10 * rnd + k)
                want = existing_paths(plan, alpha, A, beta, B0)
                got = B0.copy()
                a_before = A.copy()
                launches = ttc.ttc_launch_count()
                ttc.ttc_execute_host_static(plan, alpha, A, beta, got)
                assert ttc.ttc_launch_count() - launches == 1
                assert np.array_equal(bits(got), bits(want)), "case %d round %d" % (k, rnd)
                assert np.array_equal(bits(A), bits(a_before))
    finally:
        for p in plans:
            ttc.ttc_destroy(p)


def test_static_scratch_allocates_no_device_memory():
    da, db, sizes, perm, lda, ldb, alpha, beta = CASES[0]
    plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    try:
        A, B0 = buffers(da, db, sizes, perm, lda, ldb, 77)
        want = existing_paths(plan, alpha, A, beta, B0)
        got = B0.copy()
        ttc.ttc_execute_host_static(plan, alpha, A, beta, got)       # loads the module that holds the array
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for _ in range(2):
            got = B0.copy()
            ttc.ttc_execute_host_static(plan, alpha, A, beta, got)
            assert np.array_equal(bits(got), bits(want))
        assert torch.cuda.mem_get_info()[0] == free0
    finally:
        ttc.ttc_destroy(plan)


def test_static_scratch_atomic_counter_candidates():
    """Candidates with the atomic work distribution (sched == 2) take their tile counter from the array."""
    old = os.environ.get("TTC_SCHED")
    os.environ["TTC_SCHED"] = "all"
    try:
        da, db, sizes, perm, lda, ldb, alpha, beta = CASES[0]
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    finally:
        if old is None:
            del os.environ["TTC_SCHED"]
        else:
            os.environ["TTC_SCHED"] = old
    try:
        picked = {}
        for i in range(ttc.ttc_plan_num_candidates(plan, 1)):
            c = ttc.ttc_plan_candidate(plan, 1, i)
            if c.sched == 2:
                picked.setdefault(c.kernel, i)
        assert picked, "no atomic-sched candidate"
        for rep, idx in enumerate(list(picked.values()) * 2):          # each of them twice in a row
            A, B0 = buffers(da, db, sizes, perm, lda, ldb, 200 + rep)
            ttc.ttc_plan_select(plan, 1, idx)
            want = existing_paths(plan, alpha, A, beta, B0)
            got = B0.copy()
            ttc.ttc_execute_host_static(plan, alpha, A, beta, got)
            assert np.array_equal(bits(got), bits(want)), "candidate %d" % idx
    finally:
        ttc.ttc_destroy(plan)


def test_static_scratch_rejects_what_does_not_fit():
    limit = ttc.TTC_STATIC_SCRATCH_BYTES
    # 1024 x 1025 fp32: A and B are 4.2 MB each -> 8.4 MB > 8 MiB
    plan = ttc.ttc_plan(wl.F32, 2, (1024, 1025), (1, 0))
    try:
        A = np.zeros(1024 * 1025, dtype=np.float32)
        B = np.full(1024 * 1025, 3.0, dtype=np.float32)
        assert 2 * A.nbytes > limit
        with pytest.raises(ttc.TTCError) as err:
            ttc.ttc_execute_host_static(plan, 1.0, A, 0.0, B)
        assert err.value.status == ttc.TTC_ERR_SCRATCH_LIMIT and "TTC_ERR_SCRATCH_LIMIT" in str(err.value)
        assert np.all(B == 3.0)                                       # nothing touched
        ttc.ttc_execute_host(plan, 1.0, A, 0.0, B)                    # the allocating path takes it
        assert np.all(B == 0.0)
    finally:
        ttc.ttc_destroy(plan)
    # the boundary: 256 + round256(|A|) + round256(|B|) <= the limit.  32767 x 32 fp32 is 4194176 bytes a side, which
    # rounds up to 4 MiB: one 256-byte block too many; 16383 x 64 (4194048 bytes a side) is the largest that fits
    plan = ttc.ttc_plan(wl.F32, 2, (32767, 32), (1, 0))
    try:
        A = np.zeros(32767 * 32, dtype=np.float32)
        assert 256 + 2 * A.nbytes == limit
        with pytest.raises(ttc.TTCError) as err:
            ttc.ttc_execute_host_static(plan, 1.0, A, 0.0, A.copy())
        assert err.value.status == ttc.TTC_ERR_SCRATCH_LIMIT
    finally:
        ttc.ttc_destroy(plan)
    n = 16383 * 64
    plan = ttc.ttc_plan(wl.F32, 2, (16383, 64), (1, 0))
    try:
        A = wl.uniform_values(wl.SEED_A, n, wl.F32)
        B0 = wl.uniform_values(wl.SEED_B, n, wl.F32)
        assert 256 + 2 * A.nbytes == limit - 256
        want = existing_paths(plan, 2.0, A, 1.0, B0)
        got = B0.copy()
        ttc.ttc_execute_host_static(plan, 2.0, A, 1.0, got)
        assert np.array_equal(bits(got), bits(want))
    finally:
        ttc.ttc_destroy(plan)
    empty = ttc.ttc_plan(wl.F64, 2, (0, 5), (1, 0))
    ttc.ttc_execute_host_static(empty, 1.0, 0, 0.0, 0)                # empty tensors: no-op whatever the pointers
    ttc.ttc_destroy(empty)
