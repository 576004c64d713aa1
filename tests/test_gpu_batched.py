"""``-m gpu``: ttc_execute_batched and the GEMM packing pair
against the oracle (``oracle.transpose_batched`` = the single-pair definition applied pair by pair; pins P8,
P8b in tests/test_oracle_pins.py), bit for bit, every kernel class forced through the batched launch."""
import numpy as np
import pytest
import torch

import oracle
from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import bits

pytestmark = pytest.mark.gpu
NP = wl.NP_DTYPE


def run_batched(da, db, sizes, perm, lda, ldb, alpha, beta, batch, plan=None, candidate=None, views=False):
    """``views``: all blocks live in ONE big device buffer (as the blocks of a GEMM operand do)."""
    n = int(np.prod(sizes))
    szb = tuple(sizes[p] for p in perm)
    As = [wl.embed(wl.uniform_values(wl.SEED_A + i, n, da), sizes, lda) for i in range(batch)]
    Bs = [wl.embed(wl.uniform_values(wl.SEED_B + i, n, db), szb, ldb) for i in range(batch)]
    want = [b.copy() for b in Bs]
    if da == db:
        oracle.transpose_batched(db, sizes, perm, lda, ldb, alpha, As, beta, want)
    else:
        for a, w in zip(As, want):
            oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, alpha, a, beta, w)
    own = plan is None
    if own:
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    which = 1 if complex(beta) != 0 else 0
    try:
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, candidate)
        if views:
            la, lb = As[0].size + 4, Bs[0].size + 4        # 4 elements between blocks: stays 16-byte aligned
            big_a = torch.full((batch * la,), -7.0, dtype=torch.from_numpy(As[0]).dtype, device="cuda")
            big_b = torch.full((batch * lb,), -7.0, dtype=torch.from_numpy(Bs[0]).dtype, device="cuda")
            a_dev = [big_a[i * la:i * la + As[0].size] for i in range(batch)]
            b_dev = [big_b[i * lb:i * lb + Bs[0].size] for i in range(batch)]
            for d, h in zip(a_dev, As):
                d.copy_(torch.from_numpy(h))
            for d, h in zip(b_dev, Bs):
                d.copy_(torch.from_numpy(h))
        else:
            a_dev = [torch.from_numpy(a).cuda() for a in As]
            b_dev = [torch.from_numpy(b).cuda() for b in Bs]
        launches = ttc.ttc_launch_count()
        ttc.ttc_execute_batched(plan, alpha, a_dev, beta, b_dev)
        torch.cuda.synchronize()
        assert ttc.ttc_launch_count() - launches == (batch + 63) // 64      # ONE launch per 64 pairs
        for i in range(batch):
            got = b_dev[i].cpu().numpy()
            assert np.array_equal(bits(got), bits(want[i])), "pair %d of %d, candidate %s" % (i, batch, candidate)
        if views:     # nothing written between the blocks
            gaps = big_b.cpu().numpy().reshape(batch, lb)[:, Bs[0].size:]
            assert np.all(gaps == -7.0)
    finally:
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, -1)
        if own:
            ttc.ttc_destroy(plan)


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64, wl.C128])
@pytest.mark.parametrize("beta", [0.0, 0.5])
def test_batched_every_kernel_class(dtype, beta):
    """One candidate of every kernel flavour (direct, tile, ring bulk / staggered / shifted / peeled), 5 pairs."""
    for sizes, perm, lda, ldb in (((40, 18, 24), (2, 1, 0), None, None), ((33, 9, 21), (2, 0, 1), (35, 9, 21), None)):
        plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm, lda, ldb)
        try:
            which = 1 if beta else 0
            seen = {}
            for i in range(ttc.ttc_plan_num_candidates(plan, which)):
                c = ttc.ttc_plan_candidate(plan, which, i)
                seen.setdefault((c.kernel, c.flags, c.vec_a > 1, c.vec_b > 1), i)
            assert len(seen) >= 3
            for idx in seen.values():
                run_batched(dtype, dtype, sizes, perm, lda, ldb, 1.5, beta, 5, plan=plan, candidate=idx)
            run_batched(dtype, dtype, sizes, perm, lda, ldb, 1.5, beta, 5, plan=plan)        # the tuned winner
        finally:
            ttc.ttc_destroy(plan)


@pytest.mark.parametrize("dtype", [wl.F32, wl.F64, wl.C64, wl.C128])
@pytest.mark.parametrize("beta", [0.0, 0.5])
def test_batched_tensormap_candidates(dtype, beta):
    """Tensor-map candidates serve a batch through ONE pair of maps (the batch offset is the fifth map coordinate, stride
    16 bytes) when the canonical rank is <= 4: transposing and copy-class flavours, blocks of one big buffer and separately
    allocated tensors, 1 .. 70 pairs; a rank-5 plan's tensor-map candidates are replaced (their fifth dimension is taken)."""
    for sizes, perm, lda, ldb in (((40, 20, 24), (2, 1, 0), None, None), ((48, 12, 20), (0, 2, 1), (52, 12, 20), None),
                                  ((36, 8, 12, 20), (3, 1, 0, 2), None, None)):
        plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm, lda, ldb)
        try:
            which = 1 if beta else 0
            tm = [i for i in range(ttc.ttc_plan_num_candidates(plan, which)) if ttc.ttc_plan_candidate(plan, which, i).kernel == 6]
            assert tm
            for idx in tm[:3]:
                for batch, views in ((5, True), (3, False), (70, True)):
                    run_batched(dtype, dtype, sizes, perm, lda, ldb, 1.5, beta, batch, plan=plan, candidate=idx, views=views)
        finally:
            ttc.ttc_destroy(plan)
    sizes, perm = (20, 4, 12, 8, 16), (4, 2, 0, 3, 1)          # rank 5: no free map dimension
    plan = ttc.ttc_plan(dtype, 5, sizes, perm)
    try:
        which = 1 if beta else 0
        tm = [i for i in range(ttc.ttc_plan_num_candidates(plan, which)) if ttc.ttc_plan_candidate(plan, which, i).kernel == 6]
        assert tm
        run_batched(dtype, dtype, sizes, perm, None, None, 1.5, beta, 4, plan=plan, candidate=tm[0], views=True)
    finally:
        ttc.ttc_destroy(plan)


def test_batch_sizes_and_edge_cases():
    sizes, perm = (24, 10, 12), (1, 2, 0)
    for batch in (1, 2, 63, 64, 65, 130):
        run_batched(wl.F32, wl.F32, sizes, perm, None, None, 1.0, 0.0, batch, views=True)
    plan = ttc.ttc_plan(wl.F32, 3, sizes, perm)
    ttc.ttc_execute_batched(plan, 1.0, [], 0.0, [])                 # batch == 0: no-op
    assert ttc.lib.ttc_execute_batched(plan, None, None, None, None, 2, None) == 1          # TTC_ERR_INVALID_ARG
    one = np.ones(1, dtype=np.float32)
    assert ttc.lib.ttc_execute_batched(plan, one.ctypes.data, None, one.ctypes.data, None, -1, None) == 1
    ttc.ttc_destroy(plan)
    empty = ttc.ttc_plan(wl.F64, 2, (0, 5), (1, 0))
    ttc.ttc_execute_batched(empty, 1.0, [0, 0], 0.0, [0, 0])        # empty tensors: no-op whatever the pointers
    ttc.ttc_destroy(empty)


@pytest.mark.parametrize("mr", [4, 6, 8, 16])
@pytest.mark.parametrize("pair", [(wl.F64, wl.F64), (wl.F32, wl.F64), (wl.F64, wl.F32)], ids=["d", "sd", "ds"])
def test_gemm_packing_pair_batched(mr, pair):
    """A-panel pack (Fig. 3: M_{m1,m2,k} -> P_{m1,k,m2}) and B-panel pack (M_{k,n1,n2} -> P_{n1,k,n2})
    of mc x kc / kc x nc blocks of a padded matrix, 6 blocks per call, for register-block sizes mr = nr in
    {4, 6, 8, 16}, fp64 and the mixed pairs sd / ds (mixed-precision BLAS through packing)."""
    da, db = pair
    kc, panels, ld_extra = 40, 5, 3
    mc = mr * panels
    # A block: mc x kc inside a matrix with leading dimension mc + mr*ld_extra (a multiple of mr)
    run_batched(da, db, (mr, panels, kc), (0, 2, 1), (mr, panels + ld_extra, kc), None, 1.0, 0.0, 6, views=True)
    # B block: kc x nc, nc = mr*panels, leading dimension kc + 5
    run_batched(da, db, (kc, mr, panels), (1, 0, 2), (kc + 5, mr, panels), None, 1.0, 0.0, 6, views=True)


def test_batched_full_size_small_packs():
    """The shape bench.py --detail times: 256 A-panel packs of 8 x 32 x 1024 fp64 (2 MB each) in 4 launches."""
    run_batched(wl.F64, wl.F64, (8, 32, 1024), (0, 2, 1), (8, 40, 1024), None, 1.0, 0.0, 256, views=True)
