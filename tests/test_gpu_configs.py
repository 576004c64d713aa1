"""``-m gpu``: BASELINE.json's five configs at FULL size, in the launch configuration bench.py
times (the tuned winner of a default ttc_plan), against the CPU oracle on the whole tensor
(the oracle needs ~0.2-1 s per config, so no sampling is needed), plus the properties that
hold at any size (exact-permutation multiset, NaN padding never read, guards intact)."""
import numpy as np
import pytest

from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import bits, check_bit_exact, gpu_transpose, oracle_transpose

pytestmark = pytest.mark.gpu


def test_config1_bit_exact():
    check_bit_exact(wl.config1())


@pytest.mark.parametrize("perm", wl.config2_perms(), ids=lambda p: "".join(map(str, p)))
def test_config2_bit_exact(perm):
    check_bit_exact(wl.config2(perm))


def test_config3_bit_exact_and_tolerance():
    """alpha=1.5, beta=0.5: bit-exact because the kernels never contract to FMA (reading A7);
    the contractual bound of north_star (reading A8: relative to |alpha||a|+|beta||b|,
    2^-22 for fp32) is asserted as well."""
    w = wl.config3()
    A, B0 = w.make_a(), w.make_b()
    want = oracle_transpose(w, A, B0)
    got, guards_ok = gpu_transpose(w, A, B0)
    assert guards_ok
    # tolerance form (A8): magnitude from the oracle's own inputs, permuted by the oracle
    one = wl.Workload("mag", w.dtype, w.sizes, w.perm, abs(w.alpha), abs(w.beta))
    mag = oracle_transpose(one, np.abs(A), np.abs(B0))
    assert np.all(np.abs(got.astype(np.float64) - want) <= 2.0 ** -22 * mag.astype(np.float64))
    assert np.array_equal(bits(got), bits(want))


def test_config4_packing_no_nan():
    """Fig. 3 packing: NaN padding rows of A must never reach B."""
    w = wl.config4()
    A, B0 = w.make_a(), w.make_b()
    assert np.isnan(A).sum() == (6208 - 6144) * 4096
    want = oracle_transpose(w, A, B0)
    got, guards_ok = gpu_transpose(w, A, B0)
    assert guards_ok
    assert not np.isnan(got).any()
    assert np.array_equal(bits(got), bits(want))
    # independent restatement P8: B[i0 + 8*(k + 4096*p)] = A[(i0 + 8*p) + 6208*k]
    rng = np.random.default_rng(4)
    i0, p, k = rng.integers(0, 8, 4096), rng.integers(0, 768, 4096), rng.integers(0, 4096, 4096)
    assert np.array_equal(got[i0 + 8 * (k + 4096 * p)], A[(i0 + 8 * p) + 6208 * k])


def test_config5_bit_exact():
    check_bit_exact(wl.config5())


def test_config1_beta_nonzero_and_nan_b():
    w = wl.config1()
    check_bit_exact(w, b_init="nan")
    check_bit_exact(wl.Workload("c1b", w.dtype, w.sizes, w.perm, -0.75, 1.25))


def test_config2_top_candidates_full_size():
    """The 8 best-ranked candidates of three c2 permutations (2-D, 3-D and 4-D canonical
    forms) at full size, so that the tuner can never pick an unverified kernel shape."""
    for perm in [(2, 3, 0, 1), (3, 1, 2, 0), (1, 3, 0, 2)]:
        w = wl.config2(perm)
        A, B0 = w.make_a(), w.make_b()
        want = oracle_transpose(w, A, B0)
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
        try:
            for i in range(min(8, ttc.ttc_plan_num_candidates(plan, 0))):
                got, ok = gpu_transpose(w, A, B0, plan=plan, candidate=i)
                assert ok and np.array_equal(bits(got), bits(want)), (perm, i)
        finally:
            ttc.ttc_destroy(plan)


def test_exact_permutation_multiset_full_size():
    """P2 at full size, no oracle involved: alpha=1, beta=0 permutes bit patterns."""
    w = wl.config2((3, 1, 0, 2))
    A, B0 = w.make_a(), w.make_b()
    got, _ = gpu_transpose(w, A, B0)
    assert np.array_equal(np.sort(A.view(np.uint64)), np.sort(got.view(np.uint64)))
