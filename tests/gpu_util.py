"""Helpers of the ``-m gpu`` parity tests: run one transposition through the C ABI on cuda:0
and through the CPU oracle on the same seeded buffers, and compare bit for bit."""
import numpy as np
import torch

import oracle
from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

GUARD = 64  # guard elements before and after each device buffer


def to_dev(flat: np.ndarray, guard_fill, misalign: int = 0):
    """Copy a flat host buffer to the device between two guard bands; returns (whole, view).
    ``misalign`` shifts the payload by that many elements (pointer no longer 16-byte aligned)."""
    n = flat.size
    host = np.full(n + 2 * GUARD + misalign, guard_fill, dtype=flat.dtype)
    host[GUARD + misalign:GUARD + misalign + n] = flat
    whole = torch.from_numpy(host).cuda()
    return whole, whole[GUARD + misalign:GUARD + misalign + n]


def bits(x: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(x).view(np.uint8)


def gpu_transpose(w: wl.Workload, A: np.ndarray, B0: np.ndarray, plan=None, candidate=None,
                  misalign_a: int = 0, misalign_b: int = 0):
    """Returns (B after the GPU call as a flat host array, guards_intact)."""
    own = plan is None
    if own:
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
    try:
        which = 1 if w.beta_nonzero else 0
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, candidate)
        guard = np.array(-77.25, dtype=A.dtype)
        a_whole, a_dev = to_dev(A, guard, misalign_a)
        b_whole, b_dev = to_dev(B0, guard, misalign_b)
        ttc.ttc_execute(plan, w.alpha, a_dev, w.beta, b_dev)
        torch.cuda.synchronize()
        out = b_whole.cpu().numpy()
        lo = GUARD + misalign_b
        guards_ok = bool(np.all(out[:lo] == guard) and np.all(out[lo + B0.size:] == guard))
        a_after = a_whole.cpu().numpy()[GUARD + misalign_a:GUARD + misalign_a + A.size]
        guards_ok = guards_ok and np.array_equal(bits(a_after), bits(A))
        return out[lo:lo + B0.size].copy(), guards_ok
    finally:
        if candidate is not None:
            ttc.ttc_plan_select(plan, which, -1)
        if own:
            ttc.ttc_destroy(plan)


def oracle_transpose(w: wl.Workload, A: np.ndarray, B0: np.ndarray) -> np.ndarray:
    B = B0.copy()
    oracle.transpose(w.dtype, w.sizes, w.perm, w.lda, w.ldb, w.alpha, A, w.beta, B)
    return B


def check_bit_exact(w: wl.Workload, plan=None, candidate=None, b_init="auto", misalign_a=0, misalign_b=0):
    A = w.make_a()
    B0 = w.make_b(init=b_init)
    want = oracle_transpose(w, A, B0)
    got, guards_ok = gpu_transpose(w, A, B0, plan=plan, candidate=candidate,
                                   misalign_a=misalign_a, misalign_b=misalign_b)
    assert guards_ok, "guard band or A modified: %s cand=%s" % (w.name, candidate)
    if not np.array_equal(bits(got), bits(want)):
        bad = np.nonzero(bits(got).reshape(got.size, -1) != bits(want).reshape(want.size, -1))[0]
        raise AssertionError("%s cand=%s: %d of %d elements differ, first at %d: got %r want %r" % (
            w.name, candidate, np.unique(bad).size, got.size, bad[0], got[bad[0]], want[bad[0]]))
