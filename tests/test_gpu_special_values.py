"""``-m gpu``: IEEE-754 special values through every kernel class of the CUDA path.

Readings A7/A10 say: no FTZ, every product and sum rounded once, so subnormals, signed
zeros and infinities among the *logical* elements of A and B must come out of ``direct_kernel``,
``tile_kernel`` and ``ring_kernel`` (bulk rows, cp.async rows, peeled store phase, transposing
micro-tile) exactly as the oracle computes them.  Reading M1 says the narrowing pairs ds/zc convert
with ONE round-to-nearest-even (ties to even, overflow to +-inf, gradual underflow): the hand-derived
boundary inputs of pin MP2 (tests/test_oracle_mixed_pins.py) are fed to the kernels here.

NaN: where the oracle's result is a NaN the GPU's must be a NaN too (which NaN -- sign and payload --
is not fixed by IEEE-754 for an arithmetic result, and x86 and the GPU differ there); every other
element is compared bit for bit.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1607_01249_b200 import ttc
from paper_1607_01249_b200 import workloads as wl

from gpu_util import GUARD, to_dev

pytestmark = pytest.mark.gpu

NP = wl.NP_DTYPE
REAL = {wl.F32: np.float32, wl.F64: np.float64, wl.C64: np.float32, wl.C128: np.float64}
ALL_DTYPES = (wl.F32, wl.F64, wl.C64, wl.C128)


def specials(real):
    fi = np.finfo(real)
    tiny_sub = np.nextafter(real(0), real(1))           # smallest subnormal
    return np.array([tiny_sub, -tiny_sub, 3 * tiny_sub, fi.tiny - tiny_sub, fi.tiny, -fi.tiny,
                     np.inf, -np.inf, -0.0, 0.0, np.nan, fi.max, -fi.max, 1.0, -1.0,
                     real(1) + fi.eps, real(1) - fi.eps / 2], dtype=real)


def plant(vals: np.ndarray, dtype: int, rng) -> np.ndarray:
    """Overwrite ~6 % of the real components of ``vals`` (logical elements) with special values."""
    real = REAL[dtype]
    flat = vals.view(real).copy()
    sp = specials(real)
    k = max(sp.size * 2, flat.size // 16)
    pos = rng.choice(flat.size, size=min(k, flat.size), replace=False)
    flat[pos] = sp[np.arange(pos.size) % sp.size]
    return flat.view(NP[dtype])


def assert_same(got: np.ndarray, want: np.ndarray, what: str):
    real = got.real.dtype
    g, w = np.ascontiguousarray(got).view(real), np.ascontiguousarray(want).view(real)
    nan_w = np.isnan(w)
    assert np.array_equal(np.isnan(g), nan_w), "%s: NaN positions differ" % what
    u = np.uint32 if real == np.float32 else np.uint64
    gb, wb = g.view(u), w.view(u)
    bad = np.nonzero((gb != wb) & ~nan_w)[0]
    assert bad.size == 0, "%s: %d components differ, first %d: got %r (%#x) want %r (%#x)" % (
        what, bad.size, bad[0], g[bad[0]], gb[bad[0]], w[bad[0]], wb[bad[0]])


def pick_candidates(plan, which):
    """One candidate index per kernel flavour the plan has."""
    out = {}
    for i in range(ttc.ttc_plan_num_candidates(plan, which)):
        c = ttc.ttc_plan_candidate(plan, which, i)
        if c.kernel == 1:
            key = "direct_vec" if c.vec_a > 1 else "direct_scalar"
        elif c.kernel == 5 and c.flags & 1:
            key = "ring_staggered"
        elif c.kernel == 5 and c.flags & 4:
            key = "ring_shifted_peeled" if c.vec_b > 1 else "ring_shifted"
        elif c.kernel == 5:
            if c.vec_a > 1:
                key = "ring_bulk_vec" if c.vec_b > 1 else "ring_bulk_scalar"
            else:
                key = "ring_cpasync_peeled" if c.vec_b > 1 else "ring_cpasync"
        elif c.kernel == 6:
            key = "tma"
        else:
            key = "tile_%d%d" % (int(c.vec_a > 1), int(c.vec_b > 1))
        out.setdefault(key, i)
    return out


def run_case(da, db, sizes, perm, lda, ldb, alpha, beta, a_vals, b_vals, need=()):
    szb = tuple(sizes[p] for p in perm)
    A = wl.embed(a_vals, sizes, lda)
    B0 = wl.embed(b_vals, szb, ldb)
    want = B0.copy()
    if da == db:
        oracle.transpose(db, sizes, perm, lda, ldb, alpha, A, beta, want)
        plan = ttc.ttc_plan(db, len(sizes), sizes, perm, lda, ldb)
    else:
        oracle.transpose_mixed(da, db, sizes, perm, lda, ldb, alpha, A, beta, want)
        plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    which = 1 if complex(beta) != 0 else 0
    try:
        cands = pick_candidates(plan, which)
        for k in need:
            if db == wl.C128:             # 16-byte elements: every access is one element (vec = 1); ring rows are still bulk copies
                k = {"ring_bulk_vec": "ring_cpasync", "direct_vec": "direct_scalar"}.get(k, k)
            assert k in cands, "no %s candidate for %s %s" % (k, sizes, perm)
        for key, idx in list(cands.items()) + [("winner", -1)]:
            ttc.ttc_plan_select(plan, which, idx)
            _, a_dev = to_dev(A, np.array(-77.25, dtype=A.dtype))
            b_whole, b_dev = to_dev(B0, np.array(-77.25, dtype=B0.dtype))
            ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
            torch.cuda.synchronize()
            got = b_whole.cpu().numpy()[GUARD:GUARD + B0.size]
            # padding of B is NaN on both sides and untouched; logical elements per the rule above
            assert_same(got, want, "%s dtype %d->%d %s %s alpha=%r beta=%r" % (key, da, db, sizes, perm, alpha, beta))
        return set(cands)
    finally:
        ttc.ttc_destroy(plan)


SHAPES = [
    # aligned rows: direct, tile and bulk-row ring candidates (several tiles, ragged tail on index 1)
    ((64, 25, 48), (2, 1, 0), None, None, ("direct_scalar", "ring_bulk_vec")),
    # odd extents: rows not 16-byte aligned -> cp.async rows and the peeled store phase
    ((131, 9, 67), (2, 0, 1), None, None, ("direct_scalar",)),
    # copy class with leading dimensions
    ((48, 7, 10), (0, 2, 1), (52, 7, 10), (48, 12, 7), ("direct_vec",)),
]


@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("shape", SHAPES, ids=["aligned", "odd", "copy"])
def test_special_values_same_type(dtype, shape):
    sizes, perm, lda, ldb, need = shape
    n = int(np.prod(sizes))
    rng = np.random.default_rng(1607 + dtype)
    a_vals = plant(wl.uniform_values(wl.SEED_A, n, dtype), dtype, rng)
    b_vals = plant(wl.uniform_values(wl.SEED_B, n, dtype), dtype, rng)
    cplx = dtype >= 2
    scal = [(1.0, 0.0), (-0.5, 0.0), (1.5, 0.5), (-0.0, 0.0)]
    if cplx:
        scal += [(0.5 - 0.25j, 0.0), (0.75 - 1.25j, 0.5 + 0.375j)]
    seen = set()
    for alpha, beta in scal:
        seen |= run_case(dtype, dtype, sizes, perm, lda, ldb, alpha, beta, a_vals, b_vals, need)
    if shape[0][0] == 131 and dtype != wl.C128:
        assert "ring_cpasync" in seen and "ring_cpasync_peeled" in seen, seen
        assert "ring_shifted" in seen and "ring_shifted_peeled" in seen, seen
    if shape[0][0] == 64 and dtype != wl.C128:
        assert "ring_staggered" in seen, seen


MP2_INPUTS = [1.0 + 2.0 ** -24, 1.0 + 2.0 ** -24 + 2.0 ** -50, 1.0 + 3 * 2.0 ** -24, 1.0 - 2.0 ** -25,
              -(1.0 + 2.0 ** -24 + 2.0 ** -50), 3.5e38, -3.5e38, 2.0 ** -150, 2.0 ** -150 + 2.0 ** -200,
              1.5 * 2.0 ** -149, 0.1, -(2.0 ** -150), np.finfo(np.float32).max * (1 + 2.0 ** -25),
              np.finfo(np.float32).max * (1 + 2.0 ** -24), 2.0 ** -126 - 2.0 ** -150, 5e-324, -0.0, np.inf, -np.inf, np.nan]
MP2_WANT = [1.0, 1.0 + 2.0 ** -23, 1.0 + 2.0 ** -22, 1.0, -(1.0 + 2.0 ** -23), np.inf, -np.inf, 0.0, 2.0 ** -149,
            2.0 ** -148, float.fromhex("0x1.99999ap-4")]


@pytest.mark.parametrize("da,db", [(wl.F64, wl.F32), (wl.C128, wl.C64), (wl.F32, wl.F64), (wl.C64, wl.C128)])
@pytest.mark.parametrize("shape", SHAPES[:2] + [SHAPES[2]], ids=["aligned", "odd", "copy"])
def test_special_values_mixed(da, db, shape):
    """Narrowing (ds, zc): MP2's hand-derived ties / overflow / subnormal inputs through every kernel
    flavour; widening (sd, cz): subnormal floats become normal doubles exactly."""
    sizes, perm, lda, ldb, _ = shape
    n = int(np.prod(sizes))
    rng = np.random.default_rng(75 + da)
    a_vals = wl.uniform_values(wl.SEED_A, n, da)
    ra = a_vals.view(REAL[da]).copy()
    if da in (wl.F64, wl.C128):
        ra *= 1.0 + 2.0 ** -30                     # make the narrowing inexact almost everywhere
        pos = rng.choice(ra.size, size=len(MP2_INPUTS) * 8, replace=False)
        ra[pos] = np.array(MP2_INPUTS, dtype=np.float64)[np.arange(pos.size) % len(MP2_INPUTS)]
        a_vals = ra.view(NP[da])
    else:
        a_vals = plant(a_vals, da, rng)
    b_vals = plant(wl.uniform_values(wl.SEED_B, n, db), db, rng)
    for alpha, beta in [(1.0, 0.0), (1.5, 0.5)]:
        run_case(da, db, sizes, perm, lda, ldb, alpha, beta, a_vals, b_vals, ("direct_scalar",))


def test_mp2_values_on_the_gpu_in_closed_form():
    """The expected fp32 values of pin MP2 themselves (hand-derived, no oracle involved): rank-1 ds copy."""
    a = np.array(MP2_INPUTS[:len(MP2_WANT)], dtype=np.float64)
    want = np.array(MP2_WANT, dtype=np.float32)
    plan = ttc.ttc_plan_mixed(wl.F64, wl.F32, 1, (a.size,), (0,))
    try:
        for i in range(ttc.ttc_plan_num_candidates(plan, 0)):
            ttc.ttc_plan_select(plan, 0, i)
            b_dev = torch.full((a.size,), 7.0, dtype=torch.float32, device="cuda")
            ttc.ttc_execute(plan, 1.0, torch.from_numpy(a).cuda(), 0.0, b_dev)
            torch.cuda.synchronize()
            assert np.array_equal(b_dev.cpu().numpy().view(np.uint32), want.view(np.uint32)), i
    finally:
        ttc.ttc_destroy(plan)
