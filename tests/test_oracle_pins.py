"""Pins for the CPU oracle (``oracle/ttc_oracle.c``): what the paper and the mathematics fix.

Nothing here compares the oracle with itself or with the CUDA path.  Each pin is P<n> of
SURVEY.md section 8(c) / DESIGN.md "Oracle pins"; the passage of PAPER.md it rests on is
cited at the test.  All of this runs on CPU in seconds (``-m "not gpu"``).
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from paper_1607_01249_b200 import workloads as wl

NP = wl.NP_DTYPE
ALL_DTYPES = (wl.F32, wl.F64, wl.C64, wl.C128)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_examples.txt")


# ----------------------------------------------------------------------------- helpers
def buf_len(sizes, ld):
    return int(np.prod(wl.padded_extents(sizes, ld), dtype=np.int64))


def sizes_b(sizes, perm):
    return tuple(sizes[p] for p in perm)


def small_int_values(n, dtype, seed):
    """Small integers (exact in every dtype, products and sums stay exact)."""
    rng = np.random.default_rng(seed)
    re = rng.integers(-8, 9, size=n).astype(np.float64)
    if dtype in (wl.C64, wl.C128):
        im = rng.integers(-8, 9, size=n).astype(np.float64)
        return (re + 1j * im).astype(NP[dtype])
    return re.astype(NP[dtype])


def random_ld(rng, extents):
    return tuple(int(e + rng.integers(0, 4)) for e in extents)


def run(dtype, sizes, perm, lda, ldb, alpha, beta, a_vals, b_vals=None, b_fill=np.nan):
    """Embed logical values, call the oracle, return (flat B buffer, logical B values)."""
    A = wl.embed(a_vals, sizes, lda)
    szb = sizes_b(sizes, perm)
    if b_vals is None:
        b_vals = np.full(int(np.prod(sizes, dtype=np.int64)), b_fill, dtype=NP[dtype])
    B = wl.embed(b_vals, szb, ldb)
    oracle.transpose(dtype, sizes, perm, lda, ldb, alpha, A, beta, B)
    return B, wl.extract(B, szb, ldb)


def read_golden():
    rows = {}
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, perm, sizes, lda, ldb, order, cite = [c.strip() for c in line.split("|")]
            ints = lambda s: None if s == "-" else tuple(int(x) for x in s.split(","))
            rows[name] = dict(perm=ints(perm), sizes=ints(sizes), lda=ints(lda), ldb=ints(ldb),
                              order=tuple(int(x[1:]) for x in order.split(",")), cite=cite)
    return rows


# ------------------------------------------------------------- P1: index-encoding closed form
@pytest.mark.parametrize("dtype", [wl.F32, wl.F64])
@pytest.mark.parametrize("sizes,perm", [
    ((5, 3, 4), (1, 2, 0)), ((5, 3, 4), (2, 0, 1)), ((4, 3, 2, 5), (3, 1, 0, 2)),
    ((2, 3, 4, 3, 2), (4, 2, 0, 3, 1)), ((3, 2, 2, 3, 2, 2), (5, 2, 0, 4, 1, 3)), ((7,), (0,)),
])
@pytest.mark.parametrize("padded", [False, True])
def test_p1_index_encoding(dtype, sizes, perm, padded):
    """Eq. 1 with alpha=1, beta=0.  A holds the logical linear index L(i);
    every position of B is then decoded from B's OWN offset (mixed radix of ldb, reading A4)
    and must hold L of the A-index that Pi places there (reading A1); padding stays NaN."""
    rng = np.random.default_rng(1)
    n = len(sizes)
    szb = sizes_b(sizes, perm)
    lda = random_ld(rng, sizes) if padded else None
    ldb = random_ld(rng, szb) if padded else None
    numel = int(np.prod(sizes))
    B, _ = run(dtype, sizes, perm, lda, ldb, 1.0, 0.0, np.arange(numel, dtype=NP[dtype]), b_fill=-1.0)
    ext_b = wl.padded_extents(szb, ldb)
    j = np.unravel_index(np.arange(B.size), ext_b, order="F")       # position of every B slot
    logical = np.ones(B.size, dtype=bool)
    for k in range(n):
        logical &= j[k] < szb[k]
    L = np.zeros(B.size, dtype=np.int64)
    for k in range(n):                 # j[k] is the value of A-index perm[k]
        weight = int(np.prod(sizes[:perm[k]], dtype=np.int64))
        L += j[k].astype(np.int64) * weight
    assert np.array_equal(B[logical], L[logical].astype(NP[dtype]))
    assert np.isnan(B[~logical]).all()


# ------------------------------------------------------------- P2: exact permutation
@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_p2_exact_permutation_multiset(dtype):
    """alpha=1, beta=0 is an ordinary out-of-place transposition: B's logical
    elements are A's bit patterns, permuted; B's padding is not written."""
    sizes, perm = (6, 5, 4, 3), (2, 0, 3, 1)
    w = wl.Workload("t", dtype, sizes, perm, lda=(8, 5, 6, 3), ldb=(4, 9, 3, 6))
    A = w.make_a()
    B = np.frombuffer(np.full(buf_len(w.sizes_b, w.ldb) * A.itemsize, 0xA5, dtype=np.uint8).tobytes(),
                      dtype=A.dtype).copy()
    before = B.copy()
    oracle.transpose(dtype, sizes, perm, w.lda, w.ldb, 1.0, A, 0.0, B)
    word = np.uint32 if A.itemsize // (2 if dtype >= 2 else 1) == 4 else np.uint64
    a_bits = np.sort(wl.extract(A, sizes, w.lda).view(word))
    b_bits = np.sort(wl.extract(B, w.sizes_b, w.ldb).view(word))
    assert np.array_equal(a_bits, b_bits)
    mask = wl.embed(np.zeros(w.numel, dtype=A.dtype), w.sizes_b, w.ldb, fill=1.0).real.astype(bool)
    assert np.array_equal(B.view(np.uint8).reshape(B.size, -1)[mask],
                          before.view(np.uint8).reshape(B.size, -1)[mask])


# ------------------------------------------------------------- P3: identity permutation
@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("padded", [False, True])
def test_p3_identity_is_axpby(dtype, padded):
    """Identity Pi: Eq. 1 is B <- alpha*A + beta*B element by element.  Small
    integer data and scalars make every product and sum exact, so Python's own complex
    arithmetic is the expected value (pins signs and operands of the complex product, A9)."""
    sizes = (4, 3, 5)
    perm = (0, 1, 2)
    lda = (6, 3, 7) if padded else None
    ldb = (4, 5, 5) if padded else None
    n = int(np.prod(sizes))
    a = small_int_values(n, dtype, 3)
    b = small_int_values(n, dtype, 4)
    alpha, beta = (2 - 3j, -1 + 2j) if dtype >= 2 else (3.0, -2.0)
    _, got = run(dtype, sizes, perm, lda, ldb, alpha, beta, a, b)
    want = np.array([alpha * complex(x) + beta * complex(y) for x, y in zip(a, b)])
    if dtype < 2:
        want = want.real
    assert np.array_equal(got, want.astype(NP[dtype]))


def test_p3_beta_zero_never_reads_b():
    """Reading A5: with beta = 0, NaN in B must not leak."""
    for dtype in ALL_DTYPES:
        a = small_int_values(24, dtype, 5)
        _, got = run(dtype, (2, 3, 4), (1, 2, 0), None, None, 2.0, 0.0, a, b_fill=np.nan)
        assert not np.isnan(got).any()


def test_p3_separate_roundings_no_fma():
    """Reading A7: alpha*a and beta*b are rounded separately, then added (no contraction).
    Values chosen so that fused and unfused evaluation differ in the last bit."""
    a = np.array([1.0 + 3 * 2.0**-23], dtype=np.float32)
    b = np.array([-1.0], dtype=np.float32)
    alpha, beta = np.float32(1.0 + 3 * 2.0**-23), np.float32(1.0)
    _, got = run(wl.F32, (1,), (0,), None, None, alpha, beta, a, b)
    prod = np.float32(alpha * a[0])                       # rounded product
    unfused = np.float32(prod + np.float32(beta * b[0]))
    fused = np.float32(float(alpha) * float(a[0]) + float(beta) * float(b[0]))   # exact in fp64
    assert unfused != fused
    assert got[0] == unfused


# ------------------------------------------------------------- P4: Pi then Pi^-1
@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_p4_inverse_roundtrip(dtype):
    sizes, perm = (5, 4, 3, 6), (3, 0, 2, 1)
    n = len(sizes)
    w = wl.Workload("t", dtype, sizes, perm)
    A = w.make_a()
    B = np.zeros_like(A)
    oracle.transpose(dtype, sizes, perm, None, None, 1.0, A, 0.0, B)
    inv = [0] * n
    for k in range(n):
        inv[perm[k]] = k
    C = np.zeros_like(A)
    oracle.transpose(dtype, w.sizes_b, inv, None, None, 1.0, B, 0.0, C)
    assert np.array_equal(A.view(np.uint8), C.view(np.uint8))
    assert not np.array_equal(A, B)


# ------------------------------------------------------------- P5: 2-D textbook transpose
@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_p5_matrix_transpose_bruteforce(dtype):
    m, n = 7, 5
    a = wl.uniform_values(11, m * n, dtype)
    _, got = run(dtype, (m, n), (1, 0), None, None, 1.0, 0.0, a)
    want = np.empty_like(a)
    for i in range(m):
        for j in range(n):
            want[j + n * i] = a[i + m * j]
    assert np.array_equal(got, want)


# ------------------------------------------------------------- P6: the paper's merge example
def test_p6_merge_example_from_paper():
    """Pi(i0,i1,i2)=(i1,i2,i0) is the 2-D transposition Pi(i0,i1)=(i1,i0) with
    size(i1) := size(i1)*size(i2).  Only true if perm[k] is the A-index at B position k (A1)."""
    g = read_golden()["sec21_merge"]
    s0, s1, s2 = g["sizes"]
    a = wl.uniform_values(12, s0 * s1 * s2, wl.F64)
    _, got3 = run(wl.F64, g["sizes"], g["perm"], None, None, 1.0, 0.0, a)
    want = np.ascontiguousarray(a.reshape((s0, s1 * s2), order="F").T).reshape(-1, order="F")
    assert np.array_equal(got3, want)
    # config 1's permutation (2,0,1) is the 2-D transpose of the (s0*s1) x s2 matrix
    _, got = run(wl.F64, (s0, s1, s2), (2, 0, 1), None, None, 1.0, 0.0, a)
    want = np.ascontiguousarray(a.reshape((s0 * s1, s2), order="F").T).reshape(-1, order="F")
    assert np.array_equal(got, want)
    assert not np.array_equal(got, got3)


# ------------------------------------------------------------- P7: Fig. 2 sub-tensor pack
def test_p7_fig2_subtensor_pack():
    """perm=2,1,0 size=8,16,16 lda=32,32,32 packs a sub-tensor of a 32^3
    tensor into contiguous B_{i2,i1,i0}: B[i2 + 16 i1 + 256 i0] = A[i0 + 32 i1 + 1024 i2]."""
    g = read_golden()["fig2_subtensor_pack"]
    assert g["perm"] == (2, 1, 0) and g["sizes"] == (8, 16, 16) and g["lda"] == (32, 32, 32)
    big = np.full(32 * 32 * 16, np.nan)                 # enclosing tensor, last index cut at 16
    vals = {}
    rng = np.random.default_rng(7)
    for i0 in range(8):
        for i1 in range(16):
            for i2 in range(16):
                v = float(rng.integers(1, 1 << 30))
                big[i0 + 32 * i1 + 1024 * i2] = v
                vals[(i0, i1, i2)] = v
    B = np.full(8 * 16 * 16, np.nan)
    oracle.transpose(wl.F64, g["sizes"], g["perm"], g["lda"], g["ldb"], 1.0, big, 0.0, B)
    assert not np.isnan(B).any()
    for (i0, i1, i2), v in vals.items():
        assert B[i2 + 16 * i1 + 256 * i0] == v


# ------------------------------------------------------------- P8: Fig. 3 / config 4 packing
@pytest.mark.parametrize("mr,npanel,K,lda2d", [(4, 6, 5, 24), (4, 6, 5, 28), (8, 3, 7, 32), (6, 4, 5, 30), (16, 2, 3, 48)])
def test_p8_blas_panel_pack(mr, npanel, K, lda2d):
    """A_{m,k} viewed as A_{m1,m2,k}, perm=0,2,1 -> B_{m1,k,m2}.
    Stated on the 2-D matrix alone: B[i + mr*(k + K*p)] = A2d[(i + mr*p) + lda2d*k]."""
    M = mr * npanel
    A2d = np.full(lda2d * K, np.nan)
    rng = np.random.default_rng(8)
    for k in range(K):
        A2d[lda2d * k: lda2d * k + M] = rng.integers(-99, 100, size=M)
    if lda2d % mr == 0:
        lda = (mr, lda2d // mr, K)
    else:
        pytest.skip("outer stride not expressible as a leading dimension (SURVEY 8(b) note)")
    B = np.full(M * K, np.nan)
    oracle.transpose(wl.F64, (mr, npanel, K), (0, 2, 1), lda, None, 1.0, A2d, 0.0, B)
    assert not np.isnan(B).any()
    for p in range(npanel):
        for k in range(K):
            for i in range(mr):
                assert B[i + mr * (k + K * p)] == A2d[(i + mr * p) + lda2d * k]


@pytest.mark.parametrize("nr", [4, 6, 8, 16])
@pytest.mark.parametrize("dtype", [wl.F64, wl.F32])
def test_p8b_blas_b_panel_pack_and_batched(nr, dtype):
    """The other half of a GEMM's packing pair (BLIS-style B panels of nr columns): the
    K x N matrix M (column-major, leading dimension ldm) viewed as the 3-D tensor M_{k,n1,n2} with sizes
    (K, nr, N/nr) and leading dimensions (ldm, nr, .), perm = (1,0,2) -> P_{n1,k,n2}.  Stated on the 2-D
    matrix alone: P[j + nr*(k + K*q)] = M[k + ldm*(j + nr*q)].  Rows k >= K of M (padding) are NaN and must
    not be read.  Then the batched form: several blocks in one call is the same loop block by block."""
    K, npanel, ldm = 7, 3, 9
    N = nr * npanel
    rng = np.random.default_rng(80 + nr)

    def block():
        M = np.full(ldm * N, np.nan, dtype=NP[dtype])
        for n in range(N):
            M[ldm * n: ldm * n + K] = rng.integers(-99, 100, size=K)
        return M
    blocks = [block() for _ in range(3)]
    packed = [np.full(N * K, np.nan, dtype=NP[dtype]) for _ in blocks]
    oracle.transpose_batched(dtype, (K, nr, npanel), (1, 0, 2), (ldm, nr, npanel), None, 1.0, blocks, 0.0, packed)
    for M, P in zip(blocks, packed):
        assert not np.isnan(P).any()
        for q in range(npanel):
            for k in range(K):
                for j in range(nr):
                    assert P[j + nr * (k + K * q)] == M[k + ldm * (j + nr * q)]
    with pytest.raises(ValueError):
        oracle.transpose_batched(dtype, (K, nr, npanel), (1, 0, 2), None, None, 1.0, blocks, 0.0, packed[:2])


# ------------------------------------------------------------- P9: library routine
@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_p9_numpy_transpose(dtype, n):
    """Column-major A with extents s: numpy's transpose(axes=perm) on the Fortran-order
    array is the same permutation (out[j] = in[i], i[perm[k]] = j[k]); ld via embed/extract."""
    rng = np.random.default_rng(100 + n)
    for trial in range(6):
        sizes = tuple(int(x) for x in rng.integers(1, 6, size=n))
        perm = tuple(int(x) for x in rng.permutation(n))
        lda = random_ld(rng, sizes) if trial % 2 else None
        ldb = random_ld(rng, sizes_b(sizes, perm)) if trial % 3 else None
        a = wl.uniform_values(trial, int(np.prod(sizes)), dtype)
        _, got = run(dtype, sizes, perm, lda, ldb, 1.0, 0.0, a)
        want = np.transpose(a.reshape(sizes, order="F"), perm).reshape(-1, order="F")
        assert np.array_equal(got, want)


@pytest.mark.parametrize("dtype", [wl.F32, wl.C64, wl.F64])
@pytest.mark.parametrize("n", [10, 16])
def test_p9_numpy_transpose_high_rank(dtype, n):
    """P9 at rank 10 and at the library's maximum rank 16 (extents 1..3, with and without leading
    dimensions, general alpha/beta by small integers): the oracle is the checker of the GPU's
    ``test_high_rank``, so it is pinned at those ranks too.  P1's closed form at the same ranks."""
    rng = np.random.default_rng(1000 + n)
    for trial in range(4):
        sizes = tuple(int(x) for x in rng.choice([1, 2, 2, 3], size=n))
        perm = tuple(int(x) for x in rng.permutation(n))
        szb = sizes_b(sizes, perm)
        lda = tuple(int(e + rng.integers(0, 2)) for e in sizes) if trial % 2 else None
        ldb = tuple(int(e + rng.integers(0, 2)) for e in szb) if trial >= 2 else None
        numel = int(np.prod(sizes))
        a = small_int_values(numel, dtype, trial)
        b0 = small_int_values(numel, dtype, 50 + trial)
        _, got = run(dtype, sizes, perm, lda, ldb, 2.0, -3.0, a, b0)
        want = 2 * np.transpose(a.reshape(sizes, order="F"), perm).reshape(-1, order="F") - 3 * b0
        assert np.array_equal(got, want.astype(NP[dtype]))
        # P1: A holds its logical linear index; B decoded from its own position
        if dtype == wl.F64:
            _, gotL = run(dtype, sizes, perm, lda, ldb, 1.0, 0.0, np.arange(numel, dtype=np.float64))
            j = np.unravel_index(np.arange(numel), szb, order="F")
            L = np.zeros(numel, dtype=np.int64)
            for k in range(n):
                L += j[k].astype(np.int64) * int(np.prod(sizes[:perm[k]], dtype=np.int64))
            assert np.array_equal(gotL, L.astype(np.float64))


# ------------------------------------------------------------- P9s: explicit strides
@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_p9s_strided_oracle_against_numpy_as_strided(dtype):
    """``ttc_oracle_transpose_strided`` (explicit element strides; SURVEY.md 8(b) optional extension): A and B
    are numpy ``as_strided`` views of flat buffers -- numpy does the addressing -- and the result must be
    ``B_view = 2*transpose(A_view) - 3*B_view`` (small integers: exact).  Includes config 4's description, an
    outer stride (6208-like) that is NOT a multiple of the inner ones, and A indices given out of stride order."""
    from numpy.lib.stride_tricks import as_strided
    rng = np.random.default_rng(99)
    isz = np.dtype(NP[dtype]).itemsize
    for sizes, perm, sa, sb in (((4, 3, 5), (0, 2, 1), (1, 4, 13), (1, 4, 20)),          # outer stride 13 = 4*3 + 1
                                ((3, 4, 2), (1, 0, 2), (8, 1, 30), (1, 5, 17)),          # A's index 1 is the stride-1 one
                                ((2, 3, 2, 2), (3, 1, 0, 2), (1, 2, 7, 15), (1, 3, 10, 21))):
        span_a = 1 + sum((e - 1) * s for e, s in zip(sizes, sa))
        szb = sizes_b(sizes, perm)
        span_b = 1 + sum((e - 1) * s for e, s in zip(szb, sb))
        A = small_int_values(span_a, dtype, 7)
        B = small_int_values(span_b, dtype, 8)
        B0 = B.copy()
        av = as_strided(A, shape=sizes, strides=[s * isz for s in sa])
        want = B0.copy()
        bv = as_strided(want, shape=szb, strides=[s * isz for s in sb])
        bv[...] = 2 * np.transpose(av, perm) - 3 * bv
        oracle.transpose_strided(dtype, sizes, perm, sa, sb, 2.0, A, -3.0, B)
        assert np.array_equal(B, want)
        # and it agrees with the leading-dimension oracle where both can describe the tensors
    sizes, perm, lda, ldb = (3, 4, 5), (2, 0, 1), (4, 6, 5), (5, 3, 4)
    A = small_int_values(4 * 6 * 5, dtype, 1)
    B1 = small_int_values(5 * 3 * 4, dtype, 2)
    B2 = B1.copy()
    oracle.transpose(dtype, sizes, perm, lda, ldb, 2.0, A, -3.0, B1)
    oracle.transpose_strided(dtype, sizes, perm, (1, 4, 24), (1, 5, 15), 2.0, A, -3.0, B2)
    assert np.array_equal(B1, B2)


# ------------------------------------------------------------- P10: linearity
@pytest.mark.parametrize("dtype", ALL_DTYPES)
def test_p10_linearity(dtype):
    """result(alpha, beta) = alpha (x) result(1, 0) (+) beta (x) B0, each op rounded once in the
    tensor's precision; numpy scalar ops in that precision give the same roundings for reals,
    and the hand-written 4-mul/2-add product (A9) is retyped here with numpy arrays."""
    sizes, perm = (6, 4, 5), (2, 0, 1)
    n = int(np.prod(sizes))
    a = wl.uniform_values(21, n, dtype)
    b0 = wl.uniform_values(22, n, dtype)
    alpha, beta = (1.5 - 0.75j, 0.3 + 0.2j) if dtype >= 2 else (1.7, -0.3)
    _, perm_only = run(dtype, sizes, perm, None, None, 1.0, 0.0, a)
    _, got = run(dtype, sizes, perm, None, None, alpha, beta, a, b0)
    T = NP[dtype]
    if dtype < 2:
        al, be = T(alpha), T(beta)
        want = (al * perm_only).astype(T) + (be * b0).astype(T)
    else:
        R = np.float32 if dtype == wl.C64 else np.float64
        def cmul(s, x):
            sr, si = R(s.real), R(s.imag)
            xr, xi = x.real.astype(R), x.imag.astype(R)
            return (sr * xr - si * xi).astype(R), (sr * xi + si * xr).astype(R)
        tr, ti = cmul(complex(alpha), perm_only)
        ur, ui = cmul(complex(beta), b0)
        want = ((tr + ur).astype(R) + 1j * (ti + ui).astype(R)).astype(T)
    assert np.array_equal(got.view(np.uint8), want.view(np.uint8))


# ------------------------------------------------------------- P11: composition
def test_p11_composition():
    sizes = (3, 4, 5, 2)
    p1, p2 = (2, 0, 3, 1), (1, 3, 0, 2)
    a = wl.uniform_values(31, int(np.prod(sizes)), wl.F32)
    _, b1 = run(wl.F32, sizes, p1, None, None, 1.0, 0.0, a)
    _, b2 = run(wl.F32, sizes_b(sizes, p1), p2, None, None, 1.0, 0.0, b1)
    comp = tuple(p1[p2[k]] for k in range(4))
    _, direct = run(wl.F32, sizes, comp, None, None, 1.0, 0.0, a)
    assert np.array_equal(b2, direct)


# ------------------------------------------------------------- P12: padding and guard bands
@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("beta", [0.0, 0.5])
def test_p12_padding_untouched_and_never_read(dtype, beta):
    sizes, perm = (5, 3, 4), (2, 0, 1)
    lda, ldb = (7, 5, 4), (6, 8, 3)
    guard = 16
    w = wl.Workload("t", dtype, sizes, perm, 2.0, beta, lda, ldb)
    A = np.concatenate([np.full(guard, np.nan, NP[dtype]), w.make_a(), np.full(guard, np.nan, NP[dtype])])
    Bcore = w.make_b(init="uniform")
    sentinel = NP[dtype](-12345.0)
    Bcore[np.isnan(Bcore)] = sentinel                  # padding of B: recognisable, comparable
    B = np.concatenate([np.full(guard, sentinel), Bcore, np.full(guard, sentinel)]).astype(NP[dtype])
    before = B.copy()
    oracle.transpose(dtype, sizes, perm, lda, ldb, 2.0, A[guard:-guard], beta, B[guard:-guard])
    logical = wl.embed(np.ones(w.numel, NP[dtype]), w.sizes_b, ldb, fill=0.0).real.astype(bool)
    full = np.concatenate([np.zeros(guard, bool), logical, np.zeros(guard, bool)])
    assert np.array_equal(B[~full], before[~full])       # padding + guards bit-identical
    assert not np.isnan(B[full]).any()                   # NaN padding of A never read into B
    assert not np.array_equal(B[full], before[full])


# ------------------------------------------------------------- P13: brute force, tiny, exhaustive
def _brute(dtype, sizes, perm, lda, ldb, alpha, beta, A, B):
    """Pure-Python restatement with Horner-form addresses (enclosing extents nested), scalar
    numpy arithmetic in the tensor's precision."""
    T = NP[dtype]
    R = {wl.F32: np.float32, wl.F64: np.float64, wl.C64: np.float32, wl.C128: np.float64}[dtype]
    n = len(sizes)
    ea = lda if lda is not None else sizes
    szb = [sizes[p] for p in perm]
    eb = ldb if ldb is not None else szb
    out = B.copy()
    for idx in itertools.product(*[range(s) for s in sizes]):
        oa = 0
        for k in reversed(range(n)):
            oa = oa * ea[k] + idx[k] if k < n - 1 else idx[k]
        ob = 0
        for k in reversed(range(n)):
            jk = idx[perm[k]]
            ob = ob * eb[k] + jk if k < n - 1 else jk
        x = A[oa]
        if dtype < 2:
            t = R(R(alpha) * x)
            out[ob] = t if beta == 0 else R(t + R(R(beta) * B[ob]))
        else:
            al, be = complex(alpha), complex(beta)
            def cm(s, v):
                return (R(R(R(s.real) * R(v.real)) - R(R(s.imag) * R(v.imag))),
                        R(R(R(s.real) * R(v.imag)) + R(R(s.imag) * R(v.real))))
            tr, ti = cm(al, x)
            if be != 0:
                ur, ui = cm(be, B[ob])
                tr, ti = R(tr + ur), R(ti + ui)
            out[ob] = T(complex(tr, ti))
    return out


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_p13_bruteforce_all_perms(n):
    rng = np.random.default_rng(1300 + n)
    pool = (1, 2, 3, 5, 7) if n <= 3 else (1, 2, 3, 5)
    case = 0
    for perm in itertools.permutations(range(n)):
        for rep in range(3 if n <= 3 else 1):
            sizes = tuple(int(rng.choice(pool)) for _ in range(n))
            szb = sizes_b(sizes, perm)
            lda = random_ld(rng, sizes) if case % 2 else None
            ldb = random_ld(rng, szb) if case % 3 else None
            dtype = ALL_DTYPES[case % 4]
            beta = 0.0 if (case // 4) % 2 == 0 else (0.75 if dtype < 2 else 0.75 - 0.5j)
            alpha = 1.25 if dtype < 2 else 1.25 + 0.5j
            case += 1
            w = wl.Workload("t", dtype, sizes, perm, alpha, beta, lda, ldb)
            A = w.make_a(seed=case)
            B0 = w.make_b(seed=case + 1, init="uniform")
            B0[np.isnan(B0)] = -7.0
            B = B0.copy()
            oracle.transpose(dtype, sizes, perm, lda, ldb, alpha, A, beta, B)
            want = _brute(dtype, sizes, perm, lda, ldb, alpha, beta, A, B0)
            assert np.array_equal(B.view(np.uint8), want.view(np.uint8)), (dtype, sizes, perm, lda, ldb, beta)


def test_p13_rank5_and_6_sampled():
    rng = np.random.default_rng(1356)
    for n in (5, 6):
        for _ in range(12):
            perm = tuple(int(x) for x in rng.permutation(n))
            sizes = tuple(int(rng.choice((1, 2, 3))) for _ in range(n))
            w = wl.Workload("t", wl.C64, sizes, perm, 0.5 - 0.25j, 1.0 + 1.0j,
                            random_ld(rng, sizes), random_ld(rng, sizes_b(sizes, perm)))
            A = w.make_a()
            B0 = w.make_b(init="uniform")
            B0[np.isnan(B0)] = 3.0
            B = B0.copy()
            oracle.transpose(wl.C64, sizes, perm, w.lda, w.ldb, w.alpha, A, w.beta, B)
            want = _brute(wl.C64, sizes, perm, w.lda, w.ldb, w.alpha, w.beta, A, B0)
            assert np.array_equal(B.view(np.uint8), want.view(np.uint8))


# ------------------------------------------------------------- oracle housekeeping
def test_zero_extent_is_noop_and_bad_args_rejected():
    B = np.full(4, 9.0)
    oracle.transpose(wl.F64, (2, 0, 3), (1, 0, 2), None, None, 1.0, np.zeros(1), 0.0, B)   # A13
    assert np.all(B == 9.0)
    with pytest.raises(ValueError):
        oracle.transpose(wl.F64, (2, 2), (0, 0), None, None, 1.0, np.zeros(4), 0.0, np.zeros(4))
    with pytest.raises(ValueError):
        oracle.transpose(wl.F64, (2, 2), (1, 0), (1, 2), None, 1.0, np.zeros(4), 0.0, np.zeros(4))
    with pytest.raises(ValueError):   # ldb pairs with B's position k (A4): sizes_b = (3, 2)
        oracle.transpose(wl.F64, (2, 3), (1, 0), None, (2, 3), 1.0, np.zeros(6), 0.0, np.zeros(6))


def test_offsets_helper_matches_definition():
    """oracle.offsets is used to sample single outputs of full-size problems: pin it on Fig. 2."""
    oa, ob = oracle.offsets((8, 16, 16), (2, 1, 0), (32, 32, 32), None, (3, 5, 7))
    assert (oa, ob) == (3 + 32 * 5 + 1024 * 7, 7 + 16 * 5 + 256 * 3)


@pytest.mark.parametrize("dtype", ALL_DTYPES)
@pytest.mark.parametrize("beta", [0.0, 0.5])
def test_paper_reference_loop_agrees(dtype, beta):
    """The paper's OpenMP reference loop nest, used as a second timed CPU
    baseline, computes the same thing as the definition."""
    w = wl.Workload("t", dtype, (9, 7, 5, 3), (2, 0, 3, 1), 1.5, beta, (10, 7, 6, 3), (5, 11, 3, 8))
    A = w.make_a()
    B0 = w.make_b(init="uniform")
    B0[np.isnan(B0)] = 1.0
    B1, B2 = B0.copy(), B0.copy()
    oracle.transpose(dtype, w.sizes, w.perm, w.lda, w.ldb, w.alpha, A, beta, B1)
    oracle.ref_omp_transpose(dtype, w.sizes, w.perm, w.lda, w.ldb, w.alpha, A, beta, B2)
    assert np.array_equal(B1.view(np.uint8), B2.view(np.uint8))
    assert oracle.ref_omp_threads() >= 1
    # the timed baseline: same source built with the BASELINE.md flags on this machine, arrays first-touched in parallel
    A3, B3 = oracle.first_touch_copy(A), oracle.first_touch_copy(B0)
    assert np.array_equal(A3.view(np.uint8), A.view(np.uint8))
    oracle.ref_omp_native_transpose(dtype, w.sizes, w.perm, w.lda, w.ldb, w.alpha, A3, beta, B3)
    assert np.array_equal(B1.view(np.uint8), B3.view(np.uint8))
    assert "-O3" in oracle.NATIVE_FLAGS and "-march=native" in oracle.NATIVE_FLAGS and "-fopenmp" in oracle.NATIVE_FLAGS
    assert not oracle.first_touch_zeros(A).view(np.uint8).any()


def test_generators_hold_no_nan_and_are_exact():
    for dtype in ALL_DTYPES:
        v = wl.uniform_values(wl.SEED_A, 1000, dtype)
        assert np.isfinite(v.view(np.float32 if dtype in (wl.F32, wl.C64) else np.float64)).all()
        assert v.real.min() >= -1.0 and v.real.max() < 1.0
    a = wl.uniform_values(5, 10, wl.F32)
    b = wl.uniform_values(5, 20, wl.F32)
    assert np.array_equal(a, b[:10])                     # counter-based: prefix-stable
