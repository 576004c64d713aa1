/*
 * ttc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the hot path computes:
 *
 *     B_{Pi(i_0,...,i_{N-1})}  <-  alpha * A_{i_0,...,i_{N-1}}  +  beta * B_{Pi(i_0,...,i_{N-1})}
 *
 * (Eq. 1), on column-major tensors (fn 2) with one leading
 * dimension per index.  The method reaches exactly this result,
 * only faster, so the oracle is the definition written out: one odometer over the
 * multi-index (i_0 fastest), 64-bit offsets, no tiling, no index merging, no vectorisation.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call anything in this directory.  It shares no code, header, table or
 * helper with paper_1607_01249_b200/csrc/.
 *
 * Readings of the paper taken here:
 *   A1  perm[k] is the A-index that sits at position k of B, so B's k-th extent is
 *       sizes[perm[k]]  (merge example PAPER.md:63; Fig. 2; Fig. 3).
 *   A2  sizes[] is in A's index order.
 *   A3  lda[k] / ldb[k] are extents of the enclosing tensor; element strides are their
 *       running products: sA[0]=1, sA[k]=sA[k-1]*lda[k-1].
 *   A4  ldb[k] belongs to B's POSITION k (pairs with sizes[perm[k]]); paper silent.
 *   A5  beta == 0  =>  B is never read (NaN / uninitialised B must not leak).
 *   A6  no special case for alpha == 1 or alpha == 0: A is always read and multiplied.
 *   A7  every operation is one IEEE-754 round-to-nearest-even operation in the tensor's own
 *       precision, no FMA contraction (build with -ffp-contract=off, never -ffast-math).
 *   A9  complex multiply is the textbook (ar*br - ai*bi, ar*bi + ai*br), written by hand.
 *   A13 any zero extent => nothing to do.
 *   M1  mixed precision ("different data types for the input tensor A and the
 *       output tensor B", e.g. --dataType=sd: A single, B double; PAPER.md:75 lists sd, ds, cz,
 *       zc): the paper does not say in which precision Eq. 1 is evaluated.  Reading: the element
 *       of A is first converted to B's type (exact for s->d and c->z; ONE round-to-nearest-even
 *       per real component for d->s and z->c, overflow to +-inf), then Eq. 1 is evaluated in B's
 *       precision with alpha and beta scalars of B's type (ttc_oracle_transpose_mixed below).
 * Parity pins: every entry point here is pinned by tests/test_oracle_pins.py (P1-P13 of
 * SURVEY.md 8(c)); nothing is "parity unpinned".
 *
 * Return value: 0 on success, a negative number for an invalid argument (the oracle is
 * strict about its inputs so that a wrong test cannot pass silently).
 */
#include <stdint.h>
#include <stddef.h>

#define ORACLE_MAX_RANK 32

enum { ORACLE_F32 = 0, ORACLE_F64 = 1, ORACLE_C64 = 2, ORACLE_C128 = 3 };

static int check_args(int dtype, int N, const int64_t *sizes, const int *perm,
                      const int64_t *lda, const int64_t *ldb)
{
    int seen[ORACLE_MAX_RANK];
    int k;
    if (dtype < 0 || dtype > 3) return -1;
    if (N < 1 || N > ORACLE_MAX_RANK) return -2;
    if (!sizes || !perm) return -3;
    for (k = 0; k < N; ++k) seen[k] = 0;
    for (k = 0; k < N; ++k) {
        if (perm[k] < 0 || perm[k] >= N || seen[perm[k]]) return -4;
        seen[perm[k]] = 1;
    }
    for (k = 0; k < N; ++k) {
        if (sizes[k] < 0) return -5;
        if (lda && lda[k] < sizes[k]) return -6;
        if (ldb && ldb[k] < sizes[perm[k]]) return -7;
    }
    return 0;
}

/* Strides in elements.  sA[k]: stride of A's index k.  tB[k]: stride of B's position k
 * (NULL ld => contiguous). */
static void strides(int N, const int64_t *sizes, const int *perm,
                    const int64_t *lda, const int64_t *ldb, int64_t *sA, int64_t *tB)
{
    int k;
    sA[0] = 1;
    tB[0] = 1;
    for (k = 1; k < N; ++k) {
        sA[k] = sA[k - 1] * (lda ? lda[k - 1] : sizes[k - 1]);
        tB[k] = tB[k - 1] * (ldb ? ldb[k - 1] : sizes[perm[k - 1]]);
    }
}

/* Advance the odometer i (i_0 fastest).  Returns 0 when it wraps around. */
static int next_index(int N, const int64_t *sizes, int64_t *i)
{
    int k;
    for (k = 0; k < N; ++k) {
        if (++i[k] < sizes[k]) return 1;
        i[k] = 0;
    }
    return 0;
}

#define OFFSETS()                                                   \
    int64_t offA = 0, offB = 0;                                     \
    {                                                               \
        int k_;                                                     \
        for (k_ = 0; k_ < N; ++k_) offA += i[k_] * sA[k_];          \
        for (k_ = 0; k_ < N; ++k_) offB += i[perm[k_]] * tB[k_];    \
    }

/* Eq. 1.  alpha, beta: one scalar of the tensor's dtype (complex = re, im). */
int ttc_oracle_transpose(int dtype, int N, const int64_t *sizes, const int *perm,
                         const int64_t *lda, const int64_t *ldb,
                         const void *alpha, const void *A, const void *beta, void *B)
{
    int64_t sA[ORACLE_MAX_RANK], tB[ORACLE_MAX_RANK], i[ORACLE_MAX_RANK];
    int k, rc;
    rc = check_args(dtype, N, sizes, perm, lda, ldb);
    if (rc) return rc;
    if (!alpha || !beta) return -8;
    for (k = 0; k < N; ++k)
        if (sizes[k] == 0) return 0;                 /* A13: empty tensor */
    if (!A || !B) return -9;
    strides(N, sizes, perm, lda, ldb, sA, tB);
    for (k = 0; k < N; ++k) i[k] = 0;

    if (dtype == ORACLE_F32) {
        const float a = *(const float *)alpha, b = *(const float *)beta;
        const float *pa = (const float *)A;
        float *pb = (float *)B;
        do {
            OFFSETS();
            float t = a * pa[offA];
            if (b == 0.0f) {
                pb[offB] = t;                        /* A5: B not read */
            } else {
                float u = b * pb[offB];
                pb[offB] = t + u;
            }
        } while (next_index(N, sizes, i));
    } else if (dtype == ORACLE_F64) {
        const double a = *(const double *)alpha, b = *(const double *)beta;
        const double *pa = (const double *)A;
        double *pb = (double *)B;
        do {
            OFFSETS();
            double t = a * pa[offA];
            if (b == 0.0) {
                pb[offB] = t;
            } else {
                double u = b * pb[offB];
                pb[offB] = t + u;
            }
        } while (next_index(N, sizes, i));
    } else if (dtype == ORACLE_C64) {
        const float ar = ((const float *)alpha)[0], ai = ((const float *)alpha)[1];
        const float br = ((const float *)beta)[0], bi = ((const float *)beta)[1];
        const float *pa = (const float *)A;
        float *pb = (float *)B;
        do {
            OFFSETS();
            float xr = pa[2 * offA], xi = pa[2 * offA + 1];
            float p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;   /* A9 */
            float tr = p0 - p1, ti = p2 + p3;
            if (br == 0.0f && bi == 0.0f) {
                pb[2 * offB] = tr;
                pb[2 * offB + 1] = ti;
            } else {
                float yr = pb[2 * offB], yi = pb[2 * offB + 1];
                float q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                float ur = q0 - q1, ui = q2 + q3;
                pb[2 * offB] = tr + ur;
                pb[2 * offB + 1] = ti + ui;
            }
        } while (next_index(N, sizes, i));
    } else {
        const double ar = ((const double *)alpha)[0], ai = ((const double *)alpha)[1];
        const double br = ((const double *)beta)[0], bi = ((const double *)beta)[1];
        const double *pa = (const double *)A;
        double *pb = (double *)B;
        do {
            OFFSETS();
            double xr = pa[2 * offA], xi = pa[2 * offA + 1];
            double p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;
            double tr = p0 - p1, ti = p2 + p3;
            if (br == 0.0 && bi == 0.0) {
                pb[2 * offB] = tr;
                pb[2 * offB + 1] = ti;
            } else {
                double yr = pb[2 * offB], yi = pb[2 * offB + 1];
                double q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                double ur = q0 - q1, ui = q2 + q3;
                pb[2 * offB] = tr + ur;
                pb[2 * offB + 1] = ti + ui;
            }
        } while (next_index(N, sizes, i));
    }
    return 0;
}

/* Mixed precision (reading M1 in the header): A has dtype_a, B has dtype_b,
 * alpha and beta are scalars of dtype_b.  Allowed pairs: s->d, d->s, c->z, z->c; a pair of
 * equal types is Eq. 1 itself (ttc_oracle_transpose).  Any other pair (real <-> complex) is
 * rejected: the paper lists none.  The conversion is the C cast (float)x / (double)x, which
 * is IEEE-754 convertFormat under the default rounding mode. */
int ttc_oracle_transpose_mixed(int dtype_a, int dtype_b, int N, const int64_t *sizes, const int *perm,
                               const int64_t *lda, const int64_t *ldb,
                               const void *alpha, const void *A, const void *beta, void *B)
{
    int64_t sA[ORACLE_MAX_RANK], tB[ORACLE_MAX_RANK], i[ORACLE_MAX_RANK];
    int k, rc;
    if (dtype_a == dtype_b)
        return ttc_oracle_transpose(dtype_b, N, sizes, perm, lda, ldb, alpha, A, beta, B);
    if (!((dtype_a == ORACLE_F32 && dtype_b == ORACLE_F64) || (dtype_a == ORACLE_F64 && dtype_b == ORACLE_F32) ||
          (dtype_a == ORACLE_C64 && dtype_b == ORACLE_C128) || (dtype_a == ORACLE_C128 && dtype_b == ORACLE_C64)))
        return -11;
    rc = check_args(dtype_b, N, sizes, perm, lda, ldb);
    if (rc) return rc;
    if (!alpha || !beta) return -8;
    for (k = 0; k < N; ++k)
        if (sizes[k] == 0) return 0;
    if (!A || !B) return -9;
    strides(N, sizes, perm, lda, ldb, sA, tB);
    for (k = 0; k < N; ++k) i[k] = 0;

    if (dtype_b == ORACLE_F64) {                     /* sd: A float, B double */
        const double a = *(const double *)alpha, b = *(const double *)beta;
        const float *pa = (const float *)A;
        double *pb = (double *)B;
        do {
            OFFSETS();
            double x = (double)pa[offA];             /* exact */
            double t = a * x;
            if (b == 0.0) {
                pb[offB] = t;
            } else {
                double u = b * pb[offB];
                pb[offB] = t + u;
            }
        } while (next_index(N, sizes, i));
    } else if (dtype_b == ORACLE_F32) {              /* ds: A double, B float */
        const float a = *(const float *)alpha, b = *(const float *)beta;
        const double *pa = (const double *)A;
        float *pb = (float *)B;
        do {
            OFFSETS();
            float x = (float)pa[offA];               /* one rounding */
            float t = a * x;
            if (b == 0.0f) {
                pb[offB] = t;
            } else {
                float u = b * pb[offB];
                pb[offB] = t + u;
            }
        } while (next_index(N, sizes, i));
    } else if (dtype_b == ORACLE_C128) {             /* cz: A complex float, B complex double */
        const double ar = ((const double *)alpha)[0], ai = ((const double *)alpha)[1];
        const double br = ((const double *)beta)[0], bi = ((const double *)beta)[1];
        const float *pa = (const float *)A;
        double *pb = (double *)B;
        do {
            OFFSETS();
            double xr = (double)pa[2 * offA], xi = (double)pa[2 * offA + 1];
            double p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;   /* A9 */
            double tr = p0 - p1, ti = p2 + p3;
            if (br == 0.0 && bi == 0.0) {
                pb[2 * offB] = tr;
                pb[2 * offB + 1] = ti;
            } else {
                double yr = pb[2 * offB], yi = pb[2 * offB + 1];
                double q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                double ur = q0 - q1, ui = q2 + q3;
                pb[2 * offB] = tr + ur;
                pb[2 * offB + 1] = ti + ui;
            }
        } while (next_index(N, sizes, i));
    } else {                                         /* zc: A complex double, B complex float */
        const float ar = ((const float *)alpha)[0], ai = ((const float *)alpha)[1];
        const float br = ((const float *)beta)[0], bi = ((const float *)beta)[1];
        const double *pa = (const double *)A;
        float *pb = (float *)B;
        do {
            OFFSETS();
            float xr = (float)pa[2 * offA], xi = (float)pa[2 * offA + 1];
            float p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;
            float tr = p0 - p1, ti = p2 + p3;
            if (br == 0.0f && bi == 0.0f) {
                pb[2 * offB] = tr;
                pb[2 * offB + 1] = ti;
            } else {
                float yr = pb[2 * offB], yi = pb[2 * offB + 1];
                float q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                float ur = q0 - q1, ui = q2 + q3;
                pb[2 * offB] = tr + ur;
                pb[2 * offB + 1] = ti + ui;
            }
        } while (next_index(N, sizes, i));
    }
    return 0;
}

/* Eq. 1 on tensors given by explicit element strides instead of leading dimensions (the
 * optional extension of SURVEY.md 8(b): config 4 is described "with outer stride 6208"): sA[k] is the stride
 * of A's index k, tB[k] the stride of B's position k.  Same loop, same arithmetic as ttc_oracle_transpose;
 * only where the strides come from differs.  Same-type dtypes only.  Strides must be positive. */
int ttc_oracle_transpose_strided(int dtype, int N, const int64_t *sizes, const int *perm,
                                 const int64_t *sA, const int64_t *tB,
                                 const void *alpha, const void *A, const void *beta, void *B)
{
    int64_t i[ORACLE_MAX_RANK];
    int k, rc;
    rc = check_args(dtype, N, sizes, perm, NULL, NULL);
    if (rc) return rc;
    if (!alpha || !beta || !sA || !tB) return -8;
    for (k = 0; k < N; ++k)
        if (sA[k] < 1 || tB[k] < 1) return -12;
    for (k = 0; k < N; ++k)
        if (sizes[k] == 0) return 0;
    if (!A || !B) return -9;
    for (k = 0; k < N; ++k) i[k] = 0;
    if (dtype == ORACLE_F32 || dtype == ORACLE_F64) {
        do {
            OFFSETS();
            if (dtype == ORACLE_F32) {
                const float a = *(const float *)alpha, b = *(const float *)beta;
                float t = a * ((const float *)A)[offA];
                if (b == 0.0f) ((float *)B)[offB] = t;
                else { float u = b * ((float *)B)[offB]; ((float *)B)[offB] = t + u; }
            } else {
                const double a = *(const double *)alpha, b = *(const double *)beta;
                double t = a * ((const double *)A)[offA];
                if (b == 0.0) ((double *)B)[offB] = t;
                else { double u = b * ((double *)B)[offB]; ((double *)B)[offB] = t + u; }
            }
        } while (next_index(N, sizes, i));
    } else if (dtype == ORACLE_C64) {
        const float ar = ((const float *)alpha)[0], ai = ((const float *)alpha)[1];
        const float br = ((const float *)beta)[0], bi = ((const float *)beta)[1];
        const float *pa = (const float *)A;
        float *pb = (float *)B;
        do {
            OFFSETS();
            float xr = pa[2 * offA], xi = pa[2 * offA + 1];
            float p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;   /* A9 */
            float tr = p0 - p1, ti = p2 + p3;
            if (!(br == 0.0f && bi == 0.0f)) {
                float yr = pb[2 * offB], yi = pb[2 * offB + 1];
                float q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                float ur = q0 - q1, ui = q2 + q3;
                tr = tr + ur;
                ti = ti + ui;
            }
            pb[2 * offB] = tr;
            pb[2 * offB + 1] = ti;
        } while (next_index(N, sizes, i));
    } else {
        const double ar = ((const double *)alpha)[0], ai = ((const double *)alpha)[1];
        const double br = ((const double *)beta)[0], bi = ((const double *)beta)[1];
        const double *pa = (const double *)A;
        double *pb = (double *)B;
        do {
            OFFSETS();
            double xr = pa[2 * offA], xi = pa[2 * offA + 1];
            double p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;
            double tr = p0 - p1, ti = p2 + p3;
            if (!(br == 0.0 && bi == 0.0)) {
                double yr = pb[2 * offB], yi = pb[2 * offB + 1];
                double q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                double ur = q0 - q1, ui = q2 + q3;
                tr = tr + ur;
                ti = ti + ui;
            }
            pb[2 * offB] = tr;
            pb[2 * offB + 1] = ti;
        } while (next_index(N, sizes, i));
    }
    return 0;
}

/* Offsets of one logical element, exported so that tests can sample single outputs of a
 * full-size problem: element with A multi-index i[] lives at A[*offA_out] and goes to
 * B[*offB_out].  Same formulas as above (reading A1, A3, A4). */
int ttc_oracle_offsets(int N, const int64_t *sizes, const int *perm,
                       const int64_t *lda, const int64_t *ldb, const int64_t *i,
                       int64_t *offA_out, int64_t *offB_out)
{
    int64_t sA[ORACLE_MAX_RANK], tB[ORACLE_MAX_RANK];
    int k, rc;
    rc = check_args(0, N, sizes, perm, lda, ldb);
    if (rc) return rc;
    for (k = 0; k < N; ++k)
        if (i[k] < 0 || i[k] >= sizes[k]) return -10;
    strides(N, sizes, perm, lda, ldb, sA, tB);
    {
        OFFSETS();
        *offA_out = offA;
        *offB_out = offB;
    }
    return 0;
}
