/*
 * ttc_ref_omp.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * The paper's own *reference implementation* (the denominator of its Fig. 6), restated
 * from PAPER.md:167: "d perfectly nested loops annotated with #pragma omp parallel for
 * collapse(d-1) on the outermost loop, as well as #pragma omp simd on the innermost loop;
 * moreover, the loops are ordered such that the output tensor B is accessed in a perfectly
 * linear fashion".  With N a run-time value the d-1 collapsed outer loops are written as
 * one parallel loop over the collapsed iteration space (what collapse(d-1) itself does),
 * decoded with div/mod in B's position order; the innermost loop runs over B's position 0.
 *
 * It is reported by bench.py as a second, multi-threaded CPU number next to the oracle and
 * is itself checked against ttc_oracle_transpose in tests/test_oracle_pins.py.  Same
 * arithmetic conventions as the oracle (separate roundings, hand-written complex multiply,
 * B not read when beta == 0); real dtypes only need `re`, complex are handled as pairs.
 */
#include <stdint.h>
#include <stddef.h>

#define REF_MAX_RANK 32

#define REF_LOOP(T, ...)                                                               \
    _Pragma("omp parallel for schedule(static)")                                       \
    for (int64_t outer = 0; outer < n_outer; ++outer) {                                \
        int64_t rem = outer, offA0 = 0, offB0 = 0;                                     \
        for (int k = 1; k < N; ++k) {                                                  \
            int64_t j = rem % szB[k];                                                  \
            rem /= szB[k];                                                             \
            offA0 += j * sAofB[k];                                                     \
            offB0 += j * tB[k];                                                        \
        }                                                                              \
        const T *pa = (const T *)A;                                                    \
        T *pb = (T *)B;                                                                \
        _Pragma("omp simd")                                                            \
        for (int64_t j0 = 0; j0 < n_inner; ++j0) {                                     \
            const int64_t oa = offA0 + j0 * s_inner, ob = offB0 + j0;                  \
            __VA_ARGS__                                                                \
        }                                                                              \
    }

int ttc_ref_omp_transpose(int dtype, int N, const int64_t *sizes, const int *perm,
                          const int64_t *lda, const int64_t *ldb,
                          const void *alpha, const void *A, const void *beta, void *B)
{
    int64_t sA[REF_MAX_RANK], tB[REF_MAX_RANK], szB[REF_MAX_RANK], sAofB[REF_MAX_RANK];
    int64_t n_outer = 1, n_inner, s_inner;
    if (dtype < 0 || dtype > 3 || N < 1 || N > REF_MAX_RANK) return -1;
    sA[0] = 1;
    tB[0] = 1;
    for (int k = 1; k < N; ++k) {
        sA[k] = sA[k - 1] * (lda ? lda[k - 1] : sizes[k - 1]);
        tB[k] = tB[k - 1] * (ldb ? ldb[k - 1] : sizes[perm[k - 1]]);
    }
    for (int k = 0; k < N; ++k) {
        szB[k] = sizes[perm[k]];           /* extent of B's position k            */
        sAofB[k] = sA[perm[k]];            /* stride in A of the index sitting there */
        if (szB[k] == 0) return 0;
    }
    for (int k = 1; k < N; ++k) n_outer *= szB[k];
    n_inner = szB[0];
    s_inner = sAofB[0];

    if (dtype == 0) {
        const float a = *(const float *)alpha, b = *(const float *)beta;
        if (b == 0.0f) { REF_LOOP(float, pb[ob] = a * pa[oa];) }
        else { REF_LOOP(float, { float t = a * pa[oa]; float u = b * pb[ob]; pb[ob] = t + u; }) }
    } else if (dtype == 1) {
        const double a = *(const double *)alpha, b = *(const double *)beta;
        if (b == 0.0) { REF_LOOP(double, pb[ob] = a * pa[oa];) }
        else { REF_LOOP(double, { double t = a * pa[oa]; double u = b * pb[ob]; pb[ob] = t + u; }) }
    } else if (dtype == 2) {
        const float ar = ((const float *)alpha)[0], ai = ((const float *)alpha)[1];
        const float br = ((const float *)beta)[0], bi = ((const float *)beta)[1];
        const int bz = (br == 0.0f && bi == 0.0f);
        REF_LOOP(float, {
            float xr = pa[2 * oa], xi = pa[2 * oa + 1];
            float p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;
            float tr = p0 - p1, ti = p2 + p3;
            if (!bz) {
                float yr = pb[2 * ob], yi = pb[2 * ob + 1];
                float q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                float ur = q0 - q1, ui = q2 + q3;
                tr = tr + ur; ti = ti + ui;
            }
            pb[2 * ob] = tr; pb[2 * ob + 1] = ti;
        })
    } else {
        const double ar = ((const double *)alpha)[0], ai = ((const double *)alpha)[1];
        const double br = ((const double *)beta)[0], bi = ((const double *)beta)[1];
        const int bz = (br == 0.0 && bi == 0.0);
        REF_LOOP(double, {
            double xr = pa[2 * oa], xi = pa[2 * oa + 1];
            double p0 = ar * xr, p1 = ai * xi, p2 = ar * xi, p3 = ai * xr;
            double tr = p0 - p1, ti = p2 + p3;
            if (!bz) {
                double yr = pb[2 * ob], yi = pb[2 * ob + 1];
                double q0 = br * yr, q1 = bi * yi, q2 = br * yi, q3 = bi * yr;
                double ur = q0 - q1, ui = q2 + q3;
                tr = tr + ur; ti = ti + ui;
            }
            pb[2 * ob] = tr; pb[2 * ob + 1] = ti;
        })
    }
    return 0;
}

/* Parallel copy with the same static schedule as the loop nest: a freshly mmap'ed destination is
 * thereby FIRST TOUCHED by the threads that will use it (the arrays of the
 * paper's measurements are initialised in parallel).  No arithmetic of the method in here. */
void ttc_ref_omp_parallel_copy(void *dst, const void *src, int64_t bytes)
{
    const int64_t chunk = 1 << 20;
    const int64_t n = (bytes + chunk - 1) / chunk;
    _Pragma("omp parallel for schedule(static)")
    for (int64_t c = 0; c < n; ++c) {
        const int64_t lo = c * chunk, hi = lo + chunk < bytes ? lo + chunk : bytes;
        for (int64_t i = lo; i < hi; ++i) ((unsigned char *)dst)[i] = src ? ((const unsigned char *)src)[i] : 0;
    }
}

int ttc_ref_omp_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
