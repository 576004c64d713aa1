// canon.cpp -- stage 1 of the paper's pipeline (PAPER.md:63, 95 fn 5): argument validation,
// leading dimensions -> element strides, extent-1 removal and index merging.  Host only.
#include <algorithm>

#include "ttc_internal.h"

namespace ttc {

namespace {
// a*b and a+b with overflow detection on non-negative int64 operands
inline bool mul_ok(int64_t a, int64_t b, int64_t* r) { return !__builtin_mul_overflow(a, b, r); }
inline bool add_ok(int64_t a, int64_t b, int64_t* r) { return !__builtin_add_overflow(a, b, r); }
constexpr int64_t kMaxElems = (int64_t)1 << 62;
}  // namespace

ttc_status canonicalize(int N, const int64_t* sizes, const int* perm, const int64_t* lda,
                        const int64_t* ldb, Canon* out) {
    if (!sizes || !perm || !out) return TTC_ERR_INVALID_ARG;
    if (N < 1 || N > kMaxRank) return TTC_ERR_INVALID_ARG;
    bool seen[kMaxRank] = {false};
    for (int k = 0; k < N; ++k) {
        if (perm[k] < 0 || perm[k] >= N || seen[perm[k]]) return TTC_ERR_NOT_PERMUTATION;
        seen[perm[k]] = true;
    }
    for (int k = 0; k < N; ++k)
        if (sizes[k] < 0) return TTC_ERR_INVALID_ARG;
    for (int k = 0; k < N; ++k) {
        if (lda && lda[k] < sizes[k]) return TTC_ERR_BAD_LD;
        if (ldb && ldb[k] < sizes[perm[k]]) return TTC_ERR_BAD_LD;
    }

    Canon c;
    c.numel = 1;
    for (int k = 0; k < N; ++k) {
        if (sizes[k] == 0) c.empty = true;
    }
    if (c.empty) {
        c.rank = 0;
        c.numel = 0;
        *out = c;
        return TTC_OK;
    }
    for (int k = 0; k < N; ++k) {
        if (!mul_ok(c.numel, sizes[k], &c.numel) || c.numel > kMaxElems) return TTC_ERR_UNSUPPORTED;
    }

    // Leading dimensions -> element strides (reading A3): sA[0]=1, sA[k]=sA[k-1]*lda[k-1];
    // B's strides are per POSITION (reading A4) and are carried to A's index perm[k].
    int64_t sA[kMaxRank], sB[kMaxRank];
    int64_t run = 1;
    for (int k = 0; k < N; ++k) {
        sA[k] = run;
        int64_t ld = lda ? lda[k] : sizes[k];
        if (k + 1 < N && !mul_ok(run, ld, &run)) return TTC_ERR_UNSUPPORTED;
    }
    run = 1;
    for (int k = 0; k < N; ++k) {
        sB[perm[k]] = run;
        int64_t ld = ldb ? ldb[k] : sizes[perm[k]];
        if (k + 1 < N && !mul_ok(run, ld, &run)) return TTC_ERR_UNSUPPORTED;
    }

    // Spans (1 + largest offset).  Strides of extent-1 indices matter only through the
    // strides of later indices, which are already explicit (reading A12).
    int64_t spanA = 1, spanB = 1;
    for (int k = 0; k < N; ++k) {
        int64_t t;
        if (!mul_ok(sizes[k] - 1, sA[k], &t) || !add_ok(spanA, t, &spanA)) return TTC_ERR_UNSUPPORTED;
        if (!mul_ok(sizes[k] - 1, sB[k], &t) || !add_ok(spanB, t, &spanB)) return TTC_ERR_UNSUPPORTED;
    }
    if (spanA > kMaxElems || spanB > kMaxElems) return TTC_ERR_UNSUPPORTED;
    c.spanA = spanA;
    c.spanB = spanB;

    // Drop extent-1 indices; the rest is already ascending in A-stride (lda[k] >= sizes[k] >= 2).
    int r = 0;
    for (int k = 0; k < N; ++k) {
        if (sizes[k] == 1) continue;
        c.d[r++] = CanonDim{sizes[k], sA[k], sB[k]};
    }
    // Merge d, d+1 when they are one contiguous run in A AND in B (fn 5's
    // ld(i_m) = size(i_m) has to hold in both tensors, reading A11).
    int w = 0;
    for (int k = 0; k < r; ++k) {
        if (w > 0) {
            CanonDim& p = c.d[w - 1];
            if (c.d[k].sA == p.e * p.sA && c.d[k].sB == p.e * p.sB) {
                p.e *= c.d[k].e;
                continue;
            }
        }
        c.d[w++] = c.d[k];
    }
    if (w == 0) {  // a single element
        c.d[0] = CanonDim{1, 1, 1};
        w = 1;
    }
    c.rank = w;
    for (int k = 0; k < w; ++k) c.orderB[k] = k;
    std::stable_sort(c.orderB, c.orderB + w, [&](int a, int b) { return c.d[a].sB < c.d[b].sB; });
    *out = c;
    return TTC_OK;
}

}  // namespace ttc
