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

namespace {
// Stage 1 proper, on explicit element strides per A-index: spans, extent-1 removal, ascending A-stride,
// merging (PAPER.md:63, 95 fn 5), B order.
ttc_status canon_from_strides(int N, const int64_t* sizes, const int64_t* sA, const int64_t* sB, Canon c, Canon* out) {
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

    // Drop extent-1 indices; order by ascending A-stride (already so when the strides come from leading
    // dimensions: lda[k] >= sizes[k] >= 2).
    int r = 0;
    for (int k = 0; k < N; ++k) {
        if (sizes[k] == 1) continue;
        c.d[r++] = CanonDim{sizes[k], sA[k], sB[k]};
    }
    std::stable_sort(c.d, c.d + r, [](const CanonDim& x, const CanonDim& y) { return x.sA < y.sA; });
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

    return canon_from_strides(N, sizes, sA, sB, c, out);
}

// ttc_plan_strided: explicit element strides, stride_a[k] of A's index k, stride_b[k] of B's POSITION k.
// Accepted layouts are the "nested" ones -- sorted by stride, every stride is at least the previous stride
// times the previous extent -- which is what makes the offsets of B injective (and is all a leading-dimension
// description can express, plus outer strides that are not multiples of the inner ones).
ttc_status canonicalize_strided(int N, const int64_t* sizes, const int* perm, const int64_t* stride_a,
                                const int64_t* stride_b, Canon* out) {
    if (!sizes || !perm || !stride_a || !stride_b || !out) return TTC_ERR_INVALID_ARG;
    if (N < 1 || N > kMaxRank) return TTC_ERR_INVALID_ARG;
    bool seen[kMaxRank] = {false};
    for (int k = 0; k < N; ++k) {
        if (perm[k] < 0 || perm[k] >= N || seen[perm[k]]) return TTC_ERR_NOT_PERMUTATION;
        seen[perm[k]] = true;
    }
    for (int k = 0; k < N; ++k)
        if (sizes[k] < 0) return TTC_ERR_INVALID_ARG;
    Canon c;
    c.numel = 1;
    for (int k = 0; k < N; ++k)
        if (sizes[k] == 0) c.empty = true;
    if (c.empty) {
        c.rank = 0;
        c.numel = 0;
        *out = c;
        return TTC_OK;
    }
    for (int k = 0; k < N; ++k)
        if (!mul_ok(c.numel, sizes[k], &c.numel) || c.numel > kMaxElems) return TTC_ERR_UNSUPPORTED;
    int64_t sA[kMaxRank], sB[kMaxRank];
    for (int k = 0; k < N; ++k) {
        if (stride_a[k] < 1 || stride_b[k] < 1) return TTC_ERR_BAD_LD;
        sA[k] = stride_a[k];
        sB[perm[k]] = stride_b[k];
    }
    // nestedness of each side (indices of extent 1 do not take part)
    for (int side = 0; side < 2; ++side) {
        const int64_t* st = side ? sB : sA;
        int idx[kMaxRank], n = 0;
        for (int k = 0; k < N; ++k)
            if (sizes[k] > 1) idx[n++] = k;
        std::stable_sort(idx, idx + n, [&](int x, int y) { return st[x] < st[y]; });
        for (int j = 1; j < n; ++j) {
            int64_t need;
            if (!mul_ok(st[idx[j - 1]], sizes[idx[j - 1]], &need)) return TTC_ERR_UNSUPPORTED;
            if (st[idx[j]] < need) return TTC_ERR_BAD_LD;
        }
    }
    return canon_from_strides(N, sizes, sA, sB, c, out);
}

}  // namespace ttc
