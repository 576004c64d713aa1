// plan.cpp -- stages 2-3 of the paper's pipeline: enumerate candidate
// implementations (kernel class x blocking x loop order x vector width), estimate their cost
// with heuristics and keep a bounded, ranked list.  Host only; timing happens in api.cpp.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <set>
#include <string>

#include "ttc_internal.h"

namespace ttc {

namespace {

constexpr int kFullSearch = 96;             // candidates at the head of the list that get the full padding search
constexpr int kMaxImplementations = 400;   // the paper's default bound is 200; ours holds the
                                           // ring-kernel variants as well, and a candidate costs ~1 ms to time
constexpr int64_t kInt31 = (int64_t)1 << 31;


// ----------------------------------------------------------------------------------------
// Shared-memory bank model: wavefronts needed by one warp-wide access of `sz` bytes per lane
// at byte addresses addr[0..n) (32 banks x 4 bytes; 8-byte accesses are served per half-warp,
// 16-byte accesses per quarter-warp; lanes reading the same word are broadcast).
// ----------------------------------------------------------------------------------------
int smem_wavefronts(const int64_t* addr, int n, int sz) {
    const int lanes_per_group = sz <= 4 ? 32 : (sz == 8 ? 16 : 8);
    const int wpl = std::max(1, sz / 4);                 // words per lane
    int total = 0;
    for (int g0 = 0; g0 < n; g0 += lanes_per_group) {
        // distinct words per bank (a group holds at most 32 words, so 32 slots per bank always suffice)
        int64_t seen[32][32];
        int cnt[32] = {0};
        int worst = 0;
        const int g1 = std::min(n, g0 + lanes_per_group);
        for (int l = g0; l < g1; ++l)
            for (int w = 0; w < wpl; ++w) {
                const int64_t word = addr[l] / 4 + w;
                const int bank = (int)(word & 31);
                bool dup = false;
                for (int k = 0; k < cnt[bank]; ++k) dup |= seen[bank][k] == word;
                if (dup) continue;
                seen[bank][cnt[bank]] = word;
                worst = std::max(worst, ++cnt[bank]);
            }
        total += worst;
    }
    return total;
}

// One enumerated index of a phase.  `fused`: this entry stands for the tile's two leading A
// indices taken as ONE contiguous run (smem and global stride 1), see build_tile_candidate.
struct PhaseDim { int dim; int32_t n, step; bool fused = false; };

// Enumerate entry `idx` of a phase (dims fastest first) and return its tile offset in elements.
int64_t phase_smem_offset(const std::vector<PhaseDim>& ph, const int32_t* ss, int64_t idx) {
    int64_t s = 0;
    for (const PhaseDim& p : ph) {
        const int64_t c = idx % p.n;
        idx /= p.n;
        s += c * p.step * (p.fused ? 1 : ss[p.dim]);
    }
    return s;
}

// The sampled warps of one phase: the coordinates of every sampled lane's entry, decomposed ONCE per
// candidate (the padding search only changes the strides they are multiplied with).
constexpr int kSampleWarps = 8, kMaxPhaseDims = 2 * kMaxTab;
struct PhaseSamples {
    int nk = 0;
    int dim[kMaxPhaseDims];
    bool fused[kMaxPhaseDims];
    int n[kSampleWarps];
    int32_t co[kSampleWarps][32][kMaxPhaseDims];   // coordinate * step per enumerated index
};

void sample_phase(const std::vector<PhaseDim>& ph, int64_t items, PhaseSamples* S) {
    S->nk = (int)std::min<size_t>(ph.size(), kMaxPhaseDims);
    for (int k = 0; k < S->nk; ++k) { S->dim[k] = ph[k].dim; S->fused[k] = ph[k].fused; }
    for (int w = 0; w < kSampleWarps; ++w) {
        const int64_t start = (items / 32) * w / kSampleWarps * 32;   // spread the sampled warps over the tile
        int n = 0;
        for (int l = 0; l < 32 && start + l < items; ++l, ++n) {
            int64_t idx = start + l;
            for (int k = 0; k < S->nk; ++k) {
                S->co[w][l][k] = (int32_t)((idx % ph[k].n) * ph[k].step);
                idx /= ph[k].n;
            }
        }
        S->n[w] = n;
    }
}

inline int64_t sample_offset(const PhaseSamples& S, int w, int l, const int32_t* ss) {
    int64_t o = 0;
    for (int k = 0; k < S.nk; ++k) o += (int64_t)S.co[w][l][k] * (S.fused[k] ? 1 : ss[S.dim[k]]);
    return o;
}

// Relative smem cost (>= 1) of both phases for the given tile strides.
double smem_conflict_cost(const PhaseSamples& SA, const PhaseSamples& SB,
                          const int32_t* ss, int es, int vecA, int vecB, bool same, int sstepB,
                          bool splitA, bool skipA = false, bool xp = false) {
    double got = 0, ideal = 0;
    int64_t addr[32];
    for (int w = 0; w < kSampleWarps; ++w) {
        int n = skipA ? 0 : SA.n[w];
        for (int l = 0; l < n; ++l) addr[l] = sample_offset(SA, w, l, ss) * es;
        if (n) {
            if (!splitA) {
                got += smem_wavefronts(addr, n, es * vecA);
            } else {   // the vecA elements of a global vector are stored one by one
                for (int j = 0; j < vecA; ++j) {
                    int64_t a2[32];
                    for (int l = 0; l < n; ++l) a2[l] = addr[l] + (int64_t)j * es;
                    got += smem_wavefronts(a2, n, es);
                }
            }
            ideal += std::max(1.0, n * es * vecA / 128.0);
        }
        n = SB.n[w];
        for (int l = 0; l < n; ++l) addr[l] = sample_offset(SB, w, l, ss) * es;
        if (n) {
            if (same || vecB == 1) {
                got += smem_wavefronts(addr, n, es * vecB);
                ideal += std::max(1.0, n * es * vecB / 128.0);
            } else {
                for (int j = 0; j < vecB; ++j) {
                    int64_t a2[32];
                    // xp: lane l reads its vecB rows in the rotated order (j + (l >> 3)) mod vecB
                    for (int l = 0; l < n; ++l)
                        a2[l] = addr[l] + (int64_t)(xp ? ((j + (l >> 3)) & (vecB - 1)) : j) * sstepB * es;
                    got += smem_wavefronts(a2, n, es);
                    ideal += std::max(1.0, n * es / 128.0);
                }
            }
        }
    }
    return ideal > 0 ? got / ideal : 1.0;
}

// Efficiency model of a contiguous run of `bytes` in global memory (sector / DRAM-page use).
double run_eff(double bytes, double knee = 48.0) {
    if (bytes >= 4096) return 1.0;
    return bytes / (bytes + knee) / (4096.0 / (4096.0 + knee));
}

bool split_tables(const std::vector<PhaseDim>& ph, int* split_out, int threads = 0) {
    // lo = ph[0..k), hi = ph[k..): both <= kMaxTabEntries entries and <= kMaxTab dims;
    // choose k that minimises lo.n + hi.n.  `threads` > 0 (ring kernel, B side): a lo table whose size
    // divides the consumer threads is preferred (the largest such) -- the kernel then enumerates the
    // store phase without a division, each thread keeping its lo entry in registers.
    const int n = (int)ph.size();
    int best = -1, best_fix = -1;
    int64_t best_sum = 0, best_fix_lo = 0;
    for (int k = 1; k <= n; ++k) {
        int64_t lo = 1, hi = 1;
        for (int i = 0; i < k; ++i) lo *= ph[i].n;
        for (int i = k; i < n; ++i) hi *= ph[i].n;
        if (k > kMaxTab || n - k > kMaxTab) continue;
        if (lo > kMaxTabEntries || hi > kMaxTabEntries) continue;
        if (best < 0 || lo + hi < best_sum) { best = k; best_sum = lo + hi; }
        if (threads > 0 && lo <= threads && threads % lo == 0 && lo > best_fix_lo) { best_fix = k; best_fix_lo = lo; }
    }
    *split_out = best_fix >= 0 ? best_fix : best;
    return best >= 0;
}

}  // namespace

namespace {

// Ranking cost of a tile / ring candidate from its raw features F (see the end of build_tile_candidate);
// `legacy` is the hand-written round-1 formula.  TTC_COST=legacy ranks by it (for comparisons).
double fitted_tile_cost(const float* F, double legacy) {
    static const bool use_legacy = std::getenv("TTC_COST") && !std::strcmp(std::getenv("TTC_COST"), "legacy");
    if (use_legacy) return legacy;
    // exp(w . terms): estimated time / (bytes at 6.5 TB/s).  Least-squares fit of log(time) on measured
    // times of all candidates of 71 transpositions on B200 (BASELINE.json's configs and 44 seeded random
    // 2-D..6-D cases of ~200 MB), weighted towards each case's fastest candidates; terms and weights come
    // from `python -m paper_1607_01249_b200.fit_cost fit` (same order as terms() there).  On those samples
    // the best of the 10 / 32 best-ranked candidates reaches 0.98 / 0.995 of the exhaustive search's time
    // (hand-written round-1 formula: 0.92 / 0.95).
    static const double kCostW[30] = {0.19459, 0.29221, 0.10785, -0.08450, -0.03553, 0.73929, 0.03056, 0.14005, -0.27823, 0.17293,
                                      0.15489, 0.93256, -0.16513, 0.06247, -0.06912, -0.10319, 0.40596, 0.03243, 0.13822, 0.06578,
                                      0.02644, 0.29674, -0.04683, 0.70913, 0.15136, -0.00012, -0.08401, -0.02661, 0.03885, -0.10466};
    const double runA = F[0], runB = F[1], waste = F[2], conf = F[3], tile_b = F[4], n_tiles = F[5], ring = F[6];
    const double rowmode = F[7], peel = F[8], xp = F[9], vab = F[10], vbb = F[11], beta = F[12], kern = F[13], row_b = F[14];
    const double lc = std::log(std::max(conf, 1.0));
    const double na = vab < 16 ? 1.0 : 0.0, nb = vbb < 16 ? 1.0 : 0.0;
    const double t[30] = {
        1.0,
        std::log1p(256.0 / std::max(runA, 1.0)), std::log1p(64.0 / std::max(runB, 1.0)),
        std::log1p(2048.0 / std::max(runA, 1.0)), std::log1p(512.0 / std::max(runB, 1.0)),
        std::log(std::max(waste, 1.0)), lc,
        4096.0 / std::max(tile_b, 256.0), std::max(0.0, tile_b - 32768.0) / 65536.0, std::max(0.0, tile_b - 16384.0) / 65536.0,
        std::max(0.0, 1.0 - n_tiles / 1184.0), std::max(0.0, 1.0 - n_tiles / 4736.0),
        ring > 0 ? 1.0 : 0.0, ring >= 4 ? 1.0 : 0.0,
        rowmode == 1 ? 1.0 : 0.0, rowmode == 2 ? 1.0 : 0.0, peel != 0 ? 1.0 : 0.0, xp != 0 ? 1.0 : 0.0,
        na, nb, na * (vab <= 4 ? 1.0 : 0.0), nb * (vbb <= 4 ? 1.0 : 0.0),
        beta, (rowmode == 1 ? 1.0 : 0.0) * 128.0 / std::max(row_b, 16.0), beta * std::log1p(64.0 / std::max(runB, 1.0)),
        beta * nb, (ring == 0 ? 1.0 : 0.0) * lc, lc * (xp != 0 ? 1.0 : 0.0),
        kern == 3 ? 1.0 : 0.0, kern == 4 ? 1.0 : 0.0};
    double z = 0;
    for (int i = 0; i < 30; ++i) z += kCostW[i] * t[i];
    return std::exp(z);
}

// Largest vector (in elements) legal for global accesses along canonical index `lead` of
// tensor X (strideOf gives that tensor's strides): the index is stride-1, its extent and
// tile extent are multiples of the vector, and every other stride keeps 16-byte alignment.
int legal_vec(const Canon& c, int lead, bool sideA, int32_t t_lead, int mv) {
    if (mv <= 1) return 1;
    const int64_t s = sideA ? c.d[lead].sA : c.d[lead].sB;
    if (s != 1) return 1;
    if (c.d[lead].e % mv != 0 || t_lead % mv != 0) return 1;
    for (int i = 0; i < c.rank; ++i) {
        if (i == lead) continue;
        const int64_t si = sideA ? c.d[i].sA : c.d[i].sB;
        if (si % mv != 0) return 1;
    }
    return mv;
}

// Build one tile-kernel candidate.  Returns false if the combination is not legal.
bool build_tile_candidate(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, const TileSpec& spec,
                          int loop_order, int want_va, int want_vb, int max_smem, int sched, int ring, int xp, int rowmode, bool quick,
                          Candidate* out) {
    // es: B's element and the tile's (the planner's world is B-typed); esA differs from it only for
    // the mixed-precision pairs.  There the tile kernel converts A in its load phase (the tile holds
    // B's type), while the ring kernel's bulk copies land A's bytes unconverted: its tile holds A's
    // type (esT = esA) and the consumers convert in the store phase.  Mixed ring candidates exist
    // for 16-byte bulk rows only (no cp.async rows, no peeled store phase).
    // Vectors are 16 bytes of the side's own element type (mvA elements in A, mvB in B); where one
    // vector has to serve both sides (the wide class) it has mvS = min of the two.
    const int es = elem_size(dtype), esA = elem_size(dtype_a);
    const int mvA = 16 / esA, mvB = 16 / es, mvS = std::min(mvA, mvB);
    const int mv = mvB;   // the ring kernel's peeled store phase (same-type pairs only: mvA == mvB)
    const bool mixed = dtype_a != dtype;
    const int esT = ring ? esA : es;   // element size of the shared-memory tile
    Candidate cand;
    cand.beta_nz = beta_nz;
    TileParams& P = cand.tp;
    std::memset(&P, 0, sizeof(P));

    std::vector<int> ta, tb;   // tile indices by ascending A-stride / B-stride
    for (int i = 0; i < c.rank; ++i)
        if (spec.t[i] > 1) ta.push_back(i);
    for (int k = 0; k < c.rank; ++k)
        if (spec.t[c.orderB[k]] > 1) tb.push_back(c.orderB[k]);
    if (ta.empty()) return false;
    const int A0 = ta[0], B0 = tb[0];
    int va = legal_vec(c, A0, true, spec.t[A0], want_va > 1 ? want_va : mvA);
    const int vb = legal_vec(c, B0, false, spec.t[B0], want_vb > 1 ? want_vb : mvB);
    // K3 for a tiny/odd stride-1 extent of A (c5: 7 complex64 = 56 bytes): when the tile takes the
    // leading index whole and the next one continues it in memory, the two are ONE contiguous run
    // for the load phase (7 x t1 elements), which can be vectorised although the leading extent
    // alone cannot.  The tile keeps them dense (pitch of the second = extent of the first), so a
    // loaded vector lands as one vector; the store phase still sees two indices.  Tiles never
    // straddle the end of the second index (its extent is a multiple of its tile extent), so no
    // vector is cut by a tile edge.
    bool fuseA = false;
    if (want_va > va && want_va == mvA && ta.size() >= 2 && A0 != B0) {
        const int A1 = ta[1];
        bool ok = c.d[A0].sA == 1 && spec.t[A0] == c.d[A0].e && c.d[A1].sA == c.d[A0].e &&
                  ((int64_t)spec.t[A0] * spec.t[A1]) % mvA == 0 && c.d[A1].e % spec.t[A1] == 0 && A1 != B0;
        for (int i = 0; i < c.rank && ok; ++i)
            if (i != A0 && i != A1 && c.d[i].sA % mvA != 0) ok = false;
        if (ok) { fuseA = true; va = mvA; }
    }
    // Ring kernel, peeled store phase: the B-leading index is stride-1 but its rows are not
    // 16-byte aligned (odd extent or stride): rows are cut into aligned 16-byte windows of B.
    const bool peelB = ring && !mixed && mv > 1 && want_vb == mv && vb < mv && c.d[B0].sB == 1 && A0 != B0;
    if (want_va > va || (want_vb > vb && !peelB)) return false;
    const bool same = (A0 == B0) && want_va == mvS && want_vb == mvS && mvS > 1;
    // nothing gained by mixing widths on one index -- except for a mixed ring, whose 16-byte rows of
    // A's type and 16-byte stores of B's type have different element counts
    if (A0 == B0 && want_va != want_vb && !(ring && mixed)) return false;
    P.vecA = want_va;
    P.vecB = want_vb;
    P.same = same ? 1 : 0;
    P.threads = kTileThreads;
    P.dyn = sched;

    // Phase enumerations (entries along the vectorised leading index count vectors).
    std::vector<PhaseDim> phA, phB;
    if (fuseA) {
        phA.push_back(PhaseDim{ta[1], (int32_t)((int64_t)spec.t[A0] * spec.t[ta[1]] / want_va), want_va, true});
        for (size_t k = 2; k < ta.size(); ++k) phA.push_back(PhaseDim{ta[k], spec.t[ta[k]], 1});
    } else {
        for (int i : ta) phA.push_back(PhaseDim{i, spec.t[i] / (i == A0 ? want_va : 1), i == A0 ? want_va : 1});
    }
    const int step_b = peelB ? 1 : want_vb;   // peeled: the tables enumerate single elements of the leading index
    // xp ("staggered gather", ring kernel): the store phase's fastest digit is a pair / quad of
    // COLUMNS -- neighbouring elements of a tile index X with an odd tile stride (A's leading index, or
    // the second one behind an odd fused leading extent) -- followed by the vectors of B's leading
    // index.  A warp then reads, per instruction, vecB columns x 8 rows; with the rows taken in a
    // lane-dependent rotation (kernel) and a row pitch that is an odd multiple of 16 bytes these hit
    // 32 distinct banks, which a plain gather down ONE column of 16-byte-granular rows cannot (8-byte
    // elements would need an odd element pitch).  Stores stay coalesced: 32 / vecB vectors per column.
    int X = -1;
    if (xp) {
        if (!ring || mixed || same || peelB || want_vb != mvB || mvB < 2 || ta.size() < 2) return false;
        if (spec.t[A0] % want_vb == 0 && c.d[A0].e % want_vb == 0 && A0 != B0) X = A0;
        else if (fuseA && spec.t[ta[1]] % want_vb == 0 && (spec.t[A0] & 1) && ta[1] != B0) X = ta[1];
        if (X < 0) return false;
        phB.push_back(PhaseDim{X, want_vb, 1});
        for (int i : tb) {
            if (i == X) phB.push_back(PhaseDim{i, spec.t[i] / want_vb, want_vb});
            else phB.push_back(PhaseDim{i, spec.t[i] / (i == B0 ? step_b : 1), i == B0 ? step_b : 1});
        }
    } else
    for (int i : tb) phB.push_back(PhaseDim{i, spec.t[i] / (i == B0 ? step_b : 1), i == B0 ? step_b : 1});
    int64_t itemsA = 1, itemsB = 1;
    for (auto& p : phA) itemsA *= p.n;
    for (auto& p : phB) itemsB *= p.n;
    // small tiles run in 128-thread CTAs: the same threads per SM, shorter barrier waits
    if (std::max(itemsA, itemsB) <= 4 * 256) P.threads = 128;
    int splitA, splitB;
    if (!split_tables(phA, &splitA) || !split_tables(phB, &splitB, ring ? (itemsB <= 4 * 256 ? 128 : 256) : 0)) return false;
    // Ring kernel (producer warp + consumer warps, `ring` tile buffers): every tile row along the
    // (vectorised, possibly fused) leading A index is one cp.async.bulk, so rows and addresses must
    // be 16-byte multiples, the tile layout 16-byte granular (no split stores) and the rows the hi
    // table of the A side.  Edge tiles get shorter and fewer rows.
    int row_dims = 1;
    if (ring) {
        if (c.d[A0].sA != 1) return false;     // bulk rows are contiguous runs of A's leading index
        if (same && (want_vb * es != 16 || mixed)) return false;
        if (mixed && (want_va * esA != 16 || (want_vb != mvB && want_vb != 1))) return false;   // instances: VB = mvB or 1
        if (want_va * esA != 16) {
            // rows that cannot be 16-byte bulk copies: element-sized cp.async rows, only where the
            // vector form is not legal (otherwise the bulk twin of this candidate is the better one)
            if (want_va != 1 || mv == 1 || legal_vec(c, A0, true, spec.t[A0] / mv * mv, mv) == mv || same ||
                c.d[A0].sA != 1) return false;
            // rowmode 2, "shifted rows": the 16-byte aligned body of every row is ONE bulk copy that lands in
            // the tile at the row's own misalignment (0 .. mv-1 elements, a per-row skew the consumers add),
            // only the < 16-byte head and tail are element copies; nothing outside the row is touched.
            P.row_async = rowmode == 2 ? 2 : 1;
            if (rowmode == 2 && xp) return false;
            // 4-byte elements: rows can be copied as 8-byte pairs when every row start and length is
            // even (all other A strides, the leading extent and tile extent) -- the tile rows then
            // must start at even offsets too (pitches rounded to 2 below)
            if (P.row_async == 1 && es == 4 && c.d[A0].e % 2 == 0 && spec.t[A0] % 2 == 0) {
                bool even = true;
                for (int i = 0; i < c.rank; ++i)
                    if (i != A0 && c.d[i].sA % 2 != 0) even = false;
                P.row_pairs = even ? 1 : 0;
            }
        } else if (rowmode == 2) {
            return false;     // only rows that are not 16-byte aligned have a shifted twin
        }
        // A row = the leading A indices of the tile that form ONE contiguous run in A: an index
        // extends the row when the previous one is taken whole and continues in memory; the tile
        // keeps those indices dense, so the run lands as one bulk copy (c4: 8 x t1 doubles instead
        // of 64-byte rows; c3: 24 x t1 floats).  Only the last index of a row can be cut by an edge.
        row_dims = 1;
        while (row_dims < (int)phA.size()) {
            const int pd = phA[row_dims - 1].dim, nd = phA[row_dims].dim;
            if (spec.t[pd] != c.d[pd].e || c.d[nd].sA != c.d[pd].e * c.d[pd].sA) break;
            ++row_dims;
        }
        int64_t row_items = 1, hi = 1;
        for (int k = 0; k < row_dims; ++k) row_items *= phA[k].n;
        for (size_t k = row_dims; k < phA.size(); ++k) hi *= phA[k].n;
        if (hi > kMaxTabEntries || (int)phA.size() - row_dims > kMaxTab || row_items * want_va * esA >= (1 << 20)) return false;
        splitA = row_dims;
        P.ring = ring;
        P.row_bytes = (uint32_t)(row_items * want_va * esA);
        P.threads = 32 + (itemsB <= 4 * 256 ? 128 : 256);
    }
    if (peelB) {
        int64_t rowsB = 1;
        for (size_t k = 1; k < phB.size(); ++k) rowsB *= phB[k].n;
        if (rowsB > kMaxTabEntries || (int)phB.size() - 1 > kMaxTab || phB[0].n > kMaxTabEntries) return false;
        splitB = 1;
        itemsB = rowsB * ((spec.t[B0] + mv - 1) / mv + 1);     // aligned windows that can touch a row
        P.peel = 1;
        P.peel_len = spec.t[B0];
    }
    const int dense_levels = ring ? row_dims + (fuseA ? 1 : 0) : (fuseA ? 2 : 1);   // ta[0..dense_levels) stay dense

    // Shared-memory strides: dense in A order, padded (in units that keep vector alignment)
    // where the bank model says the store phase would conflict.
    // Two ways to land a global vector of want_va elements in the tile: one vector store (rows
    // of the tile must then stay vector-aligned, so paddings are multiples of the vector) or
    // want_va element stores (any padding; this is what makes a transposing read of 8-byte
    // elements conflict-free, which needs an odd row pitch).
    int32_t ss[kMaxRank];
    int32_t best_ss[kMaxRank];
    double best_cost = 1e30;
    int64_t best_elems = 0;
    int best_split = 0;
    const int levels = (int)ta.size() - 1;
    const int search_levels = std::min(levels, 2);     // paddings of the two innermost levels decide the conflicts
    static const int pad_opts[] = {0, 1, 2, 3, 4};
    const int n_opts = 5;
    int combos = 1;
    for (int i = 0; i < search_levels; ++i) combos *= n_opts;
    const bool shifted = P.row_async == 2;
    // quick: no padding search (dense tile, paddings 0) -- the first pass of generate_candidates ranks with
    // it; only candidates that make the bounded list's head are built again with the full search
    if (quick) combos = 1;
    static thread_local PhaseSamples samplesA, samplesB;
    PhaseSamples *SA = &samplesA, *SB = &samplesB;
    if ((int)phA.size() > kMaxPhaseDims || (int)phB.size() > kMaxPhaseDims) return false;
    sample_phase(phA, itemsA, SA);
    sample_phase(phB, itemsB, SB);
    for (int split = 0; split < ((want_va > 1 && !same && !ring && !quick) ? 2 : 1); ++split) {
    const int unit = split ? 1 : std::max(std::max(std::max(want_va, same ? mvS : 1), P.row_pairs ? 2 : 1), shifted ? mv : 1);
    for (int combo = 0; combo < combos; ++combo) {
        int cc = combo;
        int64_t stride = 1;
        bool ok = true;
        for (int i = 0; i < c.rank; ++i) ss[i] = 0;
        for (size_t k = 0; k < ta.size(); ++k) {
            if (k > 0) {
                int pad = 0;
                if ((int)k <= search_levels) { pad = pad_opts[cc % n_opts] * unit; cc /= n_opts; }
                stride = stride * spec.t[ta[k - 1]];
                if (shifted && (int)k == dense_levels) stride += mv - 1;   // room for the row's skew
                if ((int)k < dense_levels) pad = 0;                  // a fused pair / a bulk row stays dense
                else stride = (stride + unit - 1) / unit * unit;
                stride += pad;
            }
            if (stride >= kInt31) { ok = false; break; }
            ss[ta[k]] = (int32_t)stride;
        }
        if (!ok) continue;
        int64_t elems = (int64_t)ss[ta.back()] * spec.t[ta.back()];
        if (shifted && (int)ta.size() <= dense_levels) elems = (elems + 2 * mv - 1) / mv * mv;   // a one-row tile
        if (elems * esT * (ring ? ring : 1) > max_smem) continue;
        const double conf = smem_conflict_cost(*SA, *SB, ss, esT, want_va, want_vb, same, ss[B0], split != 0,
                                               ring != 0 && !P.row_async, xp != 0);
        // a split store costs want_va - 1 extra instructions per item: worth it only for a real gain
        const double cost = conf + 1e-3 * (double)elems * esT / 1024.0 + (split ? 0.08 : 0.0);
        if (cost < best_cost) {
            best_cost = cost;
            best_elems = elems;
            best_split = split;
            std::memcpy(best_ss, ss, sizeof(ss));
        }
        if (conf <= 1.0 + 1e-9) break;      // conflict-free: larger paddings only cost shared memory
    }
    }
    if (best_cost >= 1e30) return false;
    std::memcpy(ss, best_ss, sizeof(ss));
    P.tile_elems = (uint32_t)best_elems;
    P.sstepB = ss[B0];
    P.shift_ld = 0;
    if (shifted) {     // skew step per element of B's leading index: its A-stride mod the vector, unless a row runs along it
        bool in_row = false;
        for (int r = 0; r < row_dims; ++r) in_row |= phA[r].dim == B0;
        if (!in_row) P.shift_ld = (int)(c.d[B0].sA % mv);
    }
    P.xp = xp ? 1 : 0;
    P.splitA = best_split;
    P.itemsA = (uint32_t)itemsA;
    P.itemsB = (uint32_t)itemsB;

    // Macro-tile grid in loop order: 0 = ascending A-stride, 1 = ascending B-stride.
    int gslot_of[kMaxRank];
    int64_t n_tiles = 1;
    P.nG = c.rank;
    // Orders 2 and 3 (TTC_LOOP_ORDERS=4; PAPER.md:137 explores all d! orders): the plane of the two leading
    // indices first -- 2: A's leading index, then B's, then the rest by A-stride; 3: B's, then A's, then the
    // rest by B-stride -- so that consecutive macro-tiles stay inside one 2-D slab of both tensors.
    int order[kMaxRank];
    for (int k = 0; k < c.rank; ++k) order[k] = (loop_order & 1) == 0 ? k : c.orderB[k];
    if (loop_order >= 2) {
        const int first = loop_order == 2 ? A0 : B0, second = loop_order == 2 ? B0 : A0;
        if (first == second) return false;
        int w = 0, tmp[kMaxRank];
        tmp[w++] = first;
        tmp[w++] = second;
        for (int k = 0; k < c.rank; ++k)
            if (order[k] != first && order[k] != second) tmp[w++] = order[k];
        bool same_as_base = true;
        for (int k = 0; k < c.rank; ++k) { same_as_base &= tmp[k] == order[k]; order[k] = tmp[k]; }
        if (same_as_base) return false;       // nothing new
    }
    for (int k = 0; k < c.rank; ++k) {
        const int i = order[k];
        if (c.d[i].e >= kInt31) return false;
        const int64_t nt = (c.d[i].e + spec.t[i] - 1) / spec.t[i];
        GridDim& g = P.g[k];
        g.div = make_fastdiv((uint32_t)nt);
        g.sA = c.d[i].sA;
        g.sB = c.d[i].sB;
        g.e = (int32_t)c.d[i].e;
        g.t = spec.t[i];
        gslot_of[i] = k;
        n_tiles *= nt;
        if (n_tiles >= kInt31) return false;
    }
    P.n_tiles = (uint32_t)n_tiles;
    if (ring) {
        P.lead_gslot = gslot_of[phA[row_dims - 1].dim];          // the only index of a row an edge can cut
        int64_t vm = phA[row_dims - 1].fused ? spec.t[A0] : 1;
        for (int k = 0; k + 1 < row_dims; ++k) vm *= (int64_t)phA[k].n * phA[k].step;
        P.lead_vmul = (int)vm;
    }

    // Offset tables.
    auto fill = [&](Table& tb_, const std::vector<PhaseDim>& ph, int lo, int hi, bool sideA) -> bool {
        tb_.nd = hi - lo;
        int64_t n = 1, span = 0;
        for (int k = lo; k < hi; ++k) {
            const PhaseDim& p = ph[k];
            TabDim& d = tb_.d[k - lo];
            d.div = make_fastdiv((uint32_t)p.n);
            d.n = p.n;
            d.step = p.step;
            d.gslot = gslot_of[p.dim];
            d.vmul = 1;
            d.sS = ss[p.dim] * p.step;
            d.aS = 0;
            if (shifted && !sideA) {       // does this index select the tile row?  (the row runs along phA[0..row_dims))
                bool in_row = false;
                for (int r = 0; r < row_dims; ++r) in_row |= phA[r].dim == p.dim;
                if (!in_row) d.aS = (int32_t)((c.d[p.dim].sA * p.step) % mv);
            }
            d.sG = (sideA ? c.d[p.dim].sA : c.d[p.dim].sB) * p.step;
            if (p.fused) {   // one run over (A0, A1): stride 1 in A and in the tile; valid up to e(A0) * vext(A1)
                d.vmul = spec.t[A0];
                d.sS = p.step;
                d.sG = p.step;
            }
            span += (int64_t)(p.n - 1) * d.sG;
            n *= p.n;
        }
        tb_.n = (int32_t)n;
        return span < kInt31 / 2;
    };
    if (!fill(P.tab[0], phA, 0, ring ? 0 : splitA, true) || !fill(P.tab[1], phA, splitA, (int)phA.size(), true) ||
        !fill(P.tab[2], phB, 0, splitB, false) || !fill(P.tab[3], phB, splitB, (int)phB.size(), false))
        return false;
    if (ring) P.tab[0].n = 0;   // the ring kernel has no lo table on the A side (rows are bulk copies)
    P.divAlo = make_fastdiv((uint32_t)std::max(1, P.tab[0].n));
    P.divBlo = make_fastdiv((uint32_t)P.tab[2].n);
    if (peelB) {
        P.divBlo = make_fastdiv((uint32_t)((spec.t[B0] + mv - 1) / mv + 1));
        P.peel_gslot = gslot_of[B0];
    }
    if ((int)tile_smem_layout(P, esT).total > max_smem) return false;

    // Contiguous runs the tile touches in A and in B (elements): leading tile indices that are
    // whole and contiguous extend the run.
    auto run_len = [&](const std::vector<int>& order, bool sideA) {
        int64_t run = 1, expect = 1;
        for (int i : order) {
            const int64_t s = sideA ? c.d[i].sA : c.d[i].sB;
            if (s != expect) break;
            run *= spec.t[i];
            if (spec.t[i] != c.d[i].e) break;
            expect = s * c.d[i].e;
        }
        return run;
    };
    const int64_t runA = run_len(ta, true), runB = run_len(tb, false);

    ttc_candidate_info& I = cand.info;
    I.kernel = ring ? TTC_KERNEL_TMA : same ? TTC_KERNEL_WIDE : (ta.size() > 2 ? TTC_KERNEL_GATHER : TTC_KERNEL_TILE);
    I.vec_a = want_va;
    I.vec_b = want_vb;
    I.tile_u = (int)std::min<int64_t>(runA, INT32_MAX);
    I.tile_w = (int)std::min<int64_t>(runB, INT32_MAX);
    I.n_u = (int)ta.size();
    I.n_w = (int)tb.size();
    I.threads = P.threads;
    I.smem_bytes = (int)tile_smem_layout(P, esT).total;
    I.loop_order = loop_order;
    I.sched = sched;
    I.flags = (xp ? TTC_CAND_STAGGERED : 0) | (shifted ? TTC_CAND_SHIFTED_ROWS : 0);
    I.grid = 0;
    I.n_tiles = n_tiles;
    for (int i = 0; i < kMaxRank; ++i) I.tile_ext[i] = i < c.rank ? spec.t[i] : 0;
    cand.align_a = P.row_pairs ? 8 : want_va * esA;
    cand.align_b = peelB ? es : want_vb * es;

    // Cost heuristic: long contiguous runs on both sides, small remainders,
    // few bank conflicts, enough bytes per tile to amortise its bookkeeping, enough tiles to
    // fill the machine.
    double waste = 1.0;
    for (int i = 0; i < c.rank; ++i) {
        const double nt = std::ceil((double)c.d[i].e / spec.t[i]);
        waste *= nt * spec.t[i] / (double)c.d[i].e;
    }
    const double tile_bytes = (double)itemsA * want_va * esT;
    const double rd = 1.0 / run_eff((double)runA * esA) * (want_va * esA >= 16 ? 1.0 : 1.15);
    // short runs cost much less on the B side than on the A side: the 126 MB L2 merges the writes of
    // neighbouring tiles before they reach DRAM (measured: 64-byte B runs win several c2 permutations)
    const double wr = (beta_nz ? 2.0 : 1.0) / run_eff((double)runB * es, 12.0) * (want_vb * es >= 16 ? 1.0 : 1.10);
    double cost = (rd + wr) * waste;
    cost *= 1.0 + 0.05 * (best_cost - 1.0);                   // smem conflicts are cheap but not free
    cost *= 1.0 + 2048.0 / tile_bytes;                        // per-tile overhead
    if (tile_bytes > 48 * 1024) cost *= 1.0 + (tile_bytes - 48 * 1024) / (256.0 * 1024);   // occupancy
    if (n_tiles < 148 * 2) cost *= 1.0 + (148.0 * 2 - n_tiles) / (148.0 * 2);
    if (ring) cost *= 0.95;   // read and write streams overlap inside the CTA
    if (P.row_async == 2) {
        cost *= 1.04;     // heads and tails; skewed reads
    } else if (P.row_async) {
        // one producer warp copies the rows 32 elements per instruction plus ~6 instructions per
        // row: short rows make the producer the bottleneck (measured: 32-element rows 2.7x, 64-element
        // rows 1.6x the time of rows of 128 and more)
        const double len = (double)P.row_bytes / es;
        cost *= std::max(1.0, 0.4 * (std::ceil(len / 32.0) + 6.0) / (len / 32.0));
    }
    // raw inputs of the heuristic, for re-fitting it against measured times (ttc_plan_candidate_features)
    float* F = cand.feat;
    F[0] = (float)((double)runA * esA);      // contiguous bytes per tile in A
    F[1] = (float)((double)runB * es);       // contiguous bytes per tile in B
    F[2] = (float)waste;                     // padded / logical elements (remainder tiles)
    F[3] = (float)best_cost;                 // shared-memory wavefronts / ideal (bank model)
    F[4] = (float)tile_bytes;
    F[5] = (float)n_tiles;
    F[6] = (float)ring;
    F[7] = (float)P.row_async;
    F[8] = (float)P.peel;
    F[9] = (float)P.xp;
    F[10] = (float)(want_va * esA);
    F[11] = (float)(want_vb * es);
    F[12] = beta_nz ? 1.f : 0.f;
    F[13] = (float)I.kernel;
    F[14] = (float)P.row_bytes;
    F[15] = (float)itemsB;
    I.est_cost = (float)fitted_tile_cost(F, cost);
    *out = cand;
    return true;
}

}  // namespace

namespace {

// One side of a tile: a prefix of the tensor's index order, all but the last taken whole.
struct SideOpt {
    std::vector<std::pair<int, int32_t>> dims;   // (canonical index, tile extent)
    int64_t elems = 1;
};

// Tile extents of index extent `e` whose side (with `cum` elements already in it) comes close
// to `target` elements: the largest divisor of e that fits, else a multiple of `mult`
// (leaves a remainder tile).
void partial_extents(int64_t e, int64_t cum, int64_t target, int mult, std::vector<int32_t>* out) {
    const int64_t want = target / cum;
    if (want < 2) return;
    if (want >= e) { out->push_back((int32_t)e); return; }
    int64_t best_div = 0;
    for (int64_t d = want; d >= 2 && d * 2 > want; --d)
        if (e % d == 0 && d % mult == 0) { best_div = d; break; }
    if (best_div) out->push_back((int32_t)best_div);
    const int64_t rounded = want / mult * mult;
    if (rounded >= 2 && rounded != best_div) out->push_back((int32_t)rounded);
}

// Options for one side.  `order` = the tensor's index order; `taken` = tile extents already
// fixed by the other side (0 = free).  Indices the other side holds whole are skipped (the run
// continues through them); an index it holds partially ends the side.
void side_options(const Canon& c, const std::vector<int>& order, const int32_t* taken, int mult,
                  int es, std::vector<SideOpt>* out) {
    static const int64_t targets_bytes[] = {32, 64, 128, 256, 512, 1024, 2048, 4096, 8192, 16384};
    SideOpt base;
    std::set<std::vector<std::pair<int, int32_t>>> seen;
    for (size_t k = 0; k < order.size(); ++k) {
        const int i = order[k];
        if (taken[i]) {
            if (taken[i] == c.d[i].e) continue;
            break;
        }
        if ((int)base.dims.size() >= kMaxTab - 1) break;
        const int m = (k == 0) ? mult : 1;
        for (int64_t tb : targets_bytes) {
            std::vector<int32_t> ext;
            partial_extents(c.d[i].e, base.elems, std::max<int64_t>(1, tb / es), m, &ext);
            for (int32_t t : ext) {
                if (t >= c.d[i].e && t != c.d[i].e) continue;
                SideOpt o = base;
                o.dims.push_back({i, t});
                o.elems = base.elems * t;
                if (seen.insert(o.dims).second) out->push_back(o);
            }
        }
        base.dims.push_back({i, (int32_t)std::min<int64_t>(c.d[i].e, INT32_MAX)});
        base.elems *= c.d[i].e;
        if (base.elems * es > 64 * 1024) break;
    }
}

void add_direct(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int loop_order, bool vector,
                int sched, std::vector<Candidate>* out) {
    const int es = elem_size(dtype), esA = elem_size(dtype_a);
    const int mv = max_vec(dtype, dtype_a);
    Candidate cand;
    cand.beta_nz = beta_nz;
    DirectParams& P = cand.dp;
    std::memset(&P, 0, sizeof(P));
    // leading index: the one that is stride-1 in both tensors if there is one, else A's
    int lead = 0;
    for (int i = 0; i < c.rank; ++i)
        if (c.d[i].sA == 1 && c.d[i].sB == 1) lead = i;
    int vec = 1;
    if (vector) {
        const int va = legal_vec(c, lead, true, (int32_t)std::min<int64_t>(c.d[lead].e, 1 << 30) / mv * mv, mv);
        const int vb = legal_vec(c, lead, false, (int32_t)std::min<int64_t>(c.d[lead].e, 1 << 30) / mv * mv, mv);
        if (va != mv || vb != mv || mv == 1 || c.d[lead].e % mv != 0) return;
        vec = mv;
    }
    std::vector<int> order;
    order.push_back(lead);
    for (int k = 0; k < c.rank; ++k) {
        const int i = loop_order == 0 ? k : c.orderB[k];
        if (i != lead) order.push_back(i);
    }
    P.nd = c.rank;
    P.vec = vec;
    uint64_t n_items = 1;
    bool idx64 = false;
    for (int k = 0; k < c.rank; ++k) {
        const int i = order[k];
        const int64_t n = c.d[i].e / (k == 0 ? vec : 1);
        const int64_t step = (k == 0 ? vec : 1);
        P.dims[k].n = (uint64_t)n;
        P.dims[k].sA = c.d[i].sA * step;
        P.dims[k].sB = c.d[i].sB * step;
        if (n >= kInt31) idx64 = true; else P.dims[k].div = make_fastdiv((uint32_t)n);
        n_items *= (uint64_t)n;
    }
    P.n_items = n_items;
    const uint64_t per_chunk = (uint64_t)kDirectThreads * kDirectUnroll;
    const uint64_t n_chunks = (n_items + per_chunk - 1) / per_chunk;
    if (n_chunks >= (uint64_t)kInt31) return;    // > 2^41 vectors: cannot be resident in HBM
    P.n_chunks = (uint32_t)n_chunks;
    P.dyn = sched;
    if (n_items >= (uint64_t)kInt31 / 2) idx64 = true;
    if (c.spanA >= kInt31 || c.spanB >= kInt31) idx64 = true;   // 32-bit element offsets otherwise
    cand.idx64 = idx64;
    cand.align_a = vec * esA;
    cand.align_b = vec * es;
    ttc_candidate_info& I = cand.info;
    I.kernel = TTC_KERNEL_COPY;
    I.vec_a = I.vec_b = vec;
    I.threads = 256;
    I.loop_order = loop_order;
    I.sched = sched;
    I.n_tiles = (int64_t)n_items;
    for (int i = 0; i < kMaxRank; ++i) I.tile_ext[i] = i < c.rank ? 1 : 0;
    // cost: contiguous runs seen by a warp on each side
    auto run_of = [&](bool sideA) {
        int64_t run = 1, expect = 1;
        // the item order is `order`; a side's run extends while its strides follow the order
        for (int k = 0; k < c.rank; ++k) {
            const int i = order[k];
            const int64_t s = sideA ? c.d[i].sA : c.d[i].sB;
            if (s != expect) break;
            run *= c.d[i].e;
            expect = s * c.d[i].e;
        }
        return run;
    };
    const double ra = (double)run_of(true) * esA, rb = (double)run_of(false) * es;
    auto eff = [&](double r) { return r <= es ? es / 32.0 * 0.5 : run_eff(r); };
    double cost = 1.0 / eff(ra) + (beta_nz ? 2.0 : 1.0) / eff(rb);
    if (vec * std::max(es, esA) < 16) cost *= 1.25;
    if (idx64) cost *= 1.5;
    cand.feat[0] = (float)ra;
    cand.feat[1] = (float)rb;
    cand.feat[2] = 1.f;
    cand.feat[10] = (float)(vec * esA);
    cand.feat[11] = (float)(vec * es);
    cand.feat[12] = beta_nz ? 1.f : 0.f;
    cand.feat[13] = (float)TTC_KERNEL_COPY;
    cand.feat[5] = (float)n_chunks;
    cand.feat[6] = idx64 ? 1.f : 0.f;
    // the tile candidates' fitted costs are time / ideal time; the direct formula is about 2.0 at its best
    static const bool legacy_cost = std::getenv("TTC_COST") && !std::strcmp(std::getenv("TTC_COST"), "legacy");
    I.est_cost = (float)(legacy_cost ? cost : 0.5 * cost);
    I.tile_u = (int)std::min<int64_t>(run_of(true), INT32_MAX);
    I.tile_w = (int)std::min<int64_t>(run_of(false), INT32_MAX);
    out->push_back(cand);
}


// ------------------------------------------------------------------------------------------
// Tensor-map candidates (TTC_KERNEL_TENSORMAP, ttc_tmap.cuh): same element type on both sides, canonical rank
// 2..5, every stride but the unit one a multiple of 16 bytes (SURVEY.md 8(d) "TMA feasibility"; the base
// addresses must be 16-byte aligned too, which align_a / align_b tell ttc_execute).
// ------------------------------------------------------------------------------------------
// Largest t in [max(1, want / 2), want] that wastes least of extent e when it is cut into pieces of t.
int32_t fit_extent(int64_t e, int32_t want) {
    if (e <= want) return (int32_t)e;
    int32_t best = want;
    double best_eff = 0.0;
    for (int32_t t = want; t >= std::max(1, want / 2); --t) {
        const double eff = (double)e / (double)(((e + t - 1) / t) * t);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = t; }
    }
    return best;
}

void add_tmap(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int sched, int max_smem, std::vector<Candidate>* out) {
    if (dtype != dtype_a || c.rank < 2 || c.rank > kTmapRank) return;
    const int es = elem_size(dtype);
    const int unit = es >= 8 ? 8 : 4, upe = es / unit;
    const int q = c.orderB[0];
    if (c.d[0].sA != 1 || c.d[q].sB != 1) return;
    const int64_t lim = (int64_t)1 << 40;
    for (int i = 0; i < c.rank; ++i) {
        if (c.d[i].e >= kInt31 / 2) return;
        if (i != 0 && ((c.d[i].sA * es) % 16 != 0 || c.d[i].sA * es >= lim)) return;
        if (i != q && ((c.d[i].sB * es) % 16 != 0 || c.d[i].sB * es >= lim)) return;
    }
    // A store clips at the tensor's edge only in whole 16-byte granules along dimension 0 (measured: a row of 3 fp32 inside a
    // leading dimension of 4 gets its padding element overwritten): B's rows must be a multiple of 16 bytes long.
    if ((c.d[q].e * es) % 16 != 0) return;
    const int flavour = q == 0 ? 1 : 0;
    // the other indices, by ascending stride in A and in B
    std::vector<int> othA, othB;
    for (int i = 0; i < c.rank; ++i) if (i != 0 && i != q) othA.push_back(i);
    for (int k = 0; k < c.rank; ++k) if (c.orderB[k] != 0 && c.orderB[k] != q) othB.push_back(c.orderB[k]);
    const int T = 128 / es;                              // flavour 0: elements per 128-byte box row
    int TA = T, TB = T;                                  // plane edges of the variant being emitted (T or T / 2: 64-byte rows)

    std::set<std::string> seen;
    int n_added = 0;
    auto emit = [&](const int32_t* pe, int32_t box0_units, int nbA, int nbB) {
        // pe[i]: box extent of canonical index i (flavour 0: the two leading ones are fixed by the swizzle)
        std::string key((const char*)pe, sizeof(int32_t) * c.rank);
        key.push_back((char)nbA);
        key.push_back((char)nbB);
        key.append((const char*)&box0_units, sizeof(box0_units));
        key.push_back((char)TA);
        key.push_back((char)TB);
        if (!seen.insert(key).second) return;
        Candidate cand;
        cand.beta_nz = beta_nz;
        TmapParams& M = cand.mp;
        TmapEncode& E = cand.me;
        std::memset(&M, 0, sizeof(M));
        std::memset(&E, 0, sizeof(E));
        int idx[kTmapRank];                                  // canonical index of A-map dimension k (-1: padding)
        int n = 0;
        if (flavour == 0) {
            idx[n++] = 0;
            idx[n++] = q;
            for (int i : othA) idx[n++] = i;
        } else {
            for (int k = 0; k < c.rank; ++k) idx[n++] = c.orderB[k];
        }
        for (; n < kTmapRank; ++n) idx[n] = -1;
        int64_t planes = 1, box_elems = 1;
        for (int k = 0; k < kTmapRank; ++k) {
            const int i = idx[k];
            const int64_t e = i < 0 ? 1 : c.d[i].e;
            int32_t bx;                                          // box extent (elements) along A-map dimension k
            if (flavour == 0) bx = k == 0 ? TA : k == 1 ? TB : (i < 0 ? 1 : pe[i]);
            else bx = k == 0 ? box0_units / upe : (i < 0 ? 1 : pe[i]);
            if (bx < 1 || bx > 256) return;
            if (flavour == 0 && k >= 2) planes *= bx;
            box_elems *= bx;
            E.dimA[k] = (uint64_t)e * (k == 0 ? upe : 1);
            E.boxA[k] = (uint32_t)bx * (k == 0 ? upe : 1);
            if (k > 0) E.strideA[k - 1] = i < 0 ? 16 : (uint64_t)(c.d[i].sA * es);
            const int nb = flavour == 0 ? (k == 0 ? nbA : k == 1 ? nbB : 1) : 1;
            M.step[k] = bx * nb;
            const int64_t nt = (e + M.step[k] - 1) / M.step[k];
            M.gdiv[k] = make_fastdiv((uint32_t)nt);
        }
        // B's map: flavour 0 swaps the two leading dimensions, flavour 1 keeps A's order
        for (int k = 0; k < kTmapRank; ++k) {
            const int ka = flavour == 0 && k < 2 ? 1 - k : k;    // A-map dimension that is B-map dimension k
            const int i = idx[ka];
            const int64_t e = i < 0 ? 1 : c.d[i].e;
            const uint32_t bx = E.boxA[ka] / (ka == 0 ? upe : 1);
            E.dimB[k] = (uint64_t)e * (k == 0 ? upe : 1);
            E.boxB[k] = bx * (k == 0 ? upe : 1);
            if (k > 0) E.strideB[k - 1] = i < 0 ? 16 : (uint64_t)(c.d[i].sB * es);
        }
        if (E.boxA[0] > 256 || E.boxB[0] > 256 || (E.boxA[0] * unit) % 16 != 0) return;
        E.unit_bytes = unit;
        auto swz = [&](int row_elems) { const int b = row_elems * es; return b >= 128 ? 3 : b == 64 ? 2 : 1; };   // CUtensorMapSwizzle values
        E.swzA = flavour == 0 ? swz(TA) : 0;
        E.swzB = flavour == 0 ? swz(TB) : 0;
        M.ca = TA * es / 16;
        M.cb = TB * es / 16;
        const int64_t box_bytes = box_elems * es;
        if (flavour == 0 && box_bytes % 1024 != 0) return;       // every box starts on a swizzle-atom boundary
        const int64_t tile_bytes = (box_bytes * nbA * nbB + 127) / 128 * 128;
        if (box_bytes < 1024 || tile_bytes > 64 * 1024 || nbA * nbB > kTmapMaxBoxes) return;
        int stages = 0;
        for (int st = 4; st >= 2; --st)
            if (st * 2 * tile_bytes + 1024 <= std::min<int64_t>(max_smem, 100 * 1024)) { stages = st; break; }   // >= 2 CTAs per SM
        if (!stages) return;
        uint64_t n_tiles = 1;
        double padded = 1.0, real = 1.0;
        for (int k = 0; k < kTmapRank; ++k) {
            n_tiles *= M.gdiv[k].d;
            if (n_tiles >= (uint64_t)kInt31) return;
            padded *= (double)M.gdiv[k].d * M.step[k];
            real *= idx[k] < 0 ? 1.0 : (double)c.d[idx[k]].e;
        }
        M.flavour = flavour;
        M.dyn = sched;
        M.n_tiles = (uint32_t)n_tiles;
        M.stages = stages;
        M.threads = 192;                                         // producer warp, store warp, 4 consumer warps
        M.nbA = nbA;
        M.nbB = nbB;
        M.planes = (int)planes;
        M.box_bytes = (uint32_t)box_bytes;
        M.buf_bytes = (uint32_t)tile_bytes;
        M.upe = upe;
        M.box0[0] = (int32_t)(E.boxA[0] / upe);
        M.box0[1] = (int32_t)E.boxA[1];
        M.batchable = idx[kTmapRank - 1] < 0 ? 1 : 0;            // the fifth map dimension is free for the batch offset
        cand.align_a = cand.align_b = 16;
        ttc_candidate_info& I = cand.info;
        I.kernel = TTC_KERNEL_TENSORMAP;
        I.flags = TTC_CAND_TENSORMAP;
        I.vec_a = I.vec_b = 16 / es;
        I.threads = M.threads;
        I.loop_order = 0;
        I.sched = sched;
        I.n_tiles = (int64_t)n_tiles;
        I.tile_u = M.step[0];
        I.tile_w = flavour == 0 ? M.step[1] : 1;
        I.n_u = 1;
        I.n_w = 1;
        for (int i = 0; i < kMaxRank; ++i) I.tile_ext[i] = i < c.rank ? 1 : 0;
        for (int k = 0; k < kTmapRank; ++k) if (idx[k] >= 0) I.tile_ext[idx[k]] = M.step[k];
        // ranked just behind the best fitted ring candidates (fitted costs are time / ideal time), tiles that stick
        // out of the tensor cost their share of wasted shared-memory work; the tuner decides
        const double waste = padded / real;
        I.est_cost = (float)((1.04 + 0.01 * n_added) * waste * (tile_bytes < 8192 ? 1.15 : 1.0));
        cand.feat[2] = (float)waste;
        cand.feat[4] = (float)tile_bytes;
        cand.feat[5] = (float)n_tiles;
        cand.feat[12] = beta_nz ? 1.f : 0.f;
        cand.feat[13] = (float)TTC_KERNEL_TENSORMAP;
        out->push_back(cand);
        ++n_added;
    };

    // Box extents over the other indices: `want` planes (flavour 0) or rows (flavour 1), handed out along `order`.
    auto fill = [&](const std::vector<int>& order, int64_t want, int32_t* pe) {
        for (int i = 0; i < c.rank; ++i) pe[i] = 1;
        int64_t left = want;
        for (int i : order) {
            if (left < 2) break;
            const int32_t t = fit_extent(c.d[i].e, (int32_t)std::min<int64_t>(left, 256));
            pe[i] = t;
            left /= t;
        }
    };
    int32_t pe[kMaxRank];
    if (flavour == 0) {
        struct Var { int dist, kb, nbA, nbB; };
        static const Var vars[] = {{0, 16, 1, 1}, {1, 16, 1, 1}, {0, 8, 2, 1}, {1, 8, 1, 2}, {2, 16, 1, 1}, {0, 8, 1, 1}, {1, 8, 1, 1},
                                   {2, 4, 2, 2}};
        // plane edges: 128-byte rows on both sides, and 64-byte rows on a side whose extent they fit with at least 20 % less
        // padding (24 fp64 = 1.5 rows of 128 bytes but 3 of 64).  Measured on c2: for 72 and 56 fp64 (4.5 and 3.5 rows,
        // 11-14 % padding) the 64-byte rows are no faster (3210: 82-84 us against 80-82), so small gains are not offered.
        auto padded_to = [](int64_t e, int t) { return (e + t - 1) / t * t; };
        std::vector<std::pair<int, int>> edges = {{T, T}};
        const bool half_a = T >= 2 && padded_to(c.d[0].e, T / 2) * 6 <= padded_to(c.d[0].e, T) * 5;
        const bool half_b = T >= 2 && ((T / 2) * es) % 16 == 0 && padded_to(c.d[q].e, T / 2) * 6 <= padded_to(c.d[q].e, T) * 5;
        if (half_b) edges.push_back({T, T / 2});
        if (half_a && ((T / 2) * es) % 16 == 0) edges.push_back({T / 2, T});
        if (half_a && half_b && ((T / 2) * es) % 16 == 0) edges.push_back({T / 2, T / 2});
        for (auto& ed : edges) {
        TA = ed.first;
        TB = ed.second;
        const int64_t plane_bytes = (int64_t)TA * TB * es;
        for (const Var& v : vars) {
            if (c.d[0].e <= (int64_t)(v.nbA - 1) * TA || c.d[q].e <= (int64_t)(v.nbB - 1) * TB) continue;
            const int64_t want = std::max<int64_t>(1, (int64_t)v.kb * 1024 / plane_bytes);
            if (v.dist == 0) fill(othA, want, pe);
            else if (v.dist == 1) fill(othB, want, pe);
            else {
                // balanced: half of the planes along A's next index, the rest along B's
                for (int i = 0; i < c.rank; ++i) pe[i] = 1;
                if (othA.empty()) continue;
                int64_t h = 1;
                while (h * h < want) h *= 2;
                const int ia = othA[0];
                pe[ia] = fit_extent(c.d[ia].e, (int32_t)h);
                int64_t left = want / pe[ia];
                for (int i : othB) {
                    if (i == ia || left < 2) continue;
                    pe[i] = fit_extent(c.d[i].e, (int32_t)std::min<int64_t>(left, 256));
                    left /= pe[i];
                }
            }
            emit(pe, 0, v.nbA, v.nbB);
        }
        if (othA.empty()) {      // 2-D: a tile is a few planes side by side
            for (int i = 0; i < c.rank; ++i) pe[i] = 1;
            static const int nb[][2] = {{2, 2}, {4, 1}, {1, 4}, {4, 2}, {2, 4}, {2, 1}, {1, 2}};
            for (auto& b : nb)
                if (c.d[0].e > (int64_t)(b[0] - 1) * TA && c.d[q].e > (int64_t)(b[1] - 1) * TB) emit(pe, 0, b[0], b[1]);
        }
        }
        TA = TB = T;
    } else {
        // copy class: rows of up to 256 map units along the shared leading index, then rows until the box has 8-32 KB
        const int gran = 16 / unit;
        const int64_t e0u = c.d[0].e * upe;
        int32_t b0 = (int32_t)std::min<int64_t>(256, (e0u + gran - 1) / gran * gran);
        if (e0u > 256) {         // cut long rows evenly
            const int64_t pieces = (e0u + 255) / 256;
            b0 = (int32_t)(((e0u + pieces - 1) / pieces + gran - 1) / gran * gran);
        }
        for (int kb : {16, 8})
            for (int dist = 0; dist < 2; ++dist) {
                const int64_t want = std::max<int64_t>(1, (int64_t)kb * 1024 / ((int64_t)b0 * unit));
                fill(dist == 0 ? othB : othA, want, pe);
                emit(pe, b0, 1, 1);
            }
    }
}


// Tensor-map candidates for more than 5 canonical indices (flavour 2, ttc_tmap.h): every index beyond the T x T plane is
// folded into one map dimension.  Strides must still be multiples of 16 bytes and the bases 16-byte aligned: the hardware
// refuses a box whose first byte is not 16-byte aligned ("illegal instruction"), so the skew the residue classes were
// designed to absorb cannot be expressed as a coordinate (round 2).
void add_tmapu(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int sched, int max_smem, std::vector<Candidate>* out) {
    if (dtype != dtype_a || c.rank <= kTmapRank) return;
    const int es = elem_size(dtype);
    if (es > 8) return;
    const int V = 16 / es, T = 128 / es;
    const int q = c.orderB[0];
    if (q == 0 || c.d[0].sA != 1 || c.d[q].sB != 1) return;
    for (int i = 0; i < c.rank; ++i) {
        if (c.d[i].e >= kInt31 / 2) return;
        if (i != 0 && (c.d[i].sA * es) % 16 != 0) return;
        if (i != q && (c.d[i].sB * es) % 16 != 0) return;
    }
    if ((c.d[q].e * es) % 16 != 0) return;               // stores clip in whole 16-byte granules (see add_tmap)
    if (c.d[0].e < T / 2 || c.d[q].e < T / 2) return;     // more than half of every plane would be padding
    const int64_t lim = (int64_t)1 << 40;
    if (c.d[q].sA * es * V >= lim || c.d[0].sB * es * V >= lim) return;
    if (c.spanA / V >= kInt31 - 4 || c.spanB / V >= kInt31 - 4) return;        // the aligned offset is an int32 coordinate
    std::vector<int> othA, othB;
    for (int i = 0; i < c.rank; ++i) if (i != 0 && i != q) othA.push_back(i);
    for (int k = 0; k < c.rank; ++k) if (c.orderB[k] != 0 && c.orderB[k] != q) othB.push_back(c.orderB[k]);
    std::set<std::string> seen;
    int n_added = 0;
    for (int kb : {16, 8, 4})
        for (int dist = 0; dist < 2; ++dist) {
            const int want = std::max(1, std::min(kTmapUMaxPlanes, kb / V));
            int32_t pe[kMaxRank];
            for (int i = 0; i < c.rank; ++i) pe[i] = 1;
            int left = want;
            for (int i : (dist == 0 ? othA : othB)) {      // planes must divide the extents: no ragged plane stacks
                if (left < 2) break;
                int t = 1;
                for (int d = std::min<int64_t>(left, c.d[i].e); d >= 1; --d)
                    if (c.d[i].e % d == 0) { t = d; break; }
                pe[i] = t;
                left /= t;
            }
            std::string key((const char*)pe, sizeof(int32_t) * c.rank);
            if (!seen.insert(key).second) continue;
            Candidate cand;
            cand.beta_nz = beta_nz;
            TmapUParams& U = cand.up;
            std::memset(&U, 0, sizeof(U));
            std::memset(&cand.mp, 0, sizeof(cand.mp));
            U.V = V;
            U.T = T;
            U.nG = c.rank;
            U.sqA = c.d[q].sA;
            U.s0B = c.d[0].sB;
            U.remA = (int)(c.d[q].e % V);
            U.remB = (int)(c.d[0].e % V);
            // tile grid: a0, b0, then the others in canonical order
            int gd[kMaxRank];
            int n = 0;
            gd[n++] = 0;
            gd[n++] = q;
            for (int i : othA) gd[n++] = i;
            uint64_t n_tiles = 1;
            double padded = 1.0, real = 1.0;
            bool ok = true;
            for (int k = 0; k < n; ++k) {
                const int i = gd[k];
                const int64_t step = k < 2 ? T : pe[i];
                const int64_t nt = (c.d[i].e + step - 1) / step;
                U.gdiv[k] = make_fastdiv((uint32_t)nt);
                U.stepA[k] = k < 2 ? 0 : step * c.d[i].sA;
                U.stepB[k] = k < 2 ? 0 : step * c.d[i].sB;
                n_tiles *= (uint64_t)nt;
                if (n_tiles >= (uint64_t)kInt31) { ok = false; break; }
                padded *= (double)nt * step;
                real *= (double)c.d[i].e;
            }
            if (!ok) continue;
            // the planes of a tile: every index combination of the box over the other indices
            int nP = 1;
            U.pA[0] = U.pB[0] = 0;
            for (int i : othA) {
                const int have = nP;
                for (int v = 1; v < pe[i]; ++v)
                    for (int h = 0; h < have; ++h) {
                        U.pA[nP] = U.pA[h] + (int64_t)v * c.d[i].sA;
                        U.pB[nP] = U.pB[h] + (int64_t)v * c.d[i].sB;
                        ++nP;
                    }
            }
            U.nP = nP;
            const int64_t buf = (int64_t)nP * V * 1024;
            int stages = 0;
            for (int st = 4; st >= 2; --st)
                if (st * 2 * buf + 1024 <= std::min<int64_t>(max_smem, 100 * 1024)) { stages = st; break; }
            if (!stages) continue;
            U.dyn = sched;
            U.n_tiles = (uint32_t)n_tiles;
            U.stages = stages;
            U.threads = 192;
            cand.mp.flavour = 2;                            // what the launcher and prepare_candidate look at
            cand.mp.dyn = sched;
            cand.mp.n_tiles = U.n_tiles;
            cand.mp.stages = stages;
            cand.mp.threads = U.threads;
            cand.ue = TmapUEncode{es, c.d[0].e, c.d[q].e, c.d[q].sA, c.d[0].sB, c.spanA, c.spanB};
            cand.align_a = cand.align_b = 16;
            ttc_candidate_info& I = cand.info;
            I.kernel = TTC_KERNEL_TENSORMAP;
            I.flags = TTC_CAND_TENSORMAP;
            I.vec_a = I.vec_b = V;
            I.threads = U.threads;
            I.loop_order = 0;
            I.sched = sched;
            I.n_tiles = (int64_t)n_tiles;
            I.tile_u = T;
            I.tile_w = T;
            I.n_u = 1;
            I.n_w = 1;
            for (int i = 0; i < kMaxRank; ++i) I.tile_ext[i] = i < c.rank ? pe[i] : 0;
            I.tile_ext[0] = T;
            I.tile_ext[q] = T;
            const double waste = padded / real;
            I.est_cost = (float)((1.06 + 0.01 * n_added) * waste * (buf < 8192 ? 1.15 : 1.0));
            cand.feat[2] = (float)waste;
            cand.feat[4] = (float)buf;
            cand.feat[5] = (float)n_tiles;
            cand.feat[12] = beta_nz ? 1.f : 0.f;
            cand.feat[13] = (float)TTC_KERNEL_TENSORMAP;
            out->push_back(cand);
            ++n_added;
        }
}


// Skew-kernel candidates (TTC_KERNEL_SKEW, ttc_skew.cuh): 4- and 8-byte elements of one type, transposing class, offered
// where a tensor map cannot express the tensors (a stride or B's row length is not a multiple of 16 bytes).
void add_skew(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int sched, int max_smem, std::vector<Candidate>* out) {
    if (dtype != dtype_a || c.rank < 2) return;
    const int es = elem_size(dtype);
    if (es > 8) return;
    const int q = c.orderB[0];
    if (q == 0 || c.d[0].sA != 1 || c.d[q].sB != 1) return;
    bool mappable = (c.d[q].e * es) % 16 == 0;
    for (int i = 0; i < c.rank; ++i) {
        if (c.d[i].e >= kInt31 / 2) return;
        if (i != 0 && (c.d[i].sA * es) % 16 != 0) mappable = false;
        if (i != q && (c.d[i].sB * es) % 16 != 0) mappable = false;
    }
    if (mappable) return;
    // Runs (ttc_skew.h): B's leading indices while they are contiguous in B, until the run has 64 positions; then A's
    // leading indices (none of them in the B-run) while they are contiguous in A, until 128 positions; at most 3 each.
    std::vector<int> runA = {0}, runB = {q};
    int64_t LA = c.d[0].e, LB = c.d[q].e;
    for (int k = 1; k < c.rank && (int)runB.size() < 3 && LB < 64; ++k) {
        const int i = c.orderB[k];
        if (i == 0 || c.d[i].sB != LB) break;                  // LB == stride the next index needs to continue the run
        runB.push_back(i);
        LB *= c.d[i].e;
    }
    auto in_run = [](const std::vector<int>& r, int i) { return std::find(r.begin(), r.end(), i) != r.end(); };
    for (int i = 1; i < c.rank && (int)runA.size() < 3 && LA < 128; ++i) {
        if (in_run(runB, i) || c.d[i].sA != LA) break;
        runA.push_back(i);
        LA *= c.d[i].e;
    }
    if (LA < 16 || LB < 16 || LA >= kInt31 / 2 || LB >= kInt31 / 2) return;
    const bool plain_runs = runA.size() == 1 && runB.size() == 1;
    std::vector<int> othA, othB;
    for (int i = 0; i < c.rank; ++i) if (!in_run(runA, i) && !in_run(runB, i)) othA.push_back(i);
    for (int k = 0; k < c.rank; ++k) if (!in_run(runA, c.orderB[k]) && !in_run(runB, c.orderB[k])) othB.push_back(c.orderB[k]);
    // direct = 1: no out-tile, the consumers store to B themselves (coalesced element stores)
    struct Var { int lgA, lgB, planes, dist, direct; };
    static const Var vars[] = {{7, 6, 1, 0, 1}, {6, 7, 1, 0, 1}, {7, 5, 1, 0, 1}, {6, 5, 1, 0, 1}, {8, 5, 1, 0, 1}, {6, 6, 1, 0, 1},
                               {5, 6, 1, 0, 1}, {5, 7, 1, 0, 1}, {5, 5, 1, 0, 1}, {5, 5, 2, 0, 1}, {6, 5, 2, 0, 1}, {6, 5, 2, 1, 1}, {5, 6, 2, 0, 1}, {5, 6, 2, 1, 1},
                               {6, 5, 1, 0, 0}, {5, 6, 1, 0, 0}, {6, 6, 1, 0, 0}, {7, 5, 1, 0, 0}, {5, 7, 1, 0, 0}, {5, 5, 2, 0, 0}, {5, 5, 2, 1, 0},
                               {6, 5, 2, 0, 0}, {5, 6, 2, 1, 0}, {5, 5, 4, 0, 0}, {5, 5, 4, 1, 0}, {7, 6, 1, 0, 0}, {6, 7, 1, 0, 0}};
    // TTC_VARIANTS bit 3 offers the direct-out variants (default), bit 4 the out-tile variants as well (measured 2x slower)
    const int variants = std::getenv("TTC_VARIANTS") ? std::atoi(std::getenv("TTC_VARIANTS")) : 15;
    std::set<std::string> seen;
    int n_added = 0;
    for (const Var& v : vars) {
        if (!v.direct && (!(variants & 16) || !plain_runs)) continue;        // the out-tile variants know single-index runs only
        const int TA = 1 << v.lgA, TB = 1 << v.lgB;
        if (LA * 2 < TA || LB * 2 < TB) continue;                             // more than half of the tile would be padding
        int32_t pe[kMaxRank];
        for (int i = 0; i < c.rank; ++i) pe[i] = 1;
        int left = v.planes;
        for (int i : (v.dist == 0 ? othA : othB)) {                            // planes divide the extents
            if (left < 2) break;
            int t = 1;
            for (int d = (int)std::min<int64_t>(left, c.d[i].e); d >= 1; --d)
                if (c.d[i].e % d == 0) { t = d; break; }
            pe[i] = t;
            left /= t;
        }
        std::string key((const char*)pe, sizeof(int32_t) * c.rank);
        key.push_back((char)v.lgA);
        key.push_back((char)v.lgB);
        key.push_back((char)v.direct);
        if (!seen.insert(key).second) continue;
        Candidate cand;
        cand.beta_nz = beta_nz;
        SkewParams& K = cand.sp;
        std::memset(&K, 0, sizeof(K));
        K.lgTA = v.lgA;
        K.lgTB = v.lgB;
        K.nA = (int)runA.size();
        K.nB = (int)runB.size();
        for (int k = 0; k < K.nA; ++k) { K.divA[k] = make_fastdiv((uint32_t)c.d[runA[k]].e); K.sBA[k] = c.d[runA[k]].sB; }
        for (int k = 0; k < K.nB; ++k) { K.divB[k] = make_fastdiv((uint32_t)c.d[runB[k]].e); K.sAB[k] = c.d[runB[k]].sA; }
        K.e0 = LA;
        K.eq = LB;
        K.spanA = c.spanA;
        K.spanB = c.spanB;
        K.pitchA = TA * es + 48;         // the aligned superset of a row (up to 12 bytes before and after it); an odd number
        K.pitchB = v.direct ? 0 : TB * es + 48;   // of 16-byte units, so that the consumers' diagonal walk spreads over all banks
        int gd[kMaxRank];
        int n = 0;
        gd[n++] = 0;
        gd[n++] = q;
        for (int i : othA) gd[n++] = i;
        uint64_t n_tiles = 1;
        double padded = 1.0, real = 1.0;
        bool ok = true;
        for (int k = 0; k < n; ++k) {
            const int i = gd[k];
            const int64_t step = k == 0 ? TA : k == 1 ? TB : pe[i];
            const int64_t ext = k == 0 ? LA : k == 1 ? LB : c.d[i].e;
            const int64_t nt = (ext + step - 1) / step;
            K.gdiv[k] = make_fastdiv((uint32_t)nt);
            K.stepA[k] = k < 2 ? 0 : step * c.d[i].sA;
            K.stepB[k] = k < 2 ? 0 : step * c.d[i].sB;
            n_tiles *= (uint64_t)nt;
            if (n_tiles >= (uint64_t)kInt31) { ok = false; break; }
            padded *= (double)nt * step;
            real *= (double)ext;
        }
        if (!ok) continue;
        K.nG = n;
        int nP = 1;
        K.pA[0] = K.pB[0] = 0;
        for (int i : othA) {
            const int have = nP;
            for (int t = 1; t < pe[i]; ++t)
                for (int h = 0; h < have; ++h) {
                    K.pA[nP] = K.pA[h] + (int64_t)t * c.d[i].sA;
                    K.pB[nP] = K.pB[h] + (int64_t)t * c.d[i].sB;
                    ++nP;
                }
        }
        if (nP > kSkewMaxPlanes || nP * TA > kSkewMaxRows || nP * TB > kSkewMaxRows) continue;
        K.nP = nP;
        const int64_t stage = (int64_t)nP * ((int64_t)TB * K.pitchA + (int64_t)TA * K.pitchB);
        int stages = 0;
        for (int st = kSkewMaxStages; st >= 2; --st)
            if (st * stage + 128 <= std::min<int64_t>(max_smem, 100 * 1024)) { stages = st; break; }
        if (!stages) continue;
        K.dyn = sched;
        K.n_tiles = (uint32_t)n_tiles;
        K.stages = stages;
        K.np = 4;
        K.ns = v.direct ? 0 : 4;
        K.threads = 384;                 // 4 producer warps, 4 store warps, 4 consumer warps: a bulk copy costs its issuing
                                         // warp ~150 cycles, so the row copies are spread over several warps
        cand.align_a = cand.align_b = es;
        ttc_candidate_info& I = cand.info;
        I.kernel = TTC_KERNEL_SKEW;
        I.flags = v.direct ? TTC_CAND_DIRECT_OUT : 0;
        I.vec_a = I.vec_b = 16 / es;
        I.threads = K.threads;
        I.loop_order = 0;
        I.sched = sched;
        I.n_tiles = (int64_t)n_tiles;
        I.tile_u = TA;
        I.tile_w = TB;
        I.n_u = 1;
        I.n_w = 1;
        for (int i = 0; i < kMaxRank; ++i) I.tile_ext[i] = i < c.rank ? pe[i] : 0;
        I.tile_ext[0] = TA;
        I.tile_ext[q] = TB;
        const double waste = padded / real;
        // measured: rows of A shorter than 256 bytes make the bulk copies too many (448 against 152 us on 27 x 179 x 115 x 94);
        // such variants rank behind the ring kernel's candidates (whose fitted costs are about 2 for unaligned rows)
        I.est_cost = (float)((1.20 + 0.01 * n_added) * waste * (std::min<int64_t>(TA, LA) * es < 256 ? 2.0 : 1.0) * (TB * es < 256 ? 1.15 : 1.0) *
                             (v.direct ? 1.0 : 1.5));
        cand.feat[2] = (float)waste;
        cand.feat[4] = (float)stage;
        cand.feat[5] = (float)n_tiles;
        cand.feat[12] = beta_nz ? 1.f : 0.f;
        cand.feat[13] = (float)TTC_KERNEL_SKEW;
        out->push_back(cand);
        ++n_added;
    }
}

}  // namespace

void generate_candidates(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int sm_count,
                         int max_smem_optin, std::vector<Candidate>* out) {
    (void)sm_count;
    out->clear();
    if (c.empty || c.rank == 0) return;
    const int es = elem_size(dtype);
    const int mvA = 16 / elem_size(dtype_a), mvB = 16 / es, mvS = std::min(mvA, mvB);
    const int max_smem = std::min(max_smem_optin > 0 ? max_smem_optin : 48 * 1024, 160 * 1024);

    // Work distribution (row H6): dynamic (cluster launch control) unless TTC_SCHED says
    // "static" (persistent grid-stride) or "both" (both variants compete in the tuner).
    std::vector<int> scheds = {1};
    if (const char* e = std::getenv("TTC_SCHED")) {
        if (!std::strcmp(e, "static")) scheds = {0};
        else if (!std::strcmp(e, "both")) scheds = {1, 0};
        else if (!std::strcmp(e, "atomic")) scheds = {2};
        else if (!std::strcmp(e, "all")) scheds = {1, 2, 0};
    }

    // TTC_VARIANTS: bit 0 = staggered-gather ring candidates, bit 1 = shifted-row ring candidates, bit 2 = tensor-map
    // candidates, bit 3 = skew-kernel candidates that store to B directly (default 15: all of these), bit 4 = the skew
    // kernel's out-tile variants (correct but measured 2x slower: only on request)
    const int variants = std::getenv("TTC_VARIANTS") ? std::atoi(std::getenv("TTC_VARIANTS")) : 15;
    const int xp_max = (variants & 1) ? 1 : 0;
    const int n_loop_orders = std::getenv("TTC_LOOP_ORDERS") ? std::max(2, std::min(4, std::atoi(std::getenv("TTC_LOOP_ORDERS")))) : 2;
    const int ring_max = std::getenv("TTC_RING") ? std::atoi(std::getenv("TTC_RING")) : 4;

    // K1 / fallback: direct kernels (always at least the scalar one, valid for any strides).
    for (int sched : scheds)
        for (int lo = 0; lo < 2; ++lo) {
            add_direct(c, dtype, dtype_a, beta_nz, lo, true, sched, out);
            add_direct(c, dtype, dtype_a, beta_nz, lo, false, sched, out);
        }

    // Tensor-map candidates (TTC_VARIANTS bit 2).
    if (variants & 4)
        for (int sched : scheds) {
            add_tmap(c, dtype, dtype_a, beta_nz, sched, max_smem, out);
            add_tmapu(c, dtype, dtype_a, beta_nz, sched, max_smem, out);
        }
    // Skew-kernel candidates (TTC_VARIANTS bits 3 and 4).
    if (variants & 8)
        for (int sched : scheds) add_skew(c, dtype, dtype_a, beta_nz, sched, max_smem, out);

    // K2 / K3: tiles.  A side = leading indices of A, B side = leading indices of B.
    std::vector<int> orderA, orderB;
    for (int i = 0; i < c.rank; ++i) { orderA.push_back(i); orderB.push_back(c.orderB[i]); }
    bool fits32 = true;
    for (int i = 0; i < c.rank; ++i) fits32 &= c.d[i].e < kInt31;
    if (fits32 && c.rank >= 2) {
        std::vector<SideOpt> optsA;
        int32_t none[kMaxRank] = {0};
        side_options(c, orderA, none, mvA, es, &optsA);
        std::set<std::string> seen;
        for (const SideOpt& ua : optsA) {
            int32_t taken[kMaxRank] = {0};
            for (auto& d : ua.dims) taken[d.first] = d.second;
            std::vector<SideOpt> optsB;
            side_options(c, orderB, taken, mvB, es, &optsB);
            for (const SideOpt& wb : optsB) {
                const int64_t bytes = ua.elems * wb.elems * es;
                if (bytes < 2048 || bytes > max_smem) continue;
                TileSpec spec;
                for (int i = 0; i < kMaxRank; ++i) spec.t[i] = 1;
                for (auto& d : ua.dims) spec.t[d.first] = d.second;
                for (auto& d : wb.dims) spec.t[d.first] = d.second;
                std::string key((const char*)spec.t, sizeof(int32_t) * c.rank);
                if (!seen.insert(key).second) continue;
                // {8, 8}: mixed precision only -- one vector width (mvS elements) on both sides
                static const int vopts[5][2] = {{16, 16}, {16, 1}, {1, 16}, {1, 1}, {8, 8}};
                for (int lo = 0; lo < n_loop_orders; ++lo) {
                    for (auto& vo : vopts) {
                        const int va = vo[0] == 16 ? mvA : vo[0] == 8 ? mvS : 1, vb = vo[1] == 16 ? mvB : vo[1] == 8 ? mvS : 1;
                        if ((mvA == 1 && vo[0] == 16) || (mvB == 1 && vo[1] == 16)) continue;
                        if (vo[0] == 8 && (mvA == mvB || mvS == 1)) continue;
                        for (int sched : scheds)
                            for (int ring = 0; ring <= ring_max; ring += 2) {
                                if (ring && bytes * ring > 64 * 1024) continue;   // 2 buffers <= 32 KB, 4 <= 16 KB
                                for (int xp = 0; xp <= (ring ? xp_max : 0); ++xp)
                                    for (int rowmode = 1; rowmode <= (ring && !xp && (variants & 2) ? 2 : 1); ++rowmode) {
                                        Candidate cand;
                                        if (build_tile_candidate(c, dtype, dtype_a, beta_nz, spec, lo, va, vb, max_smem, sched, ring, xp,
                                                                 rowmode, true, &cand)) {
                                            cand.recipe = Recipe{spec, lo, va, vb, sched, ring, xp, rowmode};
                                            out->push_back(cand);
                                        }
                                    }
                            }
                    }
                }
            }
        }
    }

    // Bounded list ordered by estimated cost.
    auto by_cost = [](const Candidate& a, const Candidate& b) { return a.info.est_cost < b.info.est_cost; };
    std::stable_sort(out->begin(), out->end(), by_cost);
    if ((int)out->size() > kMaxImplementations) {
        // keep the scalar direct fallback whatever its rank
        Candidate fallback;
        bool have = false;
        for (auto& cd : *out)
            if (cd.info.kernel == TTC_KERNEL_COPY && cd.info.vec_a == 1) { fallback = cd; have = true; break; }
        out->resize(kMaxImplementations);
        bool kept = false;
        for (auto& cd : *out) kept |= (cd.info.kernel == TTC_KERNEL_COPY && cd.info.vec_a == 1);
        if (have && !kept) out->back() = fallback;
    }
    // Second pass: the head of the list (what the tuner times by default) gets the full shared-memory padding
    // search of the bank model; the tail keeps its dense tiles (still complete, launchable candidates).
    const int n_full = std::min<int>((int)out->size(), std::getenv("TTC_FULL_SEARCH") ? std::atoi(std::getenv("TTC_FULL_SEARCH")) : kFullSearch);
    for (int i = 0; i < n_full; ++i) {
        Candidate& cd = (*out)[i];
        if (cd.info.kernel == TTC_KERNEL_COPY || cd.info.kernel == TTC_KERNEL_TENSORMAP || cd.info.kernel == TTC_KERNEL_SKEW) continue;
        const Recipe r = cd.recipe;
        Candidate full;
        if (build_tile_candidate(c, dtype, dtype_a, beta_nz, r.spec, r.loop_order, r.va, r.vb, max_smem, r.sched, r.ring, r.xp,
                                 r.rowmode, false, &full)) {
            full.recipe = r;
            cd = full;
        }
    }
    std::stable_sort(out->begin(), out->end(), by_cost);
}

}  // namespace ttc
