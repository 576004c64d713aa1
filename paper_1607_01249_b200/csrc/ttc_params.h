// ttc_params.h -- plain-old-data kernel parameter blocks and the helpers shared by host planner and device
// code.  Nothing else is included from here, so the file also compiles under NVRTC (run-time
// specialisation of a tuned kernel, specialize.cpp).  Not visible through the C ABI; not shared with oracle/.
#pragma once
#if defined(__CUDACC_RTC__)
typedef unsigned char uint8_t;
typedef int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
typedef unsigned long long uintptr_t;
#else
#include <cstdint>
#endif

#if defined(__CUDACC__)
#define TTC_HD __host__ __device__ __forceinline__
#else
#define TTC_HD inline
#endif

namespace ttc {

constexpr int kMaxRank = 16;         // == TTC_MAX_RANK of include/ttc.h (checked in ttc_internal.h)
constexpr int kMaxTab = 6;           // canonical indices enumerated by one offset table
constexpr int kMaxTabEntries = 2048; // entries of one offset table
constexpr int kTileThreads = 256;    // default CTA size of the tile kernel
constexpr int kRingMaxStages = 4;    // ring kernel: most tile buffers per CTA
constexpr int kRingThreads = 32 + 256;  // ring kernel: producer warp + consumer warps (launch bound)
constexpr int kDirectThreads = 256;  // CTA size of the direct kernel
constexpr int kDirectUnroll = 4;     // vectors per thread and work item of the direct kernel
// element types (== ttc_dtype of include/ttc.h)
constexpr int kF32 = 0, kF64 = 1, kC64 = 2, kC128 = 3;

// ---------------------------------------------------------------------------------------
// Fast division of a 31-bit numerator by a plan-time constant (Granlund-Montgomery):
//   s = ceil(log2 d), m = floor(2^32 (2^s - d) / d) + 1, n / d = (mulhi(m, n) + n) >> s
// exact for 0 <= n < 2^31 (the sum cannot overflow 32 bits).  SURVEY.md 8(a) row H6.
// ---------------------------------------------------------------------------------------
struct FastDiv {
    uint32_t d, m, s, pad;
};

#if !defined(__CUDACC_RTC__)
inline FastDiv make_fastdiv(uint32_t d) {
    FastDiv f{d, 1u, 0u, 0u};
    if (d <= 1) { f.d = 1; return f; }
    uint32_t s = 0;
    while ((1ull << s) < d) ++s;
    f.s = s;
    f.m = (uint32_t)((((1ull << s) - d) << 32) / d + 1);
    return f;
}
#endif

TTC_HD uint32_t fd_div(uint32_t n, const FastDiv& f) {
#if defined(__CUDA_ARCH__)
    return (__umulhi(f.m, n) + n) >> f.s;
#else
    return (uint32_t)(((((uint64_t)f.m * n) >> 32) + n) >> f.s);
#endif
}

TTC_HD void fd_divmod(uint32_t n, const FastDiv& f, uint32_t& q, uint32_t& r) {
    q = fd_div(n, f);
    r = n - q * f.d;
}

// ---------------------------------------------------------------------------------------
// Kernel parameter blocks (passed by value as __grid_constant__).
// ---------------------------------------------------------------------------------------

// K1 (and the always-valid fallback): direct global->global.  Item q (one vector of `vec`
// elements along dims[0], or one element) is split by successive fast-divmods over
// dims[0..nd) (dims[0] fastest; the order of the others is the candidate's loop order).
struct DirectDim {
    FastDiv div;        // by the number of items along this dim
    int64_t sA, sB;     // element stride per item step (already multiplied by vec for dim 0)
    uint64_t n;         // items along this dim (64-bit path)
};
struct DirectParams {
    int nd;
    int vec;            // elements per item
    int dyn;            // work distribution: 0 static grid-stride, 1 cluster launch control, 2 atomic counter
    uint32_t* ctr;      // dyn == 2: device counter of the plan (set at launch)
    uint32_t n_chunks;  // work items: chunks of kDirectThreads * kDirectUnroll vectors
    uint64_t n_items;
    DirectDim dims[kMaxRank];
};

// K2/K3: macro-tile = box of tile extents t_i over the canonical indices (t_i = 1 outside the
// tile).  Two enumerations of the box: phase A (ascending stride in A, used by the load) and
// phase B (ascending stride in B, used by the store).  Each enumeration is factorised into a
// fast ("lo") and a slow ("hi") group of indices; the kernel builds one table per group that
// gives (offset in the global tensor, offset in the shared-memory tile) of every group entry.
struct TabDim {
    FastDiv div;        // by `n`
    int32_t n;          // entries along this index = t / step
    int32_t step;       // elements per entry step (vec for the vectorised leading index, else 1)
    int32_t gslot;      // position of this index in TileParams::g (for edge-tile validity)
    int32_t vmul;       // entry c is valid iff c * step < vext[gslot] * vmul (vmul > 1: fused leading pair)
    int32_t sS;         // shared-memory stride per entry step (elements)
    int32_t aS;         // shifted rows (row_async == 2), B-side tables: stride in A per entry step, mod the vector
                        // width, of an index that selects the tile ROW (0 for the indices a row runs along)
    int64_t sG;         // global stride per entry step (elements)
};
struct Table {
    int32_t nd;
    int32_t n;          // product of TabDim::n
    TabDim d[kMaxTab];
};
struct GridDim {        // one coordinate of the macro-tile grid, in loop order (first = fastest)
    FastDiv div;        // by the number of tiles along this index
    int64_t sA, sB;     // element strides of the index
    int32_t e;          // full extent of the index
    int32_t t;          // tile extent (1 if the index is outside the tile)
};
struct TileParams {
    int nG;
    int vecA, vecB;     // elements per global access in the load / store phase
    int same;           // 1: the vectorised index leads A and B (chunks move unchanged)
    int sstepB;         // smem stride between the vecB elements one store gathers (!same)
    int splitA;         // 1: a loaded vector is written to the tile as vecA element stores
    int xp;             // ring kernel: 1 = staggered gather (rows of a store vector read in a lane-dependent rotation)
    int ring;           // > 0: ring kernel with this many tile buffers (producer warp + consumer warps)
    uint32_t row_bytes; // ring kernel: bytes of one tile row (one cp.async.bulk each); rows = tab[1].n
    int row_pairs;      // ring kernel, cp.async rows of 4-byte elements: 1 = every row is 8-byte aligned (copy pairs)
    int row_async;      // ring kernel, rows not 16-byte aligned: 1 = copied with element-sized cp.async; 2 = "shifted
                        // rows": the 16-byte aligned body of a row is one bulk copy, landed at the row's own
                        // misalignment (0..3 elements) in the tile, the < 16-byte head and tail are element cp.async
    int shift_ld;       // row_async == 2: A-stride of B's leading index mod the vector width (skew step per B element)
    int peel, peel_len, peel_gslot;   // ring kernel, peeled store phase: B rows cut into aligned 16-byte windows
    int lead_gslot, lead_vmul;   // ring kernel: grid slot of the row's index and its validity multiplier
    int threads;
    int dyn;            // work distribution: 0 static grid-stride, 1 cluster launch control, 2 atomic counter
    uint32_t* ctr;      // dyn == 2: device counter of the plan (set at launch)
    uint32_t n_tiles;
    uint32_t itemsA, itemsB;      // table entries per tile: Alo.n*Ahi.n, Blo.n*Bhi.n
    uint32_t tile_elems;          // shared-memory tile size in elements (with padding)
    FastDiv divAlo, divBlo;       // item -> (lo, hi)
    Table tab[4];                 // 0: A lo, 1: A hi, 2: B lo, 3: B hi
    GridDim g[kMaxRank];
};

// Batched execution (ttc_execute_batched): up to kMaxBatch problems that share one plan run in ONE launch;
// work item w belongs to problem w / per.  n == 0: a single problem, the kernel's own A and B arguments.
constexpr int kMaxBatch = 64;
struct BatchPtrs {
    int n;
    uint32_t per;               // work items (macro-tiles / chunks) per problem
    FastDiv div;                // by `per`
    const void* a[kMaxBatch];
    void* b[kMaxBatch];
};

// Shared-memory carve-up (bytes), identical on host and device.
struct TileSmemLayout {
    uint32_t tab[4];     // int2 tables
    uint32_t val[4];     // uint8 validity of each table entry (edge tiles only)
    uint32_t vext;       // int32 valid extent per grid index
    uint32_t tile;       // tile data (16-byte aligned); ring kernel: `ring` buffers of tile_stride bytes
    uint32_t tile_stride;
    uint32_t rval, rval_stride;   // ring kernel: per-buffer validity bytes of tables 2 and 3 (edge tiles)
    uint32_t rvext;               // ring kernel: per-buffer valid extents (kMaxRank int32 each)
    uint32_t total;
};
TTC_HD TileSmemLayout tile_smem_layout(const TileParams& P, int es) {
    TileSmemLayout L;
    uint32_t o = 0;
    for (int i = 0; i < 4; ++i) { L.tab[i] = o; o += 8u * (uint32_t)P.tab[i].n; }
    for (int i = 0; i < 4; ++i) { L.val[i] = o; o += ((uint32_t)P.tab[i].n + 3u) & ~3u; }
    L.vext = o; o += 4u * kMaxRank;
    L.rval = o;
    L.rval_stride = (((uint32_t)P.tab[2].n + 3u) & ~3u) + (((uint32_t)P.tab[3].n + 3u) & ~3u);
    L.rvext = L.rval + L.rval_stride * (uint32_t)(P.ring > 0 ? P.ring : 0);
    o = L.rvext + 4u * kMaxRank * (uint32_t)(P.ring > 0 ? P.ring : 0);
    o = (o + 15u) & ~15u;
    L.tile = o;
    L.tile_stride = (P.tile_elems * (uint32_t)es + 15u) & ~15u;
    o += L.tile_stride * (uint32_t)(P.ring > 0 ? P.ring : 1);
    L.total = o;
    return L;
}

struct Scalar {         // alpha or beta, as doubles (re, im); narrowed in the launcher
    double re, im;
};

}  // namespace ttc
