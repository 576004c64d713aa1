// ttc_tmap.h -- parameter blocks of the tensor-map kernel (tmap_kernel, ttc_tmap.cuh): tiles move between global and
// shared memory as <= 5-D boxes of a CUtensorMap (cp.async.bulk.tensor, SASS UTMALDG / UTMASTG) in BOTH directions;
// the threads never touch global memory.  north_star K2 "TMA tensor-map loads and stores of <= 5-D boxes where the
// strides allow"; SURVEY.md section 7 step 7 and the TMA feasibility paragraph of 8(d).  Plain data, host and device.
#pragma once
#include <cstdint>

#include "ttc_params.h"

namespace ttc {

constexpr int kTmapRank = 5;         // every map is encoded with 5 dimensions (missing ones have extent 1)
constexpr int kTmapMaxStages = 4;
constexpr int kTmapMaxBoxes = 8;     // boxes per tile (nbA * nbB)

// flavour 0 (transposing: the stride-1 index of A is not the stride-1 index of B)
//   A's map lists the canonical indices as (a0, b0, o1, o2, o3), B's map as (b0, a0, o1, o2, o3); a box has 128 bytes
//   along a0 resp. b0 (SWIZZLE_128B) and 128 / es elements along the other of the two, so it is a stack of
//   `planes` square 2-D planes (one per (o1, o2, o3) of the box) that the consumer warps transpose from the in-box
//   to the out-box with 16-byte shared-memory accesses only.
// flavour 1 (copy class: a0 == b0): both maps list the indices in B's order, in-box and out-box have the same
//   layout (no swizzle), the threads only apply alpha and beta chunk by chunk -- or nothing at all for a real
//   alpha == 1, beta == 0, when the box is stored straight from the buffer it was loaded into.
struct TmapParams {
    int flavour;
    int dyn;                  // work distribution (WorkSched mode)
    uint32_t* ctr;            // atomic work counter (mode 2), filled in at launch
    uint32_t n_tiles;
    int stages, threads;
    int nbA, nbB;             // boxes per tile along map dimension 0 of A / of B (flavour 1: nbB == 1)
    int planes;               // flavour 0: planes per box
    int ca, cb;               // flavour 0: 16-byte chunks per in-row / per out-row (8: 128-byte rows, 4: 64-byte rows)
    uint32_t box_bytes;       // bytes of one box (the same for A's and B's map)
    uint32_t buf_bytes;       // nbA * nbB * box_bytes rounded up to 128 (a box's shared-memory address must be 128-byte aligned)
    int upe;                  // map units per element along a map's dimension 0 (2 for 16-byte elements: 8-byte units)
    FastDiv gdiv[kTmapRank];  // number of tiles along A-map dimension d
    int32_t step[kTmapRank];  // tile extent (elements) along A-map dimension d
    int32_t box0[2];          // box extent (elements) along A-map dimension 0 and 1 (the step between the boxes of a tile)
    int batchable;            // the fifth map dimension is unused (planner): ttc_execute_batched can use the candidate
};

// ttc_execute_batched through ONE pair of maps: when the fifth map dimension is free (canonical rank <= 4) it gets a stride
// of 16 bytes, and problem i of the batch is addressed by the coordinate (A_i - min A) / 16 along it (B alike): a dimension
// with a 16-byte stride reaches any 16-byte aligned address.  Work item w belongs to problem w / per.
struct TmapBatch {
    int n;
    uint32_t per;
    FastDiv div;
    int32_t offA[kMaxBatch], offB[kMaxBatch];
};

// What cuTensorMapEncodeTiled needs beside the base address (filled by the planner; encoded at launch).
struct TmapEncode {
    int unit_bytes;                       // 4 or 8: CU_TENSOR_MAP_DATA_TYPE_UINT32 / UINT64
    int swzA, swzB;                       // CUtensorMapSwizzle of A's / B's map: 0 none, 1 32-byte, 2 64-byte, 3 128-byte rows
    uint64_t dimA[kTmapRank], dimB[kTmapRank];
    uint64_t strideA[kTmapRank - 1], strideB[kTmapRank - 1];   // bytes, dimensions 1..4
    uint32_t boxA[kTmapRank], boxB[kTmapRank];
};

// ------------------------------------------------------------------------------------------
// flavour 2: more than 5 canonical indices (4- and 8-byte elements).  The rows of a T x T plane (T = 128 / es) are split
// into V = 16 / es classes by row index mod V; a row's offset R = class * stride + (offset of the tile's outer indices) is
// expressed as the coordinate R / V of a map dimension with a 16-byte stride, which can address ANY 16-byte aligned offset
// and so absorbs every index beyond the plane: no rank limit.  The design also carries a skew R % V as a shift of the
// coordinate along the row (for strides that are not multiples of 16 bytes, with 2 V maps per tensor, indexed
// [skew * 2 + (0: classes with one row more, 1: the others)], for exact clipping) -- but the hardware raises "illegal
// instruction" for a box whose first byte is not 16-byte aligned (measured: coordinate 17 of an fp64 map fails, 18
// works), so only skew 0 is ever used and the planner offers this flavour for aligned strides only.  A plane is 2 V
// sub-boxes of 1 KB (8 rows of 128 bytes, 128-byte swizzle); the thread that owns micro-tile (A2, B2) reads row B2,
// chunk A2 of the V in-sub-boxes and writes row A2, chunk B2 of the V out-sub-boxes: the sub-box index IS the position
// inside the micro-tile.
// ------------------------------------------------------------------------------------------
constexpr int kTmapUMaxPlanes = 8;
constexpr int kTmapUMaxClasses = 4;

struct TmapUParams {
    int dyn;
    uint32_t* ctr;
    uint32_t n_tiles;
    int stages, threads;
    int V, T;                      // classes (= elements per 16 bytes) and plane edge (elements)
    int nP;                        // planes per tile
    int nG;                        // tile-grid dimensions: 0 = a0, 1 = b0, then the other canonical indices
    int skewA0, skewB0;            // misalignment of the base addresses in elements, filled in at launch
    int remA, remB;                // rows of A's planes (b0 extent) mod V, rows of B's planes (a0 extent) mod V: classes below have one row more
    FastDiv gdiv[kMaxRank];
    int64_t stepA[kMaxRank], stepB[kMaxRank];   // element offset per tile index of grid dimension >= 2
    int64_t pA[kTmapUMaxPlanes], pB[kTmapUMaxPlanes];   // element offsets of the tile's planes
    int64_t sqA, s0B;              // stride of b0 in A, of a0 in B (elements)
};

struct TmapUEncode {
    int es;
    int64_t e0, eq;                // extents of a0 and b0
    int64_t sqA, s0B;
    int64_t spanA, spanB;          // elements
};

}  // namespace ttc
