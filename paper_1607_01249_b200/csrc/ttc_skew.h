// ttc_skew.h -- parameter block of skew_kernel (ttc_skew.cuh): transposition of tensors whose rows are NOT 16-byte
// aligned (odd extents of 4- and 8-byte elements), with 1-D bulk copies (cp.async.bulk, UBLKCP) in BOTH directions.
// Tensor maps cannot express such tensors (a box must start on a 16-byte boundary, a store clips in
// 16-byte granules), and the ring kernel's consumers pay ~55 instructions per element for element-wise global stores of
// unaligned rows.  Here every tile row is copied as the 16-byte aligned superset of its bytes and lands in shared memory
// at its own skew (= misalignment of its first element, in elements); consumers move elements between the skewed
// in-rows and the skewed out-rows; the aligned body of every out-row goes back with one bulk store, the < 16-byte head
// and tail with element stores.  Plain data, host and device.
#pragma once
#include <cstdint>

#include "ttc_params.h"

namespace ttc {

constexpr int kSkewMaxStages = 4;
constexpr int kSkewMaxPlanes = 8;
constexpr int kSkewMaxRows = 512;      // rows of one side of a tile (planes x tile extent)

struct SkewParams {
    int dyn;
    uint32_t* ctr;
    uint32_t n_tiles;
    int stages, threads;
    int np, ns;                    // producer warps, store warps (the rest of the CTA's warps are consumers)
    int lgTA, lgTB;                // tile extents along a0 and b0 are powers of two
    int nP;                        // planes (index combinations of the other indices) per tile
    int nG;                        // tile-grid dimensions: 0 = a0, 1 = b0, then the other canonical indices
    int pitchA, pitchB;            // bytes per shared-memory row of the in-tile / out-tile (multiples of 16)
    int64_t e0, eq;                // lengths of the A-run and of the B-run
    int64_t spanA, spanB;          // elements from the first to one past the last element of A / B
    FastDiv gdiv[kMaxRank];
    int64_t stepA[kMaxRank], stepB[kMaxRank];   // element offset per tile index of grid dimension >= 2
    int64_t pA[kSkewMaxPlanes], pB[kSkewMaxPlanes];
    // Runs: the tile's a-range is a range of positions in the A-run = the first nA indices of A merged (they are
    // contiguous in A: lda == extent), its b-range a range of positions in the B-run = the first nB indices of B merged.
    // Position -> element offset in the OTHER tensor goes index by index (divX by the extents, innermost first).
    int nA, nB;
    FastDiv divA[3], divB[3];
    int64_t sBA[3];                // strides in B of the A-run's indices
    int64_t sAB[3];                // strides in A of the B-run's indices
};

}  // namespace ttc
