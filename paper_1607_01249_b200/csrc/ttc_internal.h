// ttc_internal.h -- structures shared by the host planner and the CUDA kernels of libttc.so.
// Nothing here is visible through the C ABI (include/ttc.h).  Not shared with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "ttc.h"
#include "ttc_params.h"
#include "ttc_tmap.h"
#include "ttc_skew.h"

namespace ttc {

static_assert(kMaxRank == TTC_MAX_RANK, "ttc_params.h and include/ttc.h disagree on the maximum rank");
static_assert(kF32 == TTC_F32 && kF64 == TTC_F64 && kC64 == TTC_C64 && kC128 == TTC_C128, "dtype codes");

// ---------------------------------------------------------------------------------------
// Canonical transposition (stage 1): (extent, stride in A, stride in B) per
// index, ascending stride in A, no extent-1 index, nothing left to merge.
// ---------------------------------------------------------------------------------------
struct CanonDim {
    int64_t e, sA, sB;
};

struct Canon {
    int rank = 0;
    CanonDim d[kMaxRank];
    int64_t numel = 0;
    int64_t spanA = 0, spanB = 0;  // 1 + max offset (elements); 0 if empty
    bool empty = false;
    int orderB[kMaxRank];          // canonical indices by ascending stride in B
};

ttc_status canonicalize(int N, const int64_t* sizes, const int* perm, const int64_t* lda,
                        const int64_t* ldb, Canon* out);
ttc_status canonicalize_strided(int N, const int64_t* sizes, const int* perm, const int64_t* stride_a,
                                const int64_t* stride_b, Canon* out);



// ---------------------------------------------------------------------------------------
// A candidate = kernel class + blocking + loop order + launch shape.
// ---------------------------------------------------------------------------------------
struct TileSpec {
    int32_t t[kMaxRank];   // tile extent per canonical index (1 = outside the tile)
};
struct Recipe {             // what build_tile_candidate was called with (to build the candidate again)
    TileSpec spec;
    int loop_order, va, vb, sched, ring, xp, rowmode;
};
struct Candidate {
    ttc_candidate_info info{};
    bool beta_nz = false;
    bool idx64 = false;          // K1: item count / offsets need 64-bit arithmetic
    int  align_a = 1, align_b = 1;  // required pointer alignment in bytes
    DirectParams dp{};
    TileParams tp{};
    TmapParams mp{};             // TTC_KERNEL_TENSORMAP: kernel parameters and what the two tensor maps are encoded from
    TmapEncode me{};
    SkewParams sp{};             // TTC_KERNEL_SKEW
    TmapUParams up{};            // TTC_KERNEL_TENSORMAP with mp.flavour == 2 (residue classes)
    TmapUEncode ue{};
    float feat[16] = {0};        // raw inputs of the cost heuristic (plan.cpp), exported for re-fitting
    Recipe recipe{};
    int grid_cap = 0;            // resident CTAs the device holds of this kernel (set by prepare_candidate)
};

// `dtype` is B's element type -- the type Eq. 1 is evaluated in and the type of the shared-memory
// tile; `dtype_a` is A's.  They differ only for the mixed-precision pairs sd, ds, cz, zc
// (PAPER.md:75, 87): A's elements are then converted as they are loaded (reading M1).
void generate_candidates(const Canon& c, ttc_dtype dtype, ttc_dtype dtype_a, bool beta_nz, int sm_count,
                         int max_smem_optin, std::vector<Candidate>* out);

// Launch one candidate.  Returns the CUDA error code (0 = success) as int.
int launch_candidate(const Candidate& cand, ttc_dtype dtype, ttc_dtype dtype_a, const Scalar& alpha,
                     const Scalar& beta, const void* A, void* B, void* stream, uint32_t* sched_ctr,
                     const BatchPtrs* batch = nullptr);
// Configure dynamic shared memory / occupancy-derived grid for a candidate (needs a device).
int prepare_candidate(Candidate* cand, ttc_dtype dtype, ttc_dtype dtype_a, int sm_count);

// Run-time specialisation (specialize.cpp): NVRTC twin of a prepared ring-kernel candidate.
struct SpecKernel;
bool nvrtc_available();
SpecKernel* specialize_candidate(const Candidate& c, int pair, std::string* err);
void release_specialized(SpecKernel* k);
int launch_specialized(const SpecKernel* k, const Candidate& c, const Scalar& alpha, const Scalar& beta, const void* A,
                       void* B, void* stream);
std::string spec_source(const Candidate& c, int pair, std::string* name);
bool nvrtc_compile(const std::string& src, const std::string& name, const std::string& arch, std::string* cubin,
                   std::string* lowered, std::string* log_out);
int pair_id(ttc_dtype dtype, ttc_dtype dtype_a);     // kernels.cu: 0..3 same type, 4..7 sd, ds, cz, zc

// static_scratch.cu: staging of ttc_execute_host_static inside the file-scope device array (no allocation).
bool static_scratch_fits(size_t bytes_a, size_t bytes_b);
int static_scratch_run(const Candidate& cand, ttc_dtype dtype, ttc_dtype dtype_a, const Scalar& alpha, const Scalar& beta,
                       const void* A_host, size_t bytes_a, void* B_host, size_t bytes_b, bool b_in, void* stream);

inline int elem_size(ttc_dtype t) {
    switch (t) {
        case TTC_F32: return 4;
        case TTC_F64: return 8;
        case TTC_C64: return 8;
        default: return 16;
    }
}

// Mixed-precision pairs the library accepts: sd, ds, cz, zc; equal types always.
inline bool valid_pair(ttc_dtype a, ttc_dtype b) {
    if ((int)a < 0 || (int)a > 3 || (int)b < 0 || (int)b > 3) return false;
    if (a == b) return true;
    return (a == TTC_F32 && b == TTC_F64) || (a == TTC_F64 && b == TTC_F32) ||
           (a == TTC_C64 && b == TTC_C128) || (a == TTC_C128 && b == TTC_C64);
}

// Elements per vector access: a vector is at most 16 bytes in A, in B and in the tile.
inline int max_vec(ttc_dtype dtype, ttc_dtype dtype_a) {
    const int ea = elem_size(dtype_a), eb = elem_size(dtype);
    return 16 / (ea > eb ? ea : eb);
}

}  // namespace ttc
