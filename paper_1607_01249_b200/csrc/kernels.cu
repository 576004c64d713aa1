// kernels.cu -- the sm_100a kernels of libttc.so and their launchers.
//
//   direct_kernel  K1 of SURVEY.md 8(a): global -> global, one 4..16-byte vector per item along
//                  the index that is stride-1 in A and in B ("copy a whole column
//                  at a time"); also the always-valid scalar fallback for any strides.
//   tile_kernel    K2/K3: one macro-tile per CTA iteration, staged through
//                  shared memory (the micro-tile transpose is done in shared memory
//                  on CUDA).  The tile is an N-D box, so several small leading indices can be
//                  coarsened into each side; 16-byte global accesses on both sides; the read of
//                  B for beta != 0 is fused into the store phase; persistent CTAs take macro-tiles
//                  in the candidate's loop order through WorkSched.
//   ring_kernel    K2/K3, warp-specialised: a producer warp loads the tile rows with TMA bulk copies
//                  into a ring of tile buffers, consumer warps run tile_kernel's store phase.
//   tmap_kernel    K1/K2/K3 for tensors whose strides a CUtensorMap can express (ttc_tmap.cuh): tensor-map
//                  box loads, in-register micro-tile transposition between swizzled shared-memory boxes,
//                  tensor-map box stores.
//
// Arithmetic (Eq. 1): every product and sum is rounded separately
// (__fmul_rn/__fadd_rn, never contracted into FMA) so the result is bit-identical to the
// definition evaluated in the tensor's own precision (reading A7).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <set>
#include <type_traits>

#include "ttc_internal.h"

#include "ttc_device.cuh"
#include "ttc_tmap.cuh"
#include "ttc_skew.cuh"

namespace ttc {

int pair_id(ttc_dtype dtype, ttc_dtype dtype_a) {
    if (dtype == dtype_a) return (int)dtype;
    if (dtype_a == TTC_F32 && dtype == TTC_F64) return kPairSD;
    if (dtype_a == TTC_F64 && dtype == TTC_F32) return kPairDS;
    if (dtype_a == TTC_C64 && dtype == TTC_C128) return kPairCZ;
    if (dtype_a == TTC_C128 && dtype == TTC_C64) return kPairZC;
    return -1;
}

// ------------------------------------------------------------------------------------------
// Dispatch: (dtype, vector widths, beta != 0) -> kernel instance
// ------------------------------------------------------------------------------------------
// Kernel instances are handed around as untyped entry points (their last parameter's type differs between
// the single-problem and the batched instantiation) and launched with cudaLaunchKernelExC.
using KernelFn = const void*;

template <int DT, int VA, int VB, bool SAME>
static KernelFn tile_fn_beta(bool beta, bool batched) {
    if (batched)
        return beta ? (KernelFn)tile_kernel<DT, VA, VB, SAME, true, BatchPtrs> : (KernelFn)tile_kernel<DT, VA, VB, SAME, false, BatchPtrs>;
    return beta ? (KernelFn)tile_kernel<DT, VA, VB, SAME, true, NoBatch> : (KernelFn)tile_kernel<DT, VA, VB, SAME, false, NoBatch>;
}

template <int DT>
static KernelFn tile_fn(int va, int vb, bool same, bool beta, bool batched) {
    // 16-byte vectors of each side's own type; MS: the one width that fits both (wide class, and the
    // extra equal-width variant of the mixed-precision pairs)
    constexpr int MVA = 16 / (int)sizeof(typename ElemT<DT>::TA), MVB = 16 / ElemT<DT>::ES;
    constexpr int MS = MVA < MVB ? MVA : MVB;
    if constexpr (MS > 1) {
        if (same && va == MS && vb == MS) return tile_fn_beta<DT, MS, MS, true>(beta, batched);
    }
    if (same) return nullptr;
    if constexpr (MVA > 1 && MVB > 1) {
        if (va == MVA && vb == MVB) return tile_fn_beta<DT, MVA, MVB, false>(beta, batched);
    }
    if constexpr (MVA != MVB && MS > 1) {
        if (va == MS && vb == MS) return tile_fn_beta<DT, MS, MS, false>(beta, batched);
    }
    if constexpr (MVA > 1) {
        if (va == MVA && vb == 1) return tile_fn_beta<DT, MVA, 1, false>(beta, batched);
    }
    if constexpr (MVB > 1) {
        if (va == 1 && vb == MVB) return tile_fn_beta<DT, 1, MVB, false>(beta, batched);
    }
    if (va == 1 && vb == 1) return tile_fn_beta<DT, 1, 1, false>(beta, batched);
    return nullptr;
}

template <int DT, int V>
static KernelFn direct_fn_v(bool beta, bool idx64, bool batched) {
    if (batched) {
        if (beta) return idx64 ? (KernelFn)direct_kernel<DT, V, true, true, BatchPtrs> : (KernelFn)direct_kernel<DT, V, true, false, BatchPtrs>;
        return idx64 ? (KernelFn)direct_kernel<DT, V, false, true, BatchPtrs> : (KernelFn)direct_kernel<DT, V, false, false, BatchPtrs>;
    }
    if (beta) return idx64 ? (KernelFn)direct_kernel<DT, V, true, true, NoBatch> : (KernelFn)direct_kernel<DT, V, true, false, NoBatch>;
    return idx64 ? (KernelFn)direct_kernel<DT, V, false, true, NoBatch> : (KernelFn)direct_kernel<DT, V, false, false, NoBatch>;
}

template <int DT>
static KernelFn direct_fn(int vec, bool beta, bool idx64, bool batched) {
    constexpr int MV = max_vec_of<DT>();
    if constexpr (MV > 1) {
        if (vec == MV) return direct_fn_v<DT, MV>(beta, idx64, batched);
    }
    if (vec == 1) return direct_fn_v<DT, 1>(beta, idx64, batched);
    return nullptr;
}

template <int DT, int VB, bool PEEL, bool SHIFT>
static KernelFn ring_fn_inst(bool beta, bool batched) {
    if (batched)
        return beta ? (KernelFn)ring_kernel<DT, VB, true, PEEL, SHIFT, BatchPtrs> : (KernelFn)ring_kernel<DT, VB, false, PEEL, SHIFT, BatchPtrs>;
    return beta ? (KernelFn)ring_kernel<DT, VB, true, PEEL, SHIFT, NoBatch> : (KernelFn)ring_kernel<DT, VB, false, PEEL, SHIFT, NoBatch>;
}

template <int DT>
static KernelFn ring_fn(int vb, bool beta, bool peel, bool shift, bool batched) {
    constexpr int MV = 16 / ElemT<DT>::ES;
    constexpr bool kSameType = tt_is_same<typename ElemT<DT>::T, typename ElemT<DT>::TA>::value;
    // the peeled store phase and the shifted rows exist for same-type pairs of 4- and 8-byte elements only
    if constexpr (MV > 1 && kSameType) {
        if (vb == MV && peel) return shift ? ring_fn_inst<DT, MV, true, true>(beta, batched) : ring_fn_inst<DT, MV, true, false>(beta, batched);
        if (vb == MV && shift) return ring_fn_inst<DT, MV, false, true>(beta, batched);
        if (vb == 1 && shift && !peel) return ring_fn_inst<DT, 1, false, true>(beta, batched);
    }
    if (peel || shift) return nullptr;
    if constexpr (MV > 1) {
        if (vb == MV) return ring_fn_inst<DT, MV, false, false>(beta, batched);
    }
    if (vb == 1) return ring_fn_inst<DT, 1, false, false>(beta, batched);
    return nullptr;
}

static KernelFn get_tile_fn(int dt, const Candidate& c, bool batched) {
    const TileParams& p = c.tp;
    if (p.ring > 0) {
        const bool peel = p.peel != 0, shift = p.row_async == 2;
        switch (dt) {
            case kPairSD: return ring_fn<kPairSD>(p.vecB, c.beta_nz, peel, shift, batched);
            case kPairDS: return ring_fn<kPairDS>(p.vecB, c.beta_nz, peel, shift, batched);
            case kPairCZ: return ring_fn<kPairCZ>(p.vecB, c.beta_nz, peel, shift, batched);
            case kPairZC: return ring_fn<kPairZC>(p.vecB, c.beta_nz, peel, shift, batched);
            case TTC_F32: return ring_fn<TTC_F32>(p.vecB, c.beta_nz, peel, shift, batched);
            case TTC_F64: return ring_fn<TTC_F64>(p.vecB, c.beta_nz, peel, shift, batched);
            case TTC_C64: return ring_fn<TTC_C64>(p.vecB, c.beta_nz, peel, shift, batched);
            case TTC_C128: return ring_fn<TTC_C128>(p.vecB, c.beta_nz, peel, shift, batched);
        }
        return nullptr;
    }
    switch (dt) {
        case TTC_F32: return tile_fn<TTC_F32>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case TTC_F64: return tile_fn<TTC_F64>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case TTC_C64: return tile_fn<TTC_C64>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case TTC_C128: return tile_fn<TTC_C128>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case kPairSD: return tile_fn<kPairSD>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case kPairDS: return tile_fn<kPairDS>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case kPairCZ: return tile_fn<kPairCZ>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
        case kPairZC: return tile_fn<kPairZC>(p.vecA, p.vecB, p.same != 0, c.beta_nz, batched);
    }
    return nullptr;
}

static KernelFn get_direct_fn(int dt, const Candidate& c, bool batched) {
    switch (dt) {
        case TTC_F32: return direct_fn<TTC_F32>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case TTC_F64: return direct_fn<TTC_F64>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case TTC_C64: return direct_fn<TTC_C64>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case TTC_C128: return direct_fn<TTC_C128>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case kPairSD: return direct_fn<kPairSD>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case kPairDS: return direct_fn<kPairDS>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case kPairCZ: return direct_fn<kPairCZ>(c.dp.vec, c.beta_nz, c.idx64, batched);
        case kPairZC: return direct_fn<kPairZC>(c.dp.vec, c.beta_nz, c.idx64, batched);
    }
    return nullptr;
}

template <int DT, typename BT>
static KernelFn tmap_fn_bt(bool beta, int flavour) {
    if (flavour == 0) return beta ? (KernelFn)tmap_kernel<DT, true, 0, BT> : (KernelFn)tmap_kernel<DT, false, 0, BT>;
    return beta ? (KernelFn)tmap_kernel<DT, true, 1, BT> : (KernelFn)tmap_kernel<DT, false, 1, BT>;
}

template <int DT>
static KernelFn tmap_fn_dt(bool beta, int flavour, bool batched) {
    return batched ? tmap_fn_bt<DT, TmapBatch>(beta, flavour) : tmap_fn_bt<DT, NoBatch>(beta, flavour);
}

static KernelFn get_tmap_fn(int dt, const Candidate& c, bool batched = false) {
    switch (dt) {
        case TTC_F32: return tmap_fn_dt<TTC_F32>(c.beta_nz, c.mp.flavour, batched);
        case TTC_F64: return tmap_fn_dt<TTC_F64>(c.beta_nz, c.mp.flavour, batched);
        case TTC_C64: return tmap_fn_dt<TTC_C64>(c.beta_nz, c.mp.flavour, batched);
        case TTC_C128: return tmap_fn_dt<TTC_C128>(c.beta_nz, c.mp.flavour, batched);
    }
    return nullptr;     // same-type tensors only
}

// cuTensorMapEncodeTiled through the runtime's driver entry point query (the library does not link libcuda).
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            f = nullptr;
        return (EncodeTiledFn)f;
    }();
    return fn;
}

// dim4A / dim4B > 0 (batched launch): extent of the fifth dimension, whose stride is 16 bytes: the batch offset.
static bool encode_maps(const TmapEncode& me, const void* A, void* B, CUtensorMap* mapA, CUtensorMap* mapB, uint64_t dim4A = 0,
                        uint64_t dim4B = 0) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const CUtensorMapDataType dt = me.unit_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_UINT64;
    static const CUtensorMapSwizzle kSwz[4] = {CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_SWIZZLE_128B};
    const CUtensorMapSwizzle swA = kSwz[me.swzA & 3], swB = kSwz[me.swzB & 3];
    static const cuuint32_t ones[kTmapRank] = {1, 1, 1, 1, 1};
    const CUtensorMapL2promotion l2p = CU_TENSOR_MAP_L2_PROMOTION_L2_128B;    // none / 128 B / 256 B measured: no difference
    cuuint64_t dA[kTmapRank], dB[kTmapRank], sA[kTmapRank - 1], sB[kTmapRank - 1];
    cuuint32_t bA[kTmapRank], bB[kTmapRank];
    for (int i = 0; i < kTmapRank; ++i) { dA[i] = me.dimA[i]; dB[i] = me.dimB[i]; bA[i] = me.boxA[i]; bB[i] = me.boxB[i]; }
    for (int i = 0; i < kTmapRank - 1; ++i) { sA[i] = me.strideA[i]; sB[i] = me.strideB[i]; }
    if (dim4A) { dA[4] = dim4A; sA[3] = 16; }
    if (dim4B) { dB[4] = dim4B; sB[3] = 16; }
    if (enc(mapA, dt, kTmapRank, const_cast<void*>(A), dA, sA, bA, ones, CU_TENSOR_MAP_INTERLEAVE_NONE, swA,
            l2p, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return false;
    return enc(mapB, dt, kTmapRank, B, dB, sB, bB, ones, CU_TENSOR_MAP_INTERLEAVE_NONE, swB,
               l2p, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int DT>
static KernelFn tmapu_fn_dt(bool beta) { return beta ? (KernelFn)tmapu_kernel<DT, true> : (KernelFn)tmapu_kernel<DT, false>; }

static KernelFn get_tmapu_fn(int dt, const Candidate& c) {
    switch (dt) {
        case TTC_F32: return tmapu_fn_dt<TTC_F32>(c.beta_nz);
        case TTC_F64: return tmapu_fn_dt<TTC_F64>(c.beta_nz);
        case TTC_C64: return tmapu_fn_dt<TTC_C64>(c.beta_nz);
    }
    return nullptr;     // 16-byte elements are always 16-byte aligned: flavours 0 and 1
}

// The 2 V maps per tensor of the residue-class flavour: [skew * 2 + lo] has extents (e + skew, rows of the classes with
// (lo = 0) or without (lo = 1) one row more, every aligned offset), see ttc_tmap.h.  `A` and `B` are the base addresses rounded DOWN to 16 bytes.
static bool encode_class_maps(const TmapUEncode& ue, const void* A, void* B, TmapUSet* set) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const int V = 16 / ue.es, T = 128 / ue.es;
    const CUtensorMapDataType dt = ue.es == 4 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_UINT64;
    static const cuuint32_t ones[kTmapRank] = {1, 1, 1, 1, 1};
    const cuuint32_t box[kTmapRank] = {(cuuint32_t)T, (cuuint32_t)(T / V), 1, 1, 1};
    for (int side = 0; side < 2; ++side) {
        const int64_t e_in = side == 0 ? ue.e0 : ue.eq, e_row = side == 0 ? ue.eq : ue.e0;
        const int64_t s_row = side == 0 ? ue.sqA : ue.s0B, span = side == 0 ? ue.spanA : ue.spanB;
        void* base = side == 0 ? const_cast<void*>(A) : B;
        CUtensorMap* out = side == 0 ? set->a : set->b;
        for (int sk = 0; sk < V; ++sk)
            for (int lo = 0; lo < 2; ++lo) {       // 0: the classes below e_row % V (one row more), 1: the others
                const int64_t rows = e_row / V + (lo == 0 ? 1 : 0);
                const cuuint64_t dims[kTmapRank] = {(cuuint64_t)(e_in + sk), (cuuint64_t)(rows < 1 ? 1 : rows), (cuuint64_t)(span / V + 2), 1, 1};
                const cuuint64_t strides[kTmapRank - 1] = {(cuuint64_t)(V * s_row * ue.es), 16, 16, 16};
                if (enc(&out[sk * 2 + lo], dt, kTmapRank, base, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                    return false;
            }
    }
    return true;
}

// Encoding 4 V maps costs several microseconds of host time: the sets of the last few (shape, A, B) are kept.
static bool class_maps_cached(const TmapUEncode& ue, const void* A, void* B, TmapUSet* set) {
    struct Key {
        TmapUEncode ue; const void* a; void* b;
        bool operator<(const Key& o) const { return std::memcmp(this, &o, sizeof(Key)) < 0; }
    };
    static std::mutex mu;
    static std::map<Key, TmapUSet> cache;
    Key k;
    std::memset(&k, 0, sizeof(k));
    k.ue = ue;
    k.a = A;
    k.b = B;
    std::lock_guard<std::mutex> lk(mu);
    auto it = cache.find(k);
    if (it != cache.end()) { *set = it->second; return true; }
    if (!encode_class_maps(ue, A, B, set)) return false;
    if (cache.size() >= 64) cache.clear();
    cache.emplace(k, *set);
    return true;
}

template <int DT>
static KernelFn skew_fn_dt(bool beta, bool direct) {
    if (direct) return beta ? (KernelFn)skew_kernel<DT, true, true> : (KernelFn)skew_kernel<DT, false, true>;
    return beta ? (KernelFn)skew_kernel<DT, true, false> : (KernelFn)skew_kernel<DT, false, false>;
}

static KernelFn get_skew_fn(int dt, const Candidate& c) {
    const bool direct = c.sp.ns == 0;          // no store warps: the consumers write B
    switch (dt) {
        case TTC_F32: return skew_fn_dt<TTC_F32>(c.beta_nz, direct);
        case TTC_F64: return skew_fn_dt<TTC_F64>(c.beta_nz, direct);
        case TTC_C64: return skew_fn_dt<TTC_C64>(c.beta_nz, direct);
    }
    return nullptr;
}

static uint32_t skew_smem_bytes(const SkewParams& sp) {
    const uint32_t rowsA = (uint32_t)sp.nP << sp.lgTB, rowsB = (uint32_t)sp.nP << sp.lgTA;
    return (uint32_t)sp.stages * (rowsA * (uint32_t)sp.pitchA + rowsB * (uint32_t)sp.pitchB) + 128u;
}

static uint32_t tmapu_smem_bytes(const TmapUParams& up) {
    return (uint32_t)up.stages * 2u * (uint32_t)up.nP * (uint32_t)up.V * 1024u + 1024u;
}

static uint32_t tmap_smem_bytes(const TmapParams& mp) {
    return (uint32_t)mp.stages * 2u * mp.buf_bytes + 1024u;     // + alignment slack
}

// Opt the instance in to the device's maximum of dynamic shared memory (the attribute belongs to the kernel
// function, which many candidates share); returns that maximum less the kernel's static shared memory.
static int raise_smem_limit(KernelFn fn, int* optin_out) {
    int dev = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return (int)e;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return (int)e;
    optin -= (int)fa.sharedSizeBytes;   // the scheduler's mbarrier and response are static shared memory
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    *optin_out = optin;
    return (int)e;
}

int prepare_candidate(Candidate* cand, ttc_dtype dtype, ttc_dtype dtype_a, int sm_count) {
    const int pair = pair_id(dtype, dtype_a);
    if (pair < 0) return (int)cudaErrorInvalidValue;
    if (cand->info.kernel == TTC_KERNEL_COPY) {
        KernelFn fn = get_direct_fn(pair, *cand, false);
        if (!fn) return (int)cudaErrorInvalidValue;
        int occ = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kDirectThreads, 0);
        if (e != cudaSuccess) return (int)e;
        if (occ < 1) occ = 1;
        const uint64_t need = cand->dp.n_chunks ? cand->dp.n_chunks : 1;
        const uint64_t cap = (uint64_t)sm_count * (uint64_t)occ;
        cand->info.threads = kDirectThreads;
        cand->info.smem_bytes = 0;
        cand->info.grid = (int)(cand->dp.dyn == 1 || need < cap ? need : cap);
        cand->grid_cap = (int)cap;
        return 0;
    }
    if (cand->info.kernel == TTC_KERNEL_SKEW) {
        KernelFn fn = dtype == dtype_a ? get_skew_fn((int)dtype, *cand) : nullptr;
        if (!fn) return (int)cudaErrorInvalidValue;
        const int smem = (int)skew_smem_bytes(cand->sp);
        int optin = 0;
        int rc = raise_smem_limit(fn, &optin);
        if (rc != 0) return rc;
        if (smem > optin) return (int)cudaErrorInvalidConfiguration;
        int occ = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, cand->sp.threads, smem);
        if (e != cudaSuccess) return (int)e;
        if (occ < 1) return (int)cudaErrorInvalidConfiguration;
        const uint64_t cap = (uint64_t)sm_count * (uint64_t)occ;
        cand->info.threads = cand->sp.threads;
        cand->info.smem_bytes = smem;
        cand->info.grid = (int)(cand->sp.dyn == 1 || cand->sp.n_tiles < cap ? cand->sp.n_tiles : cap);
        cand->grid_cap = (int)cap;
        return 0;
    }
    if (cand->info.kernel == TTC_KERNEL_TENSORMAP) {
        const bool classes = cand->mp.flavour == 2;
        KernelFn fn = dtype != dtype_a ? nullptr : classes ? get_tmapu_fn((int)dtype, *cand) : get_tmap_fn((int)dtype, *cand);
        if (!fn || !encode_tiled_fn()) return (int)cudaErrorInvalidValue;
        const int smem = (int)(classes ? tmapu_smem_bytes(cand->up) : tmap_smem_bytes(cand->mp));
        int optin = 0;
        int rc = raise_smem_limit(fn, &optin);
        if (rc != 0) return rc;
        if (smem > optin) return (int)cudaErrorInvalidConfiguration;
        int occ = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, cand->mp.threads, smem);
        if (e != cudaSuccess) return (int)e;
        if (occ < 1) return (int)cudaErrorInvalidConfiguration;
        const uint64_t cap = (uint64_t)sm_count * (uint64_t)occ;
        cand->info.threads = cand->mp.threads;
        cand->info.smem_bytes = smem;
        cand->info.grid = (int)(cand->mp.dyn == 1 || cand->mp.n_tiles < cap ? cand->mp.n_tiles : cap);
        cand->grid_cap = (int)cap;
        return 0;
    }
    KernelFn fn = get_tile_fn(pair, *cand, false);
    if (!fn) return (int)cudaErrorInvalidValue;
    // the ring kernel's tile holds A's type (bulk copies), the tile kernel's B's
    const int smem = (int)tile_smem_layout(cand->tp, elem_size(cand->tp.ring > 0 ? dtype_a : dtype)).total;
    int optin = 0;
    int rc = raise_smem_limit(fn, &optin);
    if (rc != 0) return rc;
    if (smem > optin) return (int)cudaErrorInvalidConfiguration;
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, cand->tp.threads, smem);
    if (e != cudaSuccess) return (int)e;
    if (occ < 1) return (int)cudaErrorInvalidConfiguration;
    const uint64_t cap = (uint64_t)sm_count * (uint64_t)occ;
    cand->info.threads = cand->tp.threads;
    cand->info.smem_bytes = smem;
    cand->info.grid = (int)(cand->tp.dyn == 1 || cand->tp.n_tiles < cap ? cand->tp.n_tiles : cap);
    cand->grid_cap = (int)cap;
    return 0;
}

int launch_candidate(const Candidate& cand, ttc_dtype dtype, ttc_dtype dtype_a, const Scalar& alpha,
                     const Scalar& beta, const void* A, void* B, void* stream, uint32_t* sched_ctr,
                     const BatchPtrs* batch) {
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int pair = pair_id(dtype, dtype_a);
    if (pair < 0) return (int)cudaErrorInvalidValue;
    if (cand.info.grid <= 0) return (int)cudaErrorInvalidConfiguration;
    // cudaLaunchKernelExC returns the launch error itself: the caller's CUDA error state is not
    // read (no cudaGetLastError, which would clear errors that are not ours).
    cudaLaunchConfig_t cfg{};
    cfg.stream = st;
    const bool batched = batch != nullptr && batch->n > 0;
    uint64_t grid = (uint64_t)cand.info.grid;
    if (batched) {     // one CTA per work item (launch control) or as many as the device holds
        const uint64_t work = (uint64_t)batch->per * (uint64_t)batch->n;
        if (cand.info.kernel == TTC_KERNEL_SKEW) return (int)cudaErrorNotSupported;
        if (cand.info.kernel == TTC_KERNEL_TENSORMAP && (cand.mp.flavour == 2 || !cand.mp.batchable)) return (int)cudaErrorNotSupported;
        const int dyn_b = cand.info.kernel == TTC_KERNEL_COPY ? cand.dp.dyn : cand.info.kernel == TTC_KERNEL_TENSORMAP ? cand.mp.dyn : cand.tp.dyn;
        grid = (dyn_b == 1 || work < (uint64_t)cand.grid_cap) ? work : (uint64_t)cand.grid_cap;
        if (grid >= (1ull << 31)) return (int)cudaErrorInvalidConfiguration;
    }
    cfg.gridDim = dim3((unsigned)grid, 1, 1);
    // Every launch carries the programmatic-stream-serialisation attribute (programmatic dependent
    // launch): the kernels call griddepcontrol.launch_dependents first thing and griddepcontrol.wait
    // before their first global access, so the prologue (scheduler set-up, offset tables) of a kernel
    // overlaps the tail of its predecessor in the stream or graph.  Measured in a graph of 20 launches
    // (198 MB): -0.3 .. -1.3 us per launch; neutral for stream launches.  A predecessor that is not one
    // of these kernels never triggers early, which degenerates to ordinary stream order.  TTC_PDL=0: off.
    cudaLaunchAttribute attr[1];
    const int dyn = cand.info.kernel == TTC_KERNEL_COPY ? cand.dp.dyn : cand.info.kernel == TTC_KERNEL_TENSORMAP ? cand.mp.dyn
                    : cand.info.kernel == TTC_KERNEL_SKEW ? cand.sp.dyn : cand.tp.dyn;
    static const int pdl_env = std::getenv("TTC_PDL") ? std::atoi(std::getenv("TTC_PDL")) : -1;
    if (dyn == 2 && !sched_ctr) return (int)cudaErrorInvalidValue;
    if (pdl_env != 0) {
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    NoBatch none;
    Scalar al = alpha, be = beta;
    if (cand.info.kernel == TTC_KERNEL_SKEW) {
        KernelFn fn = dtype == dtype_a ? get_skew_fn((int)dtype, cand) : nullptr;
        if (!fn) return (int)cudaErrorInvalidValue;
        cfg.blockDim = dim3((unsigned)cand.sp.threads, 1, 1);
        cfg.dynamicSmemBytes = (size_t)cand.info.smem_bytes;
        SkewParams sp = cand.sp;
        sp.ctr = sched_ctr;
        void* sargs[5] = {&sp, (void*)&A, (void*)&B, &al, &be};
        return (int)cudaLaunchKernelExC(&cfg, fn, sargs);
    }
    if (cand.info.kernel == TTC_KERNEL_TENSORMAP && cand.mp.flavour == 2) {
        KernelFn fn = dtype == dtype_a ? get_tmapu_fn((int)dtype, cand) : nullptr;
        if (!fn) return (int)cudaErrorInvalidValue;
        const int es = cand.ue.es;
        const uintptr_t a16 = (uintptr_t)A & ~(uintptr_t)15, b16 = (uintptr_t)B & ~(uintptr_t)15;
        alignas(64) TmapUSet set;
        if (!class_maps_cached(cand.ue, (const void*)a16, (void*)b16, &set)) return (int)cudaErrorInvalidValue;
        cfg.blockDim = dim3((unsigned)cand.up.threads, 1, 1);
        cfg.dynamicSmemBytes = (size_t)cand.info.smem_bytes;
        TmapUParams up = cand.up;
        up.ctr = sched_ctr;
        up.skewA0 = (int)(((uintptr_t)A - a16) / (uintptr_t)es);
        up.skewB0 = (int)(((uintptr_t)B - b16) / (uintptr_t)es);
        void* uargs[4] = {&up, &set, &al, &be};
        return (int)cudaLaunchKernelExC(&cfg, fn, uargs);
    }
    if (cand.info.kernel == TTC_KERNEL_TENSORMAP) {
        KernelFn fn = dtype == dtype_a ? get_tmap_fn((int)dtype, cand, batched) : nullptr;
        if (!fn) return (int)cudaErrorInvalidValue;
        alignas(64) CUtensorMap mapA, mapB;       // the descriptors carry the base addresses: encoded per call (host only)
        TmapBatch tb;
        if (batched) {
            // one pair of maps for the whole batch: based at the lowest addresses, problem i at coordinate
            // (A_i - min A) / 16 of the fifth dimension (stride 16 bytes)
            uintptr_t lo_a = (uintptr_t)batch->a[0], lo_b = (uintptr_t)batch->b[0], hi_a = lo_a, hi_b = lo_b;
            for (int i = 1; i < batch->n; ++i) {
                lo_a = std::min(lo_a, (uintptr_t)batch->a[i]);
                hi_a = std::max(hi_a, (uintptr_t)batch->a[i]);
                lo_b = std::min(lo_b, (uintptr_t)batch->b[i]);
                hi_b = std::max(hi_b, (uintptr_t)batch->b[i]);
            }
            if ((hi_a - lo_a) / 16 >= (uintptr_t)0x7fffffff || (hi_b - lo_b) / 16 >= (uintptr_t)0x7fffffff) return (int)cudaErrorNotSupported;
            tb.n = batch->n;
            tb.per = batch->per;
            tb.div = batch->div;
            for (int i = 0; i < batch->n; ++i) {
                if ((((uintptr_t)batch->a[i] | (uintptr_t)batch->b[i]) & 15) != 0) return (int)cudaErrorMisalignedAddress;
                tb.offA[i] = (int32_t)(((uintptr_t)batch->a[i] - lo_a) / 16);
                tb.offB[i] = (int32_t)(((uintptr_t)batch->b[i] - lo_b) / 16);
            }
            if (!encode_maps(cand.me, (const void*)lo_a, (void*)lo_b, &mapA, &mapB, (hi_a - lo_a) / 16 + 1, (hi_b - lo_b) / 16 + 1))
                return (int)cudaErrorInvalidValue;
            static std::mutex mu;
            static std::set<KernelFn> raised;
            std::lock_guard<std::mutex> lk(mu);
            if (!raised.count(fn)) {
                int optin = 0;
                const int rc = raise_smem_limit(fn, &optin);
                if (rc != 0) return rc;
                raised.insert(fn);
            }
        } else if (!encode_maps(cand.me, A, B, &mapA, &mapB)) {
            return (int)cudaErrorInvalidValue;
        }
        cfg.blockDim = dim3((unsigned)cand.mp.threads, 1, 1);
        cfg.dynamicSmemBytes = (size_t)cand.info.smem_bytes;
        TmapParams mp = cand.mp;
        mp.ctr = sched_ctr;
        void* targs[6] = {&mp, &mapA, &mapB, &al, &be, batched ? (void*)&tb : (void*)&none};
        return (int)cudaLaunchKernelExC(&cfg, fn, targs);
    }
    void* args[6] = {nullptr, (void*)&A, (void*)&B, (void*)&al, (void*)&be, batched ? (void*)batch : (void*)&none};
    if (cand.info.kernel == TTC_KERNEL_COPY) {
        KernelFn fn = get_direct_fn(pair, cand, batched);
        if (!fn) return (int)cudaErrorInvalidValue;
        cfg.blockDim = dim3(kDirectThreads, 1, 1);
        cfg.dynamicSmemBytes = 0;
        DirectParams dp = cand.dp;
        dp.ctr = sched_ctr;
        args[0] = &dp;
        return (int)cudaLaunchKernelExC(&cfg, fn, args);
    }
    KernelFn fn = get_tile_fn(pair, cand, batched);
    if (!fn) return (int)cudaErrorInvalidValue;
    if (batched) {      // the batched twin of the instance has its own shared-memory attribute: set it once
        static std::mutex mu;
        static std::set<KernelFn> raised;
        std::lock_guard<std::mutex> lk(mu);
        if (!raised.count(fn)) {
            int optin = 0;
            const int rc = raise_smem_limit(fn, &optin);
            if (rc != 0) return rc;
            raised.insert(fn);
        }
    }
    cfg.blockDim = dim3((unsigned)cand.tp.threads, 1, 1);
    cfg.dynamicSmemBytes = (size_t)cand.info.smem_bytes;
    TileParams tp = cand.tp;
    tp.ctr = sched_ctr;
    args[0] = &tp;
    return (int)cudaLaunchKernelExC(&cfg, fn, args);
}

}  // namespace ttc
