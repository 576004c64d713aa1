// ttc_tmap.cuh -- tmap_kernel: Eq. 1 with tiles that travel as tensor-map boxes in both directions
// (north_star K2, SURVEY.md 8(d) "TMA feasibility").  One CTA = one producer warp, one store warp, the rest consumers:
//
//   producer (lane 0)   waits for a free stage, takes the next tile from the work scheduler, arms the stage's `full`
//                       mbarrier with the box bytes and issues cp.async.bulk.tensor.5d loads (UTMALDG) of A's boxes
//                       into the stage's in-buffer and, for beta != 0, of B's boxes into its out-buffer
//   consumers           wait for `full`; flavour 0: transpose every 2-D plane of the in-boxes into the out-boxes, V x V
//                       elements per thread held in registers (V = 16 / element size: the paper's in-register micro
//                       tile), 16-byte LDS/STS only, both sides in the 128-byte swizzle so that every
//                       quarter-warp access touches all 32 banks once; flavour 1: alpha/beta chunk by chunk; then
//                       fence.proxy.async and one arrival per warp on `done`
//   store warp (lane 0) waits for `done`, issues cp.async.bulk.tensor.5d stores (UTMASTG) of the out-boxes, commits
//                       them as one bulk group and hands the PREVIOUS stage's out-buffer back (`outfree`) once its
//                       group has finished reading shared memory.  The in-buffer of a stage is free for the next load
//                       as soon as its consumers are `done`, so loads run stages - 1 tiles ahead of the consumers
//
// Boxes that stick out of the tensor need no code: loads fill with zeros, stores clip.  No thread issues a global
// load or store.  Arithmetic: products and sums rounded separately, exactly as the other kernels (readings A7/A10).
#pragma once
#include <cuda.h>

#include "ttc_device.cuh"
#include "ttc_tmap.h"

namespace ttc {

__device__ __forceinline__ void tmap_load(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tmap_store(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts128(uint32_t a, const uint4& v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// Which V x V micro-tile (A2 = 16-byte column of the in-plane, B2 = 16-byte column of the out-plane, both 0..7) lane
// `lane` takes in pass j (0, 1) of a plane.  In-plane: element (a, b) sits in row b, chunk (a / V) ^ (b & 7);
// out-plane: row a, chunk (b / V) ^ (a & 7).  The 8 lanes of a quarter-warp read rows V*B2 + d, chunk A2 and write
// rows V*A2 + d, chunk B2 (d fixed per instruction); the maps below make both chunk positions a bijection of the
// lane's low three bits for every d, i.e. conflict-free 16-byte accesses on both sides.
template <int V>
__device__ __forceinline__ void tmap_lane_map(int lane, int j, int& A2, int& B2) {
    const int i = lane & 7, q = lane >> 3;
    if constexpr (V == 1) {
        A2 = i;
        B2 = (j << 2) | q;
    } else if constexpr (V == 2) {
        A2 = i;
        B2 = ((j << 2) | q) ^ (i >> 2);
    } else {
        A2 = (j << 2) | (i & 3);
        B2 = ((q >> 1) << 2) | (((((i >> 1) ^ q) & 1)) << 1) | (i >> 2);
    }
}

template <typename T> struct tmap_is_real { static constexpr bool value = false; };
template <> struct tmap_is_real<float> { static constexpr bool value = true; };
template <> struct tmap_is_real<double> { static constexpr bool value = true; };

template <int DT, bool BETA, int FLAVOUR, typename BT>
__global__ void __launch_bounds__(256)
tmap_kernel(const __grid_constant__ TmapParams P, const __grid_constant__ CUtensorMap mapA,
            const __grid_constant__ CUtensorMap mapB, const Scalar alpha_in, const Scalar beta_in, const __grid_constant__ BT Bt) {
    using T = typename ElemT<DT>::T;
    constexpr int ES = (int)sizeof(T);
    constexpr int V = 16 / ES;
    union Chunk { uint4 u; T e[V]; };
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t raw = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;              // the 128-byte swizzle repeats every 1024 bytes
    const int nbox = P.nbA * P.nbB;
    const uint32_t tile_bytes = P.box_bytes * (uint32_t)nbox;

    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    __shared__ __align__(8) uint64_t full_bar[kTmapMaxStages], done_bar[kTmapMaxStages], outfree_bar[kTmapMaxStages];
    // tile origin and id per stage, two deep: the producer may fill a stage again (its consumers are done) before the
    // store thread has read where the stage's previous tile goes; it cannot get two uses ahead of it
    __shared__ int32_t coord[kTmapMaxStages][2][kTmapRank];
    __shared__ int32_t coord_b4[kTmapMaxStages][2];          // batched: B's coordinate along the fifth dimension (A's is coord[..][4])
    __shared__ uint32_t tile_of[kTmapMaxStages][2];

    const int tid = threadIdx.x, lane = tid & 31;
    const int S = P.stages;
    const int n_cons_warps = ((int)blockDim.x >> 5) - 2;
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&full_bar[s])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&done_bar[s])), "r"(n_cons_warps));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[s])));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();

    // A real alpha == 1 with beta == 0 in the copy class leaves nothing to compute: the box is stored from the buffer it
    // was loaded into.  (Not for complex types: (1 + 0i) * (inf + i) has 0 * inf = NaN in the oracle's formula too.)
    bool passthrough = false;
    if constexpr (FLAVOUR == 1 && !BETA && tmap_is_real<T>::value) passthrough = alpha.re == T(1);

    if (tid < 32) {
        // ------------------------------------------------------------------ producer warp
        uint32_t tile_id = blockIdx.x;
        bool more = true;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            const int u = (int)((it / (uint32_t)S) & 1u);
            const uint32_t full_a = (uint32_t)__cvta_generic_to_shared(&full_bar[s]);
            if (it >= (uint32_t)S) {
                // the in-buffer is free once the consumers are done with it; the out-buffer (which only beta != 0 loads
                // into) once the store of its last tile has read it (passthrough: that store read the in-buffer)
                mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                if (BETA || passthrough) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
            }
            if (!more) {
                if (lane == 0) {
                    tile_of[s][u] = 0xFFFFFFFFu;
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_a) : "memory");
                }
                break;
            }
            sched.prefetch();
            if (lane == 0) {
                int32_t c[kTmapRank];
                uint32_t r = tile_id;
                int32_t c4a = 0, c4b = 0;
                if constexpr (!tt_is_same<BT, NoBatch>::value) {
                    const uint32_t pair = fd_div(r, Bt.div);
                    r -= pair * Bt.per;
                    c4a = Bt.offA[pair];
                    c4b = Bt.offB[pair];
                }
#pragma unroll
                for (int d = 0; d < kTmapRank; ++d) {
                    const uint32_t qq = fd_div(r, P.gdiv[d]);
                    c[d] = (int32_t)(r - qq * P.gdiv[d].d) * P.step[d];
                    r = qq;
                }
                if constexpr (!tt_is_same<BT, NoBatch>::value) c[4] = c4a;
                else c4b = c[4];
#pragma unroll
                for (int d = 0; d < kTmapRank; ++d) coord[s][u][d] = c[d];
                coord_b4[s][u] = c4b;
                tile_of[s][u] = tile_id;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(full_a), "r"(tile_bytes * (BETA ? 2u : 1u)) : "memory");
                const uint32_t in_s = base + (uint32_t)s * 2u * P.buf_bytes, out_s = in_s + P.buf_bytes;
                int box = 0;
                for (int bj = 0; bj < P.nbB; ++bj)
                    for (int bi = 0; bi < P.nbA; ++bi, ++box) {
                        const int ca = c[0] + bi * P.box0[0];
                        if constexpr (FLAVOUR == 0) {
                            const int cb = c[1] + bj * P.box0[1];
                            tmap_load(in_s + (uint32_t)box * P.box_bytes, &mapA, full_a, ca * P.upe, cb, c[2], c[3], c[4]);
                            if constexpr (BETA) tmap_load(out_s + (uint32_t)box * P.box_bytes, &mapB, full_a, cb * P.upe, ca, c[2], c[3], c4b);
                        } else {
                            tmap_load(in_s + (uint32_t)box * P.box_bytes, &mapA, full_a, ca * P.upe, c[1], c[2], c[3], c[4]);
                            if constexpr (BETA) tmap_load(out_s + (uint32_t)box * P.box_bytes, &mapB, full_a, ca * P.upe, c[1], c[2], c[3], c4b);
                        }
                    }
            }
            more = sched.next<true>(tile_id, Bt.n ? P.n_tiles * (uint32_t)Bt.n : P.n_tiles);
            __syncwarp();
        }
    } else if (tid < 64) {
        // ------------------------------------------------------------------ store warp (one thread: bulk groups are per thread)
        if (tid == 32) {
            for (uint32_t it = 0;; ++it) {
                const int s = (int)(it % (uint32_t)S);
                const int u = (int)((it / (uint32_t)S) & 1u);
                mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), (uint32_t)u);
                if (tile_of[s][u] == 0xFFFFFFFFu) break;
                int32_t c[kTmapRank];
#pragma unroll
                for (int d = 0; d < kTmapRank; ++d) c[d] = coord[s][u][d];
                c[4] = coord_b4[s][u];
                const uint32_t in_s = base + (uint32_t)s * 2u * P.buf_bytes;
                const uint32_t src_s = passthrough ? in_s : in_s + P.buf_bytes;
                int box = 0;
                for (int bj = 0; bj < P.nbB; ++bj)
                    for (int bi = 0; bi < P.nbA; ++bi, ++box) {
                        const int ca = c[0] + bi * P.box0[0];
                        if constexpr (FLAVOUR == 0)
                            tmap_store(&mapB, src_s + (uint32_t)box * P.box_bytes, (c[1] + bj * P.box0[1]) * P.upe, ca, c[2], c[3], c[4]);
                        else
                            tmap_store(&mapB, src_s + (uint32_t)box * P.box_bytes, ca * P.upe, c[1], c[2], c[3], c[4]);
                    }
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                if (it >= 1u) {     // the group of the stage before this one has read its out-buffer: hand that buffer back
                    asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];"
                                 ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[(it - 1u) % (uint32_t)S])) : "memory");
                }
            }
            asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        }
    } else {
        // ------------------------------------------------------------------ consumer warps
        const int cw = (tid >> 5) - 2;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            mbar_wait((uint32_t)__cvta_generic_to_shared(&full_bar[s]), (it / (uint32_t)S) & 1u);
            const bool end = tile_of[s][(it / (uint32_t)S) & 1u] == 0xFFFFFFFFu;
            if (!end && !passthrough) {
                // beta == 0: nobody has waited for the store that last read this out-buffer yet
                if constexpr (!BETA)
                    if (it >= (uint32_t)S) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                const uint32_t in_s = base + (uint32_t)s * 2u * P.buf_bytes, out_s = in_s + P.buf_bytes;
                if constexpr (FLAVOUR == 0) {
                    const int n_planes = nbox * P.planes;
                    if (P.ca == 8 && P.cb == 8) {
                    constexpr uint32_t PB = 1024u * V;          // bytes of one plane: 8 V rows of 128 bytes
                    for (int pl = cw; pl < n_planes; pl += n_cons_warps) {
                        const uint32_t ip = in_s + (uint32_t)pl * PB, op = out_s + (uint32_t)pl * PB;
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            int A2, B2;
                            tmap_lane_map<V>(lane, j, A2, B2);
                            Chunk r[V];
#pragma unroll
                            for (int d = 0; d < V; ++d) {
                                const int row = V * B2 + d;
                                r[d].u = lds128(ip + (uint32_t)(row * 128 + ((A2 ^ (row & 7)) << 4)));
                            }
#pragma unroll
                            for (int d = 0; d < V; ++d) {
                                const int row = V * A2 + d;
                                const uint32_t oa = op + (uint32_t)(row * 128 + ((B2 ^ (row & 7)) << 4));
                                Chunk o, b;
                                if constexpr (BETA) b.u = lds128(oa);
#pragma unroll
                                for (int e = 0; e < V; ++e) {
                                    T x = scale(alpha, r[e].e[d]);
                                    if constexpr (BETA) x = add(x, scale(beta, b.e[e]));
                                    o.e[e] = x;
                                }
                                sts128(oa, o.u);
                            }
                        }
                    }
                    } else {
                    // 64-byte rows on one or both sides (ca, cb in {8, 4}): a plane has ca x cb micro-tiles; the hardware
                    // swizzle of a row of c chunks is chunk ^= (address >> 7) & (c - 1), computed here on the byte offset
                    // from the stage buffer (1024-byte aligned).  Up to two-way bank conflicts: the kernel is bound by
                    // DRAM, not by shared memory.
                    const uint32_t ca = (uint32_t)P.ca, cb = (uint32_t)P.cb;
                    const uint32_t pb = ca * cb * (uint32_t)V * 16u;          // bytes of one plane
                    const uint32_t n_micro = ca * cb;
                    const uint32_t lg_ca = ca == 8u ? 3u : 2u;
                    for (int pl = cw; pl < n_planes; pl += n_cons_warps) {
                        const uint32_t pbase = (uint32_t)pl * pb;
                        for (uint32_t m = (uint32_t)lane; m < n_micro; m += 32u) {
                            const uint32_t A2 = m & (ca - 1u), B2 = m >> lg_ca;
                            Chunk r[V];
#pragma unroll
                            for (int d = 0; d < V; ++d) {
                                const uint32_t L = pbase + ((uint32_t)V * B2 + (uint32_t)d) * (ca << 4) + (A2 << 4);
                                r[d].u = lds128(in_s + (L ^ (((L >> 7) & (ca - 1u)) << 4)));
                            }
#pragma unroll
                            for (int d = 0; d < V; ++d) {
                                const uint32_t L = pbase + ((uint32_t)V * A2 + (uint32_t)d) * (cb << 4) + (B2 << 4);
                                const uint32_t oa = out_s + (L ^ (((L >> 7) & (cb - 1u)) << 4));
                                Chunk o, b;
                                if constexpr (BETA) b.u = lds128(oa);
#pragma unroll
                                for (int e = 0; e < V; ++e) {
                                    T x = scale(alpha, r[e].e[d]);
                                    if constexpr (BETA) x = add(x, scale(beta, b.e[e]));
                                    o.e[e] = x;
                                }
                                sts128(oa, o.u);
                            }
                        }
                    }
                    }
                } else {
                    const int n_chunks = (int)(tile_bytes >> 4);
                    const int n_cons = n_cons_warps * 32;
                    for (int ch = cw * 32 + lane; ch < n_chunks; ch += n_cons) {
                        Chunk a, b, o;
                        a.u = lds128(in_s + ((uint32_t)ch << 4));
                        if constexpr (BETA) b.u = lds128(out_s + ((uint32_t)ch << 4));
#pragma unroll
                        for (int e = 0; e < V; ++e) {
                            T x = scale(alpha, a.e[e]);
                            if constexpr (BETA) x = add(x, scale(beta, b.e[e]));
                            o.e[e] = x;
                        }
                        sts128(out_s + ((uint32_t)ch << 4), o.u);
                    }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the stores read what was just written
            }
            __syncwarp();
            if (lane == 0)
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(&done_bar[s])) : "memory");
            if (end) break;
        }
    }
}

// ------------------------------------------------------------------------------------------
// tmapu_kernel: the residue-class flavour (ttc_tmap.h) -- strides that are not multiples of 16 bytes, any rank, any
// element-aligned base.  Same pipeline as tmap_kernel; a plane is V in- and V out-sub-boxes of 1 KB.
// ------------------------------------------------------------------------------------------
struct TmapUSet { CUtensorMap a[kTmapUMaxClasses * 2], b[kTmapUMaxClasses * 2]; };   // [skew * 2 + (0: classes with one row more, 1: the others)]

template <int DT, bool BETA>
__global__ void __launch_bounds__(256)
tmapu_kernel(const __grid_constant__ TmapUParams P, const __grid_constant__ TmapUSet M, const Scalar alpha_in, const Scalar beta_in) {
    using T = typename ElemT<DT>::T;
    constexpr int ES = (int)sizeof(T);
    constexpr int V = 16 / ES;                 // 4 or 2
    constexpr int LGV = V == 4 ? 2 : 1;
    constexpr int TE = 128 / ES;               // plane edge in elements
    static_assert(V == 4 || V == 2, "residue classes exist for 4- and 8-byte elements only");
    union Chunk { uint4 u; T e[V]; };
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t raw = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t buf_bytes = (uint32_t)P.nP * V * 1024u;

    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    __shared__ __align__(8) uint64_t full_bar[kTmapMaxStages], done_bar[kTmapMaxStages], outfree_bar[kTmapMaxStages];
    __shared__ int64_t off_of[kTmapMaxStages][2][2];      // [stage][use parity][A, B]: offset of the tile's outer indices + base skew
    __shared__ int32_t org_of[kTmapMaxStages][2][2];      // a_tile, b_tile
    __shared__ uint32_t tile_of[kTmapMaxStages][2];

    const int tid = threadIdx.x, lane = tid & 31;
    const int S = P.stages;
    const int n_cons_warps = ((int)blockDim.x >> 5) - 2;
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&full_bar[s])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&done_bar[s])), "r"(n_cons_warps));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[s])));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();

    if (tid < 32) {
        // ------------------------------------------------------------------ producer warp
        uint32_t tile_id = blockIdx.x;
        bool more = true;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            const int u = (int)((it / (uint32_t)S) & 1u);
            const uint32_t full_a = (uint32_t)__cvta_generic_to_shared(&full_bar[s]);
            if (it >= (uint32_t)S) {
                mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                if constexpr (BETA) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
            }
            if (!more) {
                if (lane == 0) {
                    tile_of[s][u] = 0xFFFFFFFFu;
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_a) : "memory");
                }
                break;
            }
            sched.prefetch();
            if (lane == 0) {
                uint32_t r = tile_id;
                int32_t org[2];
                int64_t ca = P.skewA0, cb = P.skewB0;
                for (int d = 0; d < P.nG; ++d) {
                    const uint32_t qq = fd_div(r, P.gdiv[d]);
                    const uint32_t c = r - qq * P.gdiv[d].d;
                    r = qq;
                    if (d < 2) org[d] = (int32_t)c * TE;
                    else { ca += (int64_t)c * P.stepA[d]; cb += (int64_t)c * P.stepB[d]; }
                }
                org_of[s][u][0] = org[0];
                org_of[s][u][1] = org[1];
                off_of[s][u][0] = ca;
                off_of[s][u][1] = cb;
                tile_of[s][u] = tile_id;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(full_a), "r"(buf_bytes * (BETA ? 2u : 1u)) : "memory");
                const uint32_t in_s = base + (uint32_t)s * 2u * buf_bytes, out_s = in_s + buf_bytes;
                for (int p = 0; p < P.nP; ++p)
#pragma unroll
                    for (int cl = 0; cl < V; ++cl) {
                        const int64_t ra = (int64_t)cl * P.sqA + ca + P.pA[p];
                        const int sk = (int)(ra & (V - 1));
                        tmap_load(in_s + (uint32_t)(p * V + cl) * 1024u, &M.a[sk * 2 + (cl >= P.remA ? 1 : 0)], full_a, org[0] + sk, org[1] >> LGV, (int)(ra >> LGV), 0, 0);
                        if constexpr (BETA) {
                            const int64_t rb = (int64_t)cl * P.s0B + cb + P.pB[p];
                            const int skb = (int)(rb & (V - 1));
                            tmap_load(out_s + (uint32_t)(p * V + cl) * 1024u, &M.b[skb * 2 + (cl >= P.remB ? 1 : 0)], full_a, org[1] + skb, org[0] >> LGV, (int)(rb >> LGV), 0, 0);
                        }
                    }
            }
            more = sched.next<true>(tile_id, P.n_tiles);
            __syncwarp();
        }
    } else if (tid < 64) {
        // ------------------------------------------------------------------ store thread
        if (tid == 32) {
            for (uint32_t it = 0;; ++it) {
                const int s = (int)(it % (uint32_t)S);
                const int u = (int)((it / (uint32_t)S) & 1u);
                mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), (uint32_t)u);
                if (tile_of[s][u] == 0xFFFFFFFFu) break;
                const int32_t org0 = org_of[s][u][0], org1 = org_of[s][u][1];
                const int64_t cb = off_of[s][u][1];
                const uint32_t out_s = base + (uint32_t)s * 2u * buf_bytes + buf_bytes;
                for (int p = 0; p < P.nP; ++p)
#pragma unroll
                    for (int cl = 0; cl < V; ++cl) {
                        const int64_t rb = (int64_t)cl * P.s0B + cb + P.pB[p];
                        const int skb = (int)(rb & (V - 1));
                        tmap_store(&M.b[skb * 2 + (cl >= P.remB ? 1 : 0)], out_s + (uint32_t)(p * V + cl) * 1024u, org1 + skb, org0 >> LGV, (int)(rb >> LGV), 0, 0);
                    }
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                if (it >= 1u) {
                    asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];"
                                 ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[(it - 1u) % (uint32_t)S])) : "memory");
                }
            }
            asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        }
    } else {
        // ------------------------------------------------------------------ consumer warps
        const int cw = (tid >> 5) - 2;
        const int A2 = lane & 7;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            mbar_wait((uint32_t)__cvta_generic_to_shared(&full_bar[s]), (it / (uint32_t)S) & 1u);
            const bool end = tile_of[s][(it / (uint32_t)S) & 1u] == 0xFFFFFFFFu;
            if (!end) {
                if constexpr (!BETA)
                    if (it >= (uint32_t)S) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                const uint32_t in_s = base + (uint32_t)s * 2u * buf_bytes, out_s = in_s + buf_bytes;
                for (int p = cw; p < P.nP; p += n_cons_warps) {
                    const uint32_t ip = in_s + (uint32_t)p * (V * 1024u), op = out_s + (uint32_t)p * (V * 1024u);
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const int B2 = (j << 2) | (lane >> 3);
                        Chunk r[V];
#pragma unroll
                        for (int d = 0; d < V; ++d) r[d].u = lds128(ip + (uint32_t)(d * 1024 + B2 * 128 + ((A2 ^ B2) << 4)));
#pragma unroll
                        for (int d = 0; d < V; ++d) {
                            const uint32_t oa = op + (uint32_t)(d * 1024 + A2 * 128 + ((B2 ^ A2) << 4));
                            Chunk o, b;
                            if constexpr (BETA) b.u = lds128(oa);
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                T x = scale(alpha, r[e].e[d]);
                                if constexpr (BETA) x = add(x, scale(beta, b.e[e]));
                                o.e[e] = x;
                            }
                            sts128(oa, o.u);
                        }
                    }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            }
            __syncwarp();
            if (lane == 0)
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(&done_bar[s])) : "memory");
            if (end) break;
        }
    }
}

}  // namespace ttc
