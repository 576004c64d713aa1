// ttc_skew.cuh -- skew_kernel: Eq. 1 for tensors whose rows are not 16-byte aligned, with 1-D bulk copies
// in both directions (see ttc_skew.h).  One CTA = producer warp (32 lanes, one tile row each per pass), store warp
// (32 lanes, one out-row each per pass), consumer warps; stages of (in-tile, out-tile) as in tmap_kernel.
//
//   producer   row of A (TA elements along a0, for one b0 and plane): the 16-byte aligned superset of its bytes is ONE
//              cp.async.bulk into the row's slot; element a then sits at slot + (skew + a) * es, skew = (address & 15) / es,
//              which the lane writes to a table.  beta != 0: B's rows (TB elements along b0) land in the out-tile the
//              same way.  A superset that would reach outside [first, last] element of the tensor (only rows at the very
//              ends of A or B can) is copied element by element instead.
//   consumers  out[a][skewB(a) + b] = alpha * in[b][skewA(b) + a] (+ beta * what is there): lanes along a (conflict-free
//              loads), a warp per b
//   store warp out-row = head (< 16 bytes, element stores) + aligned body (one cp.async.bulk shared -> global) + tail
//
// DIRECT = true: no out-tile and no store warps; the consumers write B themselves, a warp per row of B with its lanes
// along b0 (coalesced element stores, and element loads of B for beta != 0).  In this variant "a0" and "b0" are RUNS of
// merged leading indices (ttc_skew.h): a row of the in-tile is TA consecutive positions of the A-run (contiguous in A),
// a lane's column is one position of the B-run (contiguous in B); the offset in B of an a-position comes from a per-tile
// table (boff), the offset in A of a b-position from decoding it index by index.
#pragma once
#include "ttc_device.cuh"
#include "ttc_skew.h"

namespace ttc {

// Offset in the other tensor of position `idx` of a run (ttc_skew.h).
__device__ __forceinline__ int64_t skew_run_offset(uint32_t idx, int n, const FastDiv* div, const int64_t* stride) {
    int64_t off = 0;
    uint32_t r = idx;
    for (int k = 0; k < n; ++k) {
        const uint32_t q = fd_div(r, div[k]);
        off += (int64_t)(r - q * div[k].d) * stride[k];
        r = q;
    }
    return off;
}

template <int DT, bool BETA, bool DIRECT>
__global__ void __launch_bounds__(384)
skew_kernel(const __grid_constant__ SkewParams P, const void* __restrict__ Ain, void* __restrict__ Bout,
            const Scalar alpha_in, const Scalar beta_in) {
    using T = typename ElemT<DT>::T;
    constexpr int ES = (int)sizeof(T);
    constexpr int V = 16 / ES;
    static_assert(V == 4 || V == 2, "4- and 8-byte elements");
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t raw = (uint32_t)__cvta_generic_to_shared(smem_raw);
    unsigned char* const smem = smem_raw + ((128u - (raw & 127u)) & 127u);
    const int TA = 1 << P.lgTA, TB = 1 << P.lgTB;
    const int rowsA = P.nP << P.lgTB, rowsB = P.nP << P.lgTA;
    const uint32_t in_bytes = (uint32_t)(rowsA * P.pitchA), out_bytes = DIRECT ? 0u : (uint32_t)(rowsB * P.pitchB);
    const uint32_t stage_bytes = in_bytes + out_bytes;

    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    __shared__ __align__(8) uint64_t full_bar[kSkewMaxStages], done_bar[kSkewMaxStages], outfree_bar[kSkewMaxStages];
    __shared__ int64_t off_of[kSkewMaxStages][2][2];         // [stage][use parity][A, B]: element offset of the tile's outer indices
    __shared__ int32_t org_of[kSkewMaxStages][2][2];         // first a0, first b0 of the tile
    __shared__ uint32_t tile_of[kSkewMaxStages][2];
    __shared__ uint32_t tile_pub[2];                         // the tile the producer warps load in iteration it (slot it & 1)
    __shared__ int64_t boff[kSkewMaxStages][256];            // direct-out: offset in B of every a-position of the tile
    __shared__ uint8_t skA[kSkewMaxStages][kSkewMaxRows];    // skew of every in-row (read by the consumers only)
    __shared__ uint8_t skB[kSkewMaxStages][2][kSkewMaxRows]; // skew of every out-row (consumers and, later, the store warp)

    const int tid = threadIdx.x, lane = tid & 31;
    const int S = P.stages;
    const int NP = P.np, NS = DIRECT ? 0 : P.ns;
    const int n_cons_warps = ((int)blockDim.x >> 5) - NP - NS;
    const int warp = tid >> 5;
    const char* const A = static_cast<const char*>(Ain);
    char* const B = static_cast<char*>(Bout);
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&full_bar[s])), "r"(32 * NP));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&done_bar[s])), "r"(n_cons_warps));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[s])), "r"(NS > 0 ? 32 * NS : 1));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();

    if (warp < NP) {
        // ------------------------------------------------------------------ producer warps (warp 0 draws the tiles)
        uint32_t tile_id = blockIdx.x;
        bool more = true;
        for (uint32_t it = 0;; ++it) {
            if (NP > 1) {        // warp 0 publishes the tile of this iteration (0xFFFFFFFF: none left), the others pick it up
                if (tid == 0) tile_pub[it & 1u] = more ? tile_id : 0xFFFFFFFFu;
                asm volatile("bar.sync 1, %0;" ::"r"(32 * NP) : "memory");
                if (warp != 0) {
                    tile_id = tile_pub[it & 1u];
                    more = tile_id != 0xFFFFFFFFu;
                }
            }
            const int s = (int)(it % (uint32_t)S);
            const int u = (int)((it / (uint32_t)S) & 1u);
            const uint32_t full_a = (uint32_t)__cvta_generic_to_shared(&full_bar[s]);
            if (it >= (uint32_t)S) {
                // the in-tile is free once its consumers are done; the out-tile, which only beta != 0 loads into, once the
                // store warp's copies of its last use have read it (beta == 0: the consumers wait for that instead)
                mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                if constexpr (BETA && !DIRECT) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
            }
            if (!more) {
                if (tid == 0) tile_of[s][u] = 0xFFFFFFFFu;
                __syncwarp();
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_a) : "memory");
                break;
            }
            if (warp == 0) sched.prefetch();
            // every lane decodes the tile (cheap) and takes rows lane, lane + 32, ...
            int32_t org0 = 0, org1 = 0;
            int64_t ca = 0, cb = 0;
            {
                uint32_t r = tile_id;
                for (int d = 0; d < P.nG; ++d) {
                    const uint32_t qq = fd_div(r, P.gdiv[d]);
                    const uint32_t c = r - qq * P.gdiv[d].d;
                    r = qq;
                    if (d == 0) org0 = (int32_t)c << P.lgTA;
                    else if (d == 1) org1 = (int32_t)c << P.lgTB;
                    else { ca += (int64_t)c * P.stepA[d]; cb += (int64_t)c * P.stepB[d]; }
                }
            }
            if (tid == 0) {
                org_of[s][u][0] = org0;
                org_of[s][u][1] = org1;
                off_of[s][u][0] = ca;
                off_of[s][u][1] = cb;
                tile_of[s][u] = tile_id;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            unsigned char* const in_s = smem + (uint32_t)s * stage_bytes;
            unsigned char* const out_s = in_s + in_bytes;
            // rows of A: TA elements from (org0, org1 + b) of plane p
            {
                const int64_t left = P.e0 - org0;
                const int len = (int)(left < TA ? left : TA);
                const uintptr_t lo = (uintptr_t)A, hi = lo + (uintptr_t)P.spanA * ES;
                for (int r = warp * 32 + lane; r < rowsA; r += 32 * NP) {      // one row per lane and pass
                    const int p = r >> P.lgTB, b = r & (TB - 1);
                    const int64_t bg = (int64_t)org1 + b;
                    if (bg >= P.eq) { skA[s][r] = 0; continue; }
                    const uintptr_t addr = lo + (uintptr_t)(ca + P.pA[p] + skew_run_offset((uint32_t)bg, P.nB, P.divB, P.sAB) + org0) * ES;
                    const int sk = (int)((addr & 15u) / ES);
                    skA[s][r] = (uint8_t)sk;
                    unsigned char* const slot = in_s + (uint32_t)r * (uint32_t)P.pitchA;
                    const uintptr_t start = addr & ~(uintptr_t)15, end = (addr + (uintptr_t)len * ES + 15u) & ~(uintptr_t)15;
                    if (start >= lo && end <= hi) {
                        const uint32_t bytes = (uint32_t)(end - start);
                        asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(full_a), "r"(bytes) : "memory");
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                     ::"r"((uint32_t)__cvta_generic_to_shared(slot)), "l"(start), "r"(bytes), "r"(full_a) : "memory");
                    } else {
                        const T* src = reinterpret_cast<const T*>(addr);
                        T* dst = reinterpret_cast<T*>(slot) + sk;
                        for (int i = 0; i < len; ++i) dst[i] = src[i];
                    }
                }
            }
            if constexpr (DIRECT) {
                for (int a = warp * 32 + lane; a < TA; a += 32 * NP)
                    boff[s][a] = (int64_t)org0 + a < P.e0 ? skew_run_offset((uint32_t)(org0 + a), P.nA, P.divA, P.sBA) : 0;
            }
            // rows of B: TB elements from (org1, org0 + a) of plane p -- loaded for beta != 0, their skews always
            if constexpr (!DIRECT) {
                const int64_t left = P.eq - org1;
                const int len = (int)(left < TB ? left : TB);
                const uintptr_t lo = (uintptr_t)B, hi = lo + (uintptr_t)P.spanB * ES;
                for (int r = warp * 32 + lane; r < rowsB; r += 32 * NP) {
                    const int p = r >> P.lgTA, a = r & (TA - 1);
                    const int64_t ag = (int64_t)org0 + a;
                    if (ag >= P.e0) { skB[s][u][r] = 0; continue; }
                    const uintptr_t addr = lo + (uintptr_t)(cb + P.pB[p] + skew_run_offset((uint32_t)ag, P.nA, P.divA, P.sBA) + org1) * ES;
                    const int sk = (int)((addr & 15u) / ES);
                    skB[s][u][r] = (uint8_t)sk;
                    if constexpr (BETA) {
                        unsigned char* const slot = out_s + (uint32_t)r * (uint32_t)P.pitchB;
                        const uintptr_t start = addr & ~(uintptr_t)15, end = (addr + (uintptr_t)len * ES + 15u) & ~(uintptr_t)15;
                        if (start >= lo && end <= hi) {
                            const uint32_t bytes = (uint32_t)(end - start);
                            asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(full_a), "r"(bytes) : "memory");
                            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                         ::"r"((uint32_t)__cvta_generic_to_shared(slot)), "l"(start), "r"(bytes), "r"(full_a) : "memory");
                        } else {
                            const T* src = reinterpret_cast<const T*>(addr);
                            T* dst = reinterpret_cast<T*>(slot) + sk;
                            for (int i = 0; i < len; ++i) dst[i] = src[i];
                        }
                    }
                }
            }
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_a) : "memory");
            if (warp == 0) more = sched.next<true>(tile_id, P.n_tiles);
            __syncwarp();
        }
    } else if (!DIRECT && warp < NP + NS) {
        // ------------------------------------------------------------------ store warps
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            const int u = (int)((it / (uint32_t)S) & 1u);
            mbar_wait((uint32_t)__cvta_generic_to_shared(&done_bar[s]), (uint32_t)u);
            if (tile_of[s][u] == 0xFFFFFFFFu) break;
            const int32_t org0 = org_of[s][u][0], org1 = org_of[s][u][1];
            const int64_t cb = off_of[s][u][1];
            unsigned char* const out_s = smem + (uint32_t)s * stage_bytes + in_bytes;
            const int64_t left = P.eq - org1;
            const int len = (int)(left < TB ? left : TB);
            for (int r = (warp - NP) * 32 + lane; r < rowsB; r += 32 * NS) {      // one out-row per lane and pass
                const int p = r >> P.lgTA, a = r & (TA - 1);
                const int64_t ag = (int64_t)org0 + a;
                if (ag >= P.e0) continue;
                T* const dst = reinterpret_cast<T*>(B) + (cb + P.pB[p] + skew_run_offset((uint32_t)ag, P.nA, P.divA, P.sBA) + org1);
                const int sk = (int)skB[s][u][r];
                const T* const row = reinterpret_cast<const T*>(out_s + (uint32_t)r * (uint32_t)P.pitchB) + sk;
                int head = (V - sk) & (V - 1);
                head = head < len ? head : len;
                const int body = (len - head) & ~(V - 1);
                if (body > 0)
                    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                                 ::"l"(dst + head), "r"((uint32_t)__cvta_generic_to_shared(row + head)), "r"((uint32_t)(body * ES)) : "memory");
                for (int i = 0; i < head; ++i) dst[i] = row[i];
                for (int i = head + body; i < len; ++i) dst[i] = row[i];
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            if (it >= 1u) {     // this lane's group of the stage before has read its rows: hand that out-tile back
                asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];"
                             ::"r"((uint32_t)__cvta_generic_to_shared(&outfree_bar[(it - 1u) % (uint32_t)S])) : "memory");
            }
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    } else {
        // ------------------------------------------------------------------ consumer warps
        const int cw = warp - NP - NS;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            const int u = (int)((it / (uint32_t)S) & 1u);
            mbar_wait((uint32_t)__cvta_generic_to_shared(&full_bar[s]), (uint32_t)u);
            const bool end = tile_of[s][u] == 0xFFFFFFFFu;
            if constexpr (DIRECT) {
                // no out-tile, no store warps: a warp takes one row of B (fixed a) at a time, its lanes run along b0, so the
                // global accesses are coalesced (element-aligned); the column reads of the in-tile cost up to four wavefronts
                if (!end) {
                    const unsigned char* const in_s = smem + (uint32_t)s * stage_bytes;
                    const int32_t org0 = org_of[s][u][0], org1 = org_of[s][u][1];
                    const int64_t cb = off_of[s][u][1];
                    const int64_t la = P.e0 - org0, lb = P.eq - org1;
                    const int lenA = (int)(la < TA ? la : TA), lenB = (int)(lb < TB ? lb : TB);
                    for (int p = 0; p < P.nP; ++p) {
                        const uint8_t* const skp = &skA[s][p << P.lgTB];
                        const unsigned char* const plane = in_s + (uint32_t)(p << P.lgTB) * (uint32_t)P.pitchA;
                        // a lane owns the columns b = lane + 32 j of B's rows (its skew and its addresses are then fixed: the inner
                        // loop is a load from the in-tile, the arithmetic, a store and two pointer increments); a warp takes
                        // RA rows of B per pass, whose loads of B (beta != 0) are in flight together
                        constexpr int RA = BETA ? 8 : 4;
                        for (int b = lane; b < lenB; b += 32) {
                            const T* const srow = reinterpret_cast<const T*>(plane + (uint32_t)b * (uint32_t)P.pitchA) + skp[b];
                            T* const dcol = reinterpret_cast<T*>(B) + (cb + P.pB[p] + org1 + b);
                            const int64_t* const bo = boff[s];
                            for (int a = cw * RA; a < lenA; a += n_cons_warps * RA) {
                                if (a + RA <= lenA) {
                                    T bv[RA];
                                    if constexpr (BETA) {
#pragma unroll
                                        for (int k = 0; k < RA; ++k) bv[k] = dcol[bo[a + k]];
                                    }
#pragma unroll
                                    for (int k = 0; k < RA; ++k) {
                                        T x = scale(alpha, srow[a + k]);
                                        if constexpr (BETA) x = add(x, scale(beta, bv[k]));
                                        dcol[bo[a + k]] = x;
                                    }
                                } else {
                                    for (int k = 0; a + k < lenA; ++k) {
                                        T x = scale(alpha, srow[a + k]);
                                        if constexpr (BETA) x = add(x, scale(beta, dcol[bo[a + k]]));
                                        dcol[bo[a + k]] = x;
                                    }
                                }
                            }
                        }
                    }
                }
            } else if (!end) {
                if constexpr (!BETA)
                    if (it >= (uint32_t)S) mbar_wait((uint32_t)__cvta_generic_to_shared(&outfree_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
                unsigned char* const in_s = smem + (uint32_t)s * stage_bytes;
                unsigned char* const out_s = in_s + in_bytes;
                // 32 x 32 blocks, walked along diagonals: in step j lane l moves element (a0 + l, b0 + (l + j) % 32).  With row
                // pitches of an odd number of 16-byte units (4 mod 32 words) the 32 lanes hit banks 5 l + 4 j + skew on the
                // in-side and 5 l + j + skew on the out-side: both conflict-free up to the skews' perturbation.  The warps
                // share every block (warp w takes the steps j = w, w + warps, ...).
                const int dq = (int)(P.sAB[0] & (V - 1)), d0 = (int)(P.sBA[0] & (V - 1));      // out-tile variants: nA == nB == 1
                for (int p = 0; p < P.nP; ++p) {
                    const int sA0 = skA[s][p << P.lgTB], sB0 = skB[s][u][p << P.lgTA];      // skews of the plane's first rows
                    for (int a0 = 0; a0 < TA; a0 += 32) {
                        const int a = a0 + lane;
                        const int skb = (sB0 + a * d0) & (V - 1);
                        unsigned char* const orow = out_s + (uint32_t)((p << P.lgTA) + a) * (uint32_t)P.pitchB + skb * ES;
                        const unsigned char* const icol = in_s + (uint32_t)(p << P.lgTB) * (uint32_t)P.pitchA + a * ES;
                        for (int b0 = 0; b0 < TB; b0 += 32) {
#pragma unroll 4
                            for (int j = cw; j < 32; j += n_cons_warps) {
                                const int b = b0 + ((lane + j) & 31);
                                const int ska = (sA0 + b * dq) & (V - 1);
                                const T* const src = reinterpret_cast<const T*>(icol + (uint32_t)b * (uint32_t)P.pitchA + ska * ES);
                                T* const dst = reinterpret_cast<T*>(orow + b * ES);
                                T x = scale(alpha, *src);
                                if constexpr (BETA) x = add(x, scale(beta, *dst));
                                *dst = x;
                            }
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
