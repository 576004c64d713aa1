// ttc_device.cuh -- the device code of libttc.so: element arithmetic, the work scheduler and the three
// kernels.  Included by kernels.cu (all pre-built instances) and, as text, by specialize.cpp, which hands it
// to NVRTC to re-compile a tuned kernel with its parameter block as a compile-time constant
// (TTC generates code for one specific size).  Includes nothing but ttc_params.h.
#pragma once
#include "ttc_params.h"

// Run-time specialisation (specialize.cpp, NVRTC): TTC_SPECIALIZED is defined and ttc::kSpecP holds the
// parameter block of ONE tuned ring-kernel candidate as a constexpr object; the kernel then has no
// TileParams argument, loops over the parameter block are unrolled and every extent, stride, divisor and
// tile shape folds into the instruction stream.
// TTC_SPECIALIZED == 1: a ring-kernel candidate (kSpecP); == 2: a direct-kernel candidate (ttc::kSpecD).
#if defined(TTC_SPECIALIZED)
#define TTC_LOOP_P _Pragma("unroll")
#else
#define TTC_LOOP_P _Pragma("unroll 1")
#endif
#if defined(TTC_SPECIALIZED) && TTC_SPECIALIZED == 1
#define TTC_RING_PARAMS
#else
#define TTC_RING_PARAMS const __grid_constant__ TileParams P,
#endif
#if defined(TTC_SPECIALIZED) && TTC_SPECIALIZED == 2
#define TTC_DIRECT_PARAMS
#else
#define TTC_DIRECT_PARAMS const __grid_constant__ DirectParams P,
#endif

namespace ttc {

// <type_traits> is not available to NVRTC: the two traits the kernels use
template <bool C, typename A, typename B> struct tt_conditional { using type = A; };
template <typename A, typename B> struct tt_conditional<false, A, B> { using type = B; };
template <typename A, typename B> struct tt_is_same { static constexpr bool value = false; };
template <typename A> struct tt_is_same<A, A> { static constexpr bool value = true; };

// ------------------------------------------------------------------------------------------
// Element types and axpby
// ------------------------------------------------------------------------------------------
// DT is a "type pair": 0..3 = ttc_dtype with A and B of the same type; 4..7 = the mixed-precision
// pairs of PAPER.md:75 (sd, ds, cz, zc).  T is B's type -- the type Eq. 1 is evaluated in and the
// type of the shared-memory tile -- and TA is A's type, converted to T as it is loaded (reading M1).
constexpr int kPairSD = 4, kPairDS = 5, kPairCZ = 6, kPairZC = 7;
template <int DT> struct ElemT;
template <> struct ElemT<kF32>  { using T = float;   using TA = float;   static constexpr int ES = 4; };
template <> struct ElemT<kF64>  { using T = double;  using TA = double;  static constexpr int ES = 8; };
template <> struct ElemT<kC64>  { using T = float2;  using TA = float2;  static constexpr int ES = 8; };
template <> struct ElemT<kC128> { using T = double2; using TA = double2; static constexpr int ES = 16; };
template <> struct ElemT<kPairSD>  { using T = double;  using TA = float;   static constexpr int ES = 8; };
template <> struct ElemT<kPairDS>  { using T = float;   using TA = double;  static constexpr int ES = 4; };
template <> struct ElemT<kPairCZ>  { using T = double2; using TA = float2;  static constexpr int ES = 16; };
template <> struct ElemT<kPairZC>  { using T = float2;  using TA = double2; static constexpr int ES = 8; };
// elements per vector: at most 16 bytes in A, in B and in the tile
template <int DT> constexpr int max_vec_of() {
    return 16 / (int)(sizeof(typename ElemT<DT>::T) > sizeof(typename ElemT<DT>::TA) ? sizeof(typename ElemT<DT>::T)
                                                                                      : sizeof(typename ElemT<DT>::TA));
}


// Conversion of an element of A to B's type (reading M1): widening is exact, narrowing is one
// round-to-nearest-even per real component (cvt.rn.f32.f64), as the C cast of the oracle.
__device__ __forceinline__ float   cvt_to(float,   float a)   { return a; }
__device__ __forceinline__ double  cvt_to(double,  double a)  { return a; }
__device__ __forceinline__ float2  cvt_to(float2,  float2 a)  { return a; }
__device__ __forceinline__ double2 cvt_to(double2, double2 a) { return a; }
__device__ __forceinline__ double  cvt_to(double,  float a)   { return (double)a; }
__device__ __forceinline__ float   cvt_to(float,   double a)  { return __double2float_rn(a); }
__device__ __forceinline__ double2 cvt_to(double2, float2 a)  { return make_double2((double)a.x, (double)a.y); }
__device__ __forceinline__ float2  cvt_to(float2,  double2 a) { return make_float2(__double2float_rn(a.x), __double2float_rn(a.y)); }

// alpha / beta in the element type, converted ONCE per thread at kernel entry (the launcher passes
// doubles; converting at every use costs an F2F per element in the inner loops).
template <typename T> struct TScal;
template <> struct TScal<float>   { float re; };
template <> struct TScal<double>  { double re; };
template <> struct TScal<float2>  { float re, im; };
template <> struct TScal<double2> { double re, im; };
__device__ __forceinline__ void typed(const Scalar& s, TScal<float>& o)   { o.re = (float)s.re; }
__device__ __forceinline__ void typed(const Scalar& s, TScal<double>& o)  { o.re = s.re; }
__device__ __forceinline__ void typed(const Scalar& s, TScal<float2>& o)  { o.re = (float)s.re; o.im = (float)s.im; }
__device__ __forceinline__ void typed(const Scalar& s, TScal<double2>& o) { o.re = s.re; o.im = s.im; }

__device__ __forceinline__ float scale(const TScal<float>& s, float a) { return __fmul_rn(s.re, a); }
__device__ __forceinline__ double scale(const TScal<double>& s, double a) { return __dmul_rn(s.re, a); }
__device__ __forceinline__ float2 scale(const TScal<float2>& s, float2 a) {
    return make_float2(__fsub_rn(__fmul_rn(s.re, a.x), __fmul_rn(s.im, a.y)),
                       __fadd_rn(__fmul_rn(s.re, a.y), __fmul_rn(s.im, a.x)));
}
__device__ __forceinline__ double2 scale(const TScal<double2>& s, double2 a) {
    return make_double2(__dsub_rn(__dmul_rn(s.re, a.x), __dmul_rn(s.im, a.y)),
                        __dadd_rn(__dmul_rn(s.re, a.y), __dmul_rn(s.im, a.x)));
}
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float2 add(float2 a, float2 b) { return make_float2(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)); }
__device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(__dadd_rn(a.x, b.x), __dadd_rn(a.y, b.y)); }

// A vector of V elements moved as one 4/8/16-byte access.
template <int BYTES> struct RawT;
template <> struct RawT<4>  { using T = uint32_t; };
template <> struct RawT<8>  { using T = uint2; };
template <> struct RawT<16> { using T = uint4; };
struct __align__(16) Raw32 { uint4 lo, hi; };      // tile side only: a converted vector of a narrower A type
template <> struct RawT<32> { using T = Raw32; };

template <typename T, int V>
union Pack {
    typename RawT<sizeof(T) * V>::T raw;
    T e[V];
    __device__ Pack() {}
};

template <typename R> __device__ __forceinline__ R ld_stream(const void* p) {
    return __ldcs(reinterpret_cast<const R*>(p));    // read once: evict-first
}
template <typename R> __device__ __forceinline__ R ld_plain(const void* p) {
    return *reinterpret_cast<const R*>(p);
}
template <typename R> __device__ __forceinline__ void st_global(void* p, const R& v) {
    *reinterpret_cast<R*>(p) = v;
}

// Store a loaded vector of V elements into the tile: one vector store, or V element stores when
// the tile rows are not vector-aligned (TileParams::splitA).
template <typename T, int V, typename Raw>
__device__ __forceinline__ void st_tile(unsigned char* p, const Raw& v, bool split) {
    if (V > 1 && split) {
        Pack<T, V> u;
        u.raw = v;
#pragma unroll
        for (int j = 0; j < V; ++j) reinterpret_cast<T*>(p)[j] = u.e[j];
    } else {
        *reinterpret_cast<Raw*>(p) = v;
    }
}

// ------------------------------------------------------------------------------------------
// Work distribution.  Static: persistent grid, CTA c takes work items
// c, c + gridDim.x, ...  Dynamic: the grid has one CTA per work item and a running CTA, instead
// of exiting, cancels the launch of a not-yet-started CTA and takes over its blockIdx
// (Blackwell cluster launch control, clusterlaunchcontrol.try_cancel): still one resident set
// of CTAs whose per-CTA setup is paid once, but SMs that run faster (the two dies see different
// memory latency) take more items.  Measured on B200: a 198 MB copy runs at 6.05 TB/s with
// dynamic distribution against 5.5-5.9 TB/s for any static persistent split (profiles/).
// ------------------------------------------------------------------------------------------
struct WorkSched {
    uint32_t bar, resp, phase;
    int mode;              // 0 static, 1 cluster launch control, 2 atomic counter
    uint32_t* ctr;
    uint32_t pending;      // mode 2: the prefetched item (thread 0)
    bool dyn;
    // Call once per CTA, followed by a __syncthreads() before the first prefetch().
    __device__ __forceinline__ void init(int m, uint64_t* bar_smem, uint4* resp_smem, uint32_t* counter = nullptr) {
        mode = m;
        dyn = m != 0;
        ctr = counter;
        pending = 0;
        phase = 0;
        bar = (uint32_t)__cvta_generic_to_shared(bar_smem);
        resp = (uint32_t)__cvta_generic_to_shared(resp_smem);
        if (mode == 1 && threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    // Ask for the next item while the current one is processed.  Every thread must have left
    // the previous next() (a __syncthreads() in between) before this is called again.
    __device__ __forceinline__ void prefetch() {
        if (mode == 1 && threadIdx.x == 0) {
            asm volatile("fence.proxy.async::generic.release.sync_restrict::shared::cta.cluster;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], 16;" ::"r"(bar) : "memory");
            asm volatile("clusterlaunchcontrol.try_cancel.async.shared::cta.mbarrier::complete_tx::bytes.b128 [%0], [%1];"
                         ::"r"(resp), "r"(bar) : "memory");
        } else if (mode == 2 && threadIdx.x == 0) {
            // persistent grid: items 0..gridDim.x-1 are the CTAs' first ones, the counter hands out the rest
            pending = atomicAdd(ctr, 1u) + gridDim.x;
        }
    }
    // All threads (WARP: only the threads of warp 0): replace `item` by the next one; false when there is none.
    template <bool WARP = false>
    __device__ __forceinline__ bool next(uint32_t& item, uint32_t n_items) {
        if (mode == 0) {
            item += gridDim.x;
            return item < n_items;
        }
        if (mode == 2) {
            if (WARP) {
                item = __shfl_sync(0xFFFFFFFFu, pending, 0);
            } else {
                if (threadIdx.x == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(resp), "r"(pending) : "memory");
                __syncthreads();
                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(item) : "r"(resp) : "memory");
            }
            // The counter is taken n_items times in all (n_items - gridDim.x items + one miss per CTA):
            // whoever draws the last ticket knows nobody will draw again and resets it for the next launch.
            if (threadIdx.x == 0 && item == n_items - 1u + gridDim.x) {
                *ctr = 0;
                __threadfence();
            }
            return item < n_items;
        }
        uint32_t done = 0;
        while (!done) {
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(bar), "r"(phase) : "memory");
        }
        phase ^= 1;
        asm volatile("fence.proxy.async::generic.acquire.sync_restrict::shared::cluster.cluster;" ::: "memory");
        uint32_t ok, nx = 0;
        asm volatile("{ .reg .b128 r; .reg .pred p; ld.shared.b128 r, [%2];\n"
                     "clusterlaunchcontrol.query_cancel.is_canceled.pred.b128 p, r; selp.u32 %0, 1, 0, p;\n"
                     "@p clusterlaunchcontrol.query_cancel.get_first_ctaid::x.b32.b128 %1, r; }"
                     : "=r"(ok), "+r"(nx) : "r"(resp) : "memory");
        item = nx;
        return ok != 0;
    }
};

// Programmatic dependent launch (the launcher sets the stream-serialisation attribute for the
// persistent-grid schedulers): let the next kernel of the stream be scheduled as soon as SM resources
// free up, and wait for the previous kernel's memory before the first global access.  Both are
// no-ops for a launch without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// The kernels are instantiated twice: for a single problem (BT = NoBatch: no pointer table among the kernel
// parameters, nothing to decode) and for ttc_execute_batched (BT = BatchPtrs).
struct NoBatch { static constexpr int n = 0; };
__device__ __forceinline__ uint32_t batch_item(const NoBatch&, uint32_t w, const char*&, char*&) { return w; }
// Batched launch: work item `w` of the whole launch -> (problem, item inside it); A and B of that problem.
__device__ __forceinline__ uint32_t batch_item(const BatchPtrs& Bt, uint32_t w, const char*& A, char*& B) {
    if (Bt.n == 0) return w;
    const uint32_t bi = fd_div(w, Bt.div);
    A = static_cast<const char*>(Bt.a[bi]);
    B = static_cast<char*>(Bt.b[bi]);
    return w - bi * Bt.per;
}

// ------------------------------------------------------------------------------------------
// K1: direct kernel
// ------------------------------------------------------------------------------------------

template <int DT, int V, bool BETA, bool IDX64, typename BT>
__global__ void __launch_bounds__(kDirectThreads)
direct_kernel(TTC_DIRECT_PARAMS const void* __restrict__ Ain, void* __restrict__ Bout,
              const Scalar alpha_in, const Scalar beta_in, const __grid_constant__ BT Bt) {
#if defined(TTC_SPECIALIZED) && TTC_SPECIALIZED == 2
    constexpr const DirectParams& P = kSpecD;
#endif
    using T = typename ElemT<DT>::T;
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);
    using TA = typename ElemT<DT>::TA;
    using PackT = Pack<T, V>;
    using PackA = Pack<TA, V>;
    using Raw = typename RawT<sizeof(T) * V>::T;
    using RawA = typename RawT<sizeof(TA) * V>::T;
    using idx_t = typename tt_conditional<IDX64, uint64_t, uint32_t>::type;
    using eoff_t = typename tt_conditional<IDX64, int64_t, uint32_t>::type;   // element offsets
    const char* A = static_cast<const char*>(Ain);
    char* B = static_cast<char*>(Bout);
    const idx_t n = (idx_t)P.n_items;
    const uint32_t n_work = Bt.n ? P.n_chunks * (uint32_t)Bt.n : P.n_chunks;
    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    // work item = chunk of kDirectThreads * kDirectUnroll consecutive vectors; inside a chunk the
    // thread handles vectors tid, tid + 256, ... so every warp access is one contiguous run
    uint32_t chunk = blockIdx.x;
    for (;;) {
        sched.prefetch();
        const idx_t first = (idx_t)batch_item(Bt, chunk, A, B) * (idx_t)(kDirectThreads * kDirectUnroll) + threadIdx.x;
        PackA a[kDirectUnroll];
        PackT b[kDirectUnroll];
        eoff_t oa[kDirectUnroll], ob[kDirectUnroll];
        idx_t r[kDirectUnroll];
        bool ok[kDirectUnroll];
#pragma unroll
        for (int k = 0; k < kDirectUnroll; ++k) {
            r[k] = first + (idx_t)(k * kDirectThreads);
            ok[k] = r[k] < n;
            oa[k] = 0;
            ob[k] = 0;
        }
        // item -> offsets: the kDirectUnroll decompositions advance together (independent chains)
TTC_LOOP_P
        for (int d = 0; d < P.nd; ++d) {
            const eoff_t sA = (eoff_t)P.dims[d].sA, sB = (eoff_t)P.dims[d].sB;
#pragma unroll
            for (int k = 0; k < kDirectUnroll; ++k) {
                idx_t c;
                if (IDX64) {
                    const idx_t nn = (idx_t)P.dims[d].n;
                    const idx_t qq = r[k] / nn;
                    c = r[k] - qq * nn;
                    r[k] = qq;
                } else {
                    const uint32_t qq = fd_div((uint32_t)r[k], P.dims[d].div);
                    c = (uint32_t)r[k] - qq * P.dims[d].div.d;
                    r[k] = qq;
                }
                oa[k] += (eoff_t)c * sA;
                ob[k] += (eoff_t)c * sB;
            }
        }
#pragma unroll
        for (int k = 0; k < kDirectUnroll; ++k) {
            if (ok[k]) {
                a[k].raw = ld_stream<RawA>(A + (int64_t)oa[k] * (int64_t)sizeof(TA));
                if (BETA) b[k].raw = ld_plain<Raw>(B + (int64_t)ob[k] * (int64_t)sizeof(T));
            }
        }
#pragma unroll
        for (int k = 0; k < kDirectUnroll; ++k) {
            if (ok[k]) {
                PackT o;
#pragma unroll
                for (int j = 0; j < V; ++j) {
                    T x = scale(alpha, cvt_to(T(), a[k].e[j]));
                    if (BETA) x = add(x, scale(beta, b[k].e[j]));
                    o.e[j] = x;
                }
                st_global<Raw>(B + (int64_t)ob[k] * (int64_t)sizeof(T), o.raw);
            }
        }
        const bool more = sched.next(chunk, n_work);
        if (!more) break;
        if (sched.dyn) __syncthreads();   // everyone has read the response before the next prefetch
    }
}

// ------------------------------------------------------------------------------------------
// K2/K3: tile kernel
// ------------------------------------------------------------------------------------------
constexpr int kTileUnroll = 4;
// Register budget of the beta == 0 instances: 6 resident CTAs of 256 threads (<= 40 registers, no
// spills).  The kernel is latency bound and every experiment that traded occupancy for fewer
// instructions or deeper prefetch lost; 5 -> 6 CTAs gains 2-3 %.
// The beta != 0 instances need more registers (the B vectors in flight) and are left alone.
constexpr int kTileMinCtas = 6;

template <int DT, int VA, int VB, bool SAME, bool BETA, typename BT>
__global__ void __launch_bounds__(kTileThreads, BETA ? 4 : kTileMinCtas)
tile_kernel(const __grid_constant__ TileParams P, const void* __restrict__ Ain, void* __restrict__ Bout,
            const Scalar alpha_in, const Scalar beta_in, const __grid_constant__ BT Bt) {
    using T = typename ElemT<DT>::T;
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);
    using TA = typename ElemT<DT>::TA;
    constexpr int ES = (int)sizeof(T);       // B and the tile
    constexpr int ESA = (int)sizeof(TA);     // A
    using RawA = typename RawT<ESA * VA>::T;
    using RawS = typename RawT<ES * VA>::T;  // a loaded vector after conversion to T
    using RawB = typename RawT<ES * VB>::T;
    extern __shared__ __align__(16) unsigned char smem[];
    const TileSmemLayout L = tile_smem_layout(P, ES);
    int2* tabs[4];
    uint8_t* vals[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        tabs[i] = reinterpret_cast<int2*>(smem + L.tab[i]);
        vals[i] = smem + L.val[i];
    }
    int32_t* vext = reinterpret_cast<int32_t*>(smem + L.vext);
    unsigned char* tile = smem + L.tile;
    const int tid = threadIdx.x;
    const int NT = blockDim.x;
    const char* A = static_cast<const char*>(Ain);
    char* B = static_cast<char*>(Bout);

    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();

    // Offset tables: entry -> (global element offset, tile element offset), once per CTA.
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const Table& tb = P.tab[i];
        for (int idx = tid; idx < tb.n; idx += NT) {
            uint32_t r = (uint32_t)idx;
            int32_t g = 0, s = 0;
#pragma unroll 1
            for (int k = 0; k < tb.nd; ++k) {
                const uint32_t qq = fd_div(r, tb.d[k].div);
                const uint32_t c = r - qq * tb.d[k].div.d;
                r = qq;
                g += (int32_t)c * (int32_t)tb.d[k].sG;
                s += (int32_t)c * tb.d[k].sS;
            }
            tabs[i][idx] = make_int2(g, s);
        }
    }
    __syncthreads();
    pdl_wait();

    uint32_t tile_id = blockIdx.x;
    for (;;) {
        sched.prefetch();
        // macro-tile id -> tile coordinates in the candidate's loop order
        int64_t baseA = 0, baseB = 0;
        bool edge = false;
        {
            uint32_t r = batch_item(Bt, tile_id, A, B);
#pragma unroll 1
            for (int g = 0; g < P.nG; ++g) {
                const uint32_t qq = fd_div(r, P.g[g].div);
                const uint32_t c = r - qq * P.g[g].div.d;
                r = qq;
                const int32_t start = (int32_t)c * P.g[g].t;
                baseA += (int64_t)start * P.g[g].sA;
                baseB += (int64_t)start * P.g[g].sB;
                const int32_t left = P.g[g].e - start;
                edge |= left < P.g[g].t;
                if (tid == 0) vext[g] = left < P.g[g].t ? left : P.g[g].t;
            }
        }
        if (edge) {  // remainder tile: mark which table entries are inside the tensor
            __syncthreads();
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const Table& tb = P.tab[i];
                for (int idx = tid; idx < tb.n; idx += NT) {
                    uint32_t r = (uint32_t)idx;
                    bool ok = true;
#pragma unroll 1
                    for (int k = 0; k < tb.nd; ++k) {
                        const uint32_t qq = fd_div(r, tb.d[k].div);
                        const uint32_t c = r - qq * tb.d[k].div.d;
                        r = qq;
                        ok &= (int32_t)c * tb.d[k].step < vext[tb.d[k].gslot] * tb.d[k].vmul;
                    }
                    vals[i][idx] = ok ? 1 : 0;
                }
            }
            __syncthreads();
        }

        const char* Ab = A + baseA * ESA;
        char* Bb = B + baseB * ES;
        // ---- load phase: A -> tile, enumerated in ascending A-stride --------------------
        for (uint32_t q0 = tid; q0 < P.itemsA; q0 += NT * kTileUnroll) {
            RawA v[kTileUnroll];
            int32_t so[kTileUnroll];
            bool ok[kTileUnroll];
#pragma unroll
            for (int k = 0; k < kTileUnroll; ++k) {
                const uint32_t q = q0 + k * NT;
                ok[k] = q < P.itemsA;
                if (ok[k]) {
                    const uint32_t hi = fd_div(q, P.divAlo);
                    const uint32_t lo = q - hi * P.divAlo.d;
                    const int2 el = tabs[0][lo], eh = tabs[1][hi];
                    if (edge) ok[k] = vals[0][lo] & vals[1][hi];
                    so[k] = el.y + eh.y;
                    if (ok[k]) v[k] = ld_stream<RawA>(Ab + (int64_t)(el.x + eh.x) * ESA);
                }
            }
#pragma unroll
            for (int k = 0; k < kTileUnroll; ++k) {
                if (!ok[k]) continue;
                if constexpr (tt_is_same<T, TA>::value) {
                    st_tile<T, VA, RawA>(tile + so[k] * ES, v[k], P.splitA != 0);
                } else {   // mixed precision: the tile holds B's type
                    Pack<TA, VA> in;
                    Pack<T, VA> cv;
                    in.raw = v[k];
#pragma unroll
                    for (int j = 0; j < VA; ++j) cv.e[j] = cvt_to(T(), in.e[j]);
                    st_tile<T, VA, RawS>(tile + so[k] * ES, cv.raw, P.splitA != 0);
                }
            }
        }
        __syncthreads();

        // ---- store phase: tile -> B, enumerated in ascending B-stride -------------------
        for (uint32_t p0 = tid; p0 < P.itemsB; p0 += NT * kTileUnroll) {
            Pack<T, VB> bv[kTileUnroll];
            int32_t so[kTileUnroll], go[kTileUnroll];
            bool ok[kTileUnroll];
#pragma unroll
            for (int k = 0; k < kTileUnroll; ++k) {
                const uint32_t p = p0 + k * NT;
                ok[k] = p < P.itemsB;
                if (ok[k]) {
                    const uint32_t hi = fd_div(p, P.divBlo);
                    const uint32_t lo = p - hi * P.divBlo.d;
                    const int2 el = tabs[2][lo], eh = tabs[3][hi];
                    if (edge) ok[k] = vals[2][lo] & vals[3][hi];
                    so[k] = el.y + eh.y;
                    go[k] = el.x + eh.x;
                    if (BETA && ok[k]) bv[k].raw = ld_plain<RawB>(Bb + (int64_t)go[k] * ES);
                }
            }
#pragma unroll
            for (int k = 0; k < kTileUnroll; ++k) {
                if (ok[k]) {
                    Pack<T, VB> a, o;
                    if (SAME || VB == 1) {
                        a.raw = *reinterpret_cast<const RawB*>(tile + so[k] * ES);
                    } else {
#pragma unroll
                        for (int j = 0; j < VB; ++j)
                            a.e[j] = *reinterpret_cast<const T*>(tile + (so[k] + j * P.sstepB) * ES);
                    }
#pragma unroll
                    for (int j = 0; j < VB; ++j) {
                        T x = scale(alpha, a.e[j]);
                        if (BETA) x = add(x, scale(beta, bv[k].e[j]));
                        o.e[j] = x;
                    }
                    st_global<RawB>(Bb + (int64_t)go[k] * ES, o.raw);
                }
            }
        }
        const bool more = sched.next(tile_id, Bt.n ? P.n_tiles * (uint32_t)Bt.n : P.n_tiles);
        if (!more) break;
        __syncthreads();   // tile and scheduler response are free again
    }
}

// ------------------------------------------------------------------------------------------
// K2/K3, warp-specialised: ring kernel (class TTC_KERNEL_TMA)
//
// Warp 0 is the producer: for each macro-tile it takes from WorkSched it issues one
// cp.async.bulk (TMA bulk copy, global -> shared, completion on an mbarrier) per tile row into
// the next free buffer of a ring of `P.ring` tile buffers.  The other warps are consumers: they
// wait for a full buffer, run the store phase of tile_kernel on it (gather from the tile in
// B order, alpha/beta, 16-byte stores) and hand the buffer back.  The load of the next tiles is
// therefore in flight for the whole store phase of the current one, inside ONE CTA, instead of
// relying on many resident CTAs to overlap the two streams.  Rows that are not 16-byte multiples
// are copied with element-sized cp.async instead (P.row_async); edge tiles get shorter and fewer
// rows.  Mixed precision (DT = a type pair): the bulk copies land A's bytes, so the tile holds
// A's type and the consumers convert each element to B's type as they read it (reading M1).
// ------------------------------------------------------------------------------------------
// cp.async: global -> shared without a register stop (LDGSTS), BYTES = 4, 8 or 16.
template <int BYTES>
__device__ __forceinline__ void cp_async(unsigned char* smem_dst, const char* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    if constexpr (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
    else if constexpr (BYTES == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done = 0;
    while (!done) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    }
}

template <int DT, int VB, bool BETA, bool PEEL, bool SHIFT, typename BT>
__global__ void __launch_bounds__(kRingThreads, (PEEL || (BETA && VB == 1 && SHIFT)) ? 3 : BETA ? 4 : 5)
ring_kernel(TTC_RING_PARAMS const void* __restrict__ Ain, void* __restrict__ Bout,
            const Scalar alpha_in, const Scalar beta_in, const __grid_constant__ BT Bt) {
#if defined(TTC_SPECIALIZED) && TTC_SPECIALIZED == 1
    constexpr const TileParams& P = kSpecP;    // the tuned candidate's parameter block, a compile-time constant
#endif
    using T = typename ElemT<DT>::T;
    TScal<T> alpha, beta;
    typed(alpha_in, alpha);
    typed(beta_in, beta);         // B
    using TA = typename ElemT<DT>::TA;       // A and the tile: bulk copies land A's bytes unconverted,
    constexpr int ES = (int)sizeof(T);       // the consumers convert (mixed precision, reading M1)
    constexpr int ESA = (int)sizeof(TA);
    constexpr bool MIXED = !tt_is_same<T, TA>::value;
    using RawB = typename RawT<ES * VB>::T;
    extern __shared__ __align__(16) unsigned char smem[];
    const TileSmemLayout L = tile_smem_layout(P, ESA);
    int2* tabs[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) tabs[i] = reinterpret_cast<int2*>(smem + L.tab[i]);
    const int tid = threadIdx.x;
    const int NT = blockDim.x;
    const int S = P.ring;
    const char* A = static_cast<const char*>(Ain);
    char* B = static_cast<char*>(Bout);

    __shared__ __align__(16) uint4 sched_resp;
    __shared__ __align__(8) uint64_t sched_bar;
    __shared__ __align__(8) uint64_t full_bar[kRingMaxStages], empty_bar[kRingMaxStages];
    __shared__ uint32_t tile_of[kRingMaxStages];
    __shared__ uint32_t edge_of[kRingMaxStages];
    __shared__ uint32_t shift_of[kRingMaxStages];   // shifted rows: misalignment of the tile origin in A, << 30
    WorkSched sched;
    sched.init(P.dyn, &sched_bar, &sched_resp, P.ctr);
    pdl_launch_dependents();
    const int n_cons_warps = (NT >> 5) - 1;
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            // full: one expect_tx arrival (bulk rows) or one arrival per producer lane (cp.async rows)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&full_bar[s])), "r"(P.row_async ? 32 : 1));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&empty_bar[s])), "r"(n_cons_warps));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // Offset tables (1: rows of the A side, 2/3: lo/hi of the B side), once per CTA.
#pragma unroll
    for (int i = 1; i < 4; ++i) {
        const Table& tb = P.tab[i];
        for (int idx = tid; idx < tb.n; idx += NT) {
            uint32_t r = (uint32_t)idx;
            int32_t g = 0, s = 0;
            uint32_t a = 0;
TTC_LOOP_P
            for (int k = 0; k < tb.nd; ++k) {
                const uint32_t qq = fd_div(r, tb.d[k].div);
                const uint32_t c = r - qq * tb.d[k].div.d;
                r = qq;
                g += (int32_t)c * (int32_t)tb.d[k].sG;
                s += (int32_t)c * tb.d[k].sS;
                a += c * (uint32_t)tb.d[k].aS;
            }
            // shifted rows: bits 30-31 carry the entry's contribution to its tile row's misalignment
            // in A (mod 4 elements); the sum of lo + hi + tile origin wraps mod 4 by itself
            tabs[i][idx] = make_int2(g, s | (int32_t)(a << 30));
        }
    }
    __syncthreads();
    pdl_wait();

    if (tid < 32) {
        // ---------------- producer warp ----------------
        const int lane = tid;
        const int rows = P.tab[1].n;
        uint32_t tile_id = blockIdx.x;
        bool more = true;
        for (uint32_t it = 0;; ++it) {
            const int s = (int)(it % (uint32_t)S);
            const uint32_t full_a = (uint32_t)__cvta_generic_to_shared(&full_bar[s]);
            if (it >= (uint32_t)S)   // the consumers have handed this buffer back
                mbar_wait((uint32_t)__cvta_generic_to_shared(&empty_bar[s]), ((it / (uint32_t)S) - 1u) & 1u);
            if (!more) {             // end marker for the consumers
                if (lane == 0) tile_of[s] = 0xFFFFFFFFu;
                __syncwarp();
                if (lane == 0 || P.row_async)
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_a) : "memory");
                break;
            }
            sched.prefetch();
            int64_t baseA = 0;
            bool edge = false;
            int32_t* vx = reinterpret_cast<int32_t*>(smem + L.rvext) + s * kMaxRank;
            {
                char* Bunused = nullptr;
                uint32_t r = batch_item(Bt, tile_id, A, Bunused);
TTC_LOOP_P
                for (int g = 0; g < P.nG; ++g) {
                    const uint32_t qq = fd_div(r, P.g[g].div);
                    const uint32_t c = r - qq * P.g[g].div.d;
                    r = qq;
                    const int32_t start = (int32_t)c * P.g[g].t;
                    baseA += (int64_t)start * P.g[g].sA;
                    const int32_t left = P.g[g].e - start;
                    edge |= left < P.g[g].t;
                    if (lane == 0) vx[g] = left < P.g[g].t ? left : P.g[g].t;
                }
            }
            const char* Ab = A + baseA * ESA;
            unsigned char* tile = smem + L.tile + (uint32_t)s * L.tile_stride;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            uint32_t row_bytes = P.row_bytes;
            uint64_t row_ok = ~0ull;            // bit j: row lane + 32 j is inside the tensor
            uint32_t n_rows = (uint32_t)rows;
            if (edge) {   // remainder tile: shorter rows, fewer rows
                __syncwarp();
                const int valid = vx[P.lead_gslot] * P.lead_vmul * ESA;
                row_bytes = (uint32_t)valid < row_bytes ? (uint32_t)valid : row_bytes;
                row_ok = 0;
                const Table& tb = P.tab[1];
                int j = 0;
                for (int row = lane; row < rows; row += 32, ++j) {
                    uint32_t r = (uint32_t)row;
                    bool ok = true;
TTC_LOOP_P
                    for (int k = 0; k < tb.nd; ++k) {
                        const uint32_t qq = fd_div(r, tb.d[k].div);
                        const uint32_t c = r - qq * tb.d[k].div.d;
                        r = qq;
                        ok &= (int32_t)c * tb.d[k].step < vx[tb.d[k].gslot] * tb.d[k].vmul;
                    }
                    if (ok) row_ok |= 1ull << j;
                }
                n_rows = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)__popcll(row_ok));
            }
            if constexpr (SHIFT) {
                // Shifted rows: lane handles rows lane, lane + 32, ...  The 16-byte aligned body of a row is one
                // bulk copy that lands at the row's own misalignment sk (elements) behind its 16-byte aligned
                // slot; the < 16-byte head and tail are element-sized cp.async.  Nothing outside the row is read.
                constexpr int MVE = 16 / ESA;
                const uint32_t org = (uint32_t)((reinterpret_cast<uintptr_t>(A) / ESA + (uint64_t)baseA) & (MVE - 1));
                if (lane == 0) {
                    tile_of[s] = tile_id;
                    edge_of[s] = edge ? 1u : 0u;
                    shift_of[s] = org << 30;
                }
                const int len = (int)(row_bytes / ESA);
                int j = 0;
                for (int row = lane; row < rows; row += 32, ++j) {
                    if (!((row_ok >> j) & 1ull)) continue;
                    const int2 e = tabs[1][row];
                    const int sk = (int)((org + (uint32_t)e.x) & (MVE - 1));
                    int h = (MVE - sk) & (MVE - 1);
                    h = h < len ? h : len;
                    const int body = (len - h) & ~(MVE - 1);
                    const char* src = Ab + (int64_t)e.x * ESA;
                    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + (e.y + sk) * ESA);
                    if (body > 0) {
                        asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(full_a), "r"(body * ESA) : "memory");
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                     ::"r"(dst + h * ESA), "l"(src + h * ESA), "r"(body * ESA), "r"(full_a) : "memory");
                    }
#pragma unroll
                    for (int i = 0; i < MVE - 1; ++i) {
                        if (i < h) {
                            if constexpr (ESA == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst + i * ESA), "l"(src + i * ESA) : "memory");
                            else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + i * ESA), "l"(src + i * ESA) : "memory");
                        }
                        const int t = h + body + i;
                        if (t < len) {
                            if constexpr (ESA == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst + t * ESA), "l"(src + t * ESA) : "memory");
                            else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + t * ESA), "l"(src + t * ESA) : "memory");
                        }
                    }
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(full_a) : "memory");
            } else if (P.row_async) {
                // Rows that are not 16-byte aligned (odd extents of 4/8-byte elements): the warp copies
                // each row with element-sized cp.async (LDGSTS), 32 elements per instruction; each lane
                // then lets the mbarrier track its copies (cp.async.mbarrier.arrive.noinc).
                if (lane == 0) {
                    tile_of[s] = tile_id;
                    edge_of[s] = edge ? 1u : 0u;
                }
                const int len = (int)(row_bytes / ESA);
                for (int row = 0; row < rows; ++row) {
                    if (edge && !((__shfl_sync(0xFFFFFFFFu, (unsigned)(row_ok >> (row >> 5)), row & 31)) & 1u)) continue;
                    const int2 e = tabs[1][row];
                    // one warp instruction copies 32 consecutive elements; pointers advance by constants
                    if (ESA == 4 && P.row_pairs) {   // 4-byte elements whose rows are all 8-byte aligned: pairs
                        const char* src = Ab + ((int64_t)e.x + 2 * lane) * ESA;
                        uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + (e.y + 2 * lane) * ESA);
                        const int n = ((len >> 1) - lane + 31) >> 5;
#pragma unroll 4
                        for (int i = 0; i < n; ++i) {
                            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
                            dst += 64 * ESA;
                            src += 64 * ESA;
                        }
                        continue;
                    }
                    const char* src = Ab + ((int64_t)e.x + lane) * ESA;
                    uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + (e.y + lane) * ESA);
                    const int n = (len - lane + 31) >> 5;
#pragma unroll 4
                    for (int i = 0; i < n; ++i) {
                        if constexpr (ESA == 4)
                            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
                        else if constexpr (ESA == 8)
                            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
                        else
                            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
                        dst += 32 * ESA;
                        src += 32 * ESA;
                    }
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(full_a) : "memory");
            } else {
            if (lane == 0) {
                tile_of[s] = tile_id;
                edge_of[s] = edge ? 1u : 0u;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                             ::"r"(full_a), "r"(row_bytes * n_rows) : "memory");
            }
            __syncwarp();
            {
                int j = 0;
                for (int row = lane; row < rows; row += 32, ++j) {
                    if (!((row_ok >> j) & 1ull)) continue;
                    const int2 e = tabs[1][row];
                    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(tile + e.y * ESA);
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(dst), "l"(Ab + (int64_t)e.x * ESA), "r"(row_bytes), "r"(full_a) : "memory");
                }
            }
            }
            more = sched.next<true>(tile_id, Bt.n ? P.n_tiles * (uint32_t)Bt.n : P.n_tiles);
            __syncwarp();
        }
        return;
    }
    // ---------------- consumer warps ----------------
    const int ctid = tid - 32;
    const int NC = NT - 32;
    const int sstep = P.sstepB * ESA;
    const bool same = P.same != 0;
    const int rot = P.xp ? ((tid >> 3) & (VB - 1)) : 0;   // staggered gather: this lane's row rotation
    // Shifted rows (P.row_async == 2): tile row r sits sk(r) = 0..MVE-1 elements behind its slot, sk = the row's
    // misalignment in A.  Bits 30-31 of the table entries' tile offsets and of shift_of[] add up to it (mod 4);
    // all of them are 0 for every other kind of tile, so the decoding below is unconditional.
    constexpr uint32_t MVE = 16 / ESA, kOffMask = 0x3FFFFFFFu;
    constexpr int U = (VB == 1 && BETA && SHIFT && ES <= 8) ? 8 : kTileUnroll;
    constexpr bool shifted = SHIFT;
    const int ldm = SHIFT ? P.shift_ld : 0;
    const FastDiv dlo = P.divBlo;
    // division-free enumeration of the store phase (see the loop): needs |lo table| to divide the consumer threads
    const bool lofix = !PEEL && (uint32_t)NC % dlo.d == 0;
    const uint32_t my_lo = lofix ? (uint32_t)ctid % dlo.d : 0u, hi_first = lofix ? (uint32_t)ctid / dlo.d : 0u;
    const uint32_t hi_step = lofix ? (uint32_t)NC / dlo.d : 0u;
    const int2 el_fixed = lofix ? tabs[2][my_lo] : make_int2(0, 0);
    for (uint32_t it = 0;; ++it) {
        const int s = (int)(it % (uint32_t)S);
        mbar_wait((uint32_t)__cvta_generic_to_shared(&full_bar[s]), (it / (uint32_t)S) & 1u);
        const uint32_t tile_id = tile_of[s];
        if (tile_id == 0xFFFFFFFFu) break;
        int64_t baseB = 0;
        {
            const char* Aunused = nullptr;
            uint32_t r = batch_item(Bt, tile_id, Aunused, B);
TTC_LOOP_P
            for (int g = 0; g < P.nG; ++g) {
                const uint32_t qq = fd_div(r, P.g[g].div);
                const uint32_t c = r - qq * P.g[g].div.d;
                r = qq;
                baseB += (int64_t)((int32_t)c * P.g[g].t) * P.g[g].sB;
            }
        }
        char* Bb = B + baseB * ES;
        const unsigned char* tile = smem + L.tile + (uint32_t)s * L.tile_stride;
        const bool edge = edge_of[s] != 0;
        const uint32_t org = shifted ? shift_of[s] : 0u;
        uint8_t* v2 = smem + L.rval + (uint32_t)s * L.rval_stride;
        uint8_t* v3 = v2 + (((uint32_t)P.tab[2].n + 3u) & ~3u);
        if (edge) {   // mark which B-side table entries are inside the tensor (consumers only)
            const int32_t* vx = reinterpret_cast<const int32_t*>(smem + L.rvext) + s * kMaxRank;
#pragma unroll
            for (int i = 2; i < 4; ++i) {
                const Table& tb = P.tab[i];
                uint8_t* val = i == 2 ? v2 : v3;
                for (int idx = ctid; idx < tb.n; idx += NC) {
                    uint32_t r = (uint32_t)idx;
                    bool ok = true;
TTC_LOOP_P
                    for (int k = 0; k < tb.nd; ++k) {
                        const uint32_t qq = fd_div(r, tb.d[k].div);
                        const uint32_t c = r - qq * tb.d[k].div.d;
                        r = qq;
                        ok &= (int32_t)c * tb.d[k].step < vx[tb.d[k].gslot] * tb.d[k].vmul;
                    }
                    val[idx] = ok ? 1 : 0;
                }
            }
            asm volatile("bar.sync 1, %0;" ::"r"(NC) : "memory");
        }
        if constexpr (PEEL) {
            // Peeled store phase for B rows that are not 16-byte aligned (odd extents): a row is cut
            // into 16-byte ALIGNED windows of B; a window inside the row is one vector store, the
            // windows over the row's two ends are element stores.  Item = (row, window).
            const int len = edge ? reinterpret_cast<const int32_t*>(smem + L.rvext)[s * kMaxRank + P.peel_gslot] : P.peel_len;
            const uint32_t nch = dlo.d;                                  // windows per row (divBlo is set to it)
            const int bmis = (int)((reinterpret_cast<uintptr_t>(B) / ES) & (uintptr_t)(VB - 1));
            // element e of the B row whose table entry decodes to (base, sk): tile row (.. + e), whose skew advances by ldm
            auto tile_elem = [&](int32_t sok, int e) -> T {
                if constexpr (!SHIFT) return cvt_to(T(), *reinterpret_cast<const TA*>(tile + sok + e * sstep));
                const int sk = sok & (int)(MVE - 1);
                return cvt_to(T(), *reinterpret_cast<const TA*>(tile + (sok & ~(int)(MVE - 1)) + e * sstep +
                                                                ((sk + e * ldm) & (int)(MVE - 1)) * ESA));
            };
            // pass 1: the windows that lie inside their row -- one vector load of B (beta), VB gathers, one vector
            // store; every lane of a warp takes the same path
            for (uint32_t p0 = ctid; p0 < P.itemsB; p0 += NC * kTileUnroll) {
                Pack<T, VB> bv[kTileUnroll];
                int32_t so[kTileUnroll], go[kTileUnroll], s0[kTileUnroll];
                bool ok[kTileUnroll];
#pragma unroll
                for (int k = 0; k < kTileUnroll; ++k) {
                    const uint32_t p = p0 + k * NC;
                    ok[k] = p < P.itemsB;
                    if (ok[k]) {
                        const uint32_t row = fd_div(p, dlo);
                        const int2 eh = tabs[3][row];
                        if (edge) ok[k] = v3[row] != 0;
                        const int m = (bmis + (int)((baseB + eh.x) & (VB - 1))) & (VB - 1);
                        s0[k] = (int)(p - row * nch) * VB - m;          // first element of the window, row-relative
                        ok[k] = ok[k] && s0[k] >= 0 && s0[k] + VB <= len;
                        const uint32_t t = (uint32_t)eh.y + org;
                        so[k] = SHIFT ? (int32_t)((t & kOffMask) * ESA | ((t >> 30) & (MVE - 1)))   // low bits: the row's skew
                                      : eh.y * ESA;
                        go[k] = eh.x + s0[k];
                        if (BETA && ok[k]) bv[k].raw = ld_plain<RawB>(Bb + (int64_t)go[k] * ES);
                    }
                }
#pragma unroll
                for (int k = 0; k < kTileUnroll; ++k) {
                    if (ok[k]) {
                        Pack<T, VB> o;
#pragma unroll
                        for (int j = 0; j < VB; ++j) {
                            T x = scale(alpha, tile_elem(so[k], s0[k] + j));
                            if (BETA) x = add(x, scale(beta, bv[k].e[j]));
                            o.e[j] = x;
                        }
                        st_global<RawB>(Bb + (int64_t)go[k] * ES, o.raw);
                    }
                }
            }
            // pass 2: the two ends of every row (< VB elements each), element by element.  Item = (row, end).
            const uint32_t n_rows_b = (uint32_t)P.tab[3].n;
            for (uint32_t q = ctid; q < 2u * n_rows_b; q += NC) {
                const uint32_t row = q >> 1;
                if (edge && v3[row] == 0) continue;
                const int2 eh = tabs[3][row];
                const int m = (bmis + (int)((baseB + eh.x) & (VB - 1))) & (VB - 1);
                const int wl = (len + m - 1) / VB;                       // last window that touches the row
                int s0;
                if ((q & 1u) == 0) {           // head: window 0, partial when the row starts inside it
                    if (m == 0 && len >= VB) continue;
                    s0 = -m;
                } else {                       // tail: the last window, unless it is full or is the head's window
                    s0 = wl * VB - m;
                    if (wl == 0 || s0 + VB <= len) continue;
                }
                const uint32_t t = (uint32_t)eh.y + org;
                const int32_t sok = SHIFT ? (int32_t)((t & kOffMask) * ESA | ((t >> 30) & (MVE - 1))) : eh.y * ESA;
#pragma unroll
                for (int j = 0; j < VB; ++j) {
                    const int e = s0 + j;
                    if (e >= 0 && e < len) {
                        T* dst = reinterpret_cast<T*>(Bb + ((int64_t)eh.x + e) * ES);
                        T x = scale(alpha, tile_elem(sok, e));
                        if (BETA) x = add(x, scale(beta, *dst));
                        *dst = x;
                    }
                }
            }
        } else
        // store phase: tile -> B, enumerated in ascending B-stride (as in tile_kernel)
        // U items per thread in flight; the element-wise beta path needs 8 (4-byte loads of B: 4 of them per
        // thread cover too little of the DRAM latency -- profiles/: the first use of the loaded B stalls)
        for (uint32_t p0 = ctid, hb = hi_first; p0 < P.itemsB; p0 += NC * U, hb += hi_step * U) {
            Pack<T, VB> bv[U];
            int32_t so[U], go[U];
            bool ok[U];
#pragma unroll
            for (int k = 0; k < U; ++k) {
                const uint32_t p = p0 + k * NC;
                ok[k] = p < P.itemsB;
                if (ok[k]) {
                    // item p = hi * |lo table| + lo.  When the lo table divides the consumer threads, lo is the
                    // same for every item of a thread (its entry sits in registers) and hi advances by a constant
                    uint32_t hi, lo;
                    int2 el;
                    if (lofix) {
                        hi = hb + k * hi_step;
                        lo = my_lo;
                        el = el_fixed;
                    } else {
                        hi = fd_div(p, dlo);
                        lo = p - hi * dlo.d;
                        el = tabs[2][lo];
                    }
                    const int2 eh = tabs[3][hi];
                    if (edge) ok[k] = v2[lo] & v3[hi];
                    if constexpr (SHIFT) {
                        const uint32_t t = (uint32_t)(el.y + eh.y) + org;
                        so[k] = (int32_t)((t & kOffMask) * ESA);
                        if (VB == 1) so[k] += (int32_t)(((t >> 30) & (MVE - 1)) * ESA);     // the row's skew
                        else so[k] |= (int32_t)((t >> 30) & (MVE - 1));                      // kept in the low bits (VB > 1)
                    } else {
                        so[k] = (el.y + eh.y) * ESA;
                    }
                    go[k] = el.x + eh.x;
                    if (BETA && ok[k]) bv[k].raw = ld_plain<RawB>(Bb + (int64_t)go[k] * ES);
                }
            }
#pragma unroll
            for (int k = 0; k < U; ++k) {
                if (ok[k]) {
                    Pack<T, VB> a, o;
                    if constexpr (MIXED) {   // the tile holds A's type: convert element by element
#pragma unroll
                        for (int j = 0; j < VB; ++j) a.e[j] = cvt_to(T(), *reinterpret_cast<const TA*>(tile + so[k] + j * sstep));
                    } else if (VB == 1 || same) {   // same: the vector leads A and B, chunks move unchanged
                        a.raw = *reinterpret_cast<const RawB*>(tile + so[k]);
                    } else if constexpr (SHIFT) {      // vector of VB tile rows, each behind its slot by its own skew
                        const int sk = so[k] & (int)(MVE - 1), base = so[k] & ~(int)(MVE - 1);
#pragma unroll
                        for (int j = 0; j < VB; ++j)
                            a.e[j] = *reinterpret_cast<const T*>(tile + base + j * sstep + ((sk + j * ldm) & (int)(MVE - 1)) * ESA);
                    } else if constexpr (VB == 2) {
                        // Staggered gather (P.xp): the warp reads 2 columns x 8 row pairs per instruction; lanes
                        // 8..15 and 24..31 take their two rows in the opposite order (rot), which spreads the 16
                        // rows over all banks when the row pitch is an odd multiple of 16 bytes.  rot = 0: plain.
                        const T v0 = *reinterpret_cast<const T*>(tile + so[k] + rot * sstep);
                        const T v1 = *reinterpret_cast<const T*>(tile + so[k] + (1 - rot) * sstep);
                        a.e[0] = rot ? v1 : v0;
                        a.e[1] = rot ? v0 : v1;
                    } else {
                        T v[VB], u[VB];
#pragma unroll
                        for (int j = 0; j < VB; ++j) v[j] = *reinterpret_cast<const T*>(tile + so[k] + ((j + rot) & (VB - 1)) * sstep);
                        // v[j] holds row (j + rot) mod 4: rotate back in two conditional stages
#pragma unroll
                        for (int j = 0; j < VB; ++j) u[j] = (rot & 1) ? v[(j + VB - 1) & (VB - 1)] : v[j];
#pragma unroll
                        for (int j = 0; j < VB; ++j) a.e[j] = (rot & 2) ? u[(j + VB - 2) & (VB - 1)] : u[j];
                    }
#pragma unroll
                    for (int j = 0; j < VB; ++j) {
                        T x = scale(alpha, a.e[j]);
                        if (BETA) x = add(x, scale(beta, bv[k].e[j]));
                        o.e[j] = x;
                    }
                    st_global<RawB>(Bb + (int64_t)go[k] * ES, o.raw);
                }
            }
        }
        __syncwarp();
        if ((tid & 31) == 0)   // this warp no longer reads the buffer
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(&empty_bar[s])) : "memory");
    }
}

}  // namespace ttc
