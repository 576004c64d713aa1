/*
 * ttc.h -- C ABI of libttc.so: out-of-place N-dimensional tensor transposition-and-update
 *
 *         B_{Pi(i_0,...,i_{N-1})}  <-  alpha * A_{i_0,...,i_{N-1}}  +  beta * B_{Pi(i_0,...,i_{N-1})}
 *
 * (arXiv 1607.01249 "TTC", Eq. 1) on column-major tensors (index 0 is
 * stride-1, PAPER.md:49 fn 2) with one optional leading dimension per index (sub-tensors,
 * BLAS-style packing; Fig. 2 and Fig. 3), for the data types
 * s, d, c, z of PAPER.md:75.  Every step of the operation runs in hand-written sm_100a
 * CUDA kernels; there is no CPU fallback.
 *
 * Notation used by every call (DESIGN.md "Readings" A1-A4):
 *   sizes[k]  extent of A's index i_k
 *   perm[k]   the A-index that sits at position k of B, i.e. B's k-th extent is
 *             sizes[perm[k]]          (merge example PAPER.md:63; Fig. 2)
 *   lda[k]    leading dimension of A's index k  (>= sizes[k]);  NULL = contiguous
 *   ldb[k]    leading dimension of B's POSITION k (>= sizes[perm[k]]); NULL = contiguous
 *   element strides: sA[0]=1, sA[k]=sA[k-1]*lda[k-1];  tB[0]=1, tB[k]=tB[k-1]*ldb[k-1]
 *   lda[N-1] / ldb[N-1] are validated but never used for addressing.
 *
 * Ownership: the caller owns A, B and the stream.  A plan owns only its own small host
 * state.  ttc_execute_host uses ONE pair of device staging buffers per process, grown to the
 * largest request and freed by ttc_release_host_staging().  While
 * ttc_plan auto-tunes it allocates scratch device buffers of the real spans of A and B
 * and frees them before it returns; the caller's tensors are never touched by tuning.
 * A candidate that fails to launch during tuning is skipped and counted in ttc_info.tune_errors
 * (the error of that scratch launch is cleared; nothing else clears CUDA errors).
 *
 * Thread safety: distinct plans may be used from distinct threads.  One plan must not be
 * executed, re-tuned or destroyed concurrently from two threads.
 *
 * Environment (read when a plan is built):
 *   TTC_TUNE=0            do not time anything: the heuristic's first choice is used
 *   TTC_TUNE_TOPK=k       time only the k best-ranked candidates of each list (default 32; 0 = all, the
 *                         paper's exhaustive mode)
 *   TTC_COST=legacy       rank candidates with the hand-written round-1 cost formula instead of the fitted one
 *   TTC_TUNE_BUDGET_MS=t  after the first 16 candidates, stop timing a list after t ms (default 400)
 *   TTC_CACHE_FILE=path   solution store on disk (winners appended, reloaded by later processes)
 *   TTC_SCHED=static|both work distribution: persistent grid-stride instead of / beside the default,
 *                         dynamic distribution by cluster launch control
 *   TTC_LOOP_ORDERS=4     also generate the two plane-first macro-tile orders (default 2: A-linear, B-linear)
 *   TTC_SPECIALIZE=1      ttc_plan also runs ttc_plan_specialize (NVRTC size-specialised winners)
 *   TTC_PDL=0             launch without programmatic dependent launch (default: with)
 *   TTC_RING=0|2|4        largest ring of tile buffers of the warp-specialised kernel (0: none; default 4)
 *   TTC_VARIANTS=bits     candidate flavours to generate: 1 staggered-gather ring, 2 shifted-row ring, 4 tensor-map
 *                         kernels, 8 skew kernels that store to B directly, 16 skew kernels with an out-tile and bulk
 *                         stores (default 15; the out-tile variants are 2x slower on B200: only on request)
 */
#ifndef TTC_H_
#define TTC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TTC_MAX_RANK 16

/* s, d, c, z of PAPER.md:75.  Complex = interleaved (re, im). */
typedef enum { TTC_F32 = 0, TTC_F64 = 1, TTC_C64 = 2, TTC_C128 = 3 } ttc_dtype;

typedef enum {
    TTC_OK = 0,
    TTC_ERR_INVALID_ARG = 1,      /* NULL pointer, N < 1, N > TTC_MAX_RANK, negative size, bad dtype */
    TTC_ERR_NOT_PERMUTATION = 2,  /* perm is not a permutation of 0..N-1                             */
    TTC_ERR_BAD_LD = 3,           /* lda[k] < sizes[k] or ldb[k] < sizes[perm[k]]                    */
    TTC_ERR_UNSUPPORTED = 4,      /* spans overflow int64 / more than 2^62 elements                  */
    TTC_ERR_ALLOC = 5,            /* host or device allocation failed                                */
    TTC_ERR_CUDA = 6,             /* a CUDA call failed (no device, launch error, ...)               */
    TTC_ERR_MISALIGNED = 7,       /* A or B is not aligned to its own element size                   */
    TTC_ERR_SCRATCH_LIMIT = 8     /* ttc_execute_host_static: A and B exceed TTC_STATIC_SCRATCH_BYTES */
} ttc_status;

/* Kernel classes. */
typedef enum {
    TTC_KERNEL_NONE = 0,    /* empty tensor: ttc_execute is a no-op                                   */
    TTC_KERNEL_COPY = 1,    /* K1: direct global->global, 128-bit rows when stride-1 index is shared  */
    TTC_KERNEL_TILE = 2,    /* K2: shared-memory tiled transpose in the plane (stride-1 of A, of B)   */
    TTC_KERNEL_GATHER = 3,  /* K3: K2 whose tile sides are coarsened over several leading indices     */
    TTC_KERNEL_WIDE = 4,    /* K2 on "wide elements": a >=16-byte run that leads both A and B         */
    TTC_KERNEL_TMA = 5,     /* K2/K3 warp-specialised: a producer warp fetches the tile rows by TMA
                               bulk copies (cp.async.bulk) into a ring of buffers, consumers store  */
    TTC_KERNEL_TENSORMAP = 6, /* K1/K2/K3 through tensor maps: cp.async.bulk.tensor box loads AND stores
                               (<= 5-D, strides multiples of 16 bytes, 16-byte aligned A and B, same
                               element type), swizzled shared-memory boxes, in-register micro-tiles  */
    TTC_KERNEL_SKEW = 7     /* K2/K3 for rows that are not 16-byte aligned (odd extents): bulk copies of aligned
                               supersets in, skewed shared-memory rows, coalesced element stores out (flag
                               TTC_CAND_DIRECT_OUT) or, on request, an out-tile and bulk stores of aligned bodies */
} ttc_kernel_class;

typedef struct ttc_plan_s* ttc_plan_t;

/* What the plan decided.  All arrays are in canonical order (ascending stride in A). */
typedef struct {
    int      dtype;                       /* ttc_dtype                                             */
    int      rank;                        /* rank N as given                                       */
    int      canon_rank;                  /* rank after dropping extent-1 indices and merging      */
    int64_t  canon_extent[TTC_MAX_RANK];  /* (e, sA, sB) triples of the canonical form */
    int64_t  canon_stride_a[TTC_MAX_RANK];
    int64_t  canon_stride_b[TTC_MAX_RANK];
    int64_t  numel;                       /* logical elements |A|                                  */
    int64_t  span_a, span_b;              /* 1 + largest element offset touched in A / in B        */
    int      tuned;                       /* 1 if the winners were timed on the device             */
    int      n_candidates[2];             /* [0]: beta == 0 variants, [1]: beta != 0               */
    int      chosen[2];                   /* index of the winner in each list                      */
    float    chosen_us[2];                /* its tuned time in microseconds (0 if not tuned)       */
    int      tune_errors;                 /* candidates that failed to configure or launch while tuning
                                             (skipped, never chosen; 0 on a healthy device)         */
    float    plan_ms;                     /* wall time ttc_plan spent building this plan (ms)      */
    float    tune_ms;                     /* the part of it spent timing candidates on the device  */
    int      specialized[2];              /* 0: generic kernel; 1: a size-specialised twin exists but the generic
                                             instance measured faster and is used; 2: the twin is used */
    float    spec_us[2], generic_us[2];   /* their times from ttc_plan_specialize (0 if it was not run) */
} ttc_info;

#define TTC_CAND_STAGGERED 1   /* ring kernel: bank-conflict-free "staggered" gather from the tile      */
#define TTC_CAND_SHIFTED_ROWS 4 /* ring kernel, rows not 16-byte aligned: aligned bodies by bulk copy, skewed tile */
#define TTC_CAND_DIRECT_OUT 8  /* skew kernel without out-tile: the consumers store to B themselves            */
#define TTC_CAND_TENSORMAP 2   /* tiles moved by TMA tensor-map loads / stores (cp.async.bulk.tensor)  */

/* One candidate implementation (loop order x blocking; here also kernel class). */
typedef struct {
    int      kernel;          /* ttc_kernel_class                                              */
    int      vec_a, vec_b;    /* elements per global access on the A side / B side             */
    int      tile_u, tile_w;  /* tile extent along A's leading side / B's leading side (elements; 0 for K1) */
    int      n_u, n_w;        /* number of canonical indices coarsened into each side          */
    int      threads;         /* CTA size                                                      */
    int      smem_bytes;      /* dynamic shared memory per CTA                                 */
    int      loop_order;      /* 0: macro-tiles walk A linearly, 1: walk B linearly            */
    int      sched;           /* 0: static persistent grid-stride, 1: dynamic (cluster launch control),
                                 2: dynamic (atomic counter of the plan; TTC_SCHED=atomic)   */
    int      flags;           /* TTC_CAND_* bits                                               */
    int      grid;            /* CTAs launched, 0 if not yet fixed (dynamic: one per work item, most of
                                 which are cancelled and taken over by the resident CTAs)      */
    float    est_cost;        /* heuristic cost used for ranking (lower is better)             */
    float    tuned_us;        /* measured time, 0 if this candidate was not timed              */
    int64_t  n_tiles;         /* macro-tiles (K2/K3) or vector items (K1)                      */
    int      tile_ext[TTC_MAX_RANK];  /* tile extent per canonical index (1 = outside the tile) */
} ttc_candidate_info;

/*
 * ttc_plan -- validate, canonicalise (drop extent-1 indices, merge indices that Pi keeps
 * adjacent and that are contiguous in both tensors: PAPER.md:63, 95 fn 5), enumerate and
 * rank candidate kernels and, if a CUDA device is present and the
 * environment does not say TTC_TUNE=0, time them in rank order on the device, for beta == 0
 * and for beta != 0, and keep the fastest of each.  The search of one list ends
 * after TTC_TUNE_TOPK candidates (default 32, enough for 0.995 of the exhaustive search's result with
 * the fitted ranking; 0 = all, the paper's exhaustive mode) or, once 16 have been timed, when
 * TTC_TUNE_BUDGET_MS (default 400) milliseconds have passed.
 * Winners are remembered per process; if the environment names a file in TTC_CACHE_FILE they
 * are also appended to it and loaded by later processes (the paper's database of known
 * solutions), so that planning the same transposition again times nothing.
 * All pointers are HOST pointers, read before the call returns.
 * Returns NULL on error; ttc_last_error() then says why.  Sizes of 0 give a valid plan
 * whose execution does nothing.  Without a CUDA device the plan is still built (heuristic
 * choice, tuned = 0) so that it can be inspected; executing it returns TTC_ERR_CUDA.
 */
ttc_plan_t ttc_plan(ttc_dtype dtype, int N, const int64_t* sizes, const int* perm,
                    const int64_t* lda, const int64_t* ldb);

/*
 * ttc_plan_mixed -- ttc_plan for a mixed-precision transposition ("dataType=
 * s,d,c,z,sd,ds,cz,zc"; "different data types for the input tensor A and the output
 * tensor B", e.g. sd: A single, B double).  `dtype_a` is the element type of A, `dtype_b` of B.
 * Accepted pairs: equal types (then this IS ttc_plan(dtype_b, ...)), F32->F64 (sd), F64->F32 (ds),
 * C64->C128 (cz), C128->C64 (zc); any other pair gives NULL / TTC_ERR_UNSUPPORTED.
 * The paper does not say in which precision Eq. 1 is then evaluated; this library (DESIGN.md
 * reading M1) converts each element of A to B's type as it is loaded -- exact for sd and cz, one
 * IEEE-754 round-to-nearest-even per real component for ds and zc (overflow gives +-inf) -- and
 * evaluates Eq. 1 in B's precision, products and sum rounded separately.  For ttc_execute and
 * ttc_execute_host of such a plan, alpha and beta are scalars of B's type, A holds span_a
 * elements of dtype_a and B span_b elements of dtype_b; ttc_info.dtype reports dtype_b and
 * ttc_plan_dtype_a() reports dtype_a.  Everything else is as for ttc_plan.
 */
ttc_plan_t ttc_plan_mixed(ttc_dtype dtype_a, ttc_dtype dtype_b, int N, const int64_t* sizes,
                          const int* perm, const int64_t* lda, const int64_t* ldb);

/*
 * ttc_plan_strided -- ttc_plan_mixed for tensors described by explicit ELEMENT STRIDES instead of leading
 * dimensions (an extension: the paper's interface has leading dimensions only, which cannot
 * express an outer stride that is not a multiple of the inner ones -- BASELINE.json describes configs[3] by
 * "outer stride 6208").  stride_a[k] is the stride of A's index k, stride_b[k] the stride of B's POSITION k
 * (as ldb).  Every stride must be >= 1 and each tensor must be "nested": sorted by stride, each stride is at
 * least the previous stride times the previous extent (so that no two elements of B share an address);
 * otherwise NULL / TTC_ERR_BAD_LD.  A's indices need not be given in ascending stride.  dtype_a == dtype_b
 * gives a same-type plan.  Everything else is as for ttc_plan.
 */
ttc_plan_t ttc_plan_strided(ttc_dtype dtype_a, ttc_dtype dtype_b, int N, const int64_t* sizes, const int* perm,
                            const int64_t* stride_a, const int64_t* stride_b);

/* Element type of A for this plan (equals ttc_info.dtype unless the plan came from
 * ttc_plan_mixed); -1 for a NULL plan. */
int ttc_plan_dtype_a(ttc_plan_t plan);

/*
 * ttc_execute -- Eq. 1 as ONE kernel launch on `cuda_stream` (a cudaStream_t;
 * NULL = the legacy default stream).  Asynchronous; never synchronises.
 *   alpha, beta  HOST pointers to one scalar of the plan's dtype (complex: re, im); read
 *                before the call returns.  beta == 0 (both parts) => B is never read.
 *   A            DEVICE pointer, span_a elements; never written; padding never read.
 *   B            DEVICE pointer, span_b elements; only the elements Pi maps onto are
 *                written; padding never touched.  A and B must not overlap.
 * Pointers only have to be aligned to the element size (16 bytes for complex128); when they
 * are less aligned than the tuned candidate needs, the best candidate of the same plan whose
 * vector widths fit the actual alignment is launched instead (a tile / ring candidate with
 * narrower vectors on the misaligned side; the scalar copy kernel only if nothing else fits).
 * Errors: TTC_ERR_INVALID_ARG (NULL plan/alpha/beta, NULL A or B for a non-empty tensor),
 * TTC_ERR_MISALIGNED, TTC_ERR_CUDA (the launch failed: the code cudaLaunchKernelEx returned;
 * the library neither reads nor clears the thread's CUDA error state here, so an error left
 * by the caller's earlier work is still there afterwards).
 */
ttc_status ttc_execute(ttc_plan_t plan, const void* alpha, const void* A,
                       const void* beta, void* B, void* cuda_stream);

/*
 * ttc_execute_batched -- Eq. 1 for `batch` independent tensor pairs (A_list[i], B_list[i]) that share one
 * plan (same sizes, permutation, leading dimensions, types), in ONE kernel launch per 64 pairs: the
 * macro-tiles of all pairs form one work list for the resident CTAs.  This is how a GEMM's packing routine
 * ("packing kernels ... used by level 3 BLAS") moves many small mc x kc blocks without
 * paying a launch and a machine fill-and-drain per block.  A_list and B_list are HOST arrays of DEVICE
 * pointers, read before the call returns; the pairs must not overlap one another.  alpha, beta, alignment
 * rules (the least aligned pointer decides the candidate), errors and asynchrony are those of ttc_execute;
 * batch == 0 is a no-op, batch < 0 is TTC_ERR_INVALID_ARG.  A tensor-map winner serves the batch through ONE pair of
 * maps (the pair's distance from the lowest address, in 16-byte units, is the coordinate of the fifth map dimension)
 * when the canonical rank is <= 4 and the 64 pairs of a launch lie within 32 GB; otherwise the plan's best other
 * candidate takes the batch.
 */
ttc_status ttc_execute_batched(ttc_plan_t plan, const void* alpha, const void* const* A_list,
                               const void* beta, void* const* B_list, int batch, void* cuda_stream);

/*
 * ttc_execute_host -- the same operation for HOST buffers A (span_a elements) and B
 * (span_b elements): copies A (and B when beta != 0, or when B has padding that has to
 * survive) to the plan's private device staging buffers, runs ttc_execute, copies B back
 * and waits for it.  Synchronous.  Pinned host memory makes the copies faster but is not
 * required.  Contiguous tensors of 16 MB and more are cut into up to 8 slabs along one index:
 * slab c is copied in, transposed and copied out while slab c + 1 is on its way in (the link
 * is full duplex), on two private copy streams and the caller's stream (TTC_HOST_PIPE=0: off).
 */
ttc_status ttc_execute_host(ttc_plan_t plan, const void* alpha, const void* A_host,
                            const void* beta, void* B_host, void* cuda_stream);

/* ttc_destroy -- frees the plan.  NULL is allowed. */
ttc_status ttc_destroy(ttc_plan_t plan);

/*
 * ttc_execute_host_static -- ttc_execute_host for callers that may not allocate device memory (set-up code of
 * a captured graph, tight serving loops, harnesses that forbid cudaMalloc).  Same operation (Eq. 1,
 * PAPER.md:24), same arguments and layouts: A_host holds span_a elements of the plan's dtype_a, B_host span_b
 * elements of dtype_b, alpha and beta are host scalars of B's type.  Instead of the cudaMalloc'ed staging
 * pool, A and B are staged inside ONE file-scope __device__ array of TTC_STATIC_SCRATCH_BYTES (8 MiB) that
 * every GPU holds from the moment it loads that part of the library until the process exits; its first 256
 * bytes are the work counter of the plan's kernel (atomic tile distribution), cleared by every call.  The
 * call itself makes no cudaMalloc / cudaFree and calls no allocating library routine: it clears the counter,
 * copies A (and B when beta != 0 or B has padding) in, launches the plan's generic kernel for the given beta
 * (never an NVRTC twin), copies B back and waits for the stream.  Synchronous.
 * Limit: 256 + round256(span_a * sizeof(dtype_a)) + round256(span_b * sizeof(dtype_b)) must not exceed
 * TTC_STATIC_SCRATCH_BYTES, otherwise TTC_ERR_SCRATCH_LIMIT and nothing is touched.  Other errors as
 * ttc_execute_host (TTC_ERR_INVALID_ARG, TTC_ERR_CUDA).  Empty tensors: no-op.
 * All calls on one device share the array, which keeps the last call's contents: calls from several threads
 * are serialised by a process-wide lock (each waits for its own stream before it returns), since two of them
 * overlapping on the GPU would race on the array.  The plan must have been built beforehand (ttc_plan
 * allocates while it tunes); the first call on a device also loads the module that holds the array.
 */
#define TTC_STATIC_SCRATCH_BYTES (8u << 20)
ttc_status ttc_execute_host_static(ttc_plan_t plan, const void* alpha, const void* A_host, const void* beta,
                                   void* B_host, void* cuda_stream);

/* Frees the process-wide device staging buffers of ttc_execute_host (they are re-allocated on
 * the next call that needs them).  Must not run concurrently with ttc_execute_host. */
ttc_status ttc_release_host_staging(void);

/* Thread-local status of the last ttc_plan / ttc_canonicalize call on this thread. */
ttc_status ttc_last_error(void);
const char* ttc_status_string(ttc_status status);

/* ttc_plan_info -- fills *out.  TTC_ERR_INVALID_ARG on NULL. */
ttc_status ttc_plan_info(ttc_plan_t plan, ttc_info* out);

/* Candidate lists of a plan: which = 0 for the beta == 0 list, 1 for beta != 0. */
int        ttc_plan_num_candidates(ttc_plan_t plan, int which);
ttc_status ttc_plan_candidate(ttc_plan_t plan, int which, int index, ttc_candidate_info* out);
/* The 16 raw inputs of the ranking heuristic for one candidate (contiguous bytes per tile in A and in B,
 * remainder waste, bank-conflict factor, tile bytes, number of tiles, ring depth, row mode, peel, staggered,
 * vector bytes on each side, beta != 0, kernel class, row bytes, store items): what
 * `python -m paper_1607_01249_b200.fit_cost` regresses measured times on when the heuristic is re-fitted
 * for another device (PAPER.md:141-143 leaves the cost function to the implementation). */
ttc_status ttc_plan_candidate_features(ttc_plan_t plan, int which, int index, float* out16);
/*
 * ttc_plan_specialize -- re-compile the plan's two winners FOR THIS TRANSPOSITION (TTC generates
 * and compiles code "for a specific size", the sizes being template parameters): NVRTC compiles the library's
 * own kernel source with the winner's whole parameter block -- extents, strides, division constants, tile
 * shape, table shapes -- as a compile-time constant, so that they become immediates and the loops over them
 * unroll.  The twin is timed against the generic instance (interleaved, median of 5 x 4 launches on scratch
 * buffers) and used by ttc_execute only if it is faster; ttc_info.specialized / spec_us / generic_us report the
 * outcome.  Warp-specialised (TTC_KERNEL_TMA) and copy-class (TTC_KERNEL_COPY) winners have a twin; a tensor-map or
 * skew-kernel winner (not issue-bound: nothing to gain) is challenged by the twin of the fastest timed ring / copy candidate,
 * which becomes the plan's winner if it is faster; ttc_execute_batched and misaligned pointers keep the generic kernels.  Costs about a second of compile time per winner (cubins are kept under
 * <TTC_CACHE_FILE>.cubins/ when that variable is set); TTC_SPECIALIZE=1 makes ttc_plan call it.
 * Returns TTC_ERR_UNSUPPORTED when libnvrtc cannot be loaded or no winner is specialisable -- the plan then
 * simply keeps its generic kernels -- and TTC_ERR_CUDA / TTC_ERR_ALLOC on device trouble.
 */
ttc_status ttc_plan_specialize(ttc_plan_t plan);
/* Force a candidate (tests, search-quality experiments).  index = -1 restores the winner. */
ttc_status ttc_plan_select(ttc_plan_t plan, int which, int index);
/*
 * ttc_plan_tune -- (re-)time the `top_k` best-ranked candidates (<= 0: all) of both lists,
 * `reps` timed launches each (minimum kept), and select the fastest.
 * Needs a CUDA device.  Uses scratch buffers, never the caller's tensors.
 */
ttc_status ttc_plan_tune(ttc_plan_t plan, int top_k, int reps);

/*
 * ttc_canonicalize -- stage 1 alone, host only, no device needed: writes the
 * canonical (extent, stride in A, stride in B) triples, ascending in A-stride, into the
 * three output arrays (room for TTC_MAX_RANK each) and returns the canonical rank
 * (0 for an empty tensor, -1 on error with ttc_last_error() set).
 */
int ttc_canonicalize(int N, const int64_t* sizes, const int* perm,
                     const int64_t* lda, const int64_t* ldb,
                     int64_t* extent_out, int64_t* stride_a_out, int64_t* stride_b_out);

/* Kernels launched by this library in this process so far (bench.py's gpu_launches). */
int64_t ttc_launch_count(void);

/* Host-only self-check hook for the fast-divmod constants the kernels use:
 * returns n / d computed with the (multiplier, shift) pair the plan generator would build
 * for divisor d.  Valid for 0 <= n < 2^31, 1 <= d < 2^31. */
uint32_t ttc_debug_fastdiv(uint32_t n, uint32_t d);

/* Host-only self-check hook of the run-time specialisation: compiles (NVRTC, for sm_100a; no device needed) the
 * specialised source of candidate `index` of list `which`; returns the cubin's size in bytes, -2 if the candidate
 * has no specialisable instance (not a ring-kernel candidate), -3 if the compilation failed (`log` then holds the
 * compiler's messages, truncated to log_len), -1 on bad arguments. */
int64_t ttc_debug_specialize_compile(ttc_plan_t plan, int which, int index, char* log, int log_len);

const char* ttc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TTC_H_ */
