/*
 * lp_collectives.h -- C ABI of liblp_b200.so: Linear Pipeline (LP) collectives of
 * arXiv 1611.04255 over P *virtual* ranks (P disjoint device buffers in one
 * B200's HBM), a fused BSP-SGD step, and same-GPU MST / BE baselines.
 *
 * Citations are PAPER.md:<line> + section; "U<k>" are
 * the readings of the paper listed in DESIGN.md.
 *
 * Conventions for every entry point
 *   - `bufs` (`grads`, `weights`) is a HOST array of P DEVICE pointers (entry
 *     points ending in `_host` take a HOST array of P HOST pointers).  The array
 *     is read during the call and not retained.  The caller owns every buffer.
 *   - `n` and `block` are counted in fp32 ELEMENTS (U1; the paper counts bytes,
 *     PAPER.md:85).  Every buffer holds n contiguous floats, is 16-byte aligned
 *     and does not overlap another buffer of the same call.
 *   - `block` is the LP block size b ("we dissect a long message into
 *     fine-grained blocks"): nb = ceil(n / block), last block short (U6).
 *     Results never depend on `block`; speed does only in the copy-engine variant
 *     (profiles/r2_cost_model_fit.md).  block == 0 lets the library choose: the block
 *     that minimises the fitted cost model of PAPER.md:81-89 (lp_optimal_block) for the
 *     copy-engine variant, LP_DEFAULT_BLOCK elements for the others.
 *   - `cuda_stream` is a cudaStream_t (NULL = legacy default stream).  Work is
 *     enqueued on it and the call returns without a host sync; results are valid
 *     once the stream reaches that point.  `_host` entry points are synchronous.
 *   - Arithmetic is fp32 IEEE-754 round-to-nearest-even, no FMA contraction, no
 *     flush-to-zero.  LP sums are the left fold in rank order 0 -> P-1 whatever
 *     the root (Fig. 2b; U4), so results are bit-exact to that fold.
 *   - Return value: LP_OK or an LP_ERR_* code.  Arguments are validated before
 *     anything is enqueued: on LP_ERR_INVALID_ARG / LP_ERR_UNSUPPORTED nothing
 *     ran.  n == 0 and P == 1 are valid (no-ops, except that P == 1 reduce /
 *     allreduce / broadcast leave the single buffer unchanged).  No exceptions,
 *     no abort, nothing printed.
 *   - The library owns only internal scratch (receive buffers of the
 *     copy-engine variant, MST/BE working copies, host-staging chunks),
 *     allocated lazily and freed by lp_shutdown().
 *   - There is no CPU fallback: without a CUDA device the compute entry points
 *     return LP_ERR_CUDA.
 *   - One device per process: the library binds to the CUDA device that is current at its first compute call
 *     (scratch, tile-claim counters and streams live there); a call with another device current returns
 *     LP_ERR_UNSUPPORTED; lp_shutdown() unbinds.
 *   - Threads and streams: every entry point may be called from any host thread; calls on different streams run
 *     concurrently on the device.  The library's lock covers only its own tables (defaults, scratch, tile-claim
 *     counters), never a launch or a copy.  Tile-claim counters belong to the stream a call is enqueued on (launches
 *     of one stream are ordered); launches recorded during a CUDA-graph capture share a counter pair per capture and
 *     stream, out of LP_CAPTURE_PAIRS for the life of the process, after which captured launches fall back to the
 *     static schedule (LP_TUNE_SCHED 1: same results, a few per cent slower).  MST / BE reduce scratch is per stream
 *     as well (for captured launches: per capturing stream, so two graphs that both hold an MST / BE reduce captured
 *     on the same stream must not be replayed at the same time).
 *   - Stream order: results are those of calls executed one after the other in stream order, whatever else the caller
 *     puts on the stream between them.  With LP_TUNE_CHAIN = 1 (opt-in) a call may START before the library calls ahead
 *     of it on the stream have finished when it touches none of their buffers; it never COMPLETES before them.  That
 *     mode cannot see other kernels: see LP_TUNE_CHAIN and lp_stream_fence.
 *     lp_set_variant / lp_set_tuning change process-wide DEFAULTS, read once at the start of each call; a caller that
 *     needs its own settings (a confined comm-stream collective beside unconfined ones) uses an lp_plan.
 *     The last-error text of lp_status_string is per thread.
 */
#ifndef LP_COLLECTIVES_H
#define LP_COLLECTIVES_H

#include <stddef.h>
#include <stdint.h>

/* every entry point below has default ELF visibility; the rest of the library is hidden */
#if defined(__GNUC__)
#define LP_API __attribute__((visibility("default")))
#else
#define LP_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------- */
#define LP_OK 0
#define LP_ERR_INVALID_ARG 1 /* P<1, P>LP_MAX_P, NULL pointer, root out of range,
                                misaligned or overlapping buffers, unknown enum value */
#define LP_ERR_UNSUPPORTED 2 /* BE with non-power-of-two P (U14); cluster variant: P > 16;
                                a call from a device other than the one the library is bound to */
#define LP_ERR_CUDA 3        /* launch / allocation / copy failure, or no device */

#define LP_MAX_P 32
#define LP_DEFAULT_BLOCK 65536 /* elements; what block == 0 means outside the copy-engine variant (BASELINE.json configs) */
#define LP_CAPTURE_PAIRS 8192  /* tile-claim counter pairs for CUDA-graph captures: one per (capture, stream) */

/* ---- enums ---------------------------------------------------------------- */
/* collective, PAPER.md:57 (broadcast), :59 (reduce), :61,71 (allreduce), :144-180 (BSP-SGD Alg. 3) */
#define LP_OP_BROADCAST 0
#define LP_OP_REDUCE 1
#define LP_OP_ALLREDUCE 2
#define LP_OP_BSP_SGD 3
#define LP_OP_BSP_SGD_MOM 4  /* Alg. 3 step with momentum; for lp_plan_query / lp_min_bytes */

/* reduce operator of reduce / allreduce, PAPER.md:59 (Sec. 3, Reduce): "It supports basic arithmetic operations
 * such as summations and multiplications."  One fp32 RN operation per combine, in chain order. */
#define LP_REDUCE_SUM 0
#define LP_REDUCE_PROD 1

/* element type of the lp_*_dt calls (SURVEY 8(f)-4 "other ... dtypes"; reading U21 in DESIGN.md).  The paper's messages
 * are fp32; a chain forwards the running partial as a block of the message, so the partial has the
 * message's element type: every combine is ONE round-to-nearest-even operation in that type, no wider accumulator,
 * no flush-to-zero.  bf16 = 1 sign, 8 exponent, 7 fraction bits. */
#define LP_DT_F32 0
#define LP_DT_F16 1
#define LP_DT_BF16 2
#define LP_DT_F64 3

/* realisation of the LP pipeline used by lp_broadcast/lp_reduce/lp_allreduce/lp_bsp_sgd_step */
#define LP_VARIANT_PIPELINE 0    /* one persistent kernel; per CTA a TMA-bulk shared-memory ring
                                    with mbarrier full/empty flags handed producer warp -> add warps -> store warp */
#define LP_VARIANT_DIRECT 1      /* one kernel, one CTA per tile, 128-bit register loads/stores, chain fold in registers */
#define LP_VARIANT_CLUSTER 2     /* stage-per-rank: a thread-block cluster of P CTAs, CTA r owns rank r and hands
                                    the running partial to CTA r+1 through distributed shared memory (P <= 16) */
#define LP_VARIANT_COPY_ENGINE 3 /* the paper's own design: one cudaMemcpyAsync + one add kernel per (hop, block)
                                    on two streams */

#define LP_VARIANT_AUTO 4        /* default: DIRECT below ~2 GB of HBM traffic per call (~650 MB for a reduce over 4 or more
                                    ranks), PIPELINE above and whenever LP_TUNE_GRID_LIMIT confines the grid;
                                    lp_plan_query reports the variant that will run */

/* schedule models of lp_schedule_steps (U2, U3) */
#define LP_MODEL_STAGE 0        /* stages = the P ranks; pipeline length P - 1 + nb */
#define LP_MODEL_LINK 1         /* stages = the P-1 links, Fig. 2; allreduce redistributes by reverse flow (U3-A) */
#define LP_MODEL_LINK_RING 2    /* as LINK, allreduce redistributes by ring closure P-1 -> 0 -> ... (U3-B) */

/* tuning keys of lp_set_tuning (0 = library default) */
#define LP_TUNE_TILE_ELEMS 0    /* tile (sub-block) size in elements: 1024, 2048, 4096 or 8192 */
#define LP_TUNE_STAGES 1        /* depth of the load ring (2..32) */
#define LP_TUNE_OUT_STAGES 2    /* depth of the store ring (1..8) */
#define LP_TUNE_CTAS_PER_SM 3   /* persistent CTAs per SM (1..8); the direct variant launches one CTA per tile
                                   unless this (or LP_TUNE_GRID_LIMIT) is set */
#define LP_TUNE_CE_STREAMS 4    /* copy-engine variant: number of streams / receive slots (paper: 2) */
#define LP_TUNE_L2_HINT 5       /* 0 none, 1 evict_first on loads, 2 evict_first on loads and stores */
#define LP_TUNE_STORE_WAIT 6    /* 0: a store-ring slot is reused once its bulk stores have READ it (default);
                                   1: only once they have COMPLETED (bounds the store bytes in flight) */
#define LP_TUNE_SCHED 7         /* pipeline variant: how persistent CTAs pick tiles: 0 (default) dynamic -- each CTA claims its next tile
                                   from a device-side counter, so SMs that get more HBM bandwidth take more tiles
                                   and all finish together; 1 static round robin (tile t -> CTA t mod grid) */
#define LP_TUNE_GRID_LIMIT 8    /* at most this many persistent CTAs per launch (0 = one grid-full: SMs x CTAs per SM).
                                   A collective that runs beside compute kernels (lp_comm_*) can be confined to a
                                   few SMs' worth of CTAs, the way NCCL confines itself to a few channels */
#define LP_TUNE_NO_PDL 9        /* 1: launch kernels without programmatic dependent launch (default 0: back-to-back
                                   collectives overlap launch latency and prologue with their predecessor's tail) */
#define LP_TUNE_GRANULE_DIV 10  /* pipeline variant: a claim counts GRANULES of tile / div elements (1 (default), 2, 4, 8);
                                   a ring slot holds a run of up to div granules.  Claims shrink from LP_TUNE_CLAIM_SLOTS
                                   slots to one granule as the tile list runs out ("guided self-scheduling") */
#define LP_TUNE_CLAIM_SLOTS 11  /* pipeline variant: ring slots' worth of granules per claim while the list is long (1..16, default 1) */
#define LP_TUNE_PREFETCH 12     /* pipeline and direct variants: 0/1 a CTA prefetches its first loads into L2 before it waits for
                                   the predecessor kernel (programmatic dependent launch): the start of a call overlaps the
                                   drain of the call before it even when the two touch the same buffers; 2 = off */
#define LP_TUNE_CLUSTER_TILE 13 /* cluster variant: tile elements, 1024 / 2048 (default) / 4096 */
#define LP_TUNE_CHAIN 14        /* stream chaining: a launch whose buffers overlap none of the launches still in flight ahead
                                   of it on its stream does not wait for them before it starts (it waits before it ENDS,
                                   so completion order on the stream is kept).
                                   0 (default): only between the launches of ONE API call (MST / BE tree levels, the three
                                     launches of an Alg. 2 step) -- the library knows nothing else went into the stream
                                     between them.  Every API call's first launch waits for whatever precedes it.
                                   1: across API calls too (back-to-back collectives on different buffers -- the layers of
                                     Alg. 1, rotating buffer sets -- run into each other without a bubble, 0.5-1 us per
                                     call).  CONTRACT: the library tracks only its own launches.  If the caller enqueues
                                     other work on the stream that writes a later call's buffers (a backward GEMM producing
                                     the gradient), it must call lp_stream_fence(stream) after that work and before the
                                     library call, or the call may start reading while that work is still running
                                     (kernels that trigger programmatic completion early, as cuBLAS / CUTLASS ones do).
                                   2: off, every launch waits first.
                                   3: as 1, and long direct-variant reduces over >= 3 ranks chain as well (by default they
                                     wait first and prefetch, 1-2 % faster). */
#define LP_TUNE_DIRECT_OCC 15   /* direct variant: at most this many CTAs resident per SM (1..8; 0 = the library's choice by
                                   collective: write-heavy launches run best with few stores in flight) */
#define LP_TUNE_COUNT 16

/* ---- LP collectives (the hot path) ----------------------------------------- */

/* Broadcast, PAPER.md:57 (Sec. 3, Fig. 2a): "copies the source vector to every GPUs".
 * bufs[r][i] <- bufs[root][i] for every r != root, i in [0, n).  bufs[root] is only read. */
LP_API int lp_broadcast(float *const *bufs, int P, size_t n, size_t block, int root, void *cuda_stream);

/* Reduce, PAPER.md:59 (Sec. 3, Fig. 2b): "combines the elements provided in the vector of each GPU, and
 * returns the combined value ... to a specific GPU".  bufs[root][i] <- S[i] with
 * S[i] = ((bufs[0][i] + bufs[1][i]) + ...) + bufs[P-1][i]; buffers of the other ranks are unchanged (U5). */
LP_API int lp_reduce(float *const *bufs, int P, size_t n, size_t block, int root, void *cuda_stream);

/* Allreduce, PAPER.md:61,71 (Fig. 2c): "equivalent to a reduce followed by a broadcast", pipeline filled
 * once.  bufs[r][i] <- S[i] for every r; the same bits on every rank. */
LP_API int lp_allreduce(float *const *bufs, int P, size_t n, size_t block, void *cuda_stream);

/* Reduce / allreduce with an operator: "It supports basic arithmetic operations such as summations and
 * multiplications."  As lp_reduce / lp_allreduce with F[i] = ((bufs[0][i] op bufs[1][i]) op ...) op bufs[P-1][i],
 * op = + (LP_REDUCE_SUM, identical to the calls above) or * (LP_REDUCE_PROD); one RN operation per combine, chain
 * order whatever the root (U4).  Unknown reduce_op: LP_ERR_INVALID_ARG. */
LP_API int lp_reduce_op(float *const *bufs, int P, size_t n, size_t block, int root, int reduce_op, void *cuda_stream);
LP_API int lp_allreduce_op(float *const *bufs, int P, size_t n, size_t block, int reduce_op, void *cuda_stream);

/* Broadcast / reduce / allreduce of vectors of element type `dtype` (LP_DT_*).  As lp_broadcast / lp_reduce_op /
 * lp_allreduce_op with bufs[r] pointing at n elements of that type; n and block count ELEMENTS of that type; buffers
 * are 16-byte aligned and disjoint.  F[i] = ((bufs[0][i] op bufs[1][i]) op ...) op bufs[P-1][i] with every op one RN
 * operation IN THE ELEMENT TYPE (U21), chain order whatever the root (U4): bit-exact to that definition (NaN results are
 * NaNs; their payload bits are the hardware's).  Every LP variant takes every type.  16-bit blocks are rounded up to an
 * even number of elements (results never depend on the block).  LP_DT_F32 is the plain call.  Unknown dtype or
 * reduce_op: LP_ERR_INVALID_ARG.  Slice lists: lp_*_segments_dt; plans: lp_plan_desc.dtype.  The SGD steps and the
 * MST / BE baselines stay fp32 (the paper's). */
LP_API int lp_broadcast_dt(void *const *bufs, int P, size_t n, size_t block, int root, int dtype, void *cuda_stream);
LP_API int lp_reduce_dt(void *const *bufs, int P, size_t n, size_t block, int root, int dtype, int reduce_op,
                        void *cuda_stream);
LP_API int lp_allreduce_dt(void *const *bufs, int P, size_t n, size_t block, int dtype, int reduce_op, void *cuda_stream);
/* The layer-wise calls (Alg. 1, below) on vectors of element type `dtype`: seg_off / seg_len count elements of that type.
 * A slice of 16-bit elements must start at an even element offset (on a 4-byte word; else LP_ERR_INVALID_ARG); any
 * length is fine. */
LP_API int lp_broadcast_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len,
                                    int n_seg, size_t block, int root, int dtype, void *cuda_stream);
LP_API int lp_reduce_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                                 size_t block, int root, int dtype, int reduce_op, void *cuda_stream);
LP_API int lp_allreduce_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len,
                                    int n_seg, size_t block, int dtype, int reduce_op, void *cuda_stream);
/* bytes per element of LP_DT_*; 0 for an unknown type */
LP_API size_t lp_dtype_size(int dtype);

/* Fused BSP-SGD step = Alg. 3's communication + update (Eq. 5, 174, 180):
 *   S = chain sum of grads;  g = S * invP, invP = fl(1.0f / P) (U7);  t = lr * g;  w' = weights[root][i] - t;
 *   weights[r][i] <- w' for every r (U8).  Three separately rounded fp32 ops, no FMA.  grads are only read.
 * grads[] and weights[] are 2P distinct buffers. */
LP_API int lp_bsp_sgd_step(float *const *grads, float *const *weights, int P, size_t n, size_t block, int root,
                    float lr, void *cuda_stream);

/* Fused BSP-SGD step with momentum.  PAPER.md:216: "The solver is SGD + momentum" (no formula printed; reading
 * U18 = the solver of the system the paper modifies, Caffe): per element, five separately rounded fp32 ops,
 *   g = S * invP;  t = lr * g;  m = mu * velocity[i];  v' = m + t;  w' = weights[root][i] - v';
 *   velocity[i] <- v';  weights[r][i] <- w' for every r.
 * velocity is ONE device vector of n floats (16-byte aligned, distinct from the 2P others): it lives where the
 * update is computed.  grads are only read.  mu = 0 with a zero velocity is lp_bsp_sgd_step. */
LP_API int lp_bsp_sgd_momentum_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                    size_t block, int root, float lr, float mu, void *cuda_stream);

/* BSP-SGD step the Alg. 2 way (reading U9; prose PAPER.md:178): lp_reduce of the sub-gradients to
 * the root (grads[root] <- S, as lp_reduce does), GradientUpdate on weights[root] (the same rounded operations as
 * the fused steps; with velocity != NULL the momentum form, else mu is ignored), lp_broadcast of weights from the
 * root.  Three launches on the stream -- two synchronisation points where Alg. 3 has one.  The weights (and
 * velocity) it leaves are bit-identical to lp_bsp_sgd_step / lp_bsp_sgd_momentum_step. */
LP_API int lp_bsp_sgd_alg2_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                size_t block, int root, float lr, float mu, void *cuda_stream);

/* ---- layer-wise collectives (Alg. 1) ------------------------------------------ */
/* Alg. 1 (prose PAPER.md:182) issues one collective PER LAYER: "GPUs broadcast network parameters
 * of layer t+1 amid forward computations at layer t ... all-reduce or reduce sub-gradients of layer t+1 amidst
 * backward computations at layer t".  These calls run the collective on a LIST of slices of the rank vectors in
 * one launch: slice s is elements [seg_off[s], seg_off[s] + seg_len[s]) of every bufs[r] (r's copy of layer s).
 * Every slice is its own LP message (cut into its own blocks of `block` elements, a1), the slices are worked on in
 * list order (earlier slices finish first), elements outside every slice are not touched.  Results per slice are
 * those of lp_broadcast / lp_reduce / lp_allreduce on that slice (bit-exact, chain order).
 * seg_off / seg_len are HOST arrays of n_seg entries, read during the call; slices may start at any element
 * (no alignment rule), may be empty, must lie inside [0, n) and must not overlap (else LP_ERR_INVALID_ARG);
 * 0 <= n_seg <= LP_MAX_SEGMENTS; lists longer than 96 slices take one launch per 96 (the cluster variant: one launch
 * per slice). */
#define LP_MAX_SEGMENTS 65536
LP_API int lp_broadcast_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len,
                                 int n_seg, size_t block, int root, void *cuda_stream);
LP_API int lp_reduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len,
                              int n_seg, size_t block, int root, void *cuda_stream);
LP_API int lp_allreduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len,
                                 int n_seg, size_t block, void *cuda_stream);
/* The fused BSP-SGD step of lp_bsp_sgd_step on every slice (a layer's weights are updated as soon as its gradient
 * has been allreduced: Alg. 1's per-layer communication with Alg. 3's update); weights outside every slice keep
 * their values, grads are only read. */
LP_API int lp_bsp_sgd_step_segments(float *const *grads, float *const *weights, int P, size_t n, const size_t *seg_off,
                                    const size_t *seg_len, int n_seg, size_t block, int root, float lr,
                                    void *cuda_stream);

/* ---- non-blocking use (Alg. 1's nonblocking_* / sync_*) ------------------------- */
/* Every lp_* call above is already asynchronous to the host; "non-blocking" in the sense of Alg. 1 (PAPER.md:117-138:
 * nonblocking_broadcast / nonblocking_reduce ... sync_broadcast() / sync_reduce(), "We use the nonblocking
 * collective to achieve the overlapping") means asynchronous to the COMPUTE stream.  An lp_comm is a
 * high-priority CUDA stream owned by the library plus the two events that tie it to the caller's streams:
 *   lp_comm_after(c, s)   collectives enqueued on c from now on start after everything s holds now (the layer's
 *                         gradient is ready), without blocking s;
 *   lp_xxx(..., lp_comm_stream(c))   any collective of this library, enqueued on the comm stream;
 *   lp_comm_wait(c, s)    s waits (on the device, no host sync) for everything enqueued on c so far: sync_reduce();
 *   lp_comm_test(c, &done) host-side poll, done = 1 when the comm stream is idle.
 * lp_comm_create fails with LP_ERR_CUDA without a device.  A comm may be used from one host thread at a time. */
typedef struct lp_comm lp_comm;
LP_API int lp_comm_create(lp_comm **comm);
LP_API int lp_comm_destroy(lp_comm *comm);              /* synchronises the comm stream first */
LP_API void *lp_comm_stream(lp_comm *comm);             /* the cudaStream_t, as void* */
LP_API int lp_comm_after(lp_comm *comm, void *cuda_stream);
LP_API int lp_comm_wait(lp_comm *comm, void *cuda_stream);
LP_API int lp_comm_test(lp_comm *comm, int *done);

/* ---- MST (binomial tree) and BE (recursive halving / doubling) baselines ------ */
/* PAPER.md:93 (MST: "balanced tree of height ceil(log p)", whole-message steps) and
 * PAPER.md:95 (BE: broadcast = MST scatter + BE allgather, reduce = reduce-scatter + gather, allreduce =
 * reduce-scatter + allgather).  Same in-place semantics as the LP calls; the summation TREE differs
 * (MST on virtual ranks v = (r - root) mod P; BE butterfly), so results agree with LP to
 * |diff| <= 1e-6 * sum_r |x_r[i]| (U15), not bit for bit.  BE needs P a power of two (U14). */
LP_API int lp_mst_broadcast(float *const *bufs, int P, size_t n, int root, void *cuda_stream);
LP_API int lp_mst_reduce(float *const *bufs, int P, size_t n, int root, void *cuda_stream);
LP_API int lp_mst_allreduce(float *const *bufs, int P, size_t n, void *cuda_stream);
LP_API int lp_be_broadcast(float *const *bufs, int P, size_t n, int root, void *cuda_stream);
LP_API int lp_be_reduce(float *const *bufs, int P, size_t n, int root, void *cuda_stream);
LP_API int lp_be_allreduce(float *const *bufs, int P, size_t n, void *cuda_stream);
/* The same trees with the operator of lp_reduce_op. */
LP_API int lp_mst_reduce_op(float *const *bufs, int P, size_t n, int root, int reduce_op, void *cuda_stream);
LP_API int lp_mst_allreduce_op(float *const *bufs, int P, size_t n, int reduce_op, void *cuda_stream);
LP_API int lp_be_reduce_op(float *const *bufs, int P, size_t n, int root, int reduce_op, void *cuda_stream);
LP_API int lp_be_allreduce_op(float *const *bufs, int P, size_t n, int reduce_op, void *cuda_stream);

/* ---- the chain over real GPUs: one rank per GPU, peer memory over NVLink / NVSwitch ------ */
/* PAPER.md:55-59,71,77 (Sec. 3, Fig. 2): rank r receives a block from rank r-1 while it sends one to rank r+1; reduce
 * adds the local block to the partial on its way up the chain 0 -> 1 -> ... -> P-1 (U4: that order whatever the root),
 * allreduce sends the finished block back down (U3-A), broadcast runs root -> root+1 -> ... around the ring.  An
 * lp_chain is ONE rank's endpoint: receive rings and counters in its own device memory that its two neighbours write
 * through peer mappings (data pushed with plain stores, published with fence.acq_rel.sys + a counter in the
 * receiver's memory; slots returned by a credit counter in the sender's memory; csrc/lp_chain.cu, lp_chain_api.cu).
 *   lp_chain_create(rank, P, channels, slots, tile, &ch)   on the rank's device (current device); 0 = defaults.  Every
 *       rank must pass the same (P, channels, slots, tile).  channels: 1..LP_CHAIN_MAX_CHANNELS concurrent rings, 2 CTAs
 *       (one SM) each.  A CTA of the default kernel moves ~75 GB/s and a block costs three memory accesses on its way
 *       through a middle rank's forward CTA (and three through its return CTA), i.e. ~25 GB/s of link payload per CTA:
 *       a 900 GB/s NVLink direction takes ~36 forward + ~36 return CTAs -- hence 40, about half the SMs; slots: ring depth
 *       1..64; tile: elements per slot = the largest unit of a flag exchange, a power of two from 4096 to 262144 (default
 *       131072 floats = 512 KB; 65536 = the LP block of BASELINE.json's configs; 16384 = the paper's 64 KB).
 *   lp_chain_get_handle(ch, h)     LP_CHAIN_HANDLE_BYTES opaque bytes (a CUDA IPC handle) to all-gather over any
 *       transport (paper_1611_04255_b200/chain.py uses torch.distributed);
 *   lp_chain_connect(ch, handles)  handles = P x LP_CHAIN_HANDLE_BYTES in rank order; maps ranks (rank +- 1) mod P.
 *   lp_chain_connect_ptrs(ch, up, down)  the same for endpoints of this process (lp_chain_endpoint of the neighbours'
 *       chains; the caller enables peer access between the devices).
 *   lp_chain_run(ch, op, buf, n, block, root, reduce_op, stream)   this rank's share of LP_OP_BROADCAST / REDUCE /
 *       ALLREDUCE on its vector buf (n floats, 16-byte aligned, in place; same semantics and the same bits as
 *       lp_broadcast / lp_reduce_op / lp_allreduce_op over P virtual ranks).  Every rank calls it with the same
 *       arguments, in the same order as its other chain collectives, on one stream per endpoint.  `block` is rounded
 *       up to a multiple of 4 elements and moved in pieces of at most one tile; 0 = the library chooses: the power of two
 *       (4096 elements .. one tile) nearest to the block that minimises the paper's cost model for one channel's share
 *       of the message (Table 1: (p - 1 + n_c / b)(2 alpha + b (2 beta + gamma)); lp_optimal_block with
 *       the constants fitted to this kernel, lp_chain_fitted_constants) -- small blocks fill the chain sooner, large
 *       ones pay fewer flag exchanges.
 *   lp_chain_error(ch, &e)   synchronises; e != 0: a wait gave up (a neighbour never arrived) and the result is void.
 *       The error is sticky and the endpoint is dead: its ring counters no longer match the sequence numbers the ranks
 *       keep, so every later collective on it returns at once without touching a buffer (the kernels check the word on
 *       entry).  Destroy and re-create the endpoint on ALL ranks.
 * lp_chain_plan is the host-only part: what `rank` does in (op, P, root) -- its ring neighbours and which of the steps
 * load / receive / store / send up / send down its forward and return CTAs take.  No device needed.
 * This build's box has ONE GPU: kernels that wait for each other cannot be run there as separate launches, so what
 * the GPU tests execute is lp_chain_emulate -- the same per-rank device code for all P ranks in ONE cooperative launch
 * of P x 2 x channels co-resident CTAs over P endpoints in this device's memory, bufs = the P virtual ranks as
 * everywhere else in this header (LP_ERR_UNSUPPORTED when that many CTAs do not fit the device).  The emulated endpoints
 * belong to (P, geometry, stream) and are allocated on first use -- a call that would have to allocate while its stream is
 * being captured into a CUDA graph returns LP_ERR_UNSUPPORTED (call once outside the capture first). */
#define LP_CHAIN_HANDLE_BYTES 64
#define LP_CHAIN_MAX_CHANNELS 64
#define LP_CHAIN_DEFAULT_CHANNELS 40
#define LP_CHAIN_EMULATE_CHANNELS 16
#define LP_CHAIN_DEFAULT_SLOTS 4
#define LP_CHAIN_DEFAULT_TILE 131072
typedef struct lp_chain lp_chain;
typedef struct lp_chain_role {
    int position;     /* place in the chain of this collective: rank for reduce / allreduce, (rank - root) mod P for broadcast */
    int up, down;     /* ring neighbours: (rank + 1) mod P, (rank - 1) mod P */
    int f_active;     /* forward CTAs run */
    int f_load;       /* ... load the local block */
    int f_recv;       /* ... receive a block from `down` (and combine it with the local one when both) */
    int f_send_up;    /* ... push the result to `up` */
    int f_store;      /* ... store it to the local vector */
    int f_send_down;  /* ... chain end of allreduce / reduce to another root: push the finished block to `down` */
    int f_update;     /* ... chain end of the SGD step: apply w' = w - lr * (S * invP) before the block turns around */
    int r_active;     /* return CTAs run: receive finished blocks from `up` */
    int r_store;      /* ... store them to the local vector */
    int r_send_down;  /* ... pass them on to `down` */
} lp_chain_role;
/* Which kernel the chain launches (process-wide; the protocol between ranks is the same, so ranks may even differ):
 * TMA (default) = a producer thread streams everything a rank reads -- its vector, its receive rings -- through a deep
 * shared-memory ring with cp.async.bulk + mbarriers, 8 consumer warps fold and push with plain 128-bit stores;
 * REGISTER = 1024 threads load, fold and store from registers in 64 KB steps. */
#define LP_CHAIN_KERNEL_DEFAULT 0
#define LP_CHAIN_KERNEL_REGISTER 1
#define LP_CHAIN_KERNEL_TMA 2
LP_API int lp_chain_set_kernel(int kernel);
/* What block == 0 resolves to for a message of n elements over P ranks (elements; 0 on bad arguments), and the constants
 * behind it: alpha s per block exchange and direction, beta s per byte and channel (gamma folded in), fitted to the
 * chain kernel in its one-GPU emulation at p = 2, 4, 8 (profiles/r2_chain_cost_model.md): 2 alpha = 5.9 us whatever p --
 * what Eq. 1 assumes and the copy-engine variant on one GPU does not deliver. */
LP_API size_t lp_chain_auto_block(size_t n, int P, int channels, int tile);
LP_API void lp_chain_fitted_constants(double *alpha, double *beta);
LP_API int lp_chain_plan(int op, int P, int root, int rank, lp_chain_role *out);
/* device bytes one endpoint takes for (channels, slots, tile): 2 x channels x slots x tile x 4 for the two rings, plus
 * counters; 0 for an invalid geometry.  Host only. */
LP_API size_t lp_chain_endpoint_bytes(int channels, int slots, int tile);
LP_API int lp_chain_create(int rank, int P, int channels, int slots, int tile, lp_chain **out);
LP_API int lp_chain_get_handle(lp_chain *ch, void *handle_out);
LP_API int lp_chain_connect(lp_chain *ch, const void *handles);
LP_API int lp_chain_connect_ptrs(lp_chain *ch, void *up_endpoint, void *down_endpoint);
LP_API void *lp_chain_endpoint(lp_chain *ch);
/* How long a kernel of this endpoint polls a counter before it gives up and sets the endpoint's error word, in polls
 * (~0.3-1 us each; default 2^28, about a minute: the ranks of a job start at different times). */
LP_API int lp_chain_set_timeout(lp_chain *ch, unsigned long long polls);
LP_API int lp_chain_run(lp_chain *ch, int op, float *buf, size_t n, size_t block, int root, int reduce_op, void *cuda_stream);
/* The same on vectors of element type `dtype` (LP_DT_*, U21; n, block in elements; an f16 / bf16 vector must hold an even
 * number of elements here: a push moves whole 4-byte words). */
LP_API int lp_chain_run_dt(lp_chain *ch, int op, void *buf, size_t n, size_t block, int root, int dtype, int reduce_op,
                           void *cuda_stream);
/* Alg. 3's communication + update over the chain: the sub-gradients `grad` are folded up the chain,
 * the last rank forms w' = w - lr * (S * fl(1/P)) (three RN operations, U7) from ITS replica `weight` (all replicas hold
 * the same bits, U8) and w' travels back down; every rank stores it into its `weight`.  grad is only read; fp32. */
LP_API int lp_chain_bsp_sgd_step(lp_chain *ch, float *grad, float *weight, size_t n, size_t block, float lr,
                                 void *cuda_stream);
/* The same with momentum ("The solver is SGD + momentum"; U18): v' = mu * v + lr * (S * fl(1/P)), w' = w - v',
 * five RN operations.  The velocity is ONE vector and lives where the update is computed: the LAST rank passes it (n
 * floats, 16-byte aligned, rewritten in place), every other rank passes NULL. */
LP_API int lp_chain_bsp_sgd_momentum_step(lp_chain *ch, float *grad, float *weight, float *velocity, size_t n, size_t block,
                                          float lr, float mu, void *cuda_stream);
/* Alg. 2 over the chain (U9; prose PAPER.md:178): lp_chain reduce of `grad` to `root` (grad <- S there),
 * GradientUpdate on the root's `weight` (velocity: the root's vector or NULL for the plain step; other ranks pass NULL),
 * broadcast of `weight` from the root.  Weights (and velocity) come out bit-identical to the fused steps. */
LP_API int lp_chain_bsp_sgd_alg2_step(lp_chain *ch, float *grad, float *weight, float *velocity, size_t n, size_t block,
                                      int root, float lr, float mu, void *cuda_stream);
LP_API int lp_chain_error(lp_chain *ch, int *error_out);
/* Tear-down.  lp_chain_destroy synchronises only THIS rank's device before it unmaps its neighbours and frees its endpoint;
 * a host barrier alone does not wait for the neighbours' kernels, and a kernel finishes without waiting for its last
 * credits, so a neighbour's kernel may still be about to store a credit or a block into this endpoint.  Across ranks:
 *   1. every rank synchronises the streams it ran chain collectives on (cudaDeviceSynchronize), then a barrier;
 *   2. every rank calls lp_chain_disconnect (closes its mappings of the neighbours' endpoints), then a barrier;
 *   3. every rank calls lp_chain_destroy (frees its own, now unmapped, endpoint).
 * ChainGroup.destroy() (chain.py) does exactly this.  lp_chain_disconnect synchronises the device itself; a disconnected
 * chain refuses lp_chain_run (LP_ERR_INVALID_ARG) and may be connected again. */
LP_API int lp_chain_disconnect(lp_chain *ch);
LP_API int lp_chain_destroy(lp_chain *ch);
LP_API int lp_chain_emulate(int op, float *const *bufs, int P, size_t n, size_t block, int root, int reduce_op, int channels,
                            int slots, int tile, void *cuda_stream);
LP_API int lp_chain_emulate_dt(int op, void *const *bufs, int P, size_t n, size_t block, int root, int dtype, int reduce_op,
                               int channels, int slots, int tile, void *cuda_stream);
/* grads[r], weights[r]: rank r's vectors; equals lp_bsp_sgd_step with root = P - 1 (the replica the chain's end reads) */
LP_API int lp_chain_emulate_bsp_sgd_step(float *const *grads, float *const *weights, int P, size_t n, size_t block, float lr,
                                         int channels, int slots, int tile, void *cuda_stream);
/* ... and with momentum: equals lp_bsp_sgd_momentum_step with root = P - 1; `velocity` is the chain end's vector */
LP_API int lp_chain_emulate_bsp_sgd_momentum_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                                  size_t block, float lr, float mu, int channels, int slots, int tile,
                                                  void *cuda_stream);
LP_API int lp_chain_emulate_bsp_sgd_alg2_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                              size_t block, int root, float lr, float mu, int channels, int slots, int tile,
                                              void *cuda_stream);
/* channels per rank the emulation takes when asked for 0: LP_CHAIN_EMULATE_CHANNELS, fewer when P x 2 x channels CTAs
 * would not all be resident on the current device (1 without a device) */
LP_API int lp_chain_emulate_channels(int P, int tile);
/* synchronises the device; *error_out != 0: a wait of an emulated rank of this (P, geometry) gave up on some stream */
LP_API int lp_chain_emulate_error(int P, int channels, int slots, int tile, int *error_out);

/* ---- host-buffer entry points (end-to-end path) ------------------------------- */
/* Same results as lp_allreduce / lp_bsp_sgd_step, but the P (2P) buffers live in HOST memory (pinned for
 * full speed; pageable works).  The message is cut into chunks that flow host -> device -> kernel -> host
 * on three streams, so the upload of chunk c+1, the LP kernel on chunk c and the download of chunk c-1
 * overlap.  Synchronous: returns when every host buffer holds its result.  Host-buffer calls are serialised among
 * themselves (they share the staging chunks) but do not block device-buffer calls of other threads. */
LP_API int lp_allreduce_host(float *const *host_bufs, int P, size_t n, size_t block);
LP_API int lp_bsp_sgd_step_host(float *const *host_grads, float *const *host_weights, int P, size_t n, size_t block,
                         int root, float lr);

/* ---- schedule engine (host only; no device needed) ---------------------------- */
/* a1: nb = ceil(n / block) (U6); 0 when block == 0. */
LP_API uint64_t lp_num_blocks(size_t n, size_t block);
/* a2: block handled by rank r at tick t in the stage model, k = t - r if 0 <= k < nb, else -1. */
LP_API int64_t lp_stage_block(int P, uint64_t nb, uint64_t t, int r);
/* Number of steps of `op` (LP_OP_BROADCAST / REDUCE / ALLREDUCE) over P ranks and nb = ceil(n/block) blocks
 * under `model`: STAGE -> P - 1 + nb; LINK / LINK_RING -> the Fig. 2 schedule with one inbound
 * and one outbound transfer per rank per step.  0 steps when n == 0 (or P == 1 in the
 * link models). */
LP_API int lp_schedule_steps(int P, size_t n, size_t block, int op, int model, uint64_t *steps_out);
/* Number of whole-message levels of the MST baseline, ceil(log2 P). */
LP_API int lp_mst_levels(int P);

/* Cost model of Sec. 3.2 (Eq. 1: T = alpha + beta n + gamma n per exchange; Table 1), in
 * seconds: algo LP_ALGO_LP / MST / BE, op LP_OP_BROADCAST / REDUCE / ALLREDUCE, p ranks, message and block size in
 * BYTES (the paper's unit here), alpha s, beta and gamma s/byte.  log p = log2 p without ceiling.
 * b_bytes is ignored for MST / BE.  Returns -1 on bad arguments. */
#define LP_ALGO_LP 0
#define LP_ALGO_MST 1
#define LP_ALGO_BE 2
LP_API double lp_cost_model(int algo, int op, double p, double n_bytes, double b_bytes, double alpha, double beta,
                            double gamma);
/* The block size (bytes) that minimises lp_cost_model(LP_ALGO_LP, op, ...): sqrt(n a / ((p-1) w)), a and w the latency
 * and per-byte cost of one block exchange of `op`; clamped to n_bytes.  -1 on bad arguments. */
LP_API double lp_optimal_block(int op, double p, double n_bytes, double alpha, double beta, double gamma);
/* The block (ELEMENTS, a multiple of 4, in [4, n]) that block == 0 resolves to for `variant` (LP_VARIANT_AUTO: the
 * variant that would run): lp_optimal_block with the constants fitted on B200 (profiles/r2_cost_model_fit.md; Eq. 1
 * with A = 2 alpha per pipeline step and W = 2 beta + gamma per byte, both measured for the copy-engine variant) for
 * LP_VARIANT_COPY_ENGINE, LP_DEFAULT_BLOCK (clamped to n) otherwise -- the persistent kernels are flat in `block`.
 * 0 on bad arguments. */
LP_API size_t lp_auto_block(int op, int P, size_t n, int variant);
/* The fitted constants behind lp_auto_block, for tests and reports: alpha (s per block exchange) and beta (s/byte),
 * gamma = 0 (folded into beta), of the copy-engine variant's allreduce over P ranks on B200.  Eq. 1
 * takes them as independent of p -- every hop has its own link; on one GPU the p-1 hops of a block share two streams,
 * so alpha = 4.4 us x (p - 1) while beta = 0.5 ps/B stays put (profiles/r2_cost_model_fit.md: fits at p = 2, 6, 16).
 * With these the model's optimal block sqrt(n alpha / ((p-1) beta)) is ~46 MB for a 244 MB message at every p
 * (measured optimum: flat from 16 to 64 MB) and its times are within 35 % of the measured ones at the optimum. */
LP_API void lp_fitted_constants(int P, double *alpha, double *beta);

/* How the persistent kernel will cut and spread the work for (op, P, n, block) under the current variant
 * and tuning: tile size, tile count, grid, threads, dynamic shared memory, ring depths. */
typedef struct lp_plan_info {
    uint64_t nb;              /* a1: number of LP blocks */
    uint64_t n_tiles;         /* tiles (sub-blocks); a tile never straddles a block boundary */
    uint32_t tile_elems;      /* elements per full tile */
    uint32_t grid;            /* persistent CTAs (clusters * P for the cluster variant) */
    uint32_t threads;         /* threads per CTA */
    uint32_t smem_bytes;      /* dynamic shared memory per CTA */
    uint32_t stages;          /* load-ring depth */
    uint32_t out_stages;      /* store-ring depth */
    uint32_t variant;         /* variant that will run */
    uint32_t sm_count;        /* SMs assumed (device query, 148 when no device) */
    uint64_t block;           /* LP block in elements after block == 0 has been resolved */
    uint32_t granule_elems;   /* pipeline variant: elements per claim granule (tile_elems for the others) */
    uint32_t claim_granules;  /* pipeline variant: granules per claim while the list is long */
} lp_plan_info;
LP_API int lp_plan_query(int op, int P, size_t n, size_t block, lp_plan_info *out);

/* ---- plans: per-call settings instead of process-wide defaults ------------------- */
/* An lp_plan fixes WHAT is run (collective, operator, P, n, block, root) and HOW (variant, tuning) once; lp_plan_run
 * enqueues it on any stream with any buffers.  Two plans with different settings (say, a comm-stream allreduce
 * confined to 64 CTAs by LP_TUNE_GRID_LIMIT and an unconfined broadcast) run concurrently from different threads and
 * streams without touching each other or the process defaults.  A plan is immutable after creation and may be used
 * from several threads at once.  Results are those of the matching lp_* call (bit-exact, chain order). */
typedef struct lp_plan lp_plan;
typedef struct lp_plan_desc {
    int op;                     /* LP_OP_BROADCAST / REDUCE / ALLREDUCE / BSP_SGD / BSP_SGD_MOM */
    int reduce_op;              /* LP_REDUCE_*; must be LP_REDUCE_SUM for the SGD steps (the average) */
    int P;
    int root;                   /* ignored by allreduce */
    size_t n;                   /* elements per rank vector */
    size_t block;               /* LP block in elements, 0 = library chooses */
    int variant;                /* LP_VARIANT_* */
    int tuning[16];             /* indexed by LP_TUNE_*; 0 = library default */
    int dtype;                  /* LP_DT_*: element type of the vectors (n, block in elements of it); LP_DT_F32 for the SGD
                                   steps.  lp_plan_run then takes the P pointers as they are (cast to float *const *) */
} lp_plan_desc;
/* Fills *desc with defaults: allreduce, sum, variant LP_VARIANT_AUTO, block 0, tuning all 0; P, n left 0. */
LP_API int lp_plan_desc_init(lp_plan_desc *desc);
/* Validates the descriptor (LP_ERR_INVALID_ARG / LP_ERR_UNSUPPORTED as the matching call would) and creates the plan;
 * no device needed. */
LP_API int lp_plan_create(const lp_plan_desc *desc, lp_plan **plan);
LP_API int lp_plan_destroy(lp_plan *plan);
/* Enqueues the plan's collective on `cuda_stream`.  bufs: the P rank vectors (gradients for the SGD steps); weights:
 * the P replicas (SGD steps, else NULL); velocity: LP_OP_BSP_SGD_MOM only, else NULL; lr, mu: SGD steps. */
LP_API int lp_plan_run(const lp_plan *plan, float *const *bufs, float *const *weights, float *velocity, float lr,
                       float mu, void *cuda_stream);
/* The plan's collective on a list of slices (as lp_*_segments; not for LP_OP_BSP_SGD_MOM). */
LP_API int lp_plan_run_segments(const lp_plan *plan, float *const *bufs, float *const *weights, const size_t *seg_off,
                                const size_t *seg_len, int n_seg, float lr, void *cuda_stream);
/* What lp_plan_run will launch (as lp_plan_query, under the plan's own variant and tuning). */
LP_API int lp_plan_get_info(const lp_plan *plan, struct lp_plan_info *out);

/* ---- measurement aids: NOT part of the method ---------------------------------------------------------------- */
/* HBM ceiling probe (used by bench.py only; nothing of the LP path calls it): a plain streaming kernel, no schedule and no fold, that reads
 * n_read device vectors of n floats and writes n_write others (every thread: one 16-byte vector of each; values are
 * summed so no load can be dropped).  It puts the same read : write mix on HBM as a collective does and so measures
 * the ceiling that mix allows.  bufs: HOST array of n_read + n_write DEVICE pointers (reads first), 16-byte aligned;
 * outputs may alias inputs (the in-place mix of an allreduce). */
LP_API int lp_hbm_probe(float *const *bufs, int n_read, int n_write, size_t n, void *cuda_stream);

/* ---- a reduce for callers that must not allocate device memory (csrc/lp_static.cu) ------------------------------ */
/* lp_mst_reduce_static: the MST reduce of PAPER.md:93 (binomial tree on virtual ranks v = (r - root) mod P, whole-message
 * levels d = 1, 2, 4, ...; root <- tree sum, the other buffers unchanged, U5) -- same arguments, same validation and
 * bit-for-bit the same values as lp_mst_reduce -- for a caller that cannot let a library call cudaMalloc / cudaFree:
 * a process whose framework pool allocator already owns all of the GPU's memory (a library cudaMalloc then fails with
 * out-of-memory), a step loop that cannot take the device-wide synchronisation cudaFree implies when library scratch
 * has to grow, or a thread running while another thread holds a global-mode stream capture (cudaMalloc is refused
 * process-wide).  lp_mst_reduce keeps the non-root ranks' partial sums in library scratch it allocates on demand; this
 * entry point keeps them in a fixed array of LP_STATIC_SCRATCH_BYTES that is part of the library's device image and
 * calls no cudaMalloc, cudaFree or other allocating routine, ever.
 *   Limit: a P-rank tree needs (P - 2) / 2 working copies of n floats (none for P <= 3), each rounded up to 256 bytes;
 *     n above lp_mst_reduce_static_max_n(P) returns LP_ERR_UNSUPPORTED before anything is enqueued, with the numbers in
 *     lp_static_last_error() (P = 4: 4,194,304 floats; P = 8: 1,398,080; P = 16: 599,168; P = 32: 279,616).
 *   Cost: every GPU on which the library is loaded holds the array (16 MiB) until the process exits.
 *   Sharing: all calls on one GPU use the same array.  Calls that can overlap on the device (two streams, no event
 *     between them) race on it and produce wrong sums; calls on one stream are safe back to back.  The array keeps the
 *     last call's partial sums; none of it needs clearing -- the tree writes every word of a copy before reading it.
 *   Set-up: the first call made with a given device current looks the array's device address up
 *     (cudaGetSymbolAddress; the runtime loads the module on that device at that point) and caches it.  Make that first
 *     call on each device before any stream capture begins.  Independent of the library's one-device binding and of
 *     lp_set_variant / lp_set_tuning; plain stream-ordered launches (one per tree level) on `cuda_stream`.
 *   Errors: LP_ERR_INVALID_ARG as lp_mst_reduce; LP_ERR_UNSUPPORTED above the limit; LP_ERR_CUDA without a device or
 *     when the symbol lookup / a launch fails.  lp_static_last_error(): the calling thread's text for the last failure. */
#define LP_STATIC_SCRATCH_BYTES (16u << 20)
LP_API int lp_mst_reduce_static(float *const *bufs, int P, size_t n, int root, void *cuda_stream);
LP_API size_t lp_mst_reduce_static_max_n(int P);   /* largest n lp_mst_reduce_static takes at P ranks; 0 for a bad P; host only */
LP_API size_t lp_static_scratch_bytes(void);       /* LP_STATIC_SCRATCH_BYTES as built; host only */
LP_API const char *lp_static_last_error(void);     /* "" after a successful call; per thread */

/* Minimum HBM bytes of one call (each input read once, each output written once):
 * broadcast P*n*4, reduce (P+1)*n*4, allreduce 2*P*n*4, bsp_sgd (2P+1)*n*4, bsp_sgd with momentum (2P+3)*n*4. */
LP_API uint64_t lp_min_bytes(int op, int P, size_t n);

/* lp_stream_fence: tells the library that work it does not track went into `cuda_stream` (LP_TUNE_CHAIN = 1 / 3 only
 * need this): the next library launch on that stream waits for everything ahead of it before it starts.  Host-side
 * bookkeeping only, nothing is enqueued.  Always LP_OK. */
LP_API int lp_stream_fence(void *cuda_stream);

/* ---- control ------------------------------------------------------------------ */
/* SURVEY 8(b) sketched one selector, lp_set_algo(LP_PERSISTENT | LP_CLUSTER | LP_COPY_ENGINE | MST | BE).  It is realised
 * as lp_set_variant (the four realisations of the LP pipeline, which all return the same bits) plus separate entry points
 * for the comparison algorithms (lp_mst_*, lp_be_*), whose summation trees -- and therefore results -- differ from LP's:
 * a process-wide switch that silently changed the VALUES of lp_allreduce would be a trap. */
LP_API int lp_set_variant(int variant);             /* LP_VARIANT_*; process-wide default of the LP calls (not of plans) */
LP_API int lp_get_variant(void);
LP_API int lp_set_tuning(int key, int value);       /* LP_TUNE_*; process-wide default; value 0 restores the library's */
LP_API int lp_get_tuning(int key);
LP_API uint64_t lp_launch_count(void);              /* kernels + async copies enqueued by this library so far */
LP_API int lp_shutdown(void);                       /* frees library scratch; safe to call twice */
LP_API const char *lp_status_string(int status);    /* static or per-thread string; carries the calling thread's last CUDA
                                                       error for LP_ERR_CUDA */
LP_API int lp_version(void);                        /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* LP_COLLECTIVES_H */
