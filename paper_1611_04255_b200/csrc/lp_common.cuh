// lp_common.cuh -- kernel argument block, PTX wrappers (mbarrier, TMA bulk copies) and the
// internal launcher interface between lp_api.cu and the kernel translation units.  sm_100a only.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/lp_collectives.h"
#include "lp_schedule.h"

#define LP_MAX_IN (LP_MAX_P + 2)  // P gradient vectors + the root's weight vector + the velocity

// Epilogues of the chain fold.
#define LP_EPI_SUM 0   // out = ((in0 op in1) op ...) op in[n_sum-1], op = a.red_op
#define LP_EPI_SGD 1   // out = in[n_sum] - lr * (S * invP), three RN ops      PAPER.md:172,174 (U7)
#define LP_EPI_COPY 2  // out = in0 (broadcast)
#define LP_EPI_SGD_MOM 3  // v' = mu * in[n_sum+1] + lr * (S * invP); out = in[n_sum] - v'; vel_out = v'   PAPER.md:216 (U18)

// One launch = one collective.  in[0..n_sum) are folded in that order (rank 0 -> P-1); for LP_EPI_SGD
// in[n_sum] is weights[root]; for LP_EPI_SGD_MOM in[n_sum + 1] is the velocity as well and vel_out receives
// the new velocity; out[0..n_out) all receive the finished tile.
struct LpArgs {
    const float *in[LP_MAX_IN];
    float *out[LP_MAX_P];
    int n_sum;     // number of folded inputs (1 for broadcast)
    int n_in;      // n_sum (+1 for SGD)
    int n_out;
    int epilogue;
    int red_op;    // LP_REDUCE_SUM / LP_REDUCE_PROD: the operator of the fold
    // Element type of the vectors (LP_DT_*; U21).  Kernels address every vector in 4-byte WORDS whatever the type: an
    // f32 element is one word, an f64 element two (every offset and length the planner hands out is then even), f16 /
    // bf16 elements come two to a word (the planner rounds blocks up to whole words; an odd last element is folded by
    // lp_tail16_launch).  Only the combine and the scalar head / tail path look at the type.  SGD epilogues: f32 only.
    int dtype;
    float lr, invP, mu;
    float *vel_out;
    int l2_hint;
    int store_wait;  // LP_TUNE_STORE_WAIT
    // Dynamic tile claims (LP_TUNE_SCHED 0): sched[0] = tiles claimed beyond the first grid-full, sched[1] = CTAs
    // that have finished claiming; the last CTA to finish zeroes both for the next launch.  NULL = static round robin.
    unsigned long long *sched;
    // Pipeline kernels: part.tile is the GRANULE (the unit of a claim); a ring slot holds a run of up to slot_gran
    // consecutive granules of one block; a claim takes claim_max granules, fewer towards the end of the list
    // (remaining >> claim_shift, at least one) so that all CTAs run dry together.  Other kernels: one tile per claim.
    uint32_t slot_gran;
    uint32_t claim_max;
    uint32_t claim_shift;
    int prefetch;  // LP_TUNE_PREFETCH: L2 prefetch of a CTA's first loads before it waits for the predecessor kernel
    // Stream chaining (LP_TUNE_CHAIN, lp_chain_admit): 1 = this launch touches no buffer of the launches that may still
    // be running ahead of it on its stream, so it does not wait for them before it starts; one thread per CTA waits
    // before the CTA EXITS instead, which keeps completion order on the stream.
    int late_wait;
    uint64_t span_elems;  // elements per rank vector (the whole vector, also for a layer-wise launch): chain ranges
    lp_partition part;
};

// Second kernel parameter: the segment table of a layer-wise launch, or nothing.
struct LpNoSegs {
    int unused;
};
template <bool SEG>
struct LpSegParam {
    typedef LpNoSegs type;
};
template <>
struct LpSegParam<true> {
    typedef lp_seg_table type;
};

struct LpLaunch {
    uint32_t grid, threads, smem_bytes, stages, out_stages;
    bool pdl;
    uint32_t claim;  // pipeline variant: granules per claim while the list is long
};

// Tuning state resolved by the API layer (0 = default).
struct LpTuning {
    int v[LP_TUNE_COUNT];
};

// ---- launchers implemented in the kernel translation units ----------------------------------------
// Each fills `cfg` (always) and, unless dry_run, enqueues the kernel(s) on `stream`.  Return cudaError_t.
// `segs` != NULL: a layer-wise launch; a.part then holds block, tile and the TOTAL tile count only.
cudaError_t lp_pipeline_launch(const LpArgs &a, const lp_seg_table *segs, const LpTuning &t, int sm_count, LpLaunch *cfg,
                               bool dry_run, cudaStream_t stream);
cudaError_t lp_direct_launch(const LpArgs &a, const lp_seg_table *segs, const LpTuning &t, int sm_count, LpLaunch *cfg,
                             bool dry_run, cudaStream_t stream);
// base_off: element offset of the message inside the rank vectors (a slice of a layer-wise list; 0 = whole vectors)
cudaError_t lp_cluster_launch(const LpArgs &a, int P, int root, uint64_t base_off, const LpTuning &t, int sm_count,
                              LpLaunch *cfg, bool dry_run, cudaStream_t stream);
uint32_t lp_pipeline_tile(const LpTuning &t, const LpArgs &a, uint64_t n, uint64_t block, int sm_count);
uint32_t lp_pipeline_granule(const LpTuning &t, uint32_t tile);
uint32_t lp_direct_tile(const LpTuning &t, const LpArgs &a, uint64_t n_work, int sm_count);
uint32_t lp_cluster_tile(const LpTuning &t);
// LP_TUNE_GRID_LIMIT confines the launch to fewer CTAs than the device has SMs (a collective beside compute kernels):
// the one predicate tile choice, ring choice and variant choice share.
inline bool lp_grid_confined(const LpTuning &t, int sm_count) {
    return t.v[LP_TUNE_GRID_LIMIT] > 0 && t.v[LP_TUNE_GRID_LIMIT] <= sm_count;
}
// Function attributes (dynamic shared memory limit, non-portable cluster size) are per device: the launchers cache
// "already set" against this epoch, which lp_shutdown() advances when it unbinds the library from its device.
unsigned lp_attr_epoch();

// Segment jobs of the MST / BE baselines: dst[i] = a[i] op b[i] (b != NULL; op = red_op of the launch) or
// dst[i] = a[i], i in [0, len); len counts 4-byte words of vectors of element type `dtype` (LpArgs::dtype).
struct LpSegJob {
    float *dst;
    const float *a;
    const float *b;
    uint64_t len;
};
#define LP_MAX_JOBS 32
cudaError_t lp_seg_launch(const LpSegJob *jobs, int n_jobs, int sm_count, cudaStream_t stream, bool pdl,
                          int red_op = LP_REDUCE_SUM, bool chain = false, int dtype = LP_DT_F32);
// Alg. 2's GradientUpdate on the root: w <- w - lr * (S * invP), or with velocity != NULL the
// momentum form (U18), element-wise over n floats.
cudaError_t lp_update_launch(float *w, const float *S, float *velocity, uint64_t n, float lr, float invP, float mu,
                             cudaStream_t stream, bool pdl);

// Programmatic dependent launch: every kernel of the library is launched with the "programmatic stream
// serialization" attribute, tells the runtime when its CTAs have nothing left to claim (lp_pdl_trigger) and waits
// for its predecessor in the stream before touching global memory (lp_pdl_wait).  Back-to-back collectives (layer-wise
// lists, MST / BE levels, reduce -> update -> broadcast) then overlap their launch latency and prologue with the
// predecessor's tail; a predecessor that never triggers (any other kernel) simply completes first, as always.
// `pdl` = false (LP_TUNE_NO_PDL) launches the classic way.
template <typename... KArgs, typename... Args>
cudaError_t lp_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl,
                      Args &&...args) {
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof(lc));
    lc.gridDim = grid;
    lc.blockDim = block;
    lc.dynamicSmemBytes = smem;
    lc.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = attr;
    lc.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&lc, kernel, static_cast<KArgs>(args)...);
}

// ---- stream chaining -------------------------------------------------------------------------------------------
// With programmatic dependent launch a kernel starts when its predecessor has TRIGGERED, not when it has finished; a
// kernel of this library triggers once it has nothing left to claim and normally waits (griddepcontrol.wait) before it
// touches memory.  lp_chain_admit keeps, per stream, the byte ranges of the launches that may still be running when the
// next one starts (everything since the last launch that waited FIRST: that one cannot trigger before all its
// predecessors have completed).  A launch that overlaps none of them may defer its wait to its end -- "late": its
// fill overlaps their drain, yet it cannot complete before they do, so anything later in the stream still sees stream
// order.  Returns true for late.  A launch without PDL, an overlap, an unknown predecessor (lp_chain_reset) or a
// full table make the launch wait first, and the table restarts with it.
struct LpRange {
    uintptr_t lo, hi;  // bytes [lo, hi)
};
bool lp_chain_admit(cudaStream_t stream, const LpRange *ranges, int n, bool pdl, bool allowed);
void lp_chain_reset(cudaStream_t stream);  // something the table does not track went into the stream
// The ranges a launch described by LpArgs touches (whole rank vectors); returns their number (<= 2 * LP_MAX_IN).
inline int lp_args_ranges(const LpArgs &a, LpRange *r) {
    int m = 0;
    const uintptr_t bytes = (uintptr_t)a.span_elems * 4u;
    for (int i = 0; i < a.n_in; ++i) r[m++] = LpRange{(uintptr_t)a.in[i], (uintptr_t)a.in[i] + bytes};
    for (int i = 0; i < a.n_out; ++i) r[m++] = LpRange{(uintptr_t)a.out[i], (uintptr_t)a.out[i] + bytes};
    if (a.vel_out) r[m++] = LpRange{(uintptr_t)a.vel_out, (uintptr_t)a.vel_out + bytes};
    return m;
}

// Launch counter (kernels + async copies enqueued by the library).
void lp_count_launch(uint64_t k);
// A zeroed, self-resetting {claimed, finished} counter pair for a launch on `stream` (see LpArgs::sched): the
// stream's own pair (launches of one stream are ordered), or a pair of its own when the stream is being captured
// into a CUDA graph.  *pair = NULL (static schedule) when none can be had.
cudaError_t lp_sched_acquire(cudaStream_t stream, unsigned long long **pair);
// Library scratch for (stream, slot): grows on demand; per stream so that calls on different streams never share it.
cudaError_t lp_scratch_get(cudaStream_t stream, int slot, size_t bytes, float **ptr);
// key of scratch that is not tied to a caller's stream (host-path staging sets, copy-engine receive slots: both are
// used under a lock of their own, on streams the library owns)
#define LP_SCRATCH_SHARED ((cudaStream_t)(intptr_t)-1)

#if defined(__CUDACC__)
__device__ __forceinline__ void lp_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void lp_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- PTX wrappers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lp_smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void lp_mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lp_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void lp_fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void lp_mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(lp_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void lp_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lp_smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void lp_mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LP_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LP_DONE_%=;\n"
        "bra LP_WAIT_%=;\n"
        "LP_DONE_%=:\n"
        "}\n" ::"r"(lp_smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// generic-proxy writes to shared memory -> visible to the async proxy (TMA store)
__device__ __forceinline__ void lp_fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ uint64_t lp_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void lp_bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     lp_smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(lp_smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void lp_bulk_g2s_hint(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar,
                                                 uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
            "r"(lp_smem_u32(smem_dst)),
        "l"(gsrc), "r"(bytes), "r"(lp_smem_u32(bar)), "l"(pol)
        : "memory");
}
// TMA bulk copy shared -> global, tracked by bulk async-groups
__device__ __forceinline__ void lp_bulk_s2g(void *gdst, const void *smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
                 "r"(lp_smem_u32(smem_src)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void lp_bulk_s2g_hint(void *gdst, const void *smem_src, uint32_t bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gdst),
                 "r"(lp_smem_u32(smem_src)), "r"(bytes), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void lp_bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void lp_bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void lp_bulk_wait() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}

// 128-bit streaming global accesses (no L1 allocation; every byte is touched once)
__device__ __forceinline__ float4 lp_ldg_stream(const float *p) {
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p));
    return v;
}
__device__ __forceinline__ void lp_stg_stream(float *p, const float4 &v) {
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y),
                 "f"(v.z), "f"(v.w)
                 : "memory");
}

// fp32 RN arithmetic that ptxas may not contract into FMA
__device__ __forceinline__ float4 lp_add4(const float4 &a, const float4 &b) {
    return make_float4(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y), __fadd_rn(a.z, b.z), __fadd_rn(a.w, b.w));
}
__device__ __forceinline__ float4 lp_mul4(const float4 &a, const float4 &b) {
    return make_float4(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y), __fmul_rn(a.z, b.z), __fmul_rn(a.w, b.w));
}
// ---- partial op local block ("summations and multiplications") in the element type (U21) -----------
// `code` = (dtype << 1) | red_op, uniform over the launch: 0 / 1 = f32 sum / product (the paper's case), then f16, bf16,
// f64.  Every combine is ONE round-to-nearest-even operation in the element type: the partial travels as a block of the
// message, so it has the message's type; no wider accumulator, no flush-to-zero, no contraction (__h*2_rn, __d*_rn).
__device__ __forceinline__ int lp_fold_code(int dtype, int red_op) { return (dtype << 1) | red_op; }
__device__ __forceinline__ __half2 lp_as_h2(float w) {
    const uint32_t u = __float_as_uint(w);
    return *reinterpret_cast<const __half2 *>(&u);
}
__device__ __forceinline__ float lp_from_h2(__half2 h) { return __uint_as_float(*reinterpret_cast<const uint32_t *>(&h)); }
__device__ __forceinline__ __nv_bfloat162 lp_as_b2(float w) {
    const uint32_t u = __float_as_uint(w);
    return *reinterpret_cast<const __nv_bfloat162 *>(&u);
}
__device__ __forceinline__ float lp_from_b2(__nv_bfloat162 h) {
    return __uint_as_float(*reinterpret_cast<const uint32_t *>(&h));
}
// one 4-byte word: an f32 element, or two f16 / bf16 elements (f64 never comes here: lp_combine_f64)
template <int CODE>
__device__ __forceinline__ float lp_word_op(float a, float b) {
    if constexpr (CODE == 0) return __fadd_rn(a, b);
    if constexpr (CODE == 1) return __fmul_rn(a, b);
    if constexpr (CODE == 2) return lp_from_h2(__hadd2_rn(lp_as_h2(a), lp_as_h2(b)));
    if constexpr (CODE == 3) return lp_from_h2(__hmul2_rn(lp_as_h2(a), lp_as_h2(b)));
    if constexpr (CODE == 4) return lp_from_b2(__hadd2_rn(lp_as_b2(a), lp_as_b2(b)));
    if constexpr (CODE == 5) return lp_from_b2(__hmul2_rn(lp_as_b2(a), lp_as_b2(b)));
    return a;
}
__device__ __forceinline__ double lp_words_f64(float lo, float hi) {
    return __hiloint2double(__float_as_int(hi), __float_as_int(lo));
}
__device__ __forceinline__ double lp_combine_f64(double a, double b, bool prod) { return prod ? __dmul_rn(a, b) : __dadd_rn(a, b); }
template <int CODE>
__device__ __forceinline__ float4 lp_vec_op(const float4 &a, const float4 &b) {
    if constexpr (CODE >= 6) {  // two f64 elements
        const double r0 = lp_combine_f64(lp_words_f64(a.x, a.y), lp_words_f64(b.x, b.y), CODE == 7);
        const double r1 = lp_combine_f64(lp_words_f64(a.z, a.w), lp_words_f64(b.z, b.w), CODE == 7);
        return make_float4(__int_as_float(__double2loint(r0)), __int_as_float(__double2hiint(r0)),
                           __int_as_float(__double2loint(r1)), __int_as_float(__double2hiint(r1)));
    } else {
        return make_float4(lp_word_op<CODE>(a.x, b.x), lp_word_op<CODE>(a.y, b.y), lp_word_op<CODE>(a.z, b.z),
                           lp_word_op<CODE>(a.w, b.w));
    }
}
__device__ __forceinline__ float4 lp_combine4(const float4 &a, const float4 &b, int code) {
    if (code <= 1) return code ? lp_vec_op<1>(a, b) : lp_vec_op<0>(a, b);  // fp32, the paper's case: what it always was
    switch (code) {
        case 2: return lp_vec_op<2>(a, b);
        case 3: return lp_vec_op<3>(a, b);
        case 4: return lp_vec_op<4>(a, b);
        case 5: return lp_vec_op<5>(a, b);
        case 6: return lp_vec_op<6>(a, b);
        default: return lp_vec_op<7>(a, b);
    }
}
// acc[v] <- acc[v] op x[v] for the first nv of V vectors: the switch on the launch's code sits outside the loop
template <int V>
__device__ __forceinline__ void lp_fold_vecs(float4 (&acc)[V], const float4 (&x)[V], int nv, int code) {
#define LP_FOLD_CASE(C)                                       \
    case C:                                                   \
        _Pragma("unroll") for (int v = 0; v < V; ++v) {       \
            if (v < nv) acc[v] = lp_vec_op<C>(acc[v], x[v]);  \
        }                                                     \
        break;
    switch (code) {
        LP_FOLD_CASE(0)
        LP_FOLD_CASE(1)
        LP_FOLD_CASE(2)
        LP_FOLD_CASE(3)
        LP_FOLD_CASE(4)
        LP_FOLD_CASE(5)
        LP_FOLD_CASE(6)
        default:
            LP_FOLD_CASE(7)
    }
#undef LP_FOLD_CASE
}
// one word of an f32 / f16 / bf16 vector (codes 0..5)
__device__ __forceinline__ float lp_combine1(float a, float b, int code) {
    switch (code) {
        case 0: return lp_word_op<0>(a, b);
        case 1: return lp_word_op<1>(a, b);
        case 2: return lp_word_op<2>(a, b);
        case 3: return lp_word_op<3>(a, b);
        case 4: return lp_word_op<4>(a, b);
        default: return lp_word_op<5>(a, b);
    }
}
// dst[i] = a[i] op b[i] on WORD i of vectors of the code's element type, straight from and to global memory (the few
// words of a segment outside its 16-byte aligned body).  f64: the element that starts at an even word; odd words are
// their element's upper half and are skipped (offsets and lengths are even, so both halves lie in the same range).
__device__ __forceinline__ void lp_word_combine_store(float *dst, const float *a, const float *b, uint64_t i, int code) {
    if (code >= 6) {
        if (i & 1u) return;
        const double x = *reinterpret_cast<const double *>(a + i);
        *reinterpret_cast<double *>(dst + i) = b ? lp_combine_f64(x, *reinterpret_cast<const double *>(b + i), code == 7) : x;
        return;
    }
    dst[i] = b ? lp_combine1(a[i], b[i], code) : a[i];
}
// w' = w - lr * (s * invP): three separately rounded operations (U7)
__device__ __forceinline__ float lp_sgd1(float s, float w, float lr, float invP) {
    return __fsub_rn(w, __fmul_rn(lr, __fmul_rn(s, invP)));
}
// momentum (U18): g = s * invP; t = lr * g; m = mu * v; v' = m + t; w' = w - v' -- five separately rounded operations
__device__ __forceinline__ void lp_mom1(float s, float w, float v, float lr, float invP, float mu, float &v_new,
                                        float &w_new) {
    v_new = __fadd_rn(__fmul_rn(mu, v), __fmul_rn(lr, __fmul_rn(s, invP)));
    w_new = __fsub_rn(w, v_new);
}
__device__ __forceinline__ void lp_mom4(const float4 &s, const float4 &w, const float4 &v, float lr, float invP, float mu,
                                        float4 &v_new, float4 &w_new) {
    lp_mom1(s.x, w.x, v.x, lr, invP, mu, v_new.x, w_new.x);
    lp_mom1(s.y, w.y, v.y, lr, invP, mu, v_new.y, w_new.y);
    lp_mom1(s.z, w.z, v.z, lr, invP, mu, v_new.z, w_new.z);
    lp_mom1(s.w, w.w, v.w, lr, invP, mu, v_new.w, w_new.w);
}
__device__ __forceinline__ float4 lp_sgd4(const float4 &s, const float4 &w, float lr, float invP) {
    return make_float4(lp_sgd1(s.x, w.x, lr, invP), lp_sgd1(s.y, w.y, lr, invP), lp_sgd1(s.z, w.z, lr, invP),
                       lp_sgd1(s.w, w.w, lr, invP));
}

// The a2 schedule of one persistent CTA (lp_schedule.h): which tiles it works on next.  A claim is a range of
// consecutive tile indices.  The first claim is static (claim_max tiles from blockIdx.x * claim_max); every further
// one comes from the launch's device counter (one atomicAdd per claim, issued one claim ahead so its latency hides
// behind the current loads), or -- static schedule -- lies gridDim.x * claim_max further on.
// Why claims: SMs do not get equal shares of HBM bandwidth when the memory system is saturated; with static shares
// the slow SMs finish last and alone.  Why they shrink ("guided self-scheduling"): a CTA's ring holds work it has
// claimed but not finished, and what it claims last it finishes last; with claims of remaining / (2 * grid) tiles
// the work in hand shrinks with the list and all CTAs run dry within one small tile of each other -- on a 64 MB
// message the fixed-size tail was 2-6 us of a 20-90 us call.
struct LpClaim {
    uint64_t g0, g1;  // tiles [g0, g1); g0 >= n_tiles: none left
};
struct LpTileClaimer {
    unsigned long long *ctr;
    uint64_t n_tiles, next0, next1;
    uint32_t cmax, shift;
    __device__ __forceinline__ LpTileClaimer(unsigned long long *c, uint64_t nt, uint32_t claim_max, uint32_t claim_shift)
        : ctr(c), n_tiles(nt), cmax(claim_max ? claim_max : 1u), shift(claim_shift) {
        next0 = (uint64_t)blockIdx.x * cmax;
        next1 = next0 + cmax;
    }
    // the first claim, without consuming it (for prefetching)
    __device__ __forceinline__ LpClaim peek() const {
        LpClaim c{next0, next1 < n_tiles ? next1 : n_tiles};
        return c;
    }
    __device__ __forceinline__ LpClaim claim() {
        LpClaim c{next0, next1 < n_tiles ? next1 : n_tiles};
        if (c.g0 < n_tiles) {
            if (ctr) {
                const uint64_t rem = n_tiles > next1 ? n_tiles - next1 : 0;  // tiles nobody has claimed yet, at most
                uint64_t size = rem >> shift;
                size = size < 1 ? 1 : (size > cmax ? cmax : size);
                next0 = (uint64_t)gridDim.x * cmax + atomicAdd(ctr, (unsigned long long)size);
                next1 = next0 + size;
            } else {
                next0 += (uint64_t)gridDim.x * cmax;
                next1 = next0 + cmax;
            }
        }
        return c;
    }
    // after the last claim and BEFORE griddepcontrol.launch_dependents: count this CTA out; the last one re-arms the
    // pair for the next launch (which starts only once every CTA of this one has triggered)
    __device__ __forceinline__ void finish() {
        if (!ctr) return;
        __threadfence();
        if (atomicAdd(ctr + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) {
            atomicExch(ctr, 0ull);  // at L2, where the next launch's claims are served (it may start without waiting
            atomicExch(ctr + 1, 0ull);  // for this kernel to END, but not before every CTA has got past this point)
            __threadfence();
        }
    }
};

// a1/a2: tile index -> element range, for a single message (a.part) or a layer-wise launch (segment table).
template <bool SEG>
__device__ __forceinline__ void lp_lookup_tile(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, uint64_t t,
                                               uint64_t &off, uint32_t &len) {
    if constexpr (SEG)
        lp_seg_tile_range(segs, a.part.block, a.part.tile, t, off, len);
    else
        lp_tile_range(a.part, t, off, len);
}

// The run of tiles that starts at tile g and ends before g1, at the end of g's block or after `max_run` tiles,
// whichever comes first: one contiguous element range [off, off + len); returns the number of tiles in it.
template <bool SEG>
__device__ __forceinline__ uint64_t lp_lookup_run(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, uint64_t g,
                                                  uint64_t g1, uint32_t max_run, uint64_t &off, uint32_t &len) {
    uint64_t left, bend;
    uint32_t len1;
    if constexpr (SEG)
        lp_seg_tile_range_ex(segs, a.part.block, a.part.tile, g, off, len1, left, bend);
    else
        lp_tile_range_ex(a.part, g, off, len1, left, bend);
    uint64_t run = g1 - g;
    if (run > left) run = left;
    if (run > max_run) run = max_run;
    const uint64_t span = run * (uint64_t)a.part.tile;
    len = off + span <= bend ? (uint32_t)span : (uint32_t)(bend - off);
    return run;
}

// L2 prefetch of [p, p + bytes) (a hint: L2 is the point of coherence, so it is safe even while the predecessor
// kernel is still writing); bytes a multiple of 16.
__device__ __forceinline__ void lp_prefetch_l2(const void *p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// A tile [off, off + len) of 16-byte aligned vectors splits into a 16-byte aligned body [a0, a1) that the bulk
// copies move and at most 3 + 3 head / tail elements that take the scalar path (tiles of a slice that does not
// start on a 16-byte boundary, and the last tile of a message).
struct LpTileSpan {
    uint64_t a0;
    uint32_t body;  // elements in [a0, a1): a multiple of 4
    uint32_t head;  // elements in [off, a0)
    uint32_t tail;  // elements in [a1, off + len)
    __device__ __forceinline__ LpTileSpan(uint64_t off, uint32_t len) {
        const uint64_t end = off + len;
        uint64_t b0 = (off + 3) & ~(uint64_t)3;
        if (b0 > end) b0 = end;
        uint64_t b1 = end & ~(uint64_t)3;
        if (b1 < b0) b1 = b0;
        a0 = b0;
        body = (uint32_t)(b1 - b0);
        head = (uint32_t)(b0 - off);
        tail = (uint32_t)(end - b1);
    }
};

// Scalar path for the (at most a few) elements of a tile outside its 16-byte aligned body: the chain fold,
// epilogue and fan-out for element i, straight from and to global memory.
__device__ __forceinline__ void lp_scalar_element(const LpArgs &a, uint64_t i) {
    const int code = lp_fold_code(a.dtype, a.red_op);
    if (code >= 6) {  // f64: word i is the lower half of an element (i even) or its upper half (skipped)
        if (i & 1u) return;
        double s = *reinterpret_cast<const double *>(a.in[0] + i);
        for (int r = 1; r < a.n_sum; ++r) s = lp_combine_f64(s, *reinterpret_cast<const double *>(a.in[r] + i), code == 7);
        for (int q = 0; q < a.n_out; ++q) *reinterpret_cast<double *>(a.out[q] + i) = s;
        return;
    }
    float s = a.in[0][i];
    for (int r = 1; r < a.n_sum; ++r) s = lp_combine1(s, a.in[r][i], code);
    if (a.epilogue == LP_EPI_SGD) s = lp_sgd1(s, a.in[a.n_sum][i], a.lr, a.invP);
    if (a.epilogue == LP_EPI_SGD_MOM) {
        float v_new, w_new;
        lp_mom1(s, a.in[a.n_sum][i], a.in[a.n_sum + 1][i], a.lr, a.invP, a.mu, v_new, w_new);
        a.vel_out[i] = v_new;
        s = w_new;
    }
    for (int q = 0; q < a.n_out; ++q) a.out[q][i] = s;
}
#endif  // __CUDACC__
