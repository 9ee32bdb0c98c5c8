// lp_common.cuh -- kernel argument block, PTX wrappers (mbarrier, TMA bulk copies) and the
// internal launcher interface between lp_api.cu and the kernel translation units.  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/lp_collectives.h"
#include "lp_schedule.h"

#define LP_MAX_IN (LP_MAX_P + 2)  // P gradient vectors + the root's weight vector + the velocity

// Epilogues of the chain fold.
#define LP_EPI_SUM 0   // out = ((in0 + in1) + ...) + in[n_sum-1]
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
    float lr, invP, mu;
    float *vel_out;
    int l2_hint;
    int store_wait;  // LP_TUNE_STORE_WAIT
    // Dynamic tile claims (LP_TUNE_SCHED 0): sched[0] = tiles claimed beyond the first grid-full, sched[1] = CTAs
    // that have finished claiming; the last CTA to finish zeroes both for the next launch.  NULL = static round robin.
    unsigned long long *sched;
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
cudaError_t lp_cluster_launch(const LpArgs &a, int P, int root, const LpTuning &t, int sm_count, LpLaunch *cfg,
                              bool dry_run, cudaStream_t stream);
uint32_t lp_pipeline_tile(const LpTuning &t, const LpArgs &a, uint64_t n, uint64_t block);
uint32_t lp_direct_tile(const LpTuning &t, int n_in, uint64_t n_work);
uint32_t lp_cluster_tile(const LpTuning &t);

// Segment jobs of the MST / BE baselines: dst[i] = a[i] + b[i] (b != NULL) or dst[i] = a[i], i in [0, len).
struct LpSegJob {
    float *dst;
    const float *a;
    const float *b;
    uint64_t len;
};
#define LP_MAX_JOBS 32
cudaError_t lp_seg_launch(const LpSegJob *jobs, int n_jobs, int sm_count, cudaStream_t stream);
// Alg. 2's GradientUpdate on the root: w <- w - lr * (S * invP), or with velocity != NULL the
// momentum form (U18), element-wise over n floats.
cudaError_t lp_update_launch(float *w, const float *S, float *velocity, uint64_t n, float lr, float invP, float mu,
                             cudaStream_t stream);

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

bool lp_pdl_enabled();  // LP_TUNE_NO_PDL == 0 (read by launchers that do not get the tuning block)

// Launch counter (kernels + async copies enqueued by the library).
void lp_count_launch(uint64_t k);
// A zeroed, self-resetting {claimed, finished} counter pair for one launch (see LpArgs::sched).
cudaError_t lp_sched_acquire(unsigned long long **pair);

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

// The a2 schedule of one persistent CTA (lp_schedule.h): which tile it works on next.  Its first tile is
// blockIdx.x; after that either the next unclaimed tile of the launch (dynamic: one atomicAdd per tile, issued
// one tile ahead so its latency hides behind the current tile's loads) or blockIdx.x + k * gridDim.x (static).
// SMs do not get equal shares of HBM bandwidth when the memory system is saturated; with static shares the
// slow SMs finish last and alone, with claims every SM is busy until the tile list is empty.
struct LpTileClaimer {
    unsigned long long *ctr;
    uint64_t next, n_tiles;
    __device__ __forceinline__ LpTileClaimer(unsigned long long *c, uint64_t nt) : ctr(c), next(blockIdx.x), n_tiles(nt) {}
    // tile to work on now (>= n_tiles: none left)
    __device__ __forceinline__ uint64_t claim() {
        const uint64_t t = next;
        if (t < n_tiles) next = ctr ? (uint64_t)gridDim.x + atomicAdd(ctr, 1ull) : t + gridDim.x;
        return t;
    }
    // after the last claim: count this CTA out; the last one re-arms the pair for the next launch
    __device__ __forceinline__ void finish() {
        if (!ctr) return;
        __threadfence();
        if (atomicAdd(ctr + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) {
            ctr[0] = 0ull;
            ctr[1] = 0ull;
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
    float s = a.in[0][i];
    for (int r = 1; r < a.n_sum; ++r) s = __fadd_rn(s, a.in[r][i]);
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
