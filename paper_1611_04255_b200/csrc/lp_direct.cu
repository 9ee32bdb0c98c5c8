// lp_direct.cu -- LP_VARIANT_DIRECT: the LP collective as one kernel (one CTA per tile) that keeps the running
// partial of the chain (a0 -> a' = a0 + a1 -> a'' = a' + a2) in registers.  Each thread owns V
// 16-byte vectors of a tile, issues the 128-bit streaming loads of up to 8 ranks at once (memory-level
// parallelism replaces the paper's two DMA engines), folds them in rank order 0 -> P-1 with RN adds and
// writes the finished vector to every destination rank.  It is also the path that takes any alignment:
// a tile whose start is not a multiple of 4 elements (block % 4 != 0) gets a scalar head and tail.
#include "lp_common.cuh"

namespace {

constexpr int kThreads = 256;
// ranks whose loads are in flight together: 8, or 16 for the one-vector-per-thread kernels of the latency regime (a
// 16-rank chain then costs one HBM latency, not two)
template <int V>
struct LpRankChunk {
    static constexpr int value = V == 1 ? 16 : 8;
};

// NS > 0: number of folded inputs known at compile time (loops fully unrolled); NS == 0: runtime a.n_sum.
template <int NS, int V, bool SEG>
__global__ void __launch_bounds__(kThreads)
    lp_direct_kernel(const __grid_constant__ LpArgs a, const __grid_constant__ typename LpSegParam<SEG>::type segs) {
    const int n_sum = NS > 0 ? NS : a.n_sum;
    const int tid = threadIdx.x;
    // a2: one CTA per tile by default (grid == n_tiles): the hardware block scheduler hands the next tile to
    // whichever SM frees up first -- the same balance the pipeline kernel gets from its tile claims, with no
    // per-CTA setup at all, which is what the latency regime wants.  A confined grid (LP_TUNE_GRID_LIMIT /
    // LP_TUNE_CTAS_PER_SM) walks the tile list round robin.
    // wait first, then trigger: at most ONE successor waits behind a running kernel (triggering before the wait lets
    // a whole queue of short kernels pile up on the SMs, each blocked on its predecessor: measured 2x slower at 256 KB)
    lp_pdl_wait();
    lp_pdl_trigger();  // every CTA of this grid is resident or done once the last one gets here
    for (uint64_t t = blockIdx.x; t < a.part.n_tiles; t += gridDim.x) {
        uint64_t off;
        uint32_t len;
        lp_lookup_tile<SEG>(a, segs, t, off, len);
        const uint64_t end = off + len;
        uint64_t a0 = (off + 3) & ~(uint64_t)3;  // first 16-byte aligned element (all buffers are 16-byte aligned)
        if (a0 > end) a0 = end;
        uint64_t a1 = end & ~(uint64_t)3;
        if (a1 < a0) a1 = a0;
        const uint32_t nvec = (uint32_t)((a1 - a0) >> 2);
        if ((uint64_t)tid < a0 - off) lp_scalar_element(a, off + tid);
        if ((uint64_t)tid < end - a1) lp_scalar_element(a, a1 + tid);

        float4 acc[V];
        float4 w[V];
        bool live[V];
#pragma unroll
        for (int v = 0; v < V; ++v) live[v] = (uint32_t)(tid + v * kThreads) < nvec;
        float4 vel[V];
        if (a.epilogue == LP_EPI_SGD || a.epilogue == LP_EPI_SGD_MOM) {
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (live[v]) w[v] = lp_ldg_stream(a.in[n_sum] + a0 + 4 * (uint64_t)(tid + v * kThreads));
        }
        if (a.epilogue == LP_EPI_SGD_MOM) {
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (live[v]) vel[v] = lp_ldg_stream(a.in[n_sum + 1] + a0 + 4 * (uint64_t)(tid + v * kThreads));
        }
        constexpr int kRankChunk = LpRankChunk<V>::value;
        for (int r0 = 0; r0 < n_sum; r0 += kRankChunk) {
            float4 x[V][kRankChunk];
#pragma unroll
            for (int j = 0; j < kRankChunk; ++j) {
                if (NS > 0 ? (r0 + j < NS) : (r0 + j < n_sum)) {
#pragma unroll
                    for (int v = 0; v < V; ++v)
                        if (live[v]) x[v][j] = lp_ldg_stream(a.in[r0 + j] + a0 + 4 * (uint64_t)(tid + v * kThreads));
                }
            }
#pragma unroll
            for (int j = 0; j < kRankChunk; ++j) {
                if (NS > 0 ? (r0 + j < NS) : (r0 + j < n_sum)) {
#pragma unroll
                    for (int v = 0; v < V; ++v) acc[v] = (r0 + j == 0) ? x[v][j] : lp_add4(acc[v], x[v][j]);
                }
            }
        }
        if (a.epilogue == LP_EPI_SGD) {
#pragma unroll
            for (int v = 0; v < V; ++v) acc[v] = lp_sgd4(acc[v], w[v], a.lr, a.invP);
        }
        if (a.epilogue == LP_EPI_SGD_MOM) {  // v' to the velocity vector, w' goes on as the finished tile
#pragma unroll
            for (int v = 0; v < V; ++v) {
                lp_mom4(acc[v], w[v], vel[v], a.lr, a.invP, a.mu, vel[v], acc[v]);
                if (live[v]) lp_stg_stream(a.vel_out + a0 + 4 * (uint64_t)(tid + v * kThreads), vel[v]);
            }
        }
        for (int q = 0; q < a.n_out; ++q) {
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (live[v]) lp_stg_stream(a.out[q] + a0 + 4 * (uint64_t)(tid + v * kThreads), acc[v]);
        }
    }
}

template <int V, bool SEG>
cudaError_t launch_v(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, const LpLaunch &cfg, cudaStream_t stream) {
#define LP_DIRECT_CASE(NS)                                                                  \
    case NS:                                                                                \
        return lp_launch(lp_direct_kernel<NS, V, SEG>, dim3(cfg.grid), dim3(cfg.threads), 0, stream, cfg.pdl, a, segs);
    switch (a.n_sum) {
        LP_DIRECT_CASE(1)
        LP_DIRECT_CASE(2)
        LP_DIRECT_CASE(3)
        LP_DIRECT_CASE(4)
        LP_DIRECT_CASE(6)
        LP_DIRECT_CASE(8)
        LP_DIRECT_CASE(16)
        default:
            return lp_launch(lp_direct_kernel<0, V, SEG>, dim3(cfg.grid), dim3(cfg.threads), 0, stream, cfg.pdl, a, segs);
    }
#undef LP_DIRECT_CASE
}

template <int V>
cudaError_t launch_seg(const LpArgs &a, const lp_seg_table *segs, const LpLaunch &cfg, cudaStream_t stream) {
    if (segs) return launch_v<V, true>(a, *segs, cfg, stream);
    return launch_v<V, false>(a, LpNoSegs{0}, cfg, stream);
}

}  // namespace

// 8 KB tiles (2 vectors per thread and rank); 4 KB when the message has fewer tiles than two grid-fulls of SMs
// (latency regime: spread it over more SMs).
uint32_t lp_direct_tile(const LpTuning &t, int /*n_in*/, uint64_t n_work) {
    if (t.v[LP_TUNE_TILE_ELEMS]) {
        const uint32_t tile = (uint32_t)t.v[LP_TUNE_TILE_ELEMS];
        return (tile == 1024u || tile == 2048u || tile == 4096u) ? tile : 2048u;
    }
    uint32_t tile = 2048u;
    if ((n_work + tile - 1) / tile < 2u * 148u) tile = 1024u;
    return tile;
}

cudaError_t lp_direct_launch(const LpArgs &a, const lp_seg_table *segs, const LpTuning &t, int sm_count, LpLaunch *cfg,
                             bool dry_run, cudaStream_t stream) {
    uint64_t grid = a.part.n_tiles;  // one CTA per tile
    if (t.v[LP_TUNE_CTAS_PER_SM]) grid = (uint64_t)sm_count * (uint32_t)t.v[LP_TUNE_CTAS_PER_SM];
    if (t.v[LP_TUNE_GRID_LIMIT] && grid > (uint64_t)t.v[LP_TUNE_GRID_LIMIT]) grid = (uint64_t)t.v[LP_TUNE_GRID_LIMIT];
    if (grid > a.part.n_tiles) grid = a.part.n_tiles;
    if (grid > 0x7fffffffull) grid = 0x7fffffffull;
    cfg->grid = (uint32_t)grid;
    cfg->threads = kThreads;
    cfg->smem_bytes = 0;
    cfg->stages = 0;
    cfg->out_stages = 0;
    cfg->pdl = t.v[LP_TUNE_NO_PDL] == 0;
    if (dry_run || grid == 0) return cudaSuccess;
    lp_count_launch(1);
    switch (a.part.tile) {
        case 1024: return launch_seg<1>(a, segs, *cfg, stream);
        case 2048: return launch_seg<2>(a, segs, *cfg, stream);
        case 4096: return launch_seg<4>(a, segs, *cfg, stream);
        default: return cudaErrorInvalidValue;
    }
}
