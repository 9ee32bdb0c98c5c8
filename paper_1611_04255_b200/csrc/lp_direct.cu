// lp_direct.cu -- LP_VARIANT_DIRECT: the LP collective as one kernel (one CTA per tile) that keeps the running
// partial of the chain (a0 -> a' = a0 + a1 -> a'' = a' + a2) in registers.  Each thread owns V
// 16-byte vectors of a tile, issues the 128-bit streaming loads of up to 8 ranks at once (memory-level
// parallelism replaces the paper's two DMA engines), folds them in rank order 0 -> P-1 with RN adds and
// writes the finished vector to every destination rank.  It is also the path that takes any alignment:
// a tile whose start is not a multiple of 4 elements (block % 4 != 0) gets a scalar head and tail.
#include <atomic>

#include "lp_common.cuh"

namespace {

constexpr int kThreads = 256;

// CTAs per SM the launch is capped at (8 = no cap: 2048 threads).  A thread's stores are fire-and-forget, so a
// write-heavy launch (broadcast to several ranks) keeps far more bytes in flight per CTA than it has loaded; beyond
// ~150 KB of stores in flight per SM the extra ones only queue up in front of the L2 and the launch slows down by
// 3-5 % (profiles/r2_tuning.md: 8 KB tiles x n_out destinations x CTAs: 8 CTAs for 2 destinations, 6 for 3, 4 for 5,
// 3 for 7; 3 CTAs of 4 KB tiles from 12 destinations on).  Folds are capped by their registers long before.
uint32_t lp_direct_occupancy(const LpArgs &a) {
    if (a.epilogue != LP_EPI_COPY || a.n_out <= 2) return 8u;
    if (a.n_out >= 12) return 3u;  // with 4 KB tiles (lp_direct_tile)
    const uint32_t occ = (18u + (uint32_t)a.n_out / 2u) / (uint32_t)a.n_out;
    return occ < 2u ? 2u : (occ > 8u ? 8u : occ);
}

// ranks whose loads are in flight together: 8, or 16 for the one-vector-per-thread kernels of the latency regime (a
// 16-rank chain then costs one HBM latency, not two)
template <int V>
struct LpRankChunk {
    static constexpr int value = V == 1 ? 16 : 8;
};

// NS > 0: number of folded inputs known at compile time (loops fully unrolled); NS == 0: runtime a.n_sum.
// SGD: the launch has an SGD epilogue (plain or momentum, a.epilogue); false keeps the weight / velocity registers
// out of the copy / fold kernels (a broadcast thread then needs 8 V + ~20 registers: 4 CTAs of 8 vectors per thread
// = 128 KB of loads in flight per SM).
template <int NS, int V, bool SEG, bool SGD>
__global__ void __launch_bounds__(kThreads)
    lp_direct_kernel(const __grid_constant__ LpArgs a, const __grid_constant__ typename LpSegParam<SEG>::type segs) {
    const int n_sum = NS > 0 ? NS : a.n_sum;
    const int tid = threadIdx.x;
    const int code = lp_fold_code(a.dtype, a.red_op);
    // a2: one CTA per tile by default (grid == n_tiles): the hardware block scheduler hands the next tile to
    // whichever SM frees up first -- the same balance the pipeline kernel gets from its tile claims, with no
    // per-CTA setup at all, which is what the latency regime wants.  A confined grid (LP_TUNE_GRID_LIMIT /
    // LP_TUNE_CTAS_PER_SM) walks the tile list round robin.
    // wait first, then trigger: at most ONE successor waits behind a running kernel (triggering before the wait lets
    // a whole queue of short kernels pile up on the SMs, each blocked on its predecessor: measured 2x slower at 256 KB)
    // A launch that touches none of the buffers of the launches ahead of it (a.late_wait) waits before it exits instead.
    if (a.prefetch) {  // this CTA's first tile into L2 while the predecessor kernel drains (a hint: L2 is the point of
                       // coherence, so it is harmless even if the predecessor is still writing these vectors)
        uint64_t off;
        uint32_t len;
        if ((uint64_t)blockIdx.x < a.part.n_tiles) {
            lp_lookup_tile<SEG>(a, segs, blockIdx.x, off, len);
            const uint32_t lines = (len * 4u + 127u) / 128u;  // 128-byte lines of the tile, per input
            for (uint32_t l = tid; l < lines * (uint32_t)a.n_in; l += kThreads) {
                const uint32_t r = l / lines, k = l - r * lines;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.in[r] + off + (uint64_t)k * 32u));
            }
        }
    }
    if (!a.late_wait) lp_pdl_wait();
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
        const uint64_t e0 = a0 + 4 * (uint64_t)tid;  // this thread's first element; vector v is v * 4 * kThreads further on

        float4 acc[V];
        float4 w[SGD ? V : 1];
        float4 vel[SGD ? V : 1];
        bool live[V];
#pragma unroll
        for (int v = 0; v < V; ++v) live[v] = (uint32_t)(tid + v * kThreads) < nvec;
        if constexpr (SGD) {
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (live[v]) w[v] = lp_ldg_stream(a.in[n_sum] + e0 + (uint64_t)(v * 4 * kThreads));
            if (a.epilogue == LP_EPI_SGD_MOM) {
#pragma unroll
                for (int v = 0; v < V; ++v)
                    if (live[v]) vel[v] = lp_ldg_stream(a.in[n_sum + 1] + e0 + (uint64_t)(v * 4 * kThreads));
            }
        }
        constexpr int kRankChunk = LpRankChunk<V>::value;
        for (int r0 = 0; r0 < n_sum; r0 += kRankChunk) {
            float4 x[V][kRankChunk];
#pragma unroll
            for (int j = 0; j < kRankChunk; ++j) {
                if (NS > 0 ? (r0 + j < NS) : (r0 + j < n_sum)) {
#pragma unroll
                    for (int v = 0; v < V; ++v)
                        if (live[v]) x[v][j] = lp_ldg_stream(a.in[r0 + j] + e0 + (uint64_t)(v * 4 * kThreads));
                }
            }
#pragma unroll
            for (int j = 0; j < kRankChunk; ++j) {
                if (NS > 0 ? (r0 + j < NS) : (r0 + j < n_sum)) {
#pragma unroll
                    for (int v = 0; v < V; ++v) acc[v] = (r0 + j == 0) ? x[v][j] : lp_combine4(acc[v], x[v][j], code);
                }
            }
        }
        if constexpr (SGD) {
            if (a.epilogue == LP_EPI_SGD) {
#pragma unroll
                for (int v = 0; v < V; ++v) acc[v] = lp_sgd4(acc[v], w[v], a.lr, a.invP);
            } else {  // momentum: v' to the velocity vector, w' goes on as the finished tile
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    lp_mom4(acc[v], w[v], vel[v], a.lr, a.invP, a.mu, vel[v], acc[v]);
                    if (live[v]) lp_stg_stream(a.vel_out + e0 + (uint64_t)(v * 4 * kThreads), vel[v]);
                }
            }
        }
        for (int q = 0; q < a.n_out; ++q) {
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (live[v]) lp_stg_stream(a.out[q] + e0 + (uint64_t)(v * 4 * kThreads), acc[v]);
        }
    }
    if (a.late_wait && tid == 0) lp_pdl_wait();  // this CTA does not exit before the launches ahead of it have completed
}

// One instantiation's launch.  cfg.smem_bytes > 0 is dynamic shared memory the kernel never touches: it caps how many
// CTAs an SM holds (LP_TUNE_DIRECT_OCC), i.e. how many stores the SM keeps in flight.
template <int NS, int V, bool SEG, bool SGD>
cudaError_t launch_k(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, const LpLaunch &cfg, cudaStream_t stream) {
    if (cfg.smem_bytes > 48u * 1024u) {
        static std::atomic<int> bytes{0};
        static std::atomic<unsigned> epoch{0};
        if (epoch.load() != lp_attr_epoch() || (int)cfg.smem_bytes > bytes.load()) {
            cudaError_t e = cudaFuncSetAttribute(lp_direct_kernel<NS, V, SEG, SGD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 (int)cfg.smem_bytes);
            if (e != cudaSuccess) return e;
            epoch.store(lp_attr_epoch());
            bytes.store((int)cfg.smem_bytes);
        }
    }
    return lp_launch(lp_direct_kernel<NS, V, SEG, SGD>, dim3(cfg.grid), dim3(cfg.threads), cfg.smem_bytes, stream, cfg.pdl, a,
                     segs);
}

template <int V, bool SEG>
cudaError_t launch_v(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, const LpLaunch &cfg, cudaStream_t stream) {
    const bool sgd = a.epilogue == LP_EPI_SGD || a.epilogue == LP_EPI_SGD_MOM;
#define LP_DIRECT_CASE(NS, SGD) \
    case NS: return launch_k<NS, V, SEG, SGD>(a, segs, cfg, stream);
    if (sgd) {
        switch (a.n_sum) {
            LP_DIRECT_CASE(2, true)
            LP_DIRECT_CASE(4, true)
            LP_DIRECT_CASE(8, true)
            LP_DIRECT_CASE(16, true)
            default: return launch_k<0, V, SEG, true>(a, segs, cfg, stream);
        }
    }
    switch (a.n_sum) {
        LP_DIRECT_CASE(1, false)
        LP_DIRECT_CASE(2, false)
        LP_DIRECT_CASE(3, false)
        LP_DIRECT_CASE(4, false)
        LP_DIRECT_CASE(5, false)
        LP_DIRECT_CASE(6, false)
        LP_DIRECT_CASE(8, false)
        LP_DIRECT_CASE(16, false)
        default: return launch_k<0, V, SEG, false>(a, segs, cfg, stream);
    }
#undef LP_DIRECT_CASE
}

template <int V>
cudaError_t launch_seg(const LpArgs &a, const lp_seg_table *segs, const LpLaunch &cfg, cudaStream_t stream) {
    if (segs) return launch_v<V, true>(a, *segs, cfg, stream);
    return launch_v<V, false>(a, LpNoSegs{0}, cfg, stream);
}

}  // namespace

// Tile = V * 1024 elements, V 16-byte vectors per thread and input stream.  What the kernel needs is enough load bytes
// in flight per SM (HBM latency x the SM's share of the bandwidth: ~100 KB): a thread has V * n_sum loads outstanding
// and the registers they take decide how many CTAs an SM holds, so few streams want long tiles and many streams short
// ones -- 16 KB (V = 4, 64 registers: 4 CTAs) for a 2-rank reduce, 8 KB from 3 to 8 ranks and for broadcasts (a copy to
// one rank: 8 CTAs x 8 KB beat 8 x 16 KB by 1.5 % from 64 to 512 MB and equal the MST baseline's plain copy, which is
// the same operation at P = 2; broadcasts to several ranks: their stores in flight are what lp_direct_occupancy
// bounds), 4 KB (16 ranks' loads at once, 2 CTAs) above: ~64-128 KB in flight in every case (profiles/r2_tuning.md).
// 4 KB also when the message has fewer tiles than two grid-fulls of SMs (latency regime: spread it over more SMs).
uint32_t lp_direct_tile(const LpTuning &t, const LpArgs &a, uint64_t n_work, int sm_count) {
    if (t.v[LP_TUNE_TILE_ELEMS]) {
        const uint32_t tile = (uint32_t)t.v[LP_TUNE_TILE_ELEMS];
        return tile <= 4096u ? tile : 4096u;
    }
    const bool sgd = a.epilogue == LP_EPI_SGD || a.epilogue == LP_EPI_SGD_MOM;
    const bool reduce_only = !sgd && a.epilogue != LP_EPI_COPY && a.n_out <= 1;
    uint32_t tile = (reduce_only && a.n_sum == 2) ? 4096u : ((a.n_sum <= 8 && a.n_out < 12) || reduce_only ? 2048u : 1024u);
    // Latency regime: halve the tile while the message has fewer tiles than `few` so that more SMs share it.  A fold
    // over several ranks wants two grid-fulls of tiles (its threads have many loads in flight each: more, smaller CTAs
    // hide more latency); a copy, a two-rank fold or a reduce (one store stream) wants one CTA per SM and no more -- fewer, fatter CTAs cost less
    // to launch, and a broadcast to many ranks runs 3-4 CTAs per SM (lp_direct_occupancy), so four tiles per SM no
    // longer fit in one wave (P = 8, 2 MB broadcast: 4.06 -> 3.2 us; P = 2, 2 MB reduce: 1.92 -> 1.44 us;
    // profiles/r2_tuning.md section 8).  A reduce over more than 8 ranks (below the pipeline cut-off: < 40 MB per rank)
    // runs 5-18 % faster on 8 KB tiles than on 4 KB ones.
    uint64_t few = (a.epilogue == LP_EPI_COPY || a.n_sum <= 2 || reduce_only) ? (uint64_t)sm_count : 2ull * (uint64_t)sm_count;
    if (a.epilogue == LP_EPI_COPY && a.n_out == 1) few = (uint64_t)sm_count / 2u;  // the plain copy: half a grid-full is enough
    while (tile > 1024u && (n_work + tile - 1) / tile < few) tile /= 2u;
    return tile;
}

cudaError_t lp_direct_launch(const LpArgs &a_in, const lp_seg_table *segs, const LpTuning &t, int sm_count, LpLaunch *cfg,
                             bool dry_run, cudaStream_t stream) {
    LpArgs a = a_in;
    uint64_t grid = a.part.n_tiles;  // one CTA per tile
    if (t.v[LP_TUNE_CTAS_PER_SM]) grid = (uint64_t)sm_count * (uint32_t)t.v[LP_TUNE_CTAS_PER_SM];
    if (t.v[LP_TUNE_GRID_LIMIT] && grid > (uint64_t)t.v[LP_TUNE_GRID_LIMIT]) grid = (uint64_t)t.v[LP_TUNE_GRID_LIMIT];
    if (grid > a.part.n_tiles) grid = a.part.n_tiles;
    if (grid > 0x7fffffffull) grid = 0x7fffffffull;
    cfg->grid = (uint32_t)grid;
    cfg->threads = kThreads;
    // residency cap: unused dynamic shared memory sized so that `occ` CTAs fill an SM's 228 KB
    const uint32_t occ = t.v[LP_TUNE_DIRECT_OCC] ? (uint32_t)t.v[LP_TUNE_DIRECT_OCC] : lp_direct_occupancy(a);
    cfg->smem_bytes = occ >= 8u ? 0u : (228u * 1024u / occ - 1024u) / 1024u * 1024u - (occ == 1u ? 1024u : 0u);
    cfg->stages = 0;
    cfg->out_stages = 0;
    cfg->pdl = t.v[LP_TUNE_NO_PDL] == 0;
    cfg->claim = 1;
    if (dry_run || grid == 0) return cudaSuccess;
    lp_count_launch(1);
    {
        LpRange ranges[2 * LP_MAX_IN];
        const int nr = lp_args_ranges(a, ranges);
        // A long reduce over 3 or more ranks (read-dominated, many loads in flight per thread) runs 1-2 % faster when it
        // waits for its predecessor and prefetches than when it shares the SMs with the predecessor's tail
        // (profiles/r2_tuning.md section 9); LP_TUNE_CHAIN = 3 chains it all the same.
        const bool long_reduce = a.epilogue == LP_EPI_SUM && a.n_out <= 1 && a.n_sum >= 3 &&
                                 a.part.n_tiles >= 8ull * (uint64_t)sm_count && t.v[LP_TUNE_CHAIN] != 3;
        a.late_wait = lp_chain_admit(stream, ranges, nr, cfg->pdl, t.v[LP_TUNE_CHAIN] != 2 && !long_reduce) ? 1 : 0;
    }
    // L2 prefetch of every CTA's first tile before it waits for its predecessor (LP_TUNE_PREFETCH 2 = off): only when the
    // launch really waits first, and only for one CTA per tile (a confined grid walks many tiles per CTA)
    a.prefetch = (cfg->pdl && !a.late_wait && t.v[LP_TUNE_PREFETCH] != 2 && grid == a.part.n_tiles) ? 1 : 0;
    switch (a.part.tile) {
        case 1024: return launch_seg<1>(a, segs, *cfg, stream);
        case 2048: return launch_seg<2>(a, segs, *cfg, stream);
        case 4096: return launch_seg<4>(a, segs, *cfg, stream);
        default: return cudaErrorInvalidValue;
    }
}
