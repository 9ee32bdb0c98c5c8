// lp_pipeline.cu -- LP_VARIANT_PIPELINE: the whole LP collective as ONE persistent sm_100a kernel.
//
// What survives of the paper's design on one B200: the message is cut into
// blocks and each block flows down the chain rank 0 -> 1 -> ... -> P-1, every rank adding its
// local block to the partial it received -- but the partial never goes back to HBM between
// hops.  Per CTA:
//
//   producer warp   one thread issues TMA bulk loads (cp.async.bulk global -> shared) of (tile, rank r),
//                   r = 0..P-1 in chain order, into a ring of `stages` slots; a slot's "full" mbarrier
//                   completes when its bytes have landed (the paper's DMA1, inbound engine)
//   add warps       wait "full", fold the slot into the running partial held in registers with fp32 RN
//                   adds in rank order (the paper's per-hop reduce kernel), hand the slot back through its
//                   "empty" mbarrier; after rank P-1 the finished tile goes to a slot of the store ring
//   store warp      one thread waits "out full" and issues one TMA bulk store (shared -> global) per
//                   destination rank (root only for reduce, all P for allreduce / SGD: the broadcast half
//                   of PAPER.md:71), then returns the slot ("out empty") once the copies have read it
//                   (the paper's DMA2, outbound engine)
//
// so loads of later tiles/ranks, adds and stores of earlier tiles overlap (reduction math overlaps
// transfer), and the grid of 148 x k persistent CTAs claims tiles from the launch's tile list (lp_schedule.h; the
// list is one message cut into blocks, or -- layer-wise launches, Alg. 1 -- a list of messages).
// Broadcast has no math: its kernel is the producer and the store thread alone.
#include <atomic>

#include "lp_common.cuh"

namespace {

// Wait until all but the newest `lag` bulk-store groups have read their shared-memory source (complete ==
// false) or have fully completed (complete == true: bounds the store bytes this CTA has in flight).
__device__ __forceinline__ void wait_read_lag(int lag, bool complete) {
    if (complete) {
        switch (lag) {
            case 0: lp_bulk_wait<0>(); break;
            case 1: lp_bulk_wait<1>(); break;
            case 2: lp_bulk_wait<2>(); break;
            default: lp_bulk_wait<3>(); break;
        }
        return;
    }
    switch (lag) {
        case 0: lp_bulk_wait_read<0>(); break;
        case 1: lp_bulk_wait_read<1>(); break;
        case 2: lp_bulk_wait_read<2>(); break;
        default: lp_bulk_wait_read<3>(); break;
    }
}

// A ring slot's meta_len: the tile length (low 32 bits), in the store ring optionally marked as the momentum step's
// velocity tile; kEndLen is the end marker.
constexpr uint64_t kVelocityTag = 1ull << 62;
constexpr uint64_t kEndLen = ~0ull;

struct Ring {
    int slot;
    uint32_t phase;
    int depth;
    __device__ __forceinline__ Ring(int d) : slot(0), phase(0), depth(d) {}
    __device__ __forceinline__ void advance() {
        if (++slot == depth) {
            slot = 0;
            phase ^= 1u;
        }
    }
};

// V float4 per add thread per tile, CW add warps: TILE = V * 4 * CW * 32 elements.
// Every ring slot carries the element range of its tile (meta_off / meta_len): the producer claims granules
// (LpTileClaimer), turns a claim into runs of consecutive granules (lp_lookup_run: a1/a2, single message or
// layer-wise list; a run never leaves its block and fits one slot) and the other two roles learn the range from
// the slot; kEndLen in meta_len is the end marker that travels producer -> add warps -> store thread.
template <int V, int CW, bool SEG>
__global__ void __launch_bounds__((CW + 2) * 32)
    lp_pipeline_kernel(const __grid_constant__ LpArgs a, const __grid_constant__ typename LpSegParam<SEG>::type segs,
                       int stages, int out_stages) {
    constexpr int CT = CW * 32;
    constexpr int TILE = V * 4 * CT;
    extern __shared__ __align__(128) unsigned char lp_smem[];
    float *in_ring = reinterpret_cast<float *>(lp_smem);
    float *out_ring = in_ring + (size_t)stages * TILE;
    uint64_t *full = reinterpret_cast<uint64_t *>(out_ring + (size_t)out_stages * TILE);
    uint64_t *empty = full + stages;
    uint64_t *ofull = empty + stages;
    uint64_t *oempty = ofull + out_stages;
    uint64_t *meta_off = oempty + out_stages;  // [stages]
    uint64_t *meta_len = meta_off + stages;    // [stages]
    uint64_t *ometa_off = meta_len + stages;   // [out_stages]
    uint64_t *ometa_len = ometa_off + out_stages;

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            lp_mbar_init(&full[s], 1);    // the producer's arrive.expect_tx (+ the bytes)
            lp_mbar_init(&empty[s], CW);  // lane 0 of every add warp
        }
        for (int s = 0; s < out_stages; ++s) {
            lp_mbar_init(&ofull[s], CW);
            lp_mbar_init(&oempty[s], 1);  // the store thread
        }
        lp_fence_mbar_init();
    }
    __syncthreads();
    if (a.prefetch && threadIdx.x == 0) {  // this CTA's first loads, into L2, while the predecessor kernel drains
        const LpClaim c = LpTileClaimer(a.sched, a.part.n_tiles, a.claim_max, a.claim_shift).peek();
        if (c.g0 < c.g1) {
            uint64_t off;
            uint32_t len;
            lp_lookup_run<SEG>(a, segs, c.g0, c.g1, a.slot_gran, off, len);
            const LpTileSpan span(off, len);
            if (span.body)
                for (int r = 0; r < a.n_in; ++r) lp_prefetch_l2(a.in[r] + span.a0, span.body * 4u);
        }
    }
    // the predecessor in the stream has completed and its writes are visible (no-op without PDL); a launch that
    // touches none of its predecessors' buffers waits at its end instead (store thread)
    if (!a.late_wait) lp_pdl_wait();

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0) {
        // ---------------- producer: claims tiles, TMA bulk loads in chain order ---------------------------
        if (lane == 0) {
            const uint64_t pol = lp_policy_evict_first();
            const bool hint = a.l2_hint >= 1;
            Ring ring(stages);
            LpTileClaimer claimer(a.sched, a.part.n_tiles, a.claim_max, a.claim_shift);
            for (;;) {
                const LpClaim c = claimer.claim();
                if (c.g0 >= c.g1) {  // end marker
                    claimer.finish();
                    lp_pdl_trigger();  // nothing left to claim here: the next kernel's CTAs may start
                    lp_mbar_wait(&empty[ring.slot], ring.phase ^ 1u);
                    meta_len[ring.slot] = kEndLen;
                    lp_mbar_arrive(&full[ring.slot]);
                    break;
                }
                for (uint64_t g = c.g0; g < c.g1;) {  // the claim as runs of <= slot_gran granules inside one block
                    uint64_t off;
                    uint32_t len;
                    g += lp_lookup_run<SEG>(a, segs, g, c.g1, a.slot_gran, off, len);
                    const LpTileSpan span(off, len);
                    const uint32_t bytes = span.body * 4u;
                    for (int r = 0; r < a.n_in; ++r) {
                        lp_mbar_wait(&empty[ring.slot], ring.phase ^ 1u);
                        meta_off[ring.slot] = off;
                        meta_len[ring.slot] = len;
                        if (bytes) {
                            lp_mbar_expect_tx(&full[ring.slot], bytes);
                            float *dst = in_ring + (size_t)ring.slot * TILE;
                            if (hint)
                                lp_bulk_g2s_hint(dst, a.in[r] + span.a0, bytes, &full[ring.slot], pol);
                            else
                                lp_bulk_g2s(dst, a.in[r] + span.a0, bytes, &full[ring.slot]);
                        } else {
                            lp_mbar_arrive(&full[ring.slot]);
                        }
                        ring.advance();
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ---------------- store thread: TMA bulk stores to every destination rank -----------------------
        if (lane == 0) {
            const uint64_t pol = lp_policy_evict_first();
            const bool hint = a.l2_hint >= 2;
            const int lag = out_stages >= 3 ? 2 : (out_stages == 2 ? 1 : 0);  // < out_stages: the end marker finds a slot
            Ring ring(out_stages);
            uint64_t issued = 0;
            int free_slot = 0;  // oldest slot not yet handed back
            for (;;) {
                lp_mbar_wait(&ofull[ring.slot], ring.phase);
                const uint64_t tag = ometa_len[ring.slot];
                if (tag == kEndLen) break;
                const bool to_velocity = (tag & kVelocityTag) != 0;  // momentum: the tile of new velocities
                const LpTileSpan span(ometa_off[ring.slot], (uint32_t)(tag & 0xffffffffull));
                const uint32_t bytes = span.body * 4u;
                if (bytes) {
                    const float *src = out_ring + (size_t)ring.slot * TILE;
                    if (to_velocity) {
                        lp_bulk_s2g(a.vel_out + span.a0, src, bytes);
                    } else {
                        for (int q = 0; q < a.n_out; ++q) {
                            if (hint)
                                lp_bulk_s2g_hint(a.out[q] + span.a0, src, bytes, pol);
                            else
                                lp_bulk_s2g(a.out[q] + span.a0, src, bytes);
                        }
                    }
                }
                lp_bulk_commit();
                ++issued;
                wait_read_lag(lag, a.store_wait != 0);  // all but the newest `lag` groups are done with shared memory
                if (issued > (uint64_t)lag) {
                    lp_mbar_arrive(&oempty[free_slot]);
                    if (++free_slot == out_stages) free_slot = 0;
                }
                ring.advance();
            }
            lp_bulk_wait<0>();  // every store has completed before the CTA exits
            if (a.late_wait) lp_pdl_wait();  // ... and the CTA does not exit before the launches ahead of it have completed
        }
    } else {
        // ---------------- add warps: chain fold in registers ----------------------------------------------
        const int ctid = threadIdx.x - 64;
        const int code = lp_fold_code(a.dtype, a.red_op);
        Ring ring(stages);
        Ring oring(out_stages);
        for (;;) {
            lp_mbar_wait(&full[ring.slot], ring.phase);
            const uint64_t len64 = meta_len[ring.slot];
            if (len64 == kEndLen) {  // end marker: pass it on to the store thread
                lp_mbar_wait(&oempty[oring.slot], oring.phase ^ 1u);
                if (ctid == 0) ometa_len[oring.slot] = kEndLen;
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&ofull[oring.slot]);
                break;
            }
            const uint64_t off = meta_off[ring.slot];
            const uint32_t len = (uint32_t)len64;
            // a short run (the shrinking claims at the end of the list) fills only the first nv slabs of the slot
            const int nv = (int)((len + (uint32_t)(CT * 4 - 1)) / (uint32_t)(CT * 4));
            float4 acc[V];
            {  // rank 0: the partial starts as its block ("writing block a0 to a buffer on GPU1")
                const float4 *s = reinterpret_cast<const float4 *>(in_ring + (size_t)ring.slot * TILE);
#pragma unroll
                for (int v = 0; v < V; ++v)
                    if (v < nv) acc[v] = s[ctid + v * CT];
                // nothing consumes these loads before the slot is handed back: make sure they have returned (an
                // mbarrier arrive does not wait for queued shared-memory loads; lp_cluster.cu has the measured case)
                __threadfence_block();
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&empty[ring.slot]);
                ring.advance();
            }
            for (int r = 1; r < a.n_sum; ++r) {  // rank r: partial <- partial + local block
                lp_mbar_wait(&full[ring.slot], ring.phase);
                const float4 *s = reinterpret_cast<const float4 *>(in_ring + (size_t)ring.slot * TILE);
                float4 x[V];
#pragma unroll
                for (int v = 0; v < V; ++v)
                    if (v < nv) x[v] = s[ctid + v * CT];
                lp_fold_vecs<V>(acc, x, nv, code);
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&empty[ring.slot]);
                ring.advance();
            }
            if (a.epilogue == LP_EPI_SGD) {  // g = S/P, w' = w_root - lr g
                lp_mbar_wait(&full[ring.slot], ring.phase);
                const float4 *s = reinterpret_cast<const float4 *>(in_ring + (size_t)ring.slot * TILE);
#pragma unroll
                for (int v = 0; v < V; ++v)
                    if (v < nv) acc[v] = lp_sgd4(acc[v], s[ctid + v * CT], a.lr, a.invP);
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&empty[ring.slot]);
                ring.advance();
            }
            if (a.epilogue == LP_EPI_SGD_MOM) {  // v' = mu v + lr g, w' = w_root - v'  (U18)
                float4 w[V];
                lp_mbar_wait(&full[ring.slot], ring.phase);
                {
                    const float4 *s = reinterpret_cast<const float4 *>(in_ring + (size_t)ring.slot * TILE);
#pragma unroll
                    for (int v = 0; v < V; ++v)
                        if (v < nv) w[v] = s[ctid + v * CT];
                }
                __threadfence_block();
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&empty[ring.slot]);
                ring.advance();
                lp_mbar_wait(&full[ring.slot], ring.phase);
                float4 vel[V];
                {
                    const float4 *s = reinterpret_cast<const float4 *>(in_ring + (size_t)ring.slot * TILE);
#pragma unroll
                    for (int v = 0; v < V; ++v)
                        if (v < nv) lp_mom4(acc[v], w[v], s[ctid + v * CT], a.lr, a.invP, a.mu, vel[v], acc[v]);
                }
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&empty[ring.slot]);
                ring.advance();
                // the tile of new velocities goes through the store ring first, tagged for its own destination
                lp_mbar_wait(&oempty[oring.slot], oring.phase ^ 1u);
                float4 *ov = reinterpret_cast<float4 *>(out_ring + (size_t)oring.slot * TILE);
#pragma unroll
                for (int v = 0; v < V; ++v)
                    if (v < nv) ov[ctid + v * CT] = vel[v];
                if (ctid == 0) {
                    ometa_off[oring.slot] = off;
                    ometa_len[oring.slot] = (uint64_t)len | kVelocityTag;
                }
                lp_fence_proxy_async();
                __syncwarp();
                if (lane == 0) lp_mbar_arrive(&ofull[oring.slot]);
                oring.advance();
            }
            // finished tile -> store ring
            lp_mbar_wait(&oempty[oring.slot], oring.phase ^ 1u);
            float4 *o = reinterpret_cast<float4 *>(out_ring + (size_t)oring.slot * TILE);
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (v < nv) o[ctid + v * CT] = acc[v];
            if (ctid == 0) {
                ometa_off[oring.slot] = off;
                ometa_len[oring.slot] = len;
            }
            lp_fence_proxy_async();
            __syncwarp();
            if (lane == 0) lp_mbar_arrive(&ofull[oring.slot]);
            oring.advance();
            // the <= 3 + 3 elements outside the 16-byte aligned body of the tile
            const LpTileSpan span(off, len);
            if ((uint32_t)ctid < span.head) lp_scalar_element(a, off + ctid);
            if ((uint32_t)ctid >= 32u && (uint32_t)ctid - 32u < span.tail) lp_scalar_element(a, span.a0 + span.body + (ctid - 32));
        }
    }
}

// Broadcast: the root's tile is loaded once into the ring and stored to the P-1 other ranks
// straight from the same slot.  Warp 0 lane 0 claims tiles and loads, warp 1 lane 0 stores (and copies the
// <= 3 + 3 elements outside the 16-byte aligned body of a tile).
template <bool SEG>
__global__ void __launch_bounds__(64)
    lp_bcast_kernel(const __grid_constant__ LpArgs a, const __grid_constant__ typename LpSegParam<SEG>::type segs, int stages,
                    int tile) {
    extern __shared__ __align__(128) unsigned char lp_smem[];
    float *ring_buf = reinterpret_cast<float *>(lp_smem);
    uint64_t *full = reinterpret_cast<uint64_t *>(ring_buf + (size_t)stages * tile);
    uint64_t *empty = full + stages;
    uint64_t *meta_off = empty + stages;
    uint64_t *meta_len = meta_off + stages;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            lp_mbar_init(&full[s], 1);
            lp_mbar_init(&empty[s], 1);
        }
        lp_fence_mbar_init();
    }
    __syncthreads();
    if (a.prefetch && threadIdx.x == 0) {
        const LpClaim c = LpTileClaimer(a.sched, a.part.n_tiles, a.claim_max, a.claim_shift).peek();
        if (c.g0 < c.g1) {
            uint64_t off;
            uint32_t len;
            lp_lookup_run<SEG>(a, segs, c.g0, c.g1, a.slot_gran, off, len);
            const LpTileSpan span(off, len);
            if (span.body) lp_prefetch_l2(a.in[0] + span.a0, span.body * 4u);
        }
    }
    if (!a.late_wait) lp_pdl_wait();
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    if (warp == 0 && lane == 0) {
        const uint64_t pol = lp_policy_evict_first();
        const bool hint = a.l2_hint >= 1;
        Ring ring(stages);
        LpTileClaimer claimer(a.sched, a.part.n_tiles, a.claim_max, a.claim_shift);
        for (;;) {
            const LpClaim c = claimer.claim();
            if (c.g0 >= c.g1) {  // end marker
                claimer.finish();
                lp_pdl_trigger();
                lp_mbar_wait(&empty[ring.slot], ring.phase ^ 1u);
                meta_len[ring.slot] = kEndLen;
                lp_mbar_arrive(&full[ring.slot]);
                break;
            }
            for (uint64_t g = c.g0; g < c.g1;) {
                uint64_t off;
                uint32_t len;
                g += lp_lookup_run<SEG>(a, segs, g, c.g1, a.slot_gran, off, len);
                lp_mbar_wait(&empty[ring.slot], ring.phase ^ 1u);
                meta_off[ring.slot] = off;
                meta_len[ring.slot] = len;
                const LpTileSpan span(off, len);
                const uint32_t bytes = span.body * 4u;
                if (bytes) {
                    lp_mbar_expect_tx(&full[ring.slot], bytes);
                    float *dst = ring_buf + (size_t)ring.slot * tile;
                    if (hint)
                        lp_bulk_g2s_hint(dst, a.in[0] + span.a0, bytes, &full[ring.slot], pol);
                    else
                        lp_bulk_g2s(dst, a.in[0] + span.a0, bytes, &full[ring.slot]);
                } else {
                    lp_mbar_arrive(&full[ring.slot]);
                }
                ring.advance();
            }
        }
    } else if (warp == 1 && lane == 0) {
        const uint64_t pol = lp_policy_evict_first();
        const bool hint = a.l2_hint >= 2;
        const int lag = stages >= 4 ? 2 : 1;  // < stages - 1: loads keep a slot, and the end marker finds one
        Ring ring(stages);
        uint64_t issued = 0;
        int free_slot = 0;
        for (;;) {
            lp_mbar_wait(&full[ring.slot], ring.phase);
            const uint64_t len64 = meta_len[ring.slot];
            if (len64 == kEndLen) break;
            const uint64_t off = meta_off[ring.slot];
            const LpTileSpan span(off, (uint32_t)len64);
            const uint32_t bytes = span.body * 4u;
            if (bytes) {
                const float *src = ring_buf + (size_t)ring.slot * tile;
                for (int q = 0; q < a.n_out; ++q) {
                    if (hint)
                        lp_bulk_s2g_hint(a.out[q] + span.a0, src, bytes, pol);
                    else
                        lp_bulk_s2g(a.out[q] + span.a0, src, bytes);
                }
            }
            for (uint32_t e = 0; e < span.head; ++e) lp_scalar_element(a, off + e);
            for (uint32_t e = 0; e < span.tail; ++e) lp_scalar_element(a, span.a0 + span.body + e);
            lp_bulk_commit();
            ++issued;
            wait_read_lag(lag, a.store_wait != 0);
            if (issued > (uint64_t)lag) {
                lp_mbar_arrive(&empty[free_slot]);
                if (++free_slot == stages) free_slot = 0;
            }
            ring.advance();
        }
        lp_bulk_wait<0>();
        if (a.late_wait) lp_pdl_wait();
    }
}

// "cudaFuncAttributeMaxDynamicSharedMemorySize already raised to `bytes`" -- valid for the device the library is bound
// to (function attributes are per device): lp_shutdown() advances lp_attr_epoch() and every cache starts over.
// Racing threads at worst set the attribute twice.
struct AttrCache {
    std::atomic<int> bytes{0};
    std::atomic<unsigned> epoch{0};
    bool needs(int want) const { return epoch.load() != lp_attr_epoch() || want > bytes.load(); }
    void set(int b) {
        epoch.store(lp_attr_epoch());
        bytes.store(b);
    }
};

template <int V, int CW, bool SEG>
cudaError_t launch_fold_t(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, const LpLaunch &cfg,
                          cudaStream_t stream) {
    static AttrCache cache;  // per instantiation
    if (cache.needs((int)cfg.smem_bytes)) {
        cudaError_t e = cudaFuncSetAttribute(lp_pipeline_kernel<V, CW, SEG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)cfg.smem_bytes);
        if (e != cudaSuccess) return e;
        cache.set((int)cfg.smem_bytes);
    }
    return lp_launch(lp_pipeline_kernel<V, CW, SEG>, dim3(cfg.grid), dim3(cfg.threads), cfg.smem_bytes, stream, cfg.pdl, a,
                     segs, (int)cfg.stages, (int)cfg.out_stages);
}

template <int V, int CW>
cudaError_t launch_fold(const LpArgs &a, const lp_seg_table *segs, const LpLaunch &cfg, cudaStream_t stream) {
    if (segs) return launch_fold_t<V, CW, true>(a, *segs, cfg, stream);
    return launch_fold_t<V, CW, false>(a, LpNoSegs{0}, cfg, stream);
}

template <bool SEG>
cudaError_t launch_bcast_t(const LpArgs &a, const typename LpSegParam<SEG>::type &segs, const LpLaunch &cfg, uint32_t tile,
                           cudaStream_t stream) {
    static AttrCache cache;
    if (cache.needs((int)cfg.smem_bytes)) {
        cudaError_t e = cudaFuncSetAttribute(lp_bcast_kernel<SEG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)cfg.smem_bytes);
        if (e != cudaSuccess) return e;
        cache.set((int)cfg.smem_bytes);
    }
    return lp_launch(lp_bcast_kernel<SEG>, dim3(cfg.grid), dim3(cfg.threads), cfg.smem_bytes, stream, cfg.pdl, a, segs,
                     (int)cfg.stages, (int)tile);
}

constexpr uint32_t kSmemPerSm = 228u * 1024u;   // sm_100: 228 KB per SM, 227 KB max per CTA, 1 KB reserved per CTA
constexpr uint32_t kSmemPerCtaMax = 227u * 1024u;

}  // namespace

// Defaults measured on B200 with dynamic tile claims (profiles/r1_tuning.md).  With every SM busy until the tile
// list is empty the optimum is broad; what matters is enough load bytes in flight per SM: 64 KB for a fold that
// writes every rank back (allreduce, SGD: 8 KB tiles x 4 slots x 2 CTAs), 96 KB for the read-dominated reduce
// (6 slots), and for broadcast a ring that covers the time its slots are pinned by n_out stores each.
static bool read_dominated(const LpArgs &a) { return a.epilogue != LP_EPI_COPY && a.n_out == 1 && a.n_sum > 1; }

// Slot size (the largest run one ring slot holds): the tuned or default size, halved while a whole block still fits in
// the half (a block is never split finer than it has to be), floor 1024.
uint32_t lp_pipeline_tile(const LpTuning &t, const LpArgs &a, uint64_t n, uint64_t block, int sm_count) {
    const bool confined = lp_grid_confined(t, sm_count);
    uint32_t tile = t.v[LP_TUNE_TILE_ELEMS] ? (uint32_t)t.v[LP_TUNE_TILE_ELEMS]
                    : (confined ? (read_dominated(a) ? 8192u : 4096u)
                                : (a.epilogue == LP_EPI_COPY && a.n_out >= 9 ? 1024u : 2048u));
    uint64_t blk = block < n ? block : n;
    while (tile > 1024u && (uint64_t)(tile / 2) >= blk) tile /= 2;
    // latency regime: fewer tiles than SMs -> halve the tile so that twice as many SMs share the message
    if (!t.v[LP_TUNE_TILE_ELEMS] && tile > 1024u && (n + tile - 1) / tile < (uint64_t)sm_count) tile = 1024u;
    return tile;
}

// Granule (the unit of a claim, lp_common.cuh): the whole slot by default.  LP_TUNE_GRANULE_DIV = 2, 4, 8 makes the
// last claims of a launch that much smaller ("guided self-scheduling"); measured on B200 it buys nothing -- the ring
// of a CTA drains in ~1 us whatever the tile, and the short runs cost 1-2 % (profiles/r2_tuning.md) -- so it stays a knob.
uint32_t lp_pipeline_granule(const LpTuning &t, uint32_t tile) {
    uint32_t div = t.v[LP_TUNE_GRANULE_DIV] ? (uint32_t)t.v[LP_TUNE_GRANULE_DIV] : 1u;
    while (div > 1u && (tile / div < 256u || tile % div != 0u)) div /= 2u;
    return tile / div;
}

cudaError_t lp_pipeline_launch(const LpArgs &a_in, const lp_seg_table *segs, const LpTuning &t, int sm_count, LpLaunch *cfg,
                               bool dry_run, cudaStream_t stream) {
    LpArgs a = a_in;
    const uint32_t gran = a.part.tile;
    const uint32_t slot_gran = a.slot_gran ? a.slot_gran : 1u;
    const uint32_t tile = gran * slot_gran;  // ring slot, elements
    const uint64_t n_slots = (a.part.n_tiles + slot_gran - 1) / slot_gran;  // about: short blocks make more, shorter runs
    const bool bcast = a.epilogue == LP_EPI_COPY;
    const bool confined = lp_grid_confined(t, sm_count);
    uint32_t ctas = t.v[LP_TUNE_CTAS_PER_SM] ? (uint32_t)t.v[LP_TUNE_CTAS_PER_SM] : (bcast && a.n_out <= 2 ? 3u : 2u);
    uint32_t stages = t.v[LP_TUNE_STAGES] ? (uint32_t)t.v[LP_TUNE_STAGES]
                      : (bcast ? (a.n_out <= 2 ? 6u : 4u) : (read_dominated(a) ? 6u : 4u));
    uint32_t out_stages = bcast ? 0u : (t.v[LP_TUNE_OUT_STAGES] ? (uint32_t)t.v[LP_TUNE_OUT_STAGES] : 2u);
    // latency regime (at most one slot per SM): one CTA per SM and a ring deep enough to have the tile of every
    // rank in flight at once -- the chain's P loads cost one HBM latency instead of P / stages of them
    if (n_slots <= (uint64_t)sm_count) {
        if (!t.v[LP_TUNE_CTAS_PER_SM]) ctas = 1u;
        if (!t.v[LP_TUNE_STAGES] && !bcast && stages < (uint32_t)a.n_in) stages = a.n_in < 24 ? (uint32_t)a.n_in : 24u;
    }
    // confined to fewer CTAs than SMs (LP_TUNE_GRID_LIMIT: a collective running beside compute kernels): one CTA per
    // SM with all of its shared memory -- 16 KB tiles in a 12-deep load ring (~100 GB/s per CTA for allreduce: 64 CTAs
    // move 6.3 TB/s), 32 KB tiles x 6 for the read-dominated reduce (~130 GB/s per CTA: 7.1 TB/s); broadcast is
    // bounded by ~60 GB/s of bulk stores per SM whatever the ring (profiles/r1_tuning.md section 6)
    if (confined) {
        if (!t.v[LP_TUNE_CTAS_PER_SM]) ctas = 1u;
        if (!t.v[LP_TUNE_STAGES]) stages = read_dominated(a) ? 6u : 12u;
        if (!t.v[LP_TUNE_OUT_STAGES] && !bcast) out_stages = read_dominated(a) ? 1u : 2u;
    }
    auto smem_of = [&](uint32_t st, uint32_t ost) {
        return (st + ost) * tile * 4u + (4u * st + 4u * ost) * 8u;  // rings + full/empty barriers + tile ranges
    };
    // shrink the rings until `ctas` CTAs fit one SM; if even the shallowest rings do not, take fewer CTAs
    const uint32_t want_stages = stages, want_out = out_stages;
    for (;;) {
        const uint32_t share = kSmemPerSm / ctas - 1024u;
        const uint32_t budget = share < kSmemPerCtaMax ? share : kSmemPerCtaMax;
        stages = want_stages;
        out_stages = want_out;
        while (smem_of(stages, out_stages) > budget && stages > (bcast ? 3u : 2u)) --stages;
        while (smem_of(stages, out_stages) > budget && out_stages > 1u) --out_stages;
        if (smem_of(stages, out_stages) <= budget) break;
        if (ctas == 1) return cudaErrorInvalidConfiguration;
        --ctas;
    }

    uint32_t threads;
    if (bcast) {
        threads = 64;
    } else {
        int CW;  // add warps: tile = V * 4 * CW * 32 elements with (V, CW) = (2,4) (4,4) (4,8) (8,8)
        switch (tile) {
            case 1024:
            case 2048: CW = 4; break;
            case 4096:
            case 8192: CW = 8; break;
            default: return cudaErrorInvalidValue;
        }
        threads = (uint32_t)(CW + 2) * 32u;
    }
    uint64_t grid = (uint64_t)sm_count * ctas;
    if (t.v[LP_TUNE_GRID_LIMIT] && grid > (uint64_t)t.v[LP_TUNE_GRID_LIMIT]) grid = (uint64_t)t.v[LP_TUNE_GRID_LIMIT];
    // a2: a claim is one slot's worth of granules (LP_TUNE_CLAIM_SLOTS: more, i.e. fewer atomics; measured slower at
    // 64 MB for every P but reduce at P = 2, profiles/r2_tuning.md); it shrinks to single granules as the list runs
    // out (LpTileClaimer)
    uint32_t claim_slots = t.v[LP_TUNE_CLAIM_SLOTS] ? (uint32_t)t.v[LP_TUNE_CLAIM_SLOTS] : 1u;
    while (claim_slots > 1u && n_slots < 4ull * grid * claim_slots) claim_slots /= 2u;
    a.claim_max = claim_slots * slot_gran;
    const uint64_t n_claims = (a.part.n_tiles + a.claim_max - 1) / a.claim_max;
    if (grid > n_claims) grid = n_claims;
    uint32_t shift = 0;  // claims of remaining / (2 * grid) granules: remaining >> floor(log2(2 * grid))
    while ((4ull << shift) <= 2ull * grid) ++shift;
    a.claim_shift = shift + 1u > 1u ? shift + 1u : 1u;
    a.prefetch = t.v[LP_TUNE_PREFETCH] == 2 ? 0 : 1;
    cfg->grid = (uint32_t)grid;
    cfg->threads = threads;
    cfg->smem_bytes = smem_of(stages, out_stages);
    cfg->stages = stages;
    cfg->out_stages = out_stages;
    cfg->pdl = t.v[LP_TUNE_NO_PDL] == 0;
    cfg->claim = a.claim_max;
    if (!cfg->pdl) a.prefetch = 0;
    if (dry_run || grid == 0) return cudaSuccess;

    lp_count_launch(1);
    if (a.sched && n_claims <= grid) a.sched = nullptr;  // one claim per CTA: nothing to balance, skip the counter
    {
        LpRange ranges[2 * LP_MAX_IN];
        const int nr = lp_args_ranges(a, ranges);
        a.late_wait = lp_chain_admit(stream, ranges, nr, cfg->pdl, t.v[LP_TUNE_CHAIN] != 2) ? 1 : 0;
        if (a.late_wait) a.prefetch = 0;
    }
    if (bcast) {
        if (segs) return launch_bcast_t<true>(a, *segs, *cfg, tile, stream);
        return launch_bcast_t<false>(a, LpNoSegs{0}, *cfg, tile, stream);
    }
    switch (tile) {
        case 1024: return launch_fold<2, 4>(a, segs, *cfg, stream);
        case 2048: return launch_fold<4, 4>(a, segs, *cfg, stream);
        case 4096: return launch_fold<4, 8>(a, segs, *cfg, stream);
        default: return launch_fold<8, 8>(a, segs, *cfg, stream);
    }
}
