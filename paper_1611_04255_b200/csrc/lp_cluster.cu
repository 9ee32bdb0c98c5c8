// lp_cluster.cu -- LP_VARIANT_CLUSTER: the paper's dataflow, stage per rank, inside a thread-block cluster.
//
// A cluster of C = P CTAs is the chain of Fig. 2: CTA r plays GPU r.  For every tile of the message
//
//   reduce half   CTA r loads ITS rank's tile from HBM (TMA bulk load, its "local block"), receives the
//                               running partial from CTA r-1 in a receive slot of its own shared memory ("writing
//                               block a0 to a buffer on GPU1"), adds, and writes the new partial into a receive slot
//                               of CTA r+1 through distributed shared memory (st.async: the store itself completes
//                               transaction bytes on CTA r+1's mbarrier, the block-ready flag).  The last CTA holds a''.
//   broadcast half  the finished tile flows back down the chain, CTA x -> CTA x-1 (U3 reading A,
//                               reverse flow); every CTA on the way stores it to its own rank's buffer (TMA bulk
//                               store) -- so each rank's HBM traffic is issued by "its" CTA, as on the real machine.
//
// reduce = reduce half, the last CTA stores to the root; allreduce / BSP-SGD = both halves (the SGD update is applied
// by the last CTA before the tile turns around); broadcast = the broadcast half alone, headed by the CTA that plays
// the root (chain position j = C-1-x plays rank (root + j) mod P).  Flow control is credit based: every slot a
// neighbour writes into has a "full" mbarrier in the receiver and a "credit" mbarrier in the sender, both signalled
// remotely.  The partial never touches HBM, as in the pipeline variant; the difference is WHERE the chain lives: P
// SMs and the SM-to-SM network instead of one CTA's ring.  P <= 16 (cluster size limit; > 8 is non-portable).
#include <cooperative_groups.h>
#include <string.h>

#include <atomic>

#include "lp_common.cuh"

namespace {

constexpr int kFoldWarps = 4;
constexpr int kRetWarps = 4;
constexpr int kClThreads = (2 + kFoldWarps + kRetWarps) * 32;  // producer, store, fold, return
// Tile = KV float4 per fold / return thread: KV = 2, 4, 8 -> 1024, 2048 (default), 4096 elements (LP_TUNE_CLUSTER_TILE).
// Ring depths are launch parameters: s_in local-block slots (LP_TUNE_STAGES, default 3), s_rv receive slots for
// partials and as many for finished tiles (LP_TUNE_OUT_STAGES, default 2).  2048 x (3 + 2 + 2) x 4 B = 56 KB: three
// CTAs per SM.

struct LpClusterArgs {
    const float *in_of[16];  // what cluster CTA x loads (NULL: nothing)
    float *out_of[16];       // where cluster CTA x stores the finished tile (NULL: nowhere)
    const float *w_root;     // SGD: weights[root], loaded by the last CTA
    const float *vel_in;     // SGD + momentum: the velocity, loaded by the last CTA
    uint64_t base;           // element offset of the message inside the rank vectors (slice of a layer-wise list)
    int C;
    int fold;      // reduce half active
    int ret;       // broadcast half active
    int head_tma;  // broadcast: the head's finished tile comes straight from HBM
    int s_in, s_rv, s_fin;
};

// ---- cluster-scope PTX ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cl_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cl_map(const void *local, uint32_t cta) {  // my smem address -> that CTA's
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(lp_smem_u32(local)), "r"(cta));
    return r;
}
// Signals between neighbours.  Data goes by st.async: a 16-byte store into the neighbour's shared memory that
// completes 16 transaction bytes on the neighbour's mbarrier -- the hardware's own "block ready" flag, no fences.
// Credits ("I am done reading your slot") are plain remote arrives.  Cluster-scope acquire / release on every wait
// and arrive would be correct too and was the first version: it compiles to MEMBAR.ALL.GPU + CCTL.IVALL per hop.
__device__ __forceinline__ void cl_arrive(uint64_t *bar, uint32_t cta) {  // arrive on `bar` of CTA `cta` (may be me)
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cl_map(bar, cta)) : "memory");
}
__device__ __forceinline__ void cl_store4_async(uint32_t remote, const float4 &v, uint32_t remote_bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(remote),
                 "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"(remote_bar)
                 : "memory");
}

struct ClRing {
    int slot;
    uint32_t phase;
    int depth;
    __device__ __forceinline__ ClRing(int d) : slot(0), phase(0), depth(d) {}
    __device__ __forceinline__ void advance() {
        if (++slot == depth) {
            slot = 0;
            phase ^= 1u;
        }
    }
};

template <int kV>
__global__ void __launch_bounds__(kClThreads)
    lp_cluster_kernel(const __grid_constant__ LpArgs a, const __grid_constant__ LpClusterArgs c) {
    constexpr int kClTile = kV * 4 * kFoldWarps * 32;
    const int kSIn = c.s_in, kSRv = c.s_rv, kSFin = c.s_fin;
    extern __shared__ __align__(128) unsigned char lp_smem[];
    float *in_ring = reinterpret_cast<float *>(lp_smem);   // my rank's tiles (and, on the last CTA, the weight tiles)
    float *rv_ring = in_ring + kSIn * kClTile;              // partials written by CTA x-1
    float *fin_ring = rv_ring + kSRv * kClTile;             // finished tiles: written by CTA x+1, or produced here (head)
    uint64_t *in_full = reinterpret_cast<uint64_t *>(fin_ring + kSFin * kClTile);
    uint64_t *in_empty = in_full + kSIn;
    uint64_t *rv_full = in_empty + kSIn;        // flag "partial has arrived", signalled by CTA x-1
    uint64_t *send_credit = rv_full + kSRv;     // "your slot in me is free again", signalled by CTA x+1
    uint64_t *fin_full = send_credit + kSRv;    // "finished tile has arrived", signalled by CTA x+1 (or by me, the head)
    uint64_t *dn_credit = fin_full + kSFin;     // credits for the finished-tile ring of CTA x-1, signalled by its consumers
    uint64_t *own_credit = dn_credit + kSFin;   // head only: credits for my own finished-tile ring

    const int C = c.C;
    const int x = (int)cl_rank();
    const bool head = x == C - 1;
    const bool stores_me = c.out_of[x] != nullptr;
    const bool fwd_me = c.ret && x > 0;
    auto consumers = [&](int y) { return (c.out_of[y] != nullptr ? 1 : 0) + ((c.ret && y > 0) ? kRetWarps : 0); };

    if (threadIdx.x == 0) {
        for (int s = 0; s < kSIn; ++s) {
            lp_mbar_init(&in_full[s], 1);
            lp_mbar_init(&in_empty[s], kFoldWarps);
        }
        for (int s = 0; s < kSRv; ++s) {
            lp_mbar_init(&rv_full[s], 1);  // my own arrive.expect_tx; the bytes come from CTA x-1's st.async
            lp_mbar_init(&send_credit[s], kFoldWarps);
        }
        const int dn = x > 0 ? consumers(x - 1) : 0, own = consumers(x);
        for (int s = 0; s < kSFin; ++s) {
            lp_mbar_init(&fin_full[s], head ? (c.head_tma ? 1 : kFoldWarps) : 1);
            lp_mbar_init(&dn_credit[s], dn > 0 ? dn : 1);
            lp_mbar_init(&own_credit[s], own > 0 ? own : 1);
        }
        lp_fence_mbar_init();
        // arm the rings my neighbours write into: one tile of transaction bytes per slot and phase
        if (c.fold && x > 0)
            for (int s = 0; s < kSRv; ++s) lp_mbar_expect_tx(&rv_full[s], kClTile * 4u);
        if (c.ret && !head)
            for (int s = 0; s < kSFin; ++s) lp_mbar_expect_tx(&fin_full[s], kClTile * 4u);
    }
    cooperative_groups::this_cluster().sync();  // every barrier of the cluster exists before anyone signals remotely

    const lp_partition &part = a.part;
    const uint64_t n_clusters = gridDim.x / (unsigned)C;
    const uint64_t cid = blockIdx.x / (unsigned)C;
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const bool mom = a.epilogue == LP_EPI_SGD_MOM;
    const bool sgd = a.epilogue == LP_EPI_SGD || mom;
    const int code = lp_fold_code(a.dtype, a.red_op);

    if (warp == 0) {
        // ---------------- producer: my rank's tiles from HBM ("local block") ------------------------------------
        if (lane == 0) {
            ClRing in(kSIn), fin(kSFin);
            for (uint64_t t = cid; t < part.n_tiles; t += n_clusters) {
                uint64_t off;
                uint32_t len;
                lp_tile_range(part, t, off, len);
                off += c.base;
                const LpTileSpan span(off, len);
                const uint32_t bytes = span.body * 4u;
                if (c.fold) {
                    const int loads = (head && sgd) ? (mom ? 3 : 2) : 1;
                    for (int k = 0; k < loads; ++k) {
                        const float *src = k == 0 ? c.in_of[x] : (k == 1 ? c.w_root : c.vel_in);
                        lp_mbar_wait(&in_empty[in.slot], in.phase ^ 1u);
                        if (bytes) {
                            lp_mbar_expect_tx(&in_full[in.slot], bytes);
                            lp_bulk_g2s(in_ring + in.slot * kClTile, src + span.a0, bytes, &in_full[in.slot]);
                        } else {
                            lp_mbar_arrive(&in_full[in.slot]);
                        }
                        in.advance();
                    }
                } else if (head) {  // broadcast: the root's tile is the finished tile
                    lp_mbar_wait(&own_credit[fin.slot], fin.phase ^ 1u);
                    if (bytes) {
                        lp_mbar_expect_tx(&fin_full[fin.slot], bytes);
                        lp_bulk_g2s(fin_ring + fin.slot * kClTile, c.in_of[x] + span.a0, bytes, &fin_full[fin.slot]);
                    } else {
                        lp_mbar_arrive(&fin_full[fin.slot]);
                    }
                    fin.advance();
                    for (uint32_t e = 0; e < span.head; ++e) lp_scalar_element(a, off + e);
                    for (uint32_t e = 0; e < span.tail; ++e) lp_scalar_element(a, span.a0 + span.body + e);
                }
            }
        }
    } else if (warp == 1) {
        // ---------------- store thread: the finished tile to MY rank's buffer ------------------------------------
        if (lane == 0 && stores_me) {
            ClRing fin(kSFin);
            for (uint64_t t = cid; t < part.n_tiles; t += n_clusters) {
                uint64_t off;
                uint32_t len;
                lp_tile_range(part, t, off, len);
                off += c.base;
                const LpTileSpan span(off, len);
                lp_mbar_wait(&fin_full[fin.slot], fin.phase);
                lp_fence_proxy_async();
                if (span.body) lp_bulk_s2g(c.out_of[x] + span.a0, fin_ring + fin.slot * kClTile, span.body * 4u);
                lp_bulk_commit();
                lp_bulk_wait_read<0>();
                if (!head && !fwd_me) lp_mbar_expect_tx(&fin_full[fin.slot], kClTile * 4u);  // CTA 0: nobody else re-arms
                if (head)
                    lp_mbar_arrive(&own_credit[fin.slot]);
                else
                    cl_arrive(&dn_credit[fin.slot], (uint32_t)x + 1u);
                fin.advance();
            }
            lp_bulk_wait<0>();
        }
    } else if (warp < 2 + kFoldWarps) {
        // ---------------- fold warps: partial <- partial + local block, hand it to CTA x+1 -----------------------
        if (c.fold) {
            const int ftid = threadIdx.x - 64;
            constexpr int FT = kFoldWarps * 32;
            ClRing in(kSIn), rv(kSRv), snd(kSRv), fin(kSFin);
            for (uint64_t t = cid; t < part.n_tiles; t += n_clusters) {
                uint64_t off;
                uint32_t len;
                lp_tile_range(part, t, off, len);
                off += c.base;
                float4 acc[kV];
                lp_mbar_wait(&in_full[in.slot], in.phase);
                // A slot is handed back only after the shared-memory reads of it have RETURNED: this SM's load/store
                // queue is busy with the neighbours' st.async traffic, and an mbarrier arrive does not wait for loads
                // that are still queued (without this the refill of a slot overtook them: "rank r's term taken from
                // the tile kSIn rounds ahead" in ~1 of 10 runs at P >= 3).  So every arrive that releases a slot comes
                // after the instruction that consumes the loaded values (the add, the st.async) AND a CTA-scope fence
                // (the fence costs nothing measurable here; the instruction order alone is at the scheduler's mercy).
                const float4 *mine = reinterpret_cast<const float4 *>(in_ring + in.slot * kClTile);
                if (x > 0) {  // a' = (what GPU x-1 sent) + my block, in that order (chain order)
                    lp_mbar_wait(&rv_full[rv.slot], rv.phase);
                    const float4 *s = reinterpret_cast<const float4 *>(rv_ring + rv.slot * kClTile);
                    float4 loc[kV];
#pragma unroll
                    for (int v = 0; v < kV; ++v) {
                        acc[v] = s[ftid + v * FT];
                        loc[v] = mine[ftid + v * FT];
                    }
                    lp_fold_vecs<kV>(acc, loc, kV, code);  // the operator switch sits outside the vector loop
                    __threadfence_block();
                    __syncwarp();
                    if (lane == 0) lp_mbar_arrive(&in_empty[in.slot]);
                    if (ftid == 0) lp_mbar_expect_tx(&rv_full[rv.slot], kClTile * 4u);  // re-arm for the slot's next use
                    if (lane == 0) cl_arrive(&send_credit[rv.slot], (uint32_t)x - 1u);
                    rv.advance();
                } else {
#pragma unroll
                    for (int v = 0; v < kV; ++v) acc[v] = mine[ftid + v * FT];
                    if (head) {  // a cluster of one (P = 1): nothing consumes the loads before the slot goes back
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) lp_mbar_arrive(&in_empty[in.slot]);
                    }
                }
                const int my_in_slot = in.slot;
                in.advance();
                if (!head) {
                    lp_mbar_wait(&send_credit[snd.slot], snd.phase ^ 1u);
                    const uint32_t dst = cl_map(rv_ring + snd.slot * kClTile, (uint32_t)x + 1u);
                    const uint32_t flag = cl_map(&rv_full[snd.slot], (uint32_t)x + 1u);
#pragma unroll
                    for (int v = 0; v < kV; ++v) cl_store4_async(dst + (uint32_t)(ftid + v * FT) * 16u, acc[v], flag);
                    if (x == 0) {  // rank 0's tile went out as it was: the stores above consumed the loads
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) lp_mbar_arrive(&in_empty[my_in_slot]);
                    }
                    snd.advance();
                } else {
                    if (sgd && !mom) {  // g = S/P, w' = w_root - lr g, applied where the chain ends
                        lp_mbar_wait(&in_full[in.slot], in.phase);
                        const float4 *s = reinterpret_cast<const float4 *>(in_ring + in.slot * kClTile);
#pragma unroll
                        for (int v = 0; v < kV; ++v) acc[v] = lp_sgd4(acc[v], s[ftid + v * FT], a.lr, a.invP);
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) lp_mbar_arrive(&in_empty[in.slot]);
                        in.advance();
                    }
                    if (mom) {  // v' = mu v + lr g, w' = w_root - v' (U18); v' goes straight to the velocity vector
                        float4 w[kV];
                        lp_mbar_wait(&in_full[in.slot], in.phase);
                        {
                            const float4 *s = reinterpret_cast<const float4 *>(in_ring + in.slot * kClTile);
#pragma unroll
                            for (int v = 0; v < kV; ++v) w[v] = s[ftid + v * FT];
                        }
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) lp_mbar_arrive(&in_empty[in.slot]);
                        in.advance();
                        lp_mbar_wait(&in_full[in.slot], in.phase);
                        const LpTileSpan vspan(off, len);
                        {
                            const float4 *s = reinterpret_cast<const float4 *>(in_ring + in.slot * kClTile);
#pragma unroll
                            for (int v = 0; v < kV; ++v) {
                                float4 vel;
                                lp_mom4(acc[v], w[v], s[ftid + v * FT], a.lr, a.invP, a.mu, vel, acc[v]);
                                const uint32_t e = (uint32_t)(ftid + v * FT) * 4u;
                                if (e < vspan.body) lp_stg_stream(a.vel_out + vspan.a0 + e, vel);
                            }
                        }
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) lp_mbar_arrive(&in_empty[in.slot]);
                        in.advance();
                    }
                    lp_mbar_wait(&own_credit[fin.slot], fin.phase ^ 1u);
                    float4 *o = reinterpret_cast<float4 *>(fin_ring + fin.slot * kClTile);
#pragma unroll
                    for (int v = 0; v < kV; ++v) o[ftid + v * FT] = acc[v];
                    lp_fence_proxy_async();
                    __syncwarp();
                    if (lane == 0) lp_mbar_arrive(&fin_full[fin.slot]);
                    fin.advance();
                    const LpTileSpan span(off, len);
                    if ((uint32_t)ftid < span.head) lp_scalar_element(a, off + ftid);
                    if ((uint32_t)ftid >= 32u && (uint32_t)ftid - 32u < span.tail)
                        lp_scalar_element(a, span.a0 + span.body + (ftid - 32));
                }
            }
        }
    } else {
        // ---------------- return warps: the finished tile on to CTA x-1 (broadcast half) -------------------------
        if (fwd_me) {
            const int rtid = threadIdx.x - (2 + kFoldWarps) * 32;
            constexpr int RT = kRetWarps * 32;
            ClRing fin(kSFin), dn(kSFin);
            for (uint64_t t = cid; t < part.n_tiles; t += n_clusters) {
                float4 r4[kV];
                lp_mbar_wait(&fin_full[fin.slot], fin.phase);
                lp_mbar_wait(&dn_credit[dn.slot], dn.phase ^ 1u);
                {
                    const float4 *s = reinterpret_cast<const float4 *>(fin_ring + fin.slot * kClTile);
#pragma unroll
                    for (int v = 0; v < kV; ++v) r4[v] = s[rtid + v * RT];
                }
                const uint32_t dst = cl_map(fin_ring + dn.slot * kClTile, (uint32_t)x - 1u);
                const uint32_t flag = cl_map(&fin_full[dn.slot], (uint32_t)x - 1u);
#pragma unroll
                for (int v = 0; v < kV; ++v) cl_store4_async(dst + (uint32_t)(rtid + v * RT) * 16u, r4[v], flag);
                __threadfence_block();
                __syncwarp();  // the stores consumed the loads: my slot may go back (see the fold warps)
                if (!head && rtid == 0) lp_mbar_expect_tx(&fin_full[fin.slot], kClTile * 4u);  // re-arm (I am the one who does)
                if (lane == 0) {
                    if (head)
                        lp_mbar_arrive(&own_credit[fin.slot]);
                    else
                        cl_arrive(&dn_credit[fin.slot], (uint32_t)x + 1u);
                }
                fin.advance();
                dn.advance();
            }
        }
    }
    cooperative_groups::this_cluster().sync();  // nobody leaves while a neighbour may still write into it
}

uint32_t cl_smem(uint32_t tile, int s_in, int s_rv, int s_fin) {
    return (uint32_t)(s_in + s_rv + s_fin) * tile * 4u + (2u * s_in + 2u * s_rv + 3u * s_fin) * 8u;
}

// per kernel instantiation and device binding (lp_attr_epoch): dynamic shared memory limit + non-portable cluster size
struct ClAttrCache {
    std::atomic<int> bytes{0};
    std::atomic<unsigned> epoch{0};
};

template <int KV>
cudaError_t cl_set_attrs(uint32_t smem) {
    static ClAttrCache cache;
    if (cache.epoch.load() == lp_attr_epoch() && (int)smem <= cache.bytes.load()) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(lp_cluster_kernel<KV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(lp_cluster_kernel<KV>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
    cache.epoch.store(lp_attr_epoch());
    cache.bytes.store((int)smem);
    return cudaSuccess;
}

template <int KV>
cudaError_t cl_launch_t(const LpArgs &a, const LpClusterArgs &c, int P, const LpTuning &t, LpLaunch *cfg, cudaStream_t stream) {
    cudaError_t e = cl_set_attrs<KV>(cfg->smem_bytes);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof(lc));
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)P;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    lc.gridDim = dim3((unsigned)P, 1, 1);
    lc.blockDim = dim3(kClThreads, 1, 1);
    lc.dynamicSmemBytes = cfg->smem_bytes;
    lc.stream = stream;
    lc.attrs = attr;
    lc.numAttrs = 1;
    int max_clusters = 0;
    e = cudaOccupancyMaxActiveClusters(&max_clusters, lp_cluster_kernel<KV>, &lc);
    if (e != cudaSuccess) return e;
    if (max_clusters <= 0) return cudaErrorNotSupported;  // a cluster of P CTAs does not fit this device
    uint64_t clusters = (uint64_t)max_clusters;
    if (t.v[LP_TUNE_GRID_LIMIT] && clusters > (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P)
        clusters = (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P ? (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P : 1;
    if (clusters > a.part.n_tiles) clusters = a.part.n_tiles;
    cfg->grid = (uint32_t)(clusters * P);
    lc.gridDim = dim3(cfg->grid, 1, 1);
    lp_count_launch(1);
    return cudaLaunchKernelEx(&lc, lp_cluster_kernel<KV>, a, c);
}

}  // namespace

uint32_t lp_cluster_tile(const LpTuning &t) { return t.v[LP_TUNE_CLUSTER_TILE] ? (uint32_t)t.v[LP_TUNE_CLUSTER_TILE] : 2048u; }

// `root` is needed for the broadcast chain (position j plays rank (root + j) mod P); P = number of virtual ranks.
cudaError_t lp_cluster_launch(const LpArgs &a, int P, int root, uint64_t base_off, const LpTuning &t, int sm_count,
                              LpLaunch *cfg, bool dry_run, cudaStream_t stream) {
    cfg->grid = cfg->threads = cfg->smem_bytes = cfg->stages = cfg->out_stages = 0;
    cfg->pdl = false;
    cfg->claim = 1;
    const bool bcast = a.epilogue == LP_EPI_COPY;
    if (P > 16) return cudaErrorNotSupported;
    LpClusterArgs c;
    memset(&c, 0, sizeof(c));
    c.C = P;
    c.base = base_off;
    c.fold = bcast ? 0 : 1;
    c.ret = (bcast || a.n_out > 1) ? 1 : 0;  // allreduce / SGD / broadcast send the finished tile back down the chain
    c.head_tma = bcast ? 1 : 0;
    const uint32_t tile = a.part.tile;
    // defaults: 3 + 2 + 2 slots of 8 KB = 56 KB, three CTAs per SM (registers).  Deeper rings or larger tiles buy nothing:
    // 4.0-4.4 TB/s for every tile (4 / 8 / 16 KB) and ring depth tried (profiles/r2_cluster.md) -- the variant is bound
    // by what an SM can push into its neighbour's shared memory, not by the latency of a hop
    c.s_in = t.v[LP_TUNE_STAGES] ? t.v[LP_TUNE_STAGES] : 3;
    c.s_rv = c.s_fin = t.v[LP_TUNE_OUT_STAGES] ? t.v[LP_TUNE_OUT_STAGES] : 2;
    if (c.s_in < 3) c.s_in = 3;  // the head of a momentum step has three loads per tile
    if (c.s_rv < 2) c.s_rv = c.s_fin = 2;
    while (cl_smem(tile, c.s_in, c.s_rv, c.s_fin) > 227u * 1024u && c.s_in > 3) --c.s_in;
    while (cl_smem(tile, c.s_in, c.s_rv, c.s_fin) > 227u * 1024u && c.s_rv > 2) c.s_fin = --c.s_rv;
    if (cl_smem(tile, c.s_in, c.s_rv, c.s_fin) > 227u * 1024u) return cudaErrorInvalidConfiguration;
    if (!dry_run) {
        if (bcast) {  // CTA x is chain position j = C-1-x and plays rank (root + j) mod P; the head plays the root
            const float *src = a.in[0];
            for (int x = 0; x < P; ++x) {
                const int j = P - 1 - x;
                c.in_of[x] = j == 0 ? src : nullptr;
                c.out_of[x] = nullptr;
            }
            // a.out lists the P-1 non-root ranks in rank order: rank r != root sits at index r - (r > root)
            for (int j = 1; j < P; ++j) {
                const int r = (root + j) % P;
                c.out_of[P - 1 - j] = a.out[r - (r > root ? 1 : 0)];
            }
        } else {
            for (int x = 0; x < P; ++x) {
                c.in_of[x] = a.in[x];
                c.out_of[x] = a.n_out > 1 ? a.out[x] : (x == P - 1 ? a.out[0] : nullptr);
            }
            const bool sgd = a.epilogue == LP_EPI_SGD || a.epilogue == LP_EPI_SGD_MOM;
            c.w_root = sgd ? a.in[a.n_sum] : nullptr;
            c.vel_in = a.epilogue == LP_EPI_SGD_MOM ? a.in[a.n_sum + 1] : nullptr;
        }
    }
    cfg->threads = kClThreads;
    cfg->smem_bytes = cl_smem(tile, c.s_in, c.s_rv, c.s_fin);
    cfg->stages = (uint32_t)c.s_in;
    cfg->out_stages = (uint32_t)c.s_fin;
    uint64_t clusters = (uint64_t)(sm_count / P) * (228u * 1024u / (cfg->smem_bytes + 1024u));  // planning figure; the launch asks the occupancy calculator
    if (t.v[LP_TUNE_GRID_LIMIT] && clusters > (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P)
        clusters = (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P ? (uint64_t)t.v[LP_TUNE_GRID_LIMIT] / P : 1;
    if (clusters > a.part.n_tiles) clusters = a.part.n_tiles;
    cfg->grid = (uint32_t)(clusters * P);
    if (dry_run || a.part.n_tiles == 0) return cudaSuccess;
    switch (tile) {
        case 1024: return cl_launch_t<2>(a, c, P, t, cfg, stream);
        case 2048: return cl_launch_t<4>(a, c, P, t, cfg, stream);
        case 4096: return cl_launch_t<8>(a, c, P, t, cfg, stream);
        default: return cudaErrorInvalidValue;
    }
}
