// lp_chain.cu -- the paper's own setting: ONE RANK PER GPU, the chain GPU r -> r+1 over peer memory (NVLink 5 /
// NVSwitch P2P), SURVEY 8(e) / 8(f)-4.  PAPER.md:55-59 (Sec. 3, Fig. 2): every GPU "receives a block from the prior
// GPU ... while sending a block to the next one"; reduce: "GPU1 reduces the received block a0 with a1 to yield a'",
// which travels on; allreduce sends the finished block back (U3 reading A, reverse flow).
//
// Each rank owns an ENDPOINT in its own HBM (one allocation, exported to its two neighbours): per channel a forward
// receive ring (partials / broadcast blocks from rank r-1) and a backward receive ring (finished blocks from rank r+1)
// of S slots of one tile, plus four monotonic 64-bit counters.  A transfer is a PUSH: the sender's SMs store the tile
// into the receiver's ring through the peer mapping (stores are fire-and-forget over NVLink; loads would pay the
// ~1 us round trip per tile), then one thread publishes it -- barrier, fence.acq_rel.sys, st.relaxed.sys of the ring's
// tail counter in the RECEIVER's memory, which the receiver polls locally.  A slot goes back by a credit counter in
// the SENDER's memory, written remotely by the receiver after it has consumed the slot's values.  Counters only ever
// grow (slot = sequence mod S), so nothing is reset between calls and a rank may run ahead of its neighbours into the
// next collective; the neighbours of a ring never change: rank r's forward ring is written by rank (r-1) mod P, its
// backward ring by rank r+1 (broadcast runs root -> root+1 -> ... around the ring in the forward direction,
// PAPER.md:77 "data always flow in one direction").
//
// The rank's kernel is 2 C CTAs: C forward CTAs (channel c takes tiles c, c + C, ...: load my block, wait for the
// partial, combine in chain order, push up; the last rank stores / turns the finished tile around) and C return CTAs
// (wait for a finished tile, store it to my vector, push it further down).  No CTA of a rank waits for another CTA of
// the same rank; a channel advances whenever its CTAs are resident on every rank, and the grid never exceeds what
// the device holds at once.  Two realisations of a rank's CTAs follow, same protocol between ranks: the register kernel
// (lp_chain_kernel: 1024 threads load, fold and store in lock-step) and, the default, the TMA-load kernel
// (lp_chain_tma_kernel: everything a rank reads is local, so a producer thread streams it through a shared-memory ring).
// Host side (endpoints, roles, launches, emulation entry points): lp_chain_api.cu.
//
// ONE GPU (this build's box): kernels that wait on each other must not run as separate launches on one device, so
// lp_chain_emulate runs the SAME per-rank code for all P ranks inside ONE cooperative launch (P x 2 C co-resident
// CTAs), every "peer" pointer then being a local one.  That is what tests/ compare with the oracle bit for bit; the
// multi-process plumbing (roles, handle exchange) is covered on the CPU.  Values: the chain order rank 0 -> P-1 (U4),
// one RN operation per combine -- the same definition as every other LP variant.
#include <cooperative_groups.h>
#include <string.h>

#include <atomic>

#include "lp_chain.cuh"

namespace {

__device__ __forceinline__ unsigned long long ld_sys(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_sys(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void fence_sys() { asm volatile("fence.acq_rel.sys;" ::: "memory"); }
// ring data is written by another GPU (or another SM): never from L1
__device__ __forceinline__ float4 ld_ring(const float *p) {
    float4 v;
    asm volatile("ld.volatile.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ float ld_ring1(const float *p) {
    float v;
    asm volatile("ld.volatile.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}

// Thread 0 polls up to three counters until each has reached its target (want == 0: nothing to wait for), then
// everybody passes the barrier.  ONE acquire fence after the polls: it is what makes the data that was published
// before the tail counter visible to the ring loads behind the barrier; the credit counters need none of their own
// (what follows them are stores into the freed slot, and a store is never performed ahead of the load it depends on).
// Returns false (for every thread) when a poll gave up or another CTA of this rank already failed.
__device__ __forceinline__ bool wait_counters(const unsigned long long *f0, unsigned long long w0, const unsigned long long *f1,
                                              unsigned long long w1, const unsigned long long *f2, unsigned long long w2,
                                              int *error, int *s_ok, unsigned long long spin_limit) {
    if (threadIdx.x == 0) {
        int ok = 1;
        const unsigned long long *f[3] = {f0, f1, f2};
        const unsigned long long w[3] = {w0, w1, w2};
        for (int i = 0; i < 3 && ok; ++i) {
            if (w[i] == 0) continue;
            unsigned long long spins = 0;
            while (ld_sys(f[i]) < w[i]) {
                if (++spins > spin_limit || ((spins & 0xfffu) == 0 && *reinterpret_cast<volatile int *>(error) != 0)) {
                    ok = 0;
                    atomicCAS(error, 0, 1);
                    break;
                }
            }
        }
        if (w0) fence_sys();  // f0 is the tail counter of a receive ring
        *s_ok = ok;
    }
    __syncthreads();
    const bool ok = *s_ok != 0;
    __syncthreads();  // s_ok may be rewritten by the next wait
    return ok;
}

// After every thread's stores into the neighbour's ring: publish the new sequence number in the neighbour's memory.
__device__ __forceinline__ void publish(unsigned long long *remote_flag, unsigned long long seq) {
    __syncthreads();
    if (threadIdx.x == 0) {
        fence_sys();  // release, cumulative over the barrier: the tile is visible before the counter
        st_sys(remote_flag, seq);
    }
}
// After every thread has CONSUMED the values it loaded from a slot (they went into an add or a store): credit.
__device__ __forceinline__ void credit(unsigned long long *remote_flag, unsigned long long seq) {
    __syncthreads();
    if (threadIdx.x == 0) st_sys(remote_flag, seq);
}

// A slot (one tile of L.tile elements: the unit of a flag exchange) is worked through in STEPS of kStep elements, kV
// 16-byte vectors per thread: between two flag exchanges nothing synchronises, so the loads of one step overlap the
// stores of the step before.  `nfull` whole vectors, then `rem` (< 4) single elements (the message's last tile only:
// every tile starts on a 16-byte boundary because the chain rounds blocks up to a multiple of 4 elements).
constexpr int kV = 4;
#define kStep ((uint32_t)(kV * 4) * blockDim.x)  // 16384 elements = 64 KB with 1024 threads
struct StepRegs {
    float4 v[kV];
};

__device__ __forceinline__ void load_step(StepRegs &t, const float *src, uint32_t len, bool ring) {
    const uint32_t nfull = len >> 2, rem = len & 3u;
#pragma unroll
    for (int k = 0; k < kV; ++k) {
        const uint32_t j = threadIdx.x + (uint32_t)k * blockDim.x;
        if (j < nfull) {
            t.v[k] = ring ? ld_ring(src + 4 * j) : lp_ldg_stream(src + 4 * j);
        } else if (j == nfull && rem) {
            float e[3] = {0.f, 0.f, 0.f};
            for (uint32_t q = 0; q < rem; ++q) e[q] = ring ? ld_ring1(src + 4 * j + q) : src[4 * j + q];
            t.v[k] = make_float4(e[0], e[1], e[2], 0.f);
        }
    }
}

__device__ __forceinline__ void store_step(const StepRegs &t, float *dst, uint32_t len) {
    const uint32_t nfull = len >> 2, rem = len & 3u;
#pragma unroll
    for (int k = 0; k < kV; ++k) {
        const uint32_t j = threadIdx.x + (uint32_t)k * blockDim.x;
        if (j < nfull) {
            lp_stg_stream(dst + 4 * j, t.v[k]);
        } else if (j == nfull && rem) {
            const float e[3] = {t.v[k].x, t.v[k].y, t.v[k].z};
            for (uint32_t q = 0; q < rem; ++q) dst[4 * j + q] = e[q];
        }
    }
}

__device__ __forceinline__ unsigned long long slot_free_at(unsigned long long sent, int S) {
    return sent + 1 > (unsigned)S ? sent + 1 - (unsigned)S : 0;  // send number sent + 1 reuses the slot of send sent + 1 - S
}

// Forward CTA of channel c: the reduce half of Fig. 2b (and the whole of a broadcast, Fig. 2a).
__device__ void chain_forward(const LpChainRank &A, const LpChainLaunch &L, int c, int *s_ok) {
    unsigned long long *st = A.state + (size_t)c * 4;
    unsigned long long recv = st[ST_RECV_FWD], sent_up = st[ST_SENT_UP], sent_down = st[ST_SENT_DOWN];
    unsigned long long *my = A.flags + (size_t)c * kFlagsPerChannel;
    unsigned long long *up = A.up_flags + (size_t)c * kFlagsPerChannel;
    unsigned long long *down = A.down_flags + (size_t)c * kFlagsPerChannel;
    const size_t ring_c = (size_t)c * L.S * L.tile;
    __syncthreads();  // everybody has read the sequence numbers before thread 0 may write them back
    bool ok = true;
    for (uint64_t t = (uint64_t)c; ok && t < L.part.n_tiles; t += (uint64_t)L.C) {
        uint64_t off;
        uint32_t len;
        lp_tile_range(L.part, t, off, len);
        // every flag this tile needs, then the tile itself without a single barrier
        ok = wait_counters(my + F_FWD_TAIL, A.f_recv ? recv + 1 : 0, my + F_UP_CREDIT,
                           A.f_send_up ? slot_free_at(sent_up, L.S) : 0, my + F_DOWN_CREDIT,
                           A.f_send_down ? slot_free_at(sent_down, L.S) : 0, A.error, s_ok, L.spin_limit);
        if (!ok) break;
        const float *in_slot = A.fwd_ring + ring_c + (size_t)(recv % (unsigned)L.S) * L.tile;
        float *up_slot = A.up_fwd_ring + ring_c + (size_t)(sent_up % (unsigned)L.S) * L.tile;
        float *down_slot = A.down_bwd_ring + ring_c + (size_t)(sent_down % (unsigned)L.S) * L.tile;
        for (uint32_t s0 = 0; s0 < len; s0 += kStep) {
            const uint32_t sl = len - s0 < kStep ? len - s0 : kStep;
            StepRegs acc, mine;
            if (A.f_load) load_step(A.f_recv ? mine : acc, A.buf + off + s0, sl, false);
            if (A.f_recv) {  // "GPU1 reduces the received block a0 with a1 to yield a'": partial op mine, in that order
                load_step(acc, in_slot + s0, sl, true);
                if (A.f_load) lp_fold_vecs<kV>(acc.v, mine.v, kV, L.code);
            }
            if (A.f_update) {  // Alg. 3's update where the global gradient S is complete: three RN operations
                StepRegs w;
                load_step(w, A.w_in + off + s0, sl, false);
                if (A.vel) {  // five with momentum; the velocity lives where the update is computed (U18)
                    StepRegs v;
                    load_step(v, A.vel + off + s0, sl, false);
#pragma unroll
                    for (int k = 0; k < kV; ++k) lp_mom4(acc.v[k], w.v[k], v.v[k], L.lr, L.invP, L.mu, v.v[k], acc.v[k]);
                    store_step(v, A.vel + off + s0, sl);
                } else {
#pragma unroll
                    for (int k = 0; k < kV; ++k) acc.v[k] = lp_sgd4(acc.v[k], w.v[k], L.lr, L.invP);
                }
            }
            if (A.f_send_up) store_step(acc, up_slot + s0, sl);
            if (A.f_store) store_step(acc, A.out + off + s0, sl);
            if (A.f_send_down) store_step(acc, down_slot + s0, sl);  // the chain's end: the tile turns around
        }
        if (A.f_send_up) publish(up + F_FWD_TAIL, ++sent_up);
        if (A.f_send_down) publish(down + F_BWD_TAIL, ++sent_down);
        // the slot's values have been consumed by the stores / the fold above: hand it back to rank r-1
        if (A.f_recv) credit(down + F_UP_CREDIT, ++recv);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st[ST_RECV_FWD] = recv;
        st[ST_SENT_UP] = sent_up;
        if (A.f_send_down) st[ST_SENT_DOWN] = sent_down;
    }
}

// Return CTA of channel c: the broadcast half of allreduce (and the way a reduced tile reaches a root that is not
// the chain's end): finished tiles flow rank r+1 -> r.
__device__ void chain_return(const LpChainRank &A, const LpChainLaunch &L, int c, int *s_ok) {
    unsigned long long *st = A.state + (size_t)c * 4;
    unsigned long long recv = st[ST_RECV_BWD], sent_down = st[ST_SENT_DOWN];
    unsigned long long *my = A.flags + (size_t)c * kFlagsPerChannel;
    unsigned long long *up = A.up_flags + (size_t)c * kFlagsPerChannel;
    unsigned long long *down = A.down_flags + (size_t)c * kFlagsPerChannel;
    const size_t ring_c = (size_t)c * L.S * L.tile;
    __syncthreads();
    bool ok = true;
    for (uint64_t t = (uint64_t)c; ok && t < L.part.n_tiles; t += (uint64_t)L.C) {
        uint64_t off;
        uint32_t len;
        lp_tile_range(L.part, t, off, len);
        ok = wait_counters(my + F_BWD_TAIL, recv + 1, my + F_DOWN_CREDIT, A.r_send_down ? slot_free_at(sent_down, L.S) : 0,
                           nullptr, 0, A.error, s_ok, L.spin_limit);
        if (!ok) break;
        const float *in_slot = A.bwd_ring + ring_c + (size_t)(recv % (unsigned)L.S) * L.tile;
        float *down_slot = A.down_bwd_ring + ring_c + (size_t)(sent_down % (unsigned)L.S) * L.tile;
        for (uint32_t s0 = 0; s0 < len; s0 += kStep) {
            const uint32_t sl = len - s0 < kStep ? len - s0 : kStep;
            StepRegs fin;
            load_step(fin, in_slot + s0, sl, true);
            if (A.r_store) store_step(fin, A.out + off + s0, sl);
            if (A.r_send_down) store_step(fin, down_slot + s0, sl);
        }
        if (A.r_send_down) publish(down + F_BWD_TAIL, ++sent_down);
        credit(up + F_DOWN_CREDIT, ++recv);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st[ST_RECV_BWD] = recv;
        if (A.r_send_down) st[ST_SENT_DOWN] = sent_down;
    }
}

// grid = n_local x 2 C: CTA b plays local rank b / (2 C); of a rank's 2 C CTAs the first C are forward, the rest return.
// Fail fast: after a wait gave up (the endpoint's sticky error word) the counters of the rings no longer match the
// sequence numbers the host keeps, so a later collective could be satisfied by stale flags and deliver old slots.  Every
// CTA checks the word on entry -- one thread reads it, all take the same decision -- and does nothing once it is set; the
// endpoint has to be destroyed and created again on all ranks.
__device__ __forceinline__ bool chain_endpoint_dead(const int *error) {
    __shared__ int s_dead;
    if (threadIdx.x == 0) s_dead = *reinterpret_cast<const volatile int *>(error);
    __syncthreads();
    return s_dead != 0;
}

__global__ void __launch_bounds__(kChainThreads, 1) lp_chain_kernel(const __grid_constant__ LpChainLaunch L) {
    __shared__ int s_ok;
    const int per_rank = 2 * L.C;
    const int lr = (int)blockIdx.x / per_rank;
    const int j = (int)blockIdx.x - lr * per_rank;
    const LpChainRank &A = L.rank[lr];
    if (chain_endpoint_dead(A.error)) return;
    if (j < L.C) {
        if (A.f_active) chain_forward(A, L, j, &s_ok);
    } else {
        if (A.r_active) chain_return(A, L, j - L.C, &s_ok);
    }
}

// ---- the same roles with TMA on the load side (the default kernel) ---------------------------------------------------
// Everything a rank READS is local -- its vector, its weight replica, its receive rings -- so the load side can be the
// TMA pipeline of lp_pipeline.cu: a producer thread waits for the ring's tail counter, then issues cp.async.bulk loads
// of the tile, step by step, into a deep shared-memory ring (192 KB in flight per CTA; mbarrier full / empty flags),
// running several steps and, across tiles, several flags ahead of the consumers.  What a rank WRITES to a neighbour
// stays plain 128-bit stores (generic proxy, fire-and-forget over NVLink) published with fence.acq_rel.sys + the
// tail counter, exactly as in the register kernel above: the protocol between ranks is unchanged, only the inside
// of a CTA is.  One CTA: 1 producer warp + 16 consumer warps (8 consumer warps: 16 % slower; measured in the one-GPU
// emulation, 64 MB allreduce over 2 ranks x 32 channels: 496 GB/s per emulated link direction against 302 for the
// register kernel, profiles/r2_dtypes_chain.md).
constexpr int kTmaConsumers = 512;
constexpr int kTmaThreads = 32 + kTmaConsumers;
constexpr int kTmaVec = 2;                                               // 16-byte vectors per consumer thread and step
constexpr uint32_t kTmaStep = kTmaVec * 4 * kTmaConsumers;               // 4096 elements = 16 KB per source
constexpr uint32_t kTmaRingBytes = 192u * 1024u;
constexpr int kTmaMaxStages = 12;

// What one CTA does with every tile of its channel: up to three local sources, folded in this order, to up to three
// destinations.
struct ChainStream {
    const float *src_ring;               // my receive ring of this channel (partial / finished block), or NULL
    const unsigned long long *src_tail;  // its tail counter (my memory)
    unsigned long long *src_credit;      // where its slots are handed back (the sender's memory)
    int st_recv;
    const float *src_local;              // my vector, or NULL
    const float *src_w;                  // SGD step at the chain's end: my weight replica, or NULL
    float *vel;                          // ... with momentum: the velocity (a fourth source, rewritten in place), or NULL
    float *dst_local;                    // where the finished block is stored, or NULL
    float *dst_ring[2];                  // a neighbour's ring of this channel, or NULL
    unsigned long long *dst_tail[2];     // its tail counter (the neighbour's memory)
    const unsigned long long *dst_credit[2];  // my credit counter for it (my memory)
    int st_sent[2];
};

__device__ __forceinline__ bool mbar_try(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(lp_smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// mbarrier wait that gives up when the CTA has been aborted (a counter poll ran into its limit)
__device__ __forceinline__ bool mbar_wait_abortable(uint64_t *bar, uint32_t parity, volatile int *abort_flag) {
    while (!mbar_try(bar, parity))
        if (*abort_flag) return false;
    return true;
}
__device__ __forceinline__ bool poll_counter(const unsigned long long *flag, unsigned long long want, int *error,
                                             volatile int *abort_flag, unsigned long long spin_limit) {
    unsigned long long spins = 0;
    while (ld_sys(flag) < want) {
        if (++spins > spin_limit || ((spins & 0xffu) == 0 && (*abort_flag || *reinterpret_cast<volatile int *>(error) != 0))) {
            atomicCAS(error, 0, 1);
            *abort_flag = 1;
            return false;
        }
    }
    return true;
}
__device__ __forceinline__ void consumer_barrier() { asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory"); }
// barrier over the consumer warps that also tells every one of them whether ANY of them passed `pred` (a uniform
// decision: a thread that gave up mid-tile and one that did not must leave the tile loop together)
__device__ __forceinline__ bool consumer_any(bool pred) {
    uint32_t r;
    asm volatile(
        "{\n"
        ".reg .pred p, q;\n"
        "setp.ne.u32 p, %1, 0;\n"
        "bar.red.or.pred q, 1, %2, p;\n"
        "selp.u32 %0, 1, 0, q;\n"
        "}\n"
        : "=r"(r)
        : "r"((uint32_t)pred), "n"(kTmaConsumers)
        : "memory");
    return r != 0;
}

__device__ void chain_stream_tma(const ChainStream &X, const LpChainRank &A, const LpChainLaunch &L, int c) {
    extern __shared__ __align__(128) unsigned char lp_smem[];
    float *ring = reinterpret_cast<float *>(lp_smem);
    uint64_t *full = reinterpret_cast<uint64_t *>(lp_smem + kTmaRingBytes);
    uint64_t *empty = full + kTmaMaxStages;
    volatile int *abort_flag = reinterpret_cast<volatile int *>(empty + kTmaMaxStages);
    const int nsrc = (X.src_ring ? 1 : 0) + (X.src_local ? 1 : 0) + (X.src_w ? 1 : 0) + (X.vel ? 1 : 0);
    const int stages = (int)(kTmaRingBytes / ((uint32_t)nsrc * kTmaStep * 4u));
    const uint32_t stage_floats = (uint32_t)nsrc * kTmaStep;
    unsigned long long *st = A.state + (size_t)c * 4;
    const unsigned long long recv0 = X.src_ring ? st[X.st_recv] : 0;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            lp_mbar_init(&full[s], 1);
            lp_mbar_init(&empty[s], kTmaConsumers / 32);
        }
        *abort_flag = 0;
        lp_fence_mbar_init();
    }
    __syncthreads();
    const size_t ring_c = (size_t)c * L.S * L.tile;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0) {
        // ---------------- producer: counters of my receive ring, TMA bulk loads of every source ------------------------
        if (lane == 0) {
            unsigned long long recv = recv0;
            int stage = 0;
            uint32_t phase = 0;
            bool ok = true;
            for (uint64_t t = (uint64_t)c; ok && t < L.part.n_tiles; t += (uint64_t)L.C) {
                uint64_t off;
                uint32_t len;
                lp_tile_range(L.part, t, off, len);
                const float *slot = nullptr;
                if (X.src_ring) {
                    ok = poll_counter(X.src_tail, recv + 1, A.error, abort_flag, L.spin_limit);
                    if (!ok) break;
                    fence_sys();  // acquire: the block published before the counter ...
                    asm volatile("fence.proxy.async;" ::: "memory");  // ... is what the bulk copies (async proxy) read
                    slot = X.src_ring + ring_c + (size_t)(recv % (unsigned)L.S) * L.tile;
                    ++recv;
                }
                for (uint32_t s0 = 0; s0 < len; s0 += kTmaStep) {
                    const uint32_t sl = len - s0 < kTmaStep ? len - s0 : kTmaStep;
                    const uint32_t bytes = (sl & ~3u) * 4u;  // the 16-byte aligned body; <= 3 tail elements go by hand
                    ok = mbar_wait_abortable(&empty[stage], phase ^ 1u, abort_flag);
                    if (!ok) break;
                    float *dst = ring + (size_t)stage * stage_floats;
                    if (bytes) {
                        lp_mbar_expect_tx(&full[stage], bytes * (uint32_t)nsrc);
                        if (X.src_ring) {
                            lp_bulk_g2s(dst, slot + s0, bytes, &full[stage]);
                            dst += kTmaStep;
                        }
                        if (X.src_local) {
                            lp_bulk_g2s(dst, X.src_local + off + s0, bytes, &full[stage]);
                            dst += kTmaStep;
                        }
                        if (X.src_w) {
                            lp_bulk_g2s(dst, X.src_w + off + s0, bytes, &full[stage]);
                            dst += kTmaStep;
                        }
                        if (X.vel) lp_bulk_g2s(dst, X.vel + off + s0, bytes, &full[stage]);
                    } else {
                        lp_mbar_arrive(&full[stage]);
                    }
                    if (++stage == stages) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
            if (X.src_ring && ok) st[X.st_recv] = recv;
        }
        return;
    }
    // -------------------- consumers: fold in chain order, store to every destination, publish, credit --------------------
    const int ctid = (int)threadIdx.x - 32;
    unsigned long long sent[2] = {X.dst_ring[0] ? st[X.st_sent[0]] : 0, X.dst_ring[1] ? st[X.st_sent[1]] : 0};
    unsigned long long recv = recv0;
    int stage = 0;
    uint32_t phase = 0;
    bool ok = true;
    for (uint64_t t = (uint64_t)c; ok && t < L.part.n_tiles; t += (uint64_t)L.C) {
        uint64_t off;
        uint32_t len;
        lp_tile_range(L.part, t, off, len);
        bool failed = false;
        if (ctid == 0) {  // the slots this tile is pushed into must be free
            for (int j = 0; j < 2 && !failed; ++j)
                if (X.dst_ring[j] && slot_free_at(sent[j], L.S))
                    failed = !poll_counter(X.dst_credit[j], slot_free_at(sent[j], L.S), A.error, abort_flag, L.spin_limit);
        }
        if (consumer_any(failed)) {
            ok = false;
            break;
        }
        float *push[2] = {X.dst_ring[0] ? X.dst_ring[0] + ring_c + (size_t)(sent[0] % (unsigned)L.S) * L.tile : nullptr,
                          X.dst_ring[1] ? X.dst_ring[1] + ring_c + (size_t)(sent[1] % (unsigned)L.S) * L.tile : nullptr};
        const float *in_slot = X.src_ring ? X.src_ring + ring_c + (size_t)(recv % (unsigned)L.S) * L.tile : nullptr;
        for (uint32_t s0 = 0; s0 < len; s0 += kTmaStep) {
            const uint32_t sl = len - s0 < kTmaStep ? len - s0 : kTmaStep;
            const uint32_t nvec = sl >> 2;
            ok = mbar_wait_abortable(&full[stage], phase, abort_flag);
            if (!ok) break;
            const float4 *src = reinterpret_cast<const float4 *>(ring + (size_t)stage * stage_floats);
            float4 acc[kTmaVec];
#pragma unroll
            for (int k = 0; k < kTmaVec; ++k) {
                const uint32_t j = (uint32_t)ctid + (uint32_t)k * kTmaConsumers;
                if (j < nvec) {
                    const float4 *p = src + j;
                    acc[k] = *p;  // the partial (or the finished block), else my block
                    if (X.src_ring && X.src_local) {  // "reduces the received block a0 with a1": partial op mine
                        p += kTmaStep / 4;
                        acc[k] = lp_combine4(acc[k], *p, L.code);
                    }
                    if (X.src_w) {  // Alg. 3's update where the global gradient is complete: three RN operations
                        p += kTmaStep / 4;
                        if (X.vel) {  // five with momentum (U18): the new velocity goes straight back to its vector
                            float4 vn;
                            lp_mom4(acc[k], *p, p[kTmaStep / 4], L.lr, L.invP, L.mu, vn, acc[k]);
                            lp_stg_stream(X.vel + off + s0 + 4 * j, vn);
                        } else {
                            acc[k] = lp_sgd4(acc[k], *p, L.lr, L.invP);
                        }
                    }
                }
            }
            // the shared-memory reads above have returned (their values went into the fold, or -- a plain copy -- are
            // consumed by the stores below only after this fence): the slot may be refilled
            __threadfence_block();
            __syncwarp();
            if (lane == 0) lp_mbar_arrive(&empty[stage]);
            if (++stage == stages) {
                stage = 0;
                phase ^= 1u;
            }
#pragma unroll
            for (int k = 0; k < kTmaVec; ++k) {
                const uint32_t j = (uint32_t)ctid + (uint32_t)k * kTmaConsumers;
                if (j < nvec) {
                    if (push[0]) lp_stg_stream(push[0] + s0 + 4 * j, acc[k]);
                    if (X.dst_local) lp_stg_stream(X.dst_local + off + s0 + 4 * j, acc[k]);
                    if (push[1]) lp_stg_stream(push[1] + s0 + 4 * j, acc[k]);
                }
            }
            if (ctid == 0 && (sl & 3u) && L.code >= 6) {
                // f64 (codes 6 / 7): the last two words are ONE element (lengths and offsets are even) -- lp_combine1 knows
                // only the one-word types, so the pair is folded as a double, like lp_word_combine_store does
                for (uint32_t e = sl & ~3u; e + 1 < sl; e += 2) {
                    float lo = X.src_ring ? ld_ring1(in_slot + s0 + e) : X.src_local[off + s0 + e];
                    float hi = X.src_ring ? ld_ring1(in_slot + s0 + e + 1) : X.src_local[off + s0 + e + 1];
                    if (X.src_ring && X.src_local) {
                        const double r = lp_combine_f64(lp_words_f64(lo, hi),
                                                        lp_words_f64(X.src_local[off + s0 + e], X.src_local[off + s0 + e + 1]),
                                                        L.code == 7);
                        lo = __int_as_float(__double2loint(r));
                        hi = __int_as_float(__double2hiint(r));
                    }
                    if (push[0]) push[0][s0 + e] = lo, push[0][s0 + e + 1] = hi;
                    if (X.dst_local) X.dst_local[off + s0 + e] = lo, X.dst_local[off + s0 + e + 1] = hi;
                    if (push[1]) push[1][s0 + e] = lo, push[1][s0 + e + 1] = hi;
                }
            } else if (ctid == 0 && (sl & 3u)) {  // the message's last <= 3 elements: by hand, straight from and to global memory
                for (uint32_t e = sl & ~3u; e < sl; ++e) {
                    float v = X.src_ring ? ld_ring1(in_slot + s0 + e) : X.src_local[off + s0 + e];
                    if (X.src_ring && X.src_local) v = lp_combine1(v, X.src_local[off + s0 + e], L.code);
                    if (X.src_w && X.vel) {
                        float vn, wn;
                        lp_mom1(v, X.src_w[off + s0 + e], X.vel[off + s0 + e], L.lr, L.invP, L.mu, vn, wn);
                        X.vel[off + s0 + e] = vn;
                        v = wn;
                    } else if (X.src_w) {
                        v = lp_sgd1(v, X.src_w[off + s0 + e], L.lr, L.invP);
                    }
                    if (push[0]) push[0][s0 + e] = v;
                    if (X.dst_local) X.dst_local[off + s0 + e] = v;
                    if (push[1]) push[1][s0 + e] = v;
                }
            }
        }
        // every consumer's stores of this tile have been issued -- or somebody gave up: then all leave together
        if (consumer_any(!ok)) {
            ok = false;
            break;
        }
        if (push[0]) ++sent[0];
        if (push[1]) ++sent[1];
        ++recv;
        if (ctid == 0) {
            if (push[0] || push[1]) fence_sys();  // release, cumulative over the barrier: the tile before its counter
            if (push[0]) st_sys(X.dst_tail[0], sent[0]);
            if (push[1]) st_sys(X.dst_tail[1], sent[1]);
            if (X.src_ring) st_sys(X.src_credit, recv);  // the bulk loads of this slot completed long ago
        }
    }
    consumer_barrier();
    if (ctid == 0 && ok) {
        if (X.dst_ring[0]) st[X.st_sent[0]] = sent[0];
        if (X.dst_ring[1]) st[X.st_sent[1]] = sent[1];
    }
}

__global__ void __launch_bounds__(kTmaThreads, 1) lp_chain_tma_kernel(const __grid_constant__ LpChainLaunch L) {
    const int per_rank = 2 * L.C;
    const int lr = (int)blockIdx.x / per_rank;
    const int j = (int)blockIdx.x - lr * per_rank;
    const LpChainRank &A = L.rank[lr];
    if (chain_endpoint_dead(A.error)) return;
    ChainStream X;
    memset(&X, 0, sizeof(X));
    int c;
    if (j < L.C) {
        if (!A.f_active) return;
        c = j;
        unsigned long long *my = A.flags + (size_t)c * kFlagsPerChannel;
        if (A.f_recv) {
            X.src_ring = A.fwd_ring;
            X.src_tail = my + F_FWD_TAIL;
            X.src_credit = A.down_flags + (size_t)c * kFlagsPerChannel + F_UP_CREDIT;
            X.st_recv = ST_RECV_FWD;
        }
        if (A.f_load) X.src_local = A.buf;
        if (A.f_update) {
            X.src_w = A.w_in;
            X.vel = A.vel;
        }
        if (A.f_store) X.dst_local = A.out;
        if (A.f_send_up) {
            X.dst_ring[0] = A.up_fwd_ring;
            X.dst_tail[0] = A.up_flags + (size_t)c * kFlagsPerChannel + F_FWD_TAIL;
            X.dst_credit[0] = my + F_UP_CREDIT;
            X.st_sent[0] = ST_SENT_UP;
        }
        if (A.f_send_down) {
            X.dst_ring[1] = A.down_bwd_ring;
            X.dst_tail[1] = A.down_flags + (size_t)c * kFlagsPerChannel + F_BWD_TAIL;
            X.dst_credit[1] = my + F_DOWN_CREDIT;
            X.st_sent[1] = ST_SENT_DOWN;
        }
    } else {
        if (!A.r_active) return;
        c = j - L.C;
        unsigned long long *my = A.flags + (size_t)c * kFlagsPerChannel;
        X.src_ring = A.bwd_ring;
        X.src_tail = my + F_BWD_TAIL;
        X.src_credit = A.up_flags + (size_t)c * kFlagsPerChannel + F_DOWN_CREDIT;
        X.st_recv = ST_RECV_BWD;
        if (A.r_store) X.dst_local = A.out;
        if (A.r_send_down) {
            X.dst_ring[1] = A.down_bwd_ring;
            X.dst_tail[1] = A.down_flags + (size_t)c * kFlagsPerChannel + F_BWD_TAIL;
            X.dst_credit[1] = my + F_DOWN_CREDIT;
            X.st_sent[1] = ST_SENT_DOWN;
        }
    }
    chain_stream_tma(X, A, L, c);
}

// ---- launch helpers ---------------------------------------------------------------------------------------------
// 1024 threads, one CTA per SM.  (512-thread CTAs, two per SM, on twice the channels: 5-20 % more per SM in the one-GPU
// emulation, for twice the ring memory -- profiles/r2_dtypes_chain.md.)
int chain_threads() { return kChainThreads; }

constexpr uint32_t kTmaSmem = kTmaRingBytes + 2u * kTmaMaxStages * 8u + 16u;

cudaError_t tma_attr() {  // per device binding (lp_attr_epoch): the dynamic shared memory limit of the TMA kernel
    static std::atomic<unsigned> epoch{0};
    if (epoch.load() == lp_attr_epoch()) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(lp_chain_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTmaSmem);
    if (e == cudaSuccess) epoch.store(lp_attr_epoch());
    return e;
}

}  // namespace

cudaError_t lp_chain_resident(bool tma, int *ctas) {
    int per_sm = 0, dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess && tma) {
        e = tma_attr();
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_chain_tma_kernel, kTmaThreads, kTmaSmem);
    } else if (e == cudaSuccess) {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_chain_kernel, chain_threads(), 0);
    }
    *ctas = per_sm * sms;
    return e;
}

cudaError_t lp_chain_launch_kernel(const LpChainLaunch &L, bool tma, bool cooperative, cudaStream_t stream) {
    const unsigned grid = (unsigned)(L.n_local * 2 * L.C);
    int cap = 0;
    cudaError_t e = lp_chain_resident(tma, &cap);
    if (e != cudaSuccess) return e;
    if ((unsigned)cap < grid) return cudaErrorCooperativeLaunchTooLarge;  // every CTA must be resident
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof(lc));
    lc.gridDim = dim3(grid);
    lc.blockDim = dim3(tma ? kTmaThreads : chain_threads());
    lc.dynamicSmemBytes = tma ? kTmaSmem : 0;
    lc.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    lc.attrs = attr;
    lc.numAttrs = cooperative ? 1 : 0;
    lp_count_launch(1);
    lp_chain_reset(stream);
    if (tma) return cudaLaunchKernelEx(&lc, lp_chain_tma_kernel, L);
    return cudaLaunchKernelEx(&lc, lp_chain_kernel, L);
}
