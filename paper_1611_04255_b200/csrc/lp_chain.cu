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
// the device holds at once.
//
// ONE GPU (this build's box): kernels that wait on each other must not run as separate launches on one device, so
// lp_chain_emulate runs the SAME per-rank code for all P ranks inside ONE cooperative launch (P x 2 C co-resident
// CTAs), every "peer" pointer then being a local one.  That is what tests/ compare with the oracle bit for bit; the
// multi-process plumbing (roles, handle exchange) is covered on the CPU.  Values: the chain order rank 0 -> P-1 (U4),
// one RN operation per combine -- the same definition as every other LP variant.
#include <cooperative_groups.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "lp_common.cuh"

namespace {

constexpr int kChainThreads = 1024;
constexpr int kFlagStride = 16;           // unsigned long longs between two counters: one 128-byte line each
constexpr int kFlagsPerChannel = 4 * kFlagStride;
enum { F_FWD_TAIL = 0, F_BWD_TAIL = kFlagStride, F_UP_CREDIT = 2 * kFlagStride, F_DOWN_CREDIT = 3 * kFlagStride };
enum { ST_RECV_FWD = 0, ST_SENT_UP = 1, ST_RECV_BWD = 2, ST_SENT_DOWN = 3 };

// What one rank's CTAs need: its vector, its endpoint, its two neighbours' endpoints, its roles in this call.
struct LpChainRank {
    float *buf;         // my vector: what the forward CTAs load
    float *out;         // where finished blocks are stored: buf (in place), or my weight replica for the SGD step
    const float *w_in;  // SGD step, chain end only: the weight replica the update reads
    float *vel;         // SGD step with momentum, chain end only: the velocity, read and rewritten in place
    unsigned long long *flags;   // my counters: [C][kFlagsPerChannel]
    unsigned long long *state;   // my private sequence numbers: [C][4]
    float *fwd_ring, *bwd_ring;  // my receive rings: [C][S][tile]
    unsigned long long *up_flags;    // endpoint of rank (r + 1) mod P
    float *up_fwd_ring;
    unsigned long long *down_flags;  // endpoint of rank (r - 1 + P) mod P
    float *down_bwd_ring;
    int *error;  // my error word (0 = fine)
    // forward CTAs
    unsigned char f_active, f_load, f_recv, f_send_up, f_store, f_send_down, f_update;
    // return CTAs
    unsigned char r_active, r_store, r_send_down;
    unsigned char pad[2];
};

struct LpChainLaunch {
    LpChainRank rank[LP_MAX_P];  // [0] alone for a real launch (one rank per GPU); all P for the one-GPU emulation
    lp_partition part;
    int n_local;  // ranks in this launch
    int C, S;
    uint32_t tile;  // elements per ring slot
    int code;  // (dtype << 1) | red_op
    float lr, invP;  // SGD step (LpChainRank::f_update): w' = w - lr * (S * invP) where the chain ends (U7)
    float mu;        // ... with momentum (LpChainRank::vel != NULL): v' = mu v + lr (S invP), w' = w - v' (U18)
    unsigned long long spin_limit;  // polls before a wait gives up and flags an error: a missing peer never hangs the GPU
};

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
__global__ void __launch_bounds__(kChainThreads, 1) lp_chain_kernel(const __grid_constant__ LpChainLaunch L) {
    __shared__ int s_ok;
    const int per_rank = 2 * L.C;
    const int lr = (int)blockIdx.x / per_rank;
    const int j = (int)blockIdx.x - lr * per_rank;
    const LpChainRank &A = L.rank[lr];
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
            if (ctid == 0 && (sl & 3u)) {  // the message's last <= 3 elements: by hand, straight from and to global memory
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

}  // namespace

// ---- host side -------------------------------------------------------------------------------------------------

// Roles of `rank` in a collective over P ranks (pure host logic: the part of the multi-process path that needs no GPU).
extern "C" int lp_chain_plan(int op, int P, int root, int rank, lp_chain_role *out) {
    if (out == nullptr || P < 1 || P > LP_MAX_P || rank < 0 || rank >= P) return LP_ERR_INVALID_ARG;
    if (op < LP_OP_BROADCAST || op > LP_OP_BSP_SGD_MOM) return LP_ERR_INVALID_ARG;
    if ((op == LP_OP_BROADCAST || op == LP_OP_REDUCE) && (root < 0 || root >= P)) return LP_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    out->up = (rank + 1) % P;
    out->down = (rank + P - 1) % P;
    if (P == 1) {  // nothing moves; the SGD step of a single rank is its own update
        if (op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM) out->f_active = out->f_load = out->f_update = out->f_store = 1;
        return LP_OK;
    }
    if (op == LP_OP_BROADCAST) {  // root -> root+1 -> ... -> root-1 around the ring, forward direction only
        const int j = (rank - root + P) % P;
        out->position = j;
        out->f_active = 1;
        out->f_load = j == 0;
        out->f_recv = j > 0;
        out->f_store = j > 0;
        out->f_send_up = j < P - 1;
        return LP_OK;
    }
    // reduce / allreduce: the chain is rank 0 -> 1 -> ... -> P-1 whatever the root (U4)
    const bool all = op != LP_OP_REDUCE;  // allreduce, and the SGD step (the new weights go to every rank)
    const bool head = rank == P - 1;
    const int ret_lo = all ? 0 : root;  // the lowest rank a finished tile travels back to
    out->position = rank;
    out->f_active = 1;
    out->f_load = 1;
    out->f_recv = rank > 0;
    out->f_send_up = !head;
    out->f_store = head && (all || root == P - 1);
    out->f_send_down = head && ret_lo < P - 1;
    out->f_update = head && (op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM);
    out->r_active = !head && rank >= ret_lo && ret_lo < P - 1;
    out->r_store = out->r_active && (all || rank == root);
    out->r_send_down = out->r_active && rank > ret_lo;
    return LP_OK;
}

struct lp_chain {
    int rank, P, C, S, tile;
    int device;
    void *base;        // my endpoint (cudaMalloc)
    size_t bytes;
    void *peer_up, *peer_down;  // mapped endpoints of the neighbours (== base of another lp_chain in the same process)
    bool up_ipc, down_ipc;      // opened with cudaIpcOpenMemHandle (to be closed)
    bool connected;
    unsigned long long spin_limit;  // polls before a wait of this endpoint's kernels gives up
};

namespace {

struct EndpointLayout {
    size_t flags_off, state_off, error_off, fwd_off, bwd_off, bytes;
};
EndpointLayout layout_of(int C, int S, int tile) {
    EndpointLayout l;
    size_t o = 0;
    l.flags_off = o;
    o += (size_t)C * kFlagsPerChannel * sizeof(unsigned long long);
    l.state_off = o;
    o += (size_t)C * 4 * sizeof(unsigned long long);
    l.error_off = o;
    o += 256;
    o = (o + 255) & ~(size_t)255;
    l.fwd_off = o;
    o += (size_t)C * S * tile * sizeof(float);
    l.bwd_off = o;
    o += (size_t)C * S * tile * sizeof(float);
    l.bytes = o;
    return l;
}

void fill_rank(LpChainRank &R, const EndpointLayout &l, float *buf, float *out, const float *w_in, float *vel, void *mine,
               void *up, void *down, const lp_chain_role &role) {
    memset(&R, 0, sizeof(R));
    char *m = (char *)mine, *u = (char *)up, *d = (char *)down;
    R.buf = buf;
    R.out = out;
    R.w_in = w_in;
    R.vel = role.f_update ? vel : nullptr;
    R.flags = (unsigned long long *)(m + l.flags_off);
    R.state = (unsigned long long *)(m + l.state_off);
    R.error = (int *)(m + l.error_off);
    R.fwd_ring = (float *)(m + l.fwd_off);
    R.bwd_ring = (float *)(m + l.bwd_off);
    R.up_flags = (unsigned long long *)(u + l.flags_off);
    R.up_fwd_ring = (float *)(u + l.fwd_off);
    R.down_flags = (unsigned long long *)(d + l.flags_off);
    R.down_bwd_ring = (float *)(d + l.bwd_off);
    R.f_active = role.f_active;
    R.f_load = role.f_load;
    R.f_recv = role.f_recv;
    R.f_send_up = role.f_send_up;
    R.f_store = role.f_store;
    R.f_send_down = role.f_send_down;
    R.f_update = role.f_update;
    R.r_active = role.r_active;
    R.r_store = role.r_store;
    R.r_send_down = role.r_send_down;
}

// 1024 threads, one CTA per SM.  (512-thread CTAs, two per SM, on twice the channels: 5-20 % more per SM in the one-GPU
// emulation, for twice the ring memory -- profiles/r2_dtypes_chain.md.)
int chain_threads() { return kChainThreads; }

std::atomic<int> g_chain_kernel{LP_CHAIN_KERNEL_DEFAULT};
bool use_tma() { return g_chain_kernel.load() != LP_CHAIN_KERNEL_REGISTER; }
constexpr uint32_t kTmaSmem = kTmaRingBytes + 2u * kTmaMaxStages * 8u + 16u;

cudaError_t tma_attr() {  // per device binding (lp_attr_epoch): the dynamic shared memory limit of the TMA kernel
    static std::atomic<unsigned> epoch{0};
    if (epoch.load() == lp_attr_epoch()) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(lp_chain_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTmaSmem);
    if (e == cudaSuccess) epoch.store(lp_attr_epoch());
    return e;
}

// CTAs of the chain kernel the current device holds at once
cudaError_t resident(int *ctas) {
    int per_sm = 0, dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess && use_tma()) {
        e = tma_attr();
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_chain_tma_kernel, kTmaThreads, kTmaSmem);
    } else if (e == cudaSuccess) {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_chain_kernel, chain_threads(), 0);
    }
    *ctas = per_sm * sms;
    return e;
}

cudaError_t launch(const LpChainLaunch &L, bool cooperative, cudaStream_t stream) {
    const unsigned grid = (unsigned)(L.n_local * 2 * L.C);
    const bool tma = use_tma();
    int cap = 0;
    cudaError_t e = resident(&cap);
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

// a1 for the chain: blocks of `block` elements rounded up to a multiple of 4 (every tile then starts on a 16-byte
// boundary; results never depend on the block), cut into tiles of at most one ring slot.  block == 0, "the library
// chooses": one slot for long messages; for short ones the power of two that still gives every channel about four
// blocks (floor 4096 elements), so that the pipeline over the ranks fills after a small block instead of after a
// whole slot -- the paper's reason for small blocks, PAPER.md:89 ((p - 1 + n/b) steps: the fill term is (p - 1) b).
lp_partition chain_partition(size_t n, size_t block, int tile, int channels) {
    if (block == 0) {
        size_t b = 4096;
        while (b < (size_t)tile && b * 4u * (size_t)channels < n) b *= 2;
        block = b;
    }
    if (block < ~(size_t)3) block = (block + 3) & ~(size_t)3;
    return lp_make_partition(n, block, (uint32_t)tile);
}

bool valid_geometry(int C, int S, int tile) {  // tile: a power of two, 4096 .. 262144 elements (16 KB .. 1 MB)
    return C >= 1 && C <= LP_CHAIN_MAX_CHANNELS && S >= 1 && S <= 64 && tile >= 4096 && tile <= 262144 &&
           (tile & (tile - 1)) == 0;
}

int chain_fail(cudaError_t e) {
    cudaGetLastError();
    return e == cudaErrorCooperativeLaunchTooLarge ? LP_ERR_UNSUPPORTED : LP_ERR_CUDA;
}

// emulation endpoints: (geometry, P, stream) -> one allocation holding P endpoints, kept for the life of the library
// binding.  Per stream: launches of one stream are ordered, launches of two streams may overlap and must not share rings.
struct EmulEndpoints {
    int P, C, S, tile;
    cudaStream_t stream;
    void *base;
};
std::mutex g_emul_mu;
std::vector<EmulEndpoints> g_emul;

}  // namespace

void lp_chain_shutdown() {
    std::lock_guard<std::mutex> lock(g_emul_mu);
    for (auto &e : g_emul) cudaFree(e.base);
    g_emul.clear();
}

extern "C" {

size_t lp_chain_endpoint_bytes(int channels, int slots, int tile) {
    return valid_geometry(channels, slots, tile) ? layout_of(channels, slots, tile).bytes : 0;
}

int lp_chain_create(int rank, int P, int channels, int slots, int tile, lp_chain **out) {
    if (out == nullptr) return LP_ERR_INVALID_ARG;
    *out = nullptr;
    if (channels == 0) channels = LP_CHAIN_DEFAULT_CHANNELS;
    if (slots == 0) slots = LP_CHAIN_DEFAULT_SLOTS;
    if (tile == 0) tile = LP_CHAIN_DEFAULT_TILE;
    if (P < 1 || P > LP_MAX_P || rank < 0 || rank >= P || !valid_geometry(channels, slots, tile)) return LP_ERR_INVALID_ARG;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return LP_ERR_CUDA;
    }
    lp_chain *ch = new lp_chain;
    memset(ch, 0, sizeof(*ch));
    ch->rank = rank;
    ch->P = P;
    ch->C = channels;
    ch->S = slots;
    ch->tile = tile;
    ch->device = dev;
    ch->bytes = layout_of(channels, slots, tile).bytes;
    ch->spin_limit = 1ull << 28;  // ~a minute of polling: ranks of different processes start at different times
    cudaError_t e = cudaMalloc(&ch->base, ch->bytes);
    if (e == cudaSuccess) e = cudaMemset(ch->base, 0, ch->bytes);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        if (ch->base) cudaFree(ch->base);
        delete ch;
        return chain_fail(e);
    }
    *out = ch;
    return LP_OK;
}

int lp_chain_get_handle(lp_chain *ch, void *handle_out) {
    if (ch == nullptr || handle_out == nullptr) return LP_ERR_INVALID_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == LP_CHAIN_HANDLE_BYTES, "handle size");
    cudaIpcMemHandle_t h;
    const cudaError_t e = cudaIpcGetMemHandle(&h, ch->base);
    if (e != cudaSuccess) return chain_fail(e);
    memcpy(handle_out, &h, sizeof(h));
    return LP_OK;
}

// handles: P x LP_CHAIN_HANDLE_BYTES, rank order (what an all-gather of lp_chain_get_handle leaves on every rank).
int lp_chain_connect(lp_chain *ch, const void *handles) {
    if (ch == nullptr || handles == nullptr || ch->connected) return LP_ERR_INVALID_ARG;
    const int up = (ch->rank + 1) % ch->P, down = (ch->rank + ch->P - 1) % ch->P;
    auto open = [&](int peer, void **ptr, bool *ipc) -> cudaError_t {
        if (peer == ch->rank) {
            *ptr = ch->base;
            *ipc = false;
            return cudaSuccess;
        }
        cudaIpcMemHandle_t h;
        memcpy(&h, (const char *)handles + (size_t)peer * LP_CHAIN_HANDLE_BYTES, sizeof(h));
        *ipc = true;
        return cudaIpcOpenMemHandle(ptr, h, cudaIpcMemLazyEnablePeerAccess);
    };
    cudaError_t e = open(up, &ch->peer_up, &ch->up_ipc);
    if (e != cudaSuccess) return chain_fail(e);
    if (down == up) {
        ch->peer_down = ch->peer_up;
        ch->down_ipc = false;
    } else {
        e = open(down, &ch->peer_down, &ch->down_ipc);
        if (e != cudaSuccess) {
            if (ch->up_ipc) cudaIpcCloseMemHandle(ch->peer_up);
            return chain_fail(e);
        }
    }
    ch->connected = true;
    return LP_OK;
}

// The same with raw device pointers: endpoints of other lp_chain objects of THIS process (one process driving several
// GPUs with peer access enabled by the caller).
int lp_chain_connect_ptrs(lp_chain *ch, void *up_endpoint, void *down_endpoint) {
    if (ch == nullptr || up_endpoint == nullptr || down_endpoint == nullptr || ch->connected) return LP_ERR_INVALID_ARG;
    ch->peer_up = up_endpoint;
    ch->peer_down = down_endpoint;
    ch->up_ipc = ch->down_ipc = false;
    ch->connected = true;
    return LP_OK;
}

void *lp_chain_endpoint(lp_chain *ch) { return ch ? ch->base : nullptr; }

int lp_chain_set_kernel(int kernel) {
    if (kernel != LP_CHAIN_KERNEL_DEFAULT && kernel != LP_CHAIN_KERNEL_REGISTER && kernel != LP_CHAIN_KERNEL_TMA)
        return LP_ERR_INVALID_ARG;
    g_chain_kernel.store(kernel);
    return LP_OK;
}

int lp_chain_set_timeout(lp_chain *ch, unsigned long long polls) {
    if (ch == nullptr || polls == 0) return LP_ERR_INVALID_ARG;
    ch->spin_limit = polls;
    return LP_OK;
}

int lp_chain_destroy(lp_chain *ch) {
    if (ch == nullptr) return LP_ERR_INVALID_ARG;
    cudaDeviceSynchronize();
    if (ch->connected) {
        if (ch->up_ipc) cudaIpcCloseMemHandle(ch->peer_up);
        if (ch->down_ipc) cudaIpcCloseMemHandle(ch->peer_down);
    }
    cudaFree(ch->base);
    cudaGetLastError();
    delete ch;
    return LP_OK;
}

// Words per element and the operator code of a typed launch; false for an unknown type.  The chain addresses vectors
// in 4-byte words like every other kernel (LpArgs::dtype): n and block arrive in elements and leave in words.  16-bit
// vectors must hold an even number of elements here (a push moves whole words).
static bool chain_words(int dtype, int reduce_op, size_t &n, size_t &block, int &code) {
    if (dtype < LP_DT_F32 || dtype > LP_DT_F64) return false;
    if (reduce_op != LP_REDUCE_SUM && reduce_op != LP_REDUCE_PROD) return false;
    code = (dtype << 1) | reduce_op;
    if (dtype == LP_DT_F64) {
        if (n > (~(size_t)0) / 8) return false;
        n *= 2;
        block = block > (~(size_t)0) / 2 ? ~(size_t)3 : 2 * block;
    } else if (dtype != LP_DT_F32) {
        if (n & 1u) return false;
        n /= 2;
        block = block / 2 + (block & 1u);
    }
    return true;
}

static bool chain_sgd(int op) { return op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM; }

static int chain_run_rank(lp_chain *ch, int op, float *buf, float *out, const float *w_in, size_t n, size_t block, int root,
                          int code, float lr, void *cuda_stream, float *vel = nullptr, float mu = 0.f) {
    if (ch == nullptr || !ch->connected) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_ALLREDUCE || chain_sgd(op)) root = 0;
    lp_chain_role role;
    int rc = lp_chain_plan(op, ch->P, root, ch->rank, &role);
    if (rc != LP_OK) return rc;
    if (buf == nullptr || ((uintptr_t)buf & 15u) || out == nullptr || ((uintptr_t)out & 15u)) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_BSP_SGD_MOM && role.f_update && (vel == nullptr || ((uintptr_t)vel & 15u))) return LP_ERR_INVALID_ARG;
    if (n == 0) return LP_OK;
    if (ch->P == 1 && !chain_sgd(op)) return LP_OK;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ch->device) {
        cudaGetLastError();
        return LP_ERR_UNSUPPORTED;
    }
    LpChainLaunch L;
    memset(&L, 0, sizeof(L));
    L.n_local = 1;
    L.C = ch->C;
    L.S = ch->S;
    L.code = code;
    L.lr = lr;
    L.mu = mu;
    L.invP = 1.0f / (float)ch->P;  // one RN division on the host (U7)
    L.spin_limit = ch->spin_limit;
    L.part = chain_partition(n, block, ch->tile, ch->C);
    L.tile = (uint32_t)ch->tile;
    fill_rank(L.rank[0], layout_of(ch->C, ch->S, ch->tile), buf, out, w_in, op == LP_OP_BSP_SGD_MOM ? vel : nullptr, ch->base,
              ch->peer_up, ch->peer_down, role);
    const cudaError_t e = launch(L, false, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? LP_OK : chain_fail(e);
}

// One rank's share of the collective: every rank of the chain calls this with the same (op, n, block, root, reduce_op),
// in the same order as its other chain collectives.
int lp_chain_run(lp_chain *ch, int op, float *buf, size_t n, size_t block, int root, int reduce_op, void *cuda_stream) {
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return LP_ERR_INVALID_ARG;
    int code;
    if (!chain_words(LP_DT_F32, reduce_op, n, block, code)) return LP_ERR_INVALID_ARG;
    return chain_run_rank(ch, op, buf, buf, nullptr, n, block, root, code, 0.f, cuda_stream);
}

int lp_chain_run_dt(lp_chain *ch, int op, void *buf, size_t n, size_t block, int root, int dtype, int reduce_op,
                    void *cuda_stream) {
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return LP_ERR_INVALID_ARG;
    int code;
    if (!chain_words(dtype, reduce_op, n, block, code)) return LP_ERR_INVALID_ARG;
    return chain_run_rank(ch, op, (float *)buf, (float *)buf, nullptr, n, block, root, code, 0.f, cuda_stream);
}

// Alg. 3's communication + update over the chain: the sub-gradients are folded up the chain, the
// last rank forms w' = w - lr * (S * invP) from ITS weight replica (all replicas hold the same bits, U8) and the new
// weights travel back down; every rank stores them into its replica.  grad is only read.
int lp_chain_bsp_sgd_step(lp_chain *ch, float *grad, float *weight, size_t n, size_t block, float lr, void *cuda_stream) {
    if (weight == nullptr || grad == weight) return LP_ERR_INVALID_ARG;
    return chain_run_rank(ch, LP_OP_BSP_SGD, grad, weight, weight, n, block, 0, LP_REDUCE_SUM, lr, cuda_stream);
}

// The same with momentum ("The solver is SGD + momentum"; U18): v' = mu v + lr (S invP), w' = w - v'.  The
// velocity is ONE vector and lives where the update is computed: on the LAST rank, which passes it; the others pass NULL.
int lp_chain_bsp_sgd_momentum_step(lp_chain *ch, float *grad, float *weight, float *velocity, size_t n, size_t block,
                                   float lr, float mu, void *cuda_stream) {
    if (weight == nullptr || grad == weight || (velocity != nullptr && (velocity == grad || velocity == weight)))
        return LP_ERR_INVALID_ARG;
    return chain_run_rank(ch, LP_OP_BSP_SGD_MOM, grad, weight, weight, n, block, 0, LP_REDUCE_SUM, lr, cuda_stream, velocity,
                          mu);
}

// Alg. 2 over the chain (PAPER.md:140-168 as read in U9, prose PAPER.md:178): reduce the sub-gradients to `root`
// (grad <- S there, as lp_reduce does, U20), the root applies GradientUpdate to its replica (the same rounded operations
// as the fused steps; velocity != NULL on the root: the momentum form), the new weights are broadcast from the root.
// Three launches on the root, two on every other rank -- the two-synchronisation-point counterpart of the fused step.
int lp_chain_bsp_sgd_alg2_step(lp_chain *ch, float *grad, float *weight, float *velocity, size_t n, size_t block, int root,
                               float lr, float mu, void *cuda_stream) {
    if (ch == nullptr || weight == nullptr || grad == weight || root < 0 || root >= ch->P) return LP_ERR_INVALID_ARG;
    int rc = chain_run_rank(ch, LP_OP_REDUCE, grad, grad, nullptr, n, block, root, LP_REDUCE_SUM, 0.f, cuda_stream);
    if (rc != LP_OK) return rc;
    if (ch->rank == root && n > 0) {
        const cudaError_t e = lp_update_launch(weight, grad, velocity, n, lr, 1.0f / (float)ch->P, mu, (cudaStream_t)cuda_stream,
                                               false);
        if (e != cudaSuccess) return chain_fail(e);
    }
    return chain_run_rank(ch, LP_OP_BROADCAST, weight, weight, nullptr, n, block, root, LP_REDUCE_SUM, 0.f, cuda_stream);
}

// 0 = no wait of this endpoint's kernels has given up so far (a peer that never arrived); synchronises the device.
int lp_chain_error(lp_chain *ch, int *error_out) {
    if (ch == nullptr || error_out == nullptr) return LP_ERR_INVALID_ARG;
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess)
        e = cudaMemcpy(error_out, (char *)ch->base + layout_of(ch->C, ch->S, ch->tile).error_off, sizeof(int), cudaMemcpyDeviceToHost);
    return e == cudaSuccess ? LP_OK : chain_fail(e);
}

// Channels per rank the emulation takes by default: LP_CHAIN_EMULATE_CHANNELS, fewer when P x 2 x channels CTAs would
// not all be resident on the current device (1 without a device).
int lp_chain_emulate_channels(int P, int tile) {
    if (tile == 0) tile = LP_CHAIN_DEFAULT_TILE;
    if (P < 1 || P > LP_MAX_P || !valid_geometry(1, 1, tile)) return 0;
    int cap = 0;
    if (resident(&cap) != cudaSuccess) {
        cudaGetLastError();
        return 1;
    }
    int c = cap / (2 * P);
    if (c > LP_CHAIN_EMULATE_CHANNELS) c = LP_CHAIN_EMULATE_CHANNELS;
    return c < 1 ? 1 : c;
}

// All P ranks of the chain on ONE device, in one cooperative launch: P x 2 x channels co-resident CTAs run the per-rank
// code above against P endpoints in this device's memory.
static int chain_emulate(int op, float *const *bufs, float *const *outs, int P, size_t n, size_t block, int root, int code,
                         size_t elem_bytes_total, float lr, int channels, int slots, int tile, void *cuda_stream,
                         float *vel = nullptr, float mu = 0.f) {
    if (slots == 0) slots = LP_CHAIN_DEFAULT_SLOTS;
    if (tile == 0) tile = LP_CHAIN_DEFAULT_TILE;
    if (channels == 0) channels = lp_chain_emulate_channels(P, tile);
    if (bufs == nullptr || P < 1 || P > LP_MAX_P || !valid_geometry(channels, slots, tile)) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_ALLREDUCE || chain_sgd(op)) root = 0;
    if (op == LP_OP_BSP_SGD_MOM && (vel == nullptr || ((uintptr_t)vel & 15u))) return LP_ERR_INVALID_ARG;
    lp_chain_role roles[LP_MAX_P];
    for (int r = 0; r < P; ++r) {
        const int rc = lp_chain_plan(op, P, root, r, &roles[r]);
        if (rc != LP_OK) return rc;
    }
    const float *all[2 * LP_MAX_P + 1];
    int m = 0;
    for (int r = 0; r < P; ++r) all[m++] = bufs[r];
    if (outs != bufs)
        for (int r = 0; r < P; ++r) all[m++] = outs[r];
    if (op == LP_OP_BSP_SGD_MOM) all[m++] = vel;
    for (int i = 0; i < m; ++i) {
        if (all[i] == nullptr || ((uintptr_t)all[i] & 15u)) return LP_ERR_INVALID_ARG;
        for (int q = 0; q < i; ++q) {
            const uintptr_t a = (uintptr_t)all[i], b = (uintptr_t)all[q];
            if (elem_bytes_total && a < b + elem_bytes_total && b < a + elem_bytes_total) return LP_ERR_INVALID_ARG;
        }
    }
    if (n == 0) return LP_OK;
    if (P == 1 && !chain_sgd(op)) return LP_OK;
    const EndpointLayout l = layout_of(channels, slots, tile);
    void *base = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_emul_mu);
        for (auto &e : g_emul)
            if (e.P == P && e.C == channels && e.S == slots && e.tile == tile && e.stream == (cudaStream_t)cuda_stream)
                base = e.base;
        if (base == nullptr) {
            // the endpoints of a (geometry, stream) are allocated and zeroed on first use: not under stream capture
            cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
            if (cudaStreamIsCapturing((cudaStream_t)cuda_stream, &cap) != cudaSuccess) cudaGetLastError();
            if (cap != cudaStreamCaptureStatusNone) return LP_ERR_UNSUPPORTED;
            cudaError_t e = cudaMalloc(&base, l.bytes * (size_t)P);
            if (e == cudaSuccess) e = cudaMemset(base, 0, l.bytes * (size_t)P);
            if (e == cudaSuccess) e = cudaDeviceSynchronize();
            if (e != cudaSuccess) {
                if (base) cudaFree(base);
                return chain_fail(e);
            }
            g_emul.push_back(EmulEndpoints{P, channels, slots, tile, (cudaStream_t)cuda_stream, base});
        }
    }
    LpChainLaunch L;
    memset(&L, 0, sizeof(L));
    L.n_local = P;
    L.C = channels;
    L.S = slots;
    L.code = code;
    L.lr = lr;
    L.mu = mu;
    L.invP = 1.0f / (float)P;
    L.spin_limit = 1ull << 23;  // all ranks start together here: a few seconds mean a bug
    L.part = chain_partition(n, block, tile, channels);
    L.tile = (uint32_t)tile;
    for (int r = 0; r < P; ++r) {
        char *b = (char *)base;
        fill_rank(L.rank[r], l, bufs[r], outs[r], chain_sgd(op) ? outs[r] : nullptr, op == LP_OP_BSP_SGD_MOM ? vel : nullptr,
                  b + l.bytes * (size_t)r,
                  b + l.bytes * (size_t)roles[r].up, b + l.bytes * (size_t)roles[r].down, roles[r]);
    }
    const cudaError_t e = launch(L, true, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? LP_OK : chain_fail(e);
}

int lp_chain_emulate(int op, float *const *bufs, int P, size_t n, size_t block, int root, int reduce_op, int channels,
                     int slots, int tile, void *cuda_stream) {
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return LP_ERR_INVALID_ARG;
    int code;
    const size_t bytes = n * sizeof(float);
    if (!chain_words(LP_DT_F32, reduce_op, n, block, code)) return LP_ERR_INVALID_ARG;
    return chain_emulate(op, bufs, bufs, P, n, block, root, code, bytes, 0.f, channels, slots, tile, cuda_stream);
}

int lp_chain_emulate_dt(int op, void *const *bufs, int P, size_t n, size_t block, int root, int dtype, int reduce_op,
                        int channels, int slots, int tile, void *cuda_stream) {
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return LP_ERR_INVALID_ARG;
    int code;
    const size_t bytes = n * (dtype == LP_DT_F64 ? 8 : (dtype == LP_DT_F32 ? 4 : 2));
    if (!chain_words(dtype, reduce_op, n, block, code)) return LP_ERR_INVALID_ARG;
    return chain_emulate(op, (float *const *)bufs, (float *const *)bufs, P, n, block, root, code, bytes, 0.f, channels, slots,
                         tile, cuda_stream);
}

int lp_chain_emulate_bsp_sgd_step(float *const *grads, float *const *weights, int P, size_t n, size_t block, float lr,
                                  int channels, int slots, int tile, void *cuda_stream) {
    if (weights == nullptr) return LP_ERR_INVALID_ARG;
    return chain_emulate(LP_OP_BSP_SGD, grads, weights, P, n, block, 0, LP_REDUCE_SUM, n * sizeof(float), lr, channels, slots,
                         tile, cuda_stream);
}

// reduce (one cooperative launch), GradientUpdate on the root's vectors, broadcast (one cooperative launch)
int lp_chain_emulate_bsp_sgd_alg2_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                       size_t block, int root, float lr, float mu, int channels, int slots, int tile,
                                       void *cuda_stream) {
    if (weights == nullptr || grads == nullptr || P < 1 || P > LP_MAX_P || root < 0 || root >= P) return LP_ERR_INVALID_ARG;
    int rc = chain_emulate(LP_OP_REDUCE, grads, grads, P, n, block, root, LP_REDUCE_SUM, n * sizeof(float), 0.f, channels, slots,
                           tile, cuda_stream);
    if (rc != LP_OK) return rc;
    if (weights[root] == nullptr || ((uintptr_t)weights[root] & 15u)) return LP_ERR_INVALID_ARG;
    if (n > 0) {
        const cudaError_t e = lp_update_launch(weights[root], grads[root], velocity, n, lr, 1.0f / (float)P, mu,
                                               (cudaStream_t)cuda_stream, false);
        if (e != cudaSuccess) return chain_fail(e);
    }
    return chain_emulate(LP_OP_BROADCAST, weights, weights, P, n, block, root, LP_REDUCE_SUM, n * sizeof(float), 0.f, channels,
                         slots, tile, cuda_stream);
}

int lp_chain_emulate_bsp_sgd_momentum_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n,
                                           size_t block, float lr, float mu, int channels, int slots, int tile,
                                           void *cuda_stream) {
    if (weights == nullptr) return LP_ERR_INVALID_ARG;
    return chain_emulate(LP_OP_BSP_SGD_MOM, grads, weights, P, n, block, 0, LP_REDUCE_SUM, n * sizeof(float), lr, channels,
                         slots, tile, cuda_stream, velocity, mu);
}

// error word of emulated rank `rank` for the geometry (P, channels, slots, tile); synchronises the device
int lp_chain_emulate_error(int P, int channels, int slots, int tile, int *error_out) {
    if (slots == 0) slots = LP_CHAIN_DEFAULT_SLOTS;
    if (tile == 0) tile = LP_CHAIN_DEFAULT_TILE;
    if (channels == 0) channels = lp_chain_emulate_channels(P, tile);
    if (error_out == nullptr || !valid_geometry(channels, slots, tile)) return LP_ERR_INVALID_ARG;
    *error_out = 0;
    std::vector<void *> bases;  // the endpoints of this geometry on every stream they were used on
    {
        std::lock_guard<std::mutex> lock(g_emul_mu);
        for (auto &e : g_emul)
            if (e.P == P && e.C == channels && e.S == slots && e.tile == tile) bases.push_back(e.base);
    }
    if (bases.empty()) return LP_OK;
    cudaError_t e = cudaDeviceSynchronize();
    const EndpointLayout l = layout_of(channels, slots, tile);
    for (void *base : bases)
        for (int r = 0; r < P && e == cudaSuccess; ++r) {
            int w = 0;
            e = cudaMemcpy(&w, (char *)base + l.bytes * (size_t)r + l.error_off, sizeof(int), cudaMemcpyDeviceToHost);
            if (w) *error_out = w;
        }
    return e == cudaSuccess ? LP_OK : chain_fail(e);
}

}  // extern "C"
