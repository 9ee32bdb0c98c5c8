// lp_chain.cuh -- what the chain's kernels (lp_chain.cu) and its host side (lp_chain_api.cu) share: the per-rank argument
// block, the launch descriptor and the two launch helpers.
#pragma once
#include "lp_common.cuh"

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


// CTAs of the selected chain kernel (tma: the default, TMA-load kernel; else the register kernel) the current device
// holds at once.
cudaError_t lp_chain_resident(bool tma, int *ctas);
// grid = n_local x 2 C CTAs; cooperative: every CTA of the grid co-resident by contract (the one-GPU emulation).
cudaError_t lp_chain_launch_kernel(const LpChainLaunch &L, bool tma, bool cooperative, cudaStream_t stream);
