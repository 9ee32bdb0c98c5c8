// lp_copy_engine.cu -- LP_VARIANT_COPY_ENGINE: the paper's own realisation of the Linear Pipeline, kept as a
// mirror and a baseline (a9).  PAPER.md:55-59: per hop and block, "a GPU receives a block from the prior GPU
// via DMA1 while sending a block to the next one via DMA2" = one cudaMemcpyAsync of the block into the next
// rank's receive buffer ("writing block a0 to a buffer on GPU1"), then one add kernel ("GPU1 reduces the
// received block a0 with a1 to yield a'").  PAPER.md:73: "the data transfers are asynchronous launched on two
// separate streams", alternating -- block k runs on stream k mod S (S = 2, U17) and uses receive slot k mod S,
// so slot reuse is ordered by the stream and consecutive blocks overlap.  Allreduce sends the finished block
// back down the chain (U3 reading A); the fused SGD step applies the update at the last rank and sends w'.
// On one B200 this is bound by launch / copy-submission overhead (2-3 operations per hop per block), which
// is exactly why the product path is the persistent kernel.
#include <mutex>

#include "lp_common.cuh"

namespace {

// The side streams, their events and the receive slots are one set per process: calls of this variant are enqueued
// one at a time (g_ce_mu) and run one after the other on the side streams, whatever streams the callers use.
std::mutex g_ce_mu;
constexpr int kMaxStreams = 8;
cudaStream_t g_side[kMaxStreams];
cudaEvent_t g_fork, g_join[kMaxStreams];
int g_n_side = 0;
bool g_events = false;

#define LP_TRY(x)                           \
    do {                                    \
        cudaError_t e__ = (x);              \
        if (e__ != cudaSuccess) return e__; \
    } while (0)

cudaError_t ensure_streams(int S) {
    if (!g_events) {
        LP_TRY(cudaEventCreateWithFlags(&g_fork, cudaEventDisableTiming));
        for (int s = 0; s < kMaxStreams; ++s) LP_TRY(cudaEventCreateWithFlags(&g_join[s], cudaEventDisableTiming));
        g_events = true;
    }
    while (g_n_side < S) {
        LP_TRY(cudaStreamCreateWithFlags(&g_side[g_n_side], cudaStreamNonBlocking));
        ++g_n_side;
    }
    return cudaSuccess;
}

// dst = w - lr * (s * invP), three RN ops (U7), or with vel != NULL the momentum form (U18: vel updated in place);
// element-wise, any alignment.
__global__ void lp_ce_sgd_kernel(float *dst, const float *s, const float *w, float *vel, uint64_t len, float lr, float invP,
                                 float mu) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < len; i += (uint64_t)gridDim.x * blockDim.x) {
        if (vel) {
            float vn, wn;
            lp_mom1(s[i], w[i], vel[i], lr, invP, mu, vn, wn);
            vel[i] = vn;
            dst[i] = wn;
        } else {
            dst[i] = lp_sgd1(s[i], w[i], lr, invP);
        }
    }
}

cudaError_t copy_block(float *dst, const float *src, uint64_t len, cudaStream_t st) {
    lp_count_launch(1);
    return cudaMemcpyAsync(dst, src, len * sizeof(float), cudaMemcpyDeviceToDevice, st);
}

}  // namespace

void lp_copy_engine_shutdown() {
    std::lock_guard<std::mutex> lock(g_ce_mu);
    for (int s = 0; s < g_n_side; ++s) cudaStreamDestroy(g_side[s]);
    g_n_side = 0;
    if (g_events) {
        cudaEventDestroy(g_fork);
        for (int s = 0; s < kMaxStreams; ++s) cudaEventDestroy(g_join[s]);
        g_events = false;
    }
}

// op: LP_OP_*.  For LP_OP_BSP_SGD `bufs` are the gradients and `weights` the replicas.
cudaError_t lp_copy_engine_run(int op, int red_op, float *const *bufs, float *const *weights, float *velocity, int P,
                               size_t n, size_t block, int root, float lr, float mu, const LpTuning &t, int sm_count,
                               cudaStream_t stream, int dtype) {
    std::lock_guard<std::mutex> lock(g_ce_mu);
    const bool sgd = (op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM);
    if (n == 0) return cudaSuccess;
    if (P == 1 && !sgd) return cudaSuccess;
    int S = t.v[LP_TUNE_CE_STREAMS] ? t.v[LP_TUNE_CE_STREAMS] : 2;
    if (S > kMaxStreams) S = kMaxStreams;
    if (block > n) block = n;
    const uint64_t nb = (n + block - 1) / block;
    LP_TRY(ensure_streams(S));

    // receive buffers: rank r >= 1 owns S slots of one block; reserved before anything is enqueued
    float *recv[LP_MAX_P] = {nullptr};
    const bool reduces = (op != LP_OP_BROADCAST);
    if (reduces)
        for (int r = (P == 1 ? 0 : 1); r < P; ++r)
            LP_TRY(lp_scratch_get(LP_SCRATCH_SHARED, LP_MAX_P + r, (size_t)S * (block + 4) * sizeof(float), &recv[r]));

    LP_TRY(cudaEventRecord(g_fork, stream));
    for (int s = 0; s < S; ++s) LP_TRY(cudaStreamWaitEvent(g_side[s], g_fork, 0));

    const float invP = 1.0f / (float)P;
    for (uint64_t k = 0; k < nb; ++k) {
        const int s = (int)(k % (uint64_t)S);
        cudaStream_t st = g_side[s];
        const uint64_t off = k * block;
        const uint64_t len = off + block <= n ? block : n - off;
        if (op == LP_OP_BROADCAST) {
            // chain root -> root+1 -> ... (GPU0 is the source, each GPU forwards what it received)
            for (int j = 0; j + 1 < P; ++j)
                LP_TRY(copy_block(bufs[(root + j + 1) % P] + off, bufs[(root + j) % P] + off, len, st));
            continue;
        }
        // reduce chain 0 -> 1 -> ... -> P-1 (U4); the slot keeps the 16-byte phase of `off`
        const float *partial = bufs[0] + off;
        for (int r = 1; r < P; ++r) {
            float *slot = recv[r] + (size_t)s * (block + 4) + (off & 3);
            LP_TRY(copy_block(slot, partial, len, st));  // DMA: partial of rank r-1 -> receive buffer of rank r
            float *dst = slot;
            if (r == P - 1 && op == LP_OP_REDUCE) dst = bufs[root] + off;  // "returns the combined value ... to a specific GPU"
            if (r == P - 1 && op == LP_OP_ALLREDUCE) dst = bufs[P - 1] + off;
            LpSegJob job{dst, slot, bufs[r] + off, len};  // partial op local block, RN
            LP_TRY(lp_seg_launch(&job, 1, sm_count, st, false, red_op, false, dtype));
            partial = dst;
        }
        if (op == LP_OP_ALLREDUCE) {
            // finished block flows back P-1 -> P-2 -> ... -> 0 ("a'' is broadcast"; U3-A)
            for (int r = P - 1; r > 0; --r) LP_TRY(copy_block(bufs[r - 1] + off, bufs[r] + off, len, st));
        } else if (sgd) {
            // last rank: w' = w_root - lr * (S / P), then w' to every replica
            float *s_ptr;
            if (P == 1) {
                s_ptr = recv[0] + (size_t)s * (block + 4) + (off & 3);
                LP_TRY(copy_block(s_ptr, bufs[0] + off, len, st));
            } else {
                s_ptr = const_cast<float *>(partial);
            }
            unsigned grid = (unsigned)((len + 255) / 256);
            if (grid > (unsigned)sm_count * 8u) grid = (unsigned)sm_count * 8u;
            lp_count_launch(1);
            lp_ce_sgd_kernel<<<grid, 256, 0, st>>>(weights[P - 1] + off, s_ptr, weights[root] + off,
                                                   op == LP_OP_BSP_SGD_MOM ? velocity + off : nullptr, len, lr, invP, mu);
            LP_TRY(cudaGetLastError());
            for (int r = P - 1; r > 0; --r) LP_TRY(copy_block(weights[r - 1] + off, weights[r] + off, len, st));
        }
    }
    for (int s = 0; s < S; ++s) {
        LP_TRY(cudaEventRecord(g_join[s], g_side[s]));
        LP_TRY(cudaStreamWaitEvent(stream, g_join[s], 0));
    }
    return cudaSuccess;
}
