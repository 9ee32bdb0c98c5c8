// lp_seg.cu -- the one kernel the MST and BE baselines are built from: a batch of whole-segment jobs
// dst = a + b (fp32 RN) or dst = a, one grid.y slice per job.  PAPER.md:200: in MST/BE "GPUs reduce the
// incoming data only after the entire data is available" -- every tree level / exchange step is one such
// launch over whole messages (MST) or whole halves (BE), reading the partner's buffer directly (the most
// favourable same-GPU realisation: no staging copy).
#include "lp_common.cuh"

namespace {

struct LpSegArgs {
    LpSegJob j[LP_MAX_JOBS];
    int code;  // (dtype << 1) | red_op: the operator of dst = a op b and the element type (lp_common.cuh)
    int late_wait;  // lp_chain_admit: wait for the launches ahead at the end of the CTA instead of at its start
};

constexpr int kSegThreads = 256;
constexpr int kSegUnroll = 4;

__device__ __forceinline__ void lp_seg_body(const LpSegArgs &s);

__global__ void __launch_bounds__(kSegThreads) lp_seg_kernel(const __grid_constant__ LpSegArgs s) {
    if (!s.late_wait) {
        // like the LP direct kernel (the baselines get every launch-side advantage LP has): this CTA's chunk of both
        // operands into L2 while the previous level drains; L2 is the point of coherence, so lines the previous level
        // is still writing end up with its values
        const LpSegJob &job = s.j[blockIdx.y];
        const uint64_t per = (uint64_t)kSegThreads * kSegUnroll * 4;
        const uint64_t lo = (uint64_t)blockIdx.x * per;
        if (lo < job.len) {
            const uint64_t n = job.len - lo < per ? job.len - lo : per;
            const uint32_t lines = (uint32_t)((n * 4u + 127u) / 128u);
            for (uint32_t l = threadIdx.x; l < 2u * lines; l += kSegThreads) {
                const float *base = l < lines ? job.a : job.b;
                if (base) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + lo + (uint64_t)(l < lines ? l : l - lines) * 32u));
            }
        }
        lp_pdl_wait();  // the previous level (or whatever precedes in the stream) has completed
    }
    lp_pdl_trigger();  // one chunk per CTA: once the last CTA is resident the next level's kernel may be scheduled
    lp_seg_body(s);
    if (s.late_wait && threadIdx.x == 0) lp_pdl_wait();
}

__device__ __forceinline__ void lp_seg_body(const LpSegArgs &s) {
    const LpSegJob &job = s.j[blockIdx.y];
    const int code = s.code;
    float *dst = job.dst;
    const float *a = job.a;
    const float *b = job.b;
    const uint64_t len = job.len;
    // One CTA per chunk of kSegThreads * kSegUnroll 16-byte vectors: the hardware block scheduler hands chunks to
    // SMs as they free up, so (as with the LP kernels' tile claims) no SM is left with a fixed share to finish alone.
    const uint32_t mis = (uint32_t)((uintptr_t)dst & 15u);
    const bool same = ((uintptr_t)a & 15u) == mis && (b == nullptr || ((uintptr_t)b & 15u) == mis);
    if (!same) {  // operands disagree on alignment: element-wise (never the case for the MST / BE segments)
        const uint64_t per = (uint64_t)kSegThreads * kSegUnroll * 4;
        const uint64_t lo = (uint64_t)blockIdx.x * per;
        const uint64_t hi = lo + per < len ? lo + per : len;
        for (uint64_t i = lo + threadIdx.x; i < hi; i += kSegThreads) lp_word_combine_store(dst, a, b, i, code);
        return;
    }
    uint64_t head = ((16u - mis) & 15u) >> 2;
    if (head > len) head = len;
    const uint64_t nvec = (len - head) >> 2;
    const uint64_t tail0 = head + (nvec << 2);
    if (blockIdx.x == 0) {
        const uint64_t i = threadIdx.x;
        if (i < head) lp_word_combine_store(dst, a, b, i, code);
        if (i < len - tail0) lp_word_combine_store(dst, a, b, tail0 + i, code);
    }
    float *d4 = dst + head;
    const float *a4 = a + head;
    const float *b4 = b ? b + head : nullptr;
    const uint64_t v0 = (uint64_t)blockIdx.x * (kSegThreads * kSegUnroll) + threadIdx.x;
    float4 x[kSegUnroll], y[kSegUnroll];
#pragma unroll
    for (int u = 0; u < kSegUnroll; ++u) {
        const uint64_t v = v0 + (uint64_t)u * kSegThreads;
        if (v < nvec) {
            x[u] = lp_ldg_stream(a4 + 4 * v);
            if (b4) y[u] = lp_ldg_stream(b4 + 4 * v);
        }
    }
#pragma unroll
    for (int u = 0; u < kSegUnroll; ++u) {
        const uint64_t v = v0 + (uint64_t)u * kSegThreads;
        if (v < nvec) lp_stg_stream(d4 + 4 * v, b4 ? lp_combine4(x[u], y[u], code) : x[u]);
    }
}

// GradientUpdate of Alg. 2 on the root replica: one thread per 16-byte vector (hardware-scheduled CTAs), scalar
// path for misaligned ends.  Same rounded operations as the fused epilogues (lp_sgd1 / lp_mom1).
__global__ void __launch_bounds__(kSegThreads) lp_update_kernel(float *w, const float *S, float *vel, uint64_t n, float lr,
                                                                float invP, float mu) {
    lp_pdl_wait();
    lp_pdl_trigger();
    const uint64_t nvec = n >> 2;
    const uint64_t v = (uint64_t)blockIdx.x * kSegThreads + threadIdx.x;
    if (v < nvec) {
        const float4 s4 = lp_ldg_stream(S + 4 * v);
        const float4 w4 = lp_ldg_stream(w + 4 * v);
        if (vel) {
            const float4 v4 = lp_ldg_stream(vel + 4 * v);
            float4 vn, wn;
            lp_mom4(s4, w4, v4, lr, invP, mu, vn, wn);
            lp_stg_stream(vel + 4 * v, vn);
            lp_stg_stream(w + 4 * v, wn);
        } else {
            lp_stg_stream(w + 4 * v, lp_sgd4(s4, w4, lr, invP));
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < (n & 3u)) {
        const uint64_t i = (nvec << 2) + threadIdx.x;
        if (vel) {
            float vn, wn;
            lp_mom1(S[i], w[i], vel[i], lr, invP, mu, vn, wn);
            vel[i] = vn;
            w[i] = wn;
        } else {
            w[i] = lp_sgd1(S[i], w[i], lr, invP);
        }
    }
}

// The odd last element of a 16-bit vector (it fills half a 4-byte word, so the word-addressed kernels stop before it):
// one thread folds element e of every input in chain order and writes it to every output.  The element rides in the
// low half of a two-element word whose high half is zero (0 op 0 raises nothing and is dropped).
__global__ void lp_tail16_kernel(const __grid_constant__ LpArgs a, uint64_t e) {
    lp_pdl_wait();
    if (threadIdx.x != 0) return;
    const int code = lp_fold_code(a.dtype, a.red_op);
    float s = __uint_as_float((uint32_t) reinterpret_cast<const unsigned short *>(a.in[0])[e]);
    for (int r = 1; r < a.n_sum; ++r)
        s = lp_combine1(s, __uint_as_float((uint32_t) reinterpret_cast<const unsigned short *>(a.in[r])[e]), code);
    for (int q = 0; q < a.n_out; ++q)
        reinterpret_cast<unsigned short *>(a.out[q])[e] = (unsigned short)(__float_as_uint(s) & 0xffffu);
}

}  // namespace

cudaError_t lp_tail16_launch(const LpArgs &a, uint64_t elem, cudaStream_t stream, bool pdl) {
    lp_count_launch(1);
    lp_chain_reset(stream);  // waits first; touches the last bytes of every vector of the launch ahead of it
    return lp_launch(lp_tail16_kernel, dim3(1), dim3(32), 0, stream, pdl, a, elem);
}

cudaError_t lp_update_launch(float *w, const float *S, float *velocity, uint64_t n, float lr, float invP, float mu,
                             cudaStream_t stream, bool pdl) {
    if (n == 0) return cudaSuccess;
    const uint64_t blocks = ((n >> 2) + kSegThreads - 1) / kSegThreads + ((n >> 2) == 0 ? 1 : 0);
    if (blocks > 0x7fffffffull) return cudaErrorInvalidValue;
    lp_count_launch(1);
    lp_chain_reset(stream);  // waits first, reads and rewrites what its neighbours in the stream touch
    return lp_launch(lp_update_kernel, dim3((unsigned)blocks), dim3(kSegThreads), 0, stream, pdl, w, S, velocity,
                     (uint64_t)n, lr, invP, mu);
}

cudaError_t lp_seg_launch(const LpSegJob *jobs, int n_jobs, int sm_count, cudaStream_t stream, bool pdl, int red_op,
                          bool chain, int dtype) {
    LpSegArgs s;
    s.code = (dtype << 1) | red_op;
    int m = 0;
    uint64_t longest = 0;
    for (int i = 0; i < n_jobs; ++i) {
        if (jobs[i].len == 0) continue;
        s.j[m++] = jobs[i];
        if (jobs[i].len > longest) longest = jobs[i].len;
    }
    if (m == 0) return cudaSuccess;
    for (int i = m; i < LP_MAX_JOBS; ++i) s.j[i] = LpSegJob{nullptr, nullptr, nullptr, 0};
    // one CTA per chunk of the longest job (shorter jobs' surplus CTAs return at once)
    (void)sm_count;
    const uint64_t chunk = (uint64_t)kSegThreads * kSegUnroll * 4;  // elements
    uint64_t per_job = (longest + chunk - 1) / chunk + 1;           // + 1: a misaligned head shifts the body
    if (per_job > 0x7fffffffull) return cudaErrorInvalidValue;
    dim3 grid((unsigned)per_job, (unsigned)m, 1);
    lp_count_launch(1);
    {
        LpRange ranges[3 * LP_MAX_JOBS];
        int nr = 0;
        for (int i = 0; i < m; ++i) {
            const uintptr_t bytes = (uintptr_t)s.j[i].len * 4u;
            ranges[nr++] = LpRange{(uintptr_t)s.j[i].dst, (uintptr_t)s.j[i].dst + bytes};
            ranges[nr++] = LpRange{(uintptr_t)s.j[i].a, (uintptr_t)s.j[i].a + bytes};
            if (s.j[i].b) ranges[nr++] = LpRange{(uintptr_t)s.j[i].b, (uintptr_t)s.j[i].b + bytes};
        }
        s.late_wait = lp_chain_admit(stream, ranges, nr, pdl, chain) ? 1 : 0;
    }
    return lp_launch(lp_seg_kernel, grid, dim3(kSegThreads), 0, stream, pdl, s);
}
