// lp_seg.cu -- the one kernel the MST and BE baselines are built from: a batch of whole-segment jobs
// dst = a + b (fp32 RN) or dst = a, one grid.y slice per job.  PAPER.md:200: in MST/BE "GPUs reduce the
// incoming data only after the entire data is available" -- every tree level / exchange step is one such
// launch over whole messages (MST) or whole halves (BE), reading the partner's buffer directly (the most
// favourable same-GPU realisation: no staging copy).
#include "lp_common.cuh"

namespace {

struct LpSegArgs {
    LpSegJob j[LP_MAX_JOBS];
};

constexpr int kSegThreads = 256;
constexpr int kSegUnroll = 4;

__global__ void __launch_bounds__(kSegThreads) lp_seg_kernel(const __grid_constant__ LpSegArgs s) {
    const LpSegJob &job = s.j[blockIdx.y];
    float *dst = job.dst;
    const float *a = job.a;
    const float *b = job.b;
    const uint64_t len = job.len;
    const uint64_t gtid = (uint64_t)blockIdx.x * kSegThreads + threadIdx.x;
    const uint64_t gsize = (uint64_t)gridDim.x * kSegThreads;
    const uint32_t mis = (uint32_t)((uintptr_t)dst & 15u);
    const bool same = ((uintptr_t)a & 15u) == mis && (b == nullptr || ((uintptr_t)b & 15u) == mis);
    if (!same) {  // operands disagree on alignment: element-wise (never the case for the MST / BE segments)
        for (uint64_t i = gtid; i < len; i += gsize) dst[i] = b ? __fadd_rn(a[i], b[i]) : a[i];
        return;
    }
    uint64_t head = ((16u - mis) & 15u) >> 2;
    if (head > len) head = len;
    const uint64_t nvec = (len - head) >> 2;
    const uint64_t tail0 = head + (nvec << 2);
    if (gtid < head) dst[gtid] = b ? __fadd_rn(a[gtid], b[gtid]) : a[gtid];
    if (gtid < len - tail0) dst[tail0 + gtid] = b ? __fadd_rn(a[tail0 + gtid], b[tail0 + gtid]) : a[tail0 + gtid];
    float *d4 = dst + head;
    const float *a4 = a + head;
    const float *b4 = b ? b + head : nullptr;
    for (uint64_t v0 = gtid; v0 < nvec; v0 += gsize * kSegUnroll) {
        float4 x[kSegUnroll], y[kSegUnroll];
#pragma unroll
        for (int u = 0; u < kSegUnroll; ++u) {
            const uint64_t v = v0 + (uint64_t)u * gsize;
            if (v < nvec) {
                x[u] = lp_ldg_stream(a4 + 4 * v);
                if (b4) y[u] = lp_ldg_stream(b4 + 4 * v);
            }
        }
#pragma unroll
        for (int u = 0; u < kSegUnroll; ++u) {
            const uint64_t v = v0 + (uint64_t)u * gsize;
            if (v < nvec) lp_stg_stream(d4 + 4 * v, b4 ? lp_add4(x[u], y[u]) : x[u]);
        }
    }
}

}  // namespace

cudaError_t lp_seg_launch(const LpSegJob *jobs, int n_jobs, int sm_count, cudaStream_t stream) {
    LpSegArgs s;
    int m = 0;
    uint64_t longest = 0;
    for (int i = 0; i < n_jobs; ++i) {
        if (jobs[i].len == 0) continue;
        s.j[m++] = jobs[i];
        if (jobs[i].len > longest) longest = jobs[i].len;
    }
    if (m == 0) return cudaSuccess;
    for (int i = m; i < LP_MAX_JOBS; ++i) s.j[i] = LpSegJob{nullptr, nullptr, nullptr, 0};
    // enough CTAs over all jobs to fill the chip 8 deep, no more than the longest job needs
    uint64_t per_job = ((uint64_t)sm_count * 8 + m - 1) / m;
    uint64_t need = (longest / 4 + (uint64_t)kSegThreads * kSegUnroll - 1) / ((uint64_t)kSegThreads * kSegUnroll);
    if (need == 0) need = 1;
    if (per_job > need) per_job = need;
    dim3 grid((unsigned)per_job, (unsigned)m, 1);
    lp_count_launch(1);
    lp_seg_kernel<<<grid, kSegThreads, 0, stream>>>(s);
    return cudaGetLastError();
}
