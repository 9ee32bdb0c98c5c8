// lp_probe.cu -- lp_hbm_probe: the HBM ceiling of a read : write mix, measured with the plainest possible kernel.
// One thread per 16-byte vector index i: it loads vector i of each of the n_read inputs (all loads issued before the
// first use), sums them so that no load can be dropped, and stores the sum to vector i of each of the n_write
// outputs.  No schedule, no shared memory, no claims, no fold order: what it reaches is what HBM + L2 give a kernel
// that asks for this mix of streams, and bench.py quotes the LP collectives against it (broadcast = 1 : P-1,
// reduce = P : 1, allreduce = P : P).  Measurement aid; not on the collectives' path.
#include "lp_common.cuh"

namespace {

struct LpProbeArgs {
    const float *in[2 * LP_MAX_P];
    float *out[2 * LP_MAX_P];
    int n_read, n_write;
    int late_wait;  // as the collectives' kernels: lp_chain_admit
    uint64_t nvec;
};

constexpr int kProbeThreads = 256;
constexpr int kProbeUnroll = 4;

template <int NR>
__device__ __forceinline__ void lp_probe_body(const LpProbeArgs &p);

template <int NR>  // NR > 0: read streams known at compile time (all loads of a thread in flight at once)
__global__ void __launch_bounds__(kProbeThreads) lp_probe_kernel(const __grid_constant__ LpProbeArgs p) {
    // launched like the collectives' kernels: programmatic dependent launch, and no wait for the launches ahead when
    // it touches none of their buffers -- the ceiling is measured under the conditions the collectives run in
    if (!p.late_wait) lp_pdl_wait();
    lp_pdl_trigger();
    lp_probe_body<NR>(p);
    if (p.late_wait && threadIdx.x == 0) lp_pdl_wait();
}

template <int NR>
__device__ __forceinline__ void lp_probe_body(const LpProbeArgs &p) {
    const uint64_t v0 = (uint64_t)blockIdx.x * (kProbeThreads * kProbeUnroll) + threadIdx.x;
    float4 acc[kProbeUnroll];
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) acc[u] = make_float4(1.f, 2.f, 3.f, 4.f);
    const int n_read = NR > 0 ? NR : p.n_read;
    for (int r0 = 0; r0 < n_read; r0 += 4) {
        float4 x[4][kProbeUnroll];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (r0 + j < n_read) {
#pragma unroll
                for (int u = 0; u < kProbeUnroll; ++u) {
                    const uint64_t v = v0 + (uint64_t)u * kProbeThreads;
                    if (v < p.nvec) x[j][u] = lp_ldg_stream(p.in[r0 + j] + 4 * v);
                }
            }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (r0 + j < n_read) {
#pragma unroll
                for (int u = 0; u < kProbeUnroll; ++u) acc[u] = lp_add4(acc[u], x[j][u]);
            }
    }
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) {
        const uint64_t v = v0 + (uint64_t)u * kProbeThreads;
        if (v >= p.nvec) continue;
        for (int q = 0; q < p.n_write; ++q) lp_stg_stream(p.out[q] + 4 * v, acc[u]);
        // read-only probe: keep the loads alive without writing (the sum of finite inputs is never this NaN pattern)
        if (p.n_write == 0 && __float_as_uint(acc[u].x) == 0x7fc12345u) lp_stg_stream(const_cast<float *>(p.in[0]) + 4 * v, acc[u]);
    }
}

}  // namespace

cudaError_t lp_probe_launch(float *const *bufs, int n_read, int n_write, size_t n, cudaStream_t stream) {
    LpProbeArgs p;
    memset(&p, 0, sizeof(p));
    for (int r = 0; r < n_read; ++r) p.in[r] = bufs[r];
    for (int q = 0; q < n_write; ++q) p.out[q] = bufs[n_read + q];
    p.n_read = n_read;
    p.n_write = n_write;
    p.nvec = (uint64_t)n >> 2;
    if (p.nvec == 0) return cudaSuccess;
    const uint64_t per = (uint64_t)kProbeThreads * kProbeUnroll;
    const uint64_t grid = (p.nvec + per - 1) / per;
    if (grid > 0x7fffffffull) return cudaErrorInvalidValue;
    lp_count_launch(1);
    {
        LpRange ranges[4 * LP_MAX_P];
        for (int i = 0; i < n_read + n_write; ++i) ranges[i] = LpRange{(uintptr_t)bufs[i], (uintptr_t)bufs[i] + (uintptr_t)n * 4u};
        p.late_wait = lp_chain_admit(stream, ranges, n_read + n_write, true, true) ? 1 : 0;
    }
    const dim3 g((unsigned)grid), b(kProbeThreads);
    switch (n_read) {
        case 1: return lp_launch(lp_probe_kernel<1>, g, b, 0, stream, true, p);
        case 2: return lp_launch(lp_probe_kernel<2>, g, b, 0, stream, true, p);
        case 4: return lp_launch(lp_probe_kernel<4>, g, b, 0, stream, true, p);
        default: return lp_launch(lp_probe_kernel<0>, g, b, 0, stream, true, p);
    }
}
