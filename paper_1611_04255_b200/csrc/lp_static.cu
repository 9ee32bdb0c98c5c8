// lp_static.cu -- lp_mst_reduce_static: the MST (binomial tree) reduce of PAPER.md:93 for callers that must not
// allocate device memory.
//
// Why it exists.  lp_mst_reduce leaves the non-root buffers unchanged (U5), so the partial sums that the non-root
// ranks of the tree build need working copies; the regular entry point takes them from library scratch that it
// cudaMallocs (and, when a longer message comes, cudaFrees and reallocates) on demand.  Some callers cannot afford that:
//   * a training process that has handed all of the GPU's memory to its framework's pool allocator -- a cudaMalloc
//     from a library then fails with out-of-memory although the pool has room;
//   * a step loop that must never stall: cudaMalloc may, and cudaFree does, synchronise the whole device, so a
//     collective that grows its scratch in iteration k stops every other stream of the process;
//   * a thread that runs while another thread of the process holds a stream capture in the default (global) capture
//     mode, where cudaMalloc from any thread is refused.
// This file gives them one entry point that calls no cudaMalloc, cudaFree or any other allocating routine: the
// working copies live in the file-scope device array below, which is part of the loaded library image.
//
// What it costs.  Every GPU on which this library's code is loaded holds LP_STATIC_SCRATCH_BYTES (16 MiB) from the
// moment the module is loaded until the process exits, whether or not this entry point is ever called, and a call
// whose working copies do not fit is refused (lp_mst_reduce_static_max_n).  All calls of the process on one GPU share
// the one array: two calls that may run at the same time on the device (different streams, or graphs replayed side by
// side) race on it and corrupt each other's partial sums -- keep calls to this entry point on one stream per GPU, or
// order them with events.  The array keeps whatever the last call left in it; the tree writes every word of a
// working copy before it reads it (level d = 1 stores x_v + x_{v+1} there), so nothing has to start at zero and
// nothing is cleared.
//
// Set-up.  In host code the array's name is not a device address (it is the host-side shadow the runtime uses to look
// the symbol up); the device address is fetched with cudaGetSymbolAddress, once per device, with that device current,
// on the first call made there, and cached.  That first call also makes the runtime load this module on the device.
// Make the first call on each device before any stream capture begins.
//
// The file shares nothing with the rest of the library (own kernel, own validation, plain stream-ordered launches, no
// tile-claim counters, no library scratch, no device binding), so it changes no existing code path.  Values: the same
// tree, the same fp32 round-to-nearest adds in the same order as lp_mst_reduce -> bit-identical results.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/lp_collectives.h"

namespace {

// The working copies of every call.  256-byte aligned so that each copy starts on the same 16-byte phase as the
// callers' (16-byte aligned) buffers and on a DRAM-friendly boundary.
static __device__ __align__(256) unsigned char lp_static_scratch[LP_STATIC_SCRATCH_BYTES];

constexpr int kThreads = 256;
constexpr int kUnroll = 4;                          // 16-byte vectors per thread
constexpr uint64_t kChunk = (uint64_t)kThreads * kUnroll * 4;  // floats per CTA
constexpr size_t kCopyAlign = 64;                   // floats: every working copy starts on a 256-byte boundary
constexpr int kMaxDevices = 64;
constexpr int kMaxJobs = LP_MAX_P / 2;              // pairs of one tree level

struct StaticJob {
    float *dst;      // x_v's new home: the root's buffer (v = 0) or a working copy
    const float *a;  // x_v
    const float *b;  // x_{v+d}
};
struct StaticLevel {
    StaticJob j[kMaxJobs];
    uint64_t n;
};

// One tree level: dst[i] = a[i] + b[i] (one fp32 RN add) for every pair of the level; blockIdx.y = pair.  All three
// pointers are 16-byte aligned (validated buffers, 256-byte aligned copies).
__global__ void __launch_bounds__(kThreads) lp_static_level_kernel(const __grid_constant__ StaticLevel L) {
    const StaticJob &job = L.j[blockIdx.y];
    const uint64_t nvec = L.n >> 2;
    const float4 *a4 = reinterpret_cast<const float4 *>(job.a);
    const float4 *b4 = reinterpret_cast<const float4 *>(job.b);
    float4 *d4 = reinterpret_cast<float4 *>(job.dst);
    const uint64_t v0 = (uint64_t)blockIdx.x * (kThreads * kUnroll) + threadIdx.x;
    float4 x[kUnroll], y[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
        const uint64_t v = v0 + (uint64_t)u * kThreads;
        if (v < nvec) {
            x[u] = a4[v];
            y[u] = b4[v];
        }
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
        const uint64_t v = v0 + (uint64_t)u * kThreads;
        if (v < nvec)
            d4[v] = make_float4(__fadd_rn(x[u].x, y[u].x), __fadd_rn(x[u].y, y[u].y), __fadd_rn(x[u].z, y[u].z),
                                __fadd_rn(x[u].w, y[u].w));
    }
    if (blockIdx.x == 0 && threadIdx.x < (L.n & 3u)) {  // the last 1..3 floats
        const uint64_t i = (nvec << 2) + threadIdx.x;
        job.dst[i] = __fadd_rn(job.a[i], job.b[i]);
    }
}

std::mutex g_static_mu;
float *g_static_base[kMaxDevices] = {nullptr};  // device address of lp_static_scratch, per device ordinal
thread_local char t_static_err[256] = "";

int fail(int status, const char *msg) {
    snprintf(t_static_err, sizeof(t_static_err), "%s", msg);
    return status;
}
int cuda_fail(cudaError_t e, const char *where) {
    snprintf(t_static_err, sizeof(t_static_err), "lp_mst_reduce_static: CUDA error in %s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();
    return LP_ERR_CUDA;
}

// Working copies a P-rank tree needs: the virtual ranks v = 2, 4, ... with v + 1 < P receive at level d = 1 and are not
// the root (every receiver of a later level is among them).
int n_copies(int P) { return P >= 4 ? (P - 2) / 2 : 0; }
size_t copy_stride(size_t n) { return (n + kCopyAlign - 1) / kCopyAlign * kCopyAlign; }  // floats

// Device address of the array on the current device; looked up on the first call there.
int scratch_base(float **base) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice (no CUDA device: there is no CPU fallback)");
    if (dev < 0 || dev >= kMaxDevices) return fail(LP_ERR_UNSUPPORTED, "lp_mst_reduce_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (g_static_base[dev] == nullptr) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, lp_static_scratch);  // NOT &lp_static_scratch: that is a host address
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(lp_static_scratch)");
        if (p == nullptr || ((uintptr_t)p & 255u) != 0)
            return fail(LP_ERR_CUDA, "lp_mst_reduce_static: the scratch symbol has no usable device address");
        g_static_base[dev] = static_cast<float *>(p);
    }
    *base = g_static_base[dev];
    return LP_OK;
}

}  // namespace

extern "C" {

size_t lp_static_scratch_bytes(void) { return (size_t)LP_STATIC_SCRATCH_BYTES; }

size_t lp_mst_reduce_static_max_n(int P) {
    if (P < 1 || P > LP_MAX_P) return 0;
    const uint64_t grid_cap = 0x7fffffffull * kChunk;  // one CTA per chunk, grid.x < 2^31
    const int c = n_copies(P);
    if (c == 0) return (size_t)grid_cap;
    const size_t floats = (size_t)LP_STATIC_SCRATCH_BYTES / sizeof(float) / (size_t)c;
    return floats / kCopyAlign * kCopyAlign;
}

const char *lp_static_last_error(void) { return t_static_err; }

int lp_mst_reduce_static(float *const *bufs, int P, size_t n, int root, void *cuda_stream) {
    t_static_err[0] = 0;
    // ---- arguments (the rules of every lp_* call: nothing is enqueued unless all of them hold) ----
    if (bufs == nullptr || P < 1 || P > LP_MAX_P || root < 0 || root >= P)
        return fail(LP_ERR_INVALID_ARG, "lp_mst_reduce_static: bad bufs / P / root");
    for (int r = 0; r < P; ++r)
        if (bufs[r] == nullptr || ((uintptr_t)bufs[r] & 15u) != 0)
            return fail(LP_ERR_INVALID_ARG, "lp_mst_reduce_static: NULL or not 16-byte aligned buffer");
    if (n > lp_mst_reduce_static_max_n(P)) {
        snprintf(t_static_err, sizeof(t_static_err),
                 "lp_mst_reduce_static: n = %zu floats is above the %zu this entry point takes at P = %d (%d working "
                 "copies in a fixed %u-byte array, no allocation); use lp_mst_reduce for longer messages",
                 n, lp_mst_reduce_static_max_n(P), P, n_copies(P), (unsigned)LP_STATIC_SCRATCH_BYTES);
        return LP_ERR_UNSUPPORTED;
    }
    const uintptr_t bytes = (uintptr_t)n * sizeof(float);
    for (int i = 0; i < P && bytes; ++i)
        for (int k = i + 1; k < P; ++k) {
            const uintptr_t a = (uintptr_t)bufs[i], b = (uintptr_t)bufs[k];
            if (a < b + bytes && b < a + bytes) return fail(LP_ERR_INVALID_ARG, "lp_mst_reduce_static: overlapping buffers");
        }
    float *base = nullptr;
    const int rc = scratch_base(&base);  // also the "is there a device" check
    if (rc != LP_OK) return rc;
    if (P == 1 || n == 0) return LP_OK;

    // ---- the tree of PAPER.md:93 on virtual ranks v = (r - root) mod P, ascending d (as lp_mst_reduce) ----
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t stride = copy_stride(n);
    const float *cur[LP_MAX_P];
    for (int v = 0; v < P; ++v) cur[v] = bufs[(v + root) % P];
    const uint64_t chunks = (((uint64_t)n >> 2) + (uint64_t)kThreads * kUnroll - 1) / ((uint64_t)kThreads * kUnroll);
    for (int d = 1; d < P; d *= 2) {
        StaticLevel L;
        L.n = n;
        int m = 0;
        for (int v = 0; v + d < P; v += 2 * d) {
            float *out = v == 0 ? bufs[root] : base + (size_t)(v / 2 - 1) * stride;
            L.j[m++] = StaticJob{out, cur[v], cur[v + d]};
            cur[v] = out;
        }
        for (int i = m; i < kMaxJobs; ++i) L.j[i] = StaticJob{nullptr, nullptr, nullptr};
        dim3 grid((unsigned)(chunks ? chunks : 1), (unsigned)m, 1);
        lp_static_level_kernel<<<grid, kThreads, 0, stream>>>(L);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
    }
    return LP_OK;
}

}  // extern "C"
