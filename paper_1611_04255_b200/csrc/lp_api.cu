// lp_api.cu -- the C ABI of include/lp_collectives.h: argument validation, the planner that turns
// (op, P, n, block) into a kernel argument block + launch shape, variant dispatch, library scratch and the
// host-buffer (end-to-end) entry points.  Every step of the path runs in the kernels of this library.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <mutex>
#include <utility>
#include <vector>

#include "lp_common.cuh"

cudaError_t lp_mst_run(int op, float *const *bufs, int P, size_t n, int root, int sm_count, cudaStream_t stream);
cudaError_t lp_be_run(int op, float *const *bufs, int P, size_t n, int root, int sm_count, cudaStream_t stream);
cudaError_t lp_copy_engine_run(int op, float *const *bufs, float *const *weights, float *velocity, int P, size_t n,
                               size_t block, int root, float lr, float mu, const LpTuning &t, int sm_count,
                               cudaStream_t stream);
void lp_copy_engine_shutdown();

namespace {

std::mutex g_mu;
int g_variant = LP_VARIANT_AUTO;
LpTuning g_tuning = {{0, 0, 0, 0, 0, 0, 0, 0, 0, 0}};
std::atomic<uint64_t> g_launches{0};
char g_err[256] = "";
int g_sm_count = 0;  // 0 = not queried yet

// Tile-claim counters (LpArgs::sched): a ring of self-resetting pairs, one per launch, so launches that overlap
// on different streams do not share a pair unless kSchedPairs of them are in flight at once.
constexpr int kSchedPairs = 1024;
constexpr int kSchedStride = 4;  // unsigned long longs per pair (32 bytes: one L2 sector each)
unsigned long long *g_sched = nullptr;
uint32_t g_sched_next = 0;

constexpr int kScratchSlots = 2 * LP_MAX_P + 8;
float *g_scratch[kScratchSlots];
size_t g_scratch_bytes[kScratchSlots];

int cuda_fail(cudaError_t e, const char *where) {
    snprintf(g_err, sizeof(g_err), "CUDA error in %s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
    return LP_ERR_CUDA;
}

// SM count of the current device; <= 0 when there is no usable device.  The library binds to the device that is
// current at its first call (its scratch, tile-claim counters and streams live there: one process per GPU); a call
// made with another device current is refused (-1) rather than allowed to touch the wrong device's memory.
int g_device = -1;
int sm_count_or_fail() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    if (g_sm_count > 0) return dev == g_device ? g_sm_count : -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    g_sm_count = sms;
    g_device = dev;
    return sms;
}

// Message for a failed sm_count_or_fail().
int no_device(int sms) {
    if (sms < 0) {
        snprintf(g_err, sizeof(g_err), "liblp_b200 is bound to CUDA device %d (one process per GPU); call lp_shutdown() before using another",
                 g_device);
        return LP_ERR_UNSUPPORTED;
    }
    snprintf(g_err, sizeof(g_err), "no CUDA device: liblp_b200 has no CPU fallback");
    return LP_ERR_CUDA;
}

bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

// NULL, alignment and pairwise-overlap checks over `count` buffers of n floats.
int check_buffers(const float *const *ptrs, int count, size_t n) {
    for (int i = 0; i < count; ++i)
        if (ptrs[i] == nullptr || !aligned16(ptrs[i])) return LP_ERR_INVALID_ARG;
    const size_t bytes = n * sizeof(float);
    if (bytes == 0) return LP_OK;
    for (int i = 0; i < count; ++i)
        for (int j = i + 1; j < count; ++j) {
            const uintptr_t a = (uintptr_t)ptrs[i], b = (uintptr_t)ptrs[j];
            if (a < b + bytes && b < a + bytes) return LP_ERR_INVALID_ARG;
        }
    return LP_OK;
}

bool is_sgd(int op) { return op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM; }

int validate(int op, float *const *bufs, float *const *weights, const float *velocity, int P, size_t n, size_t block,
             int root) {
    if (P < 1 || P > LP_MAX_P || bufs == nullptr || block == 0) return LP_ERR_INVALID_ARG;
    if (root < 0 || root >= P) return LP_ERR_INVALID_ARG;
    if (is_sgd(op) && weights == nullptr) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_BSP_SGD_MOM && velocity == nullptr) return LP_ERR_INVALID_ARG;
    const float *all[2 * LP_MAX_P + 1];
    int m = 0;
    for (int r = 0; r < P; ++r) all[m++] = bufs[r];
    if (is_sgd(op))
        for (int r = 0; r < P; ++r) all[m++] = weights[r];
    if (velocity) all[m++] = velocity;
    return check_buffers(all, m, n);
}

// The kernel argument block of one collective (which vectors are folded, in which order; where the finished
// tile goes).  The fold order is ALWAYS rank 0 -> P-1 (U4); `root` only selects sources / destinations.
void fill_args(LpArgs &a, int op, float *const *bufs, float *const *weights, float *velocity, int P, int root, float lr,
               float mu) {
    memset(&a, 0, sizeof(a));
    a.lr = lr;
    a.mu = mu;
    a.invP = 1.0f / (float)P;  // one RN division on the host (U7)
    a.l2_hint = g_tuning.v[LP_TUNE_L2_HINT];
    a.store_wait = g_tuning.v[LP_TUNE_STORE_WAIT];
    a.sched = nullptr;  // set by plan_and_run for a real launch
    switch (op) {
        case LP_OP_BROADCAST:
            a.epilogue = LP_EPI_COPY;
            a.n_sum = a.n_in = 1;
            a.in[0] = bufs[root];
            for (int r = 0; r < P; ++r)
                if (r != root) a.out[a.n_out++] = bufs[r];
            break;
        case LP_OP_REDUCE:
        case LP_OP_ALLREDUCE:
            a.epilogue = LP_EPI_SUM;
            a.n_sum = a.n_in = P;
            for (int r = 0; r < P; ++r) a.in[r] = bufs[r];
            if (op == LP_OP_REDUCE) {
                a.out[a.n_out++] = bufs[root];
            } else {
                for (int r = 0; r < P; ++r) a.out[a.n_out++] = bufs[r];
            }
            break;
        default:  // LP_OP_BSP_SGD, LP_OP_BSP_SGD_MOM
            a.epilogue = op == LP_OP_BSP_SGD_MOM ? LP_EPI_SGD_MOM : LP_EPI_SGD;
            a.n_sum = P;
            a.n_in = P + 1;
            for (int r = 0; r < P; ++r) a.in[r] = bufs[r];
            a.in[P] = weights[root];
            if (op == LP_OP_BSP_SGD_MOM) {
                a.in[P + 1] = velocity;  // read and rewritten in place, tile by tile
                a.vel_out = velocity;
                a.n_in = P + 2;
            }
            for (int r = 0; r < P; ++r) a.out[a.n_out++] = weights[r];
            break;
    }
}

// A list of slices of the rank vectors, each its own LP message (layer-wise collectives, Alg. 1); n == 0: the
// whole vector is the one message.
struct SegList {
    const size_t *off;
    const size_t *len;
    int n;  // <= LP_MAX_SEGS, every len > 0
};

// Plans (and unless dry_run, enqueues) one LP collective on device buffers.
int plan_and_run(int op, float *const *bufs, float *const *weights, float *velocity, int P, size_t n, size_t block,
                 int root, float lr, float mu, int sm_count, lp_plan_info *info, bool dry_run, cudaStream_t stream,
                 const SegList *segl = nullptr) {
    const bool layered = segl != nullptr && segl->n > 0;
    LpArgs a;
    LpLaunch cfg = {0, 0, 0, 0, 0};
    if (!dry_run)
        fill_args(a, op, bufs, weights, velocity, P, root, lr, mu);
    else {
        memset(&a, 0, sizeof(a));
        a.epilogue = op == LP_OP_BROADCAST ? LP_EPI_COPY
                     : (op == LP_OP_BSP_SGD ? LP_EPI_SGD : (op == LP_OP_BSP_SGD_MOM ? LP_EPI_SGD_MOM : LP_EPI_SUM));
        a.n_sum = op == LP_OP_BROADCAST ? 1 : P;
        a.n_in = a.n_sum + (op == LP_OP_BSP_SGD ? 1 : (op == LP_OP_BSP_SGD_MOM ? 2 : 0));
        a.n_out = op == LP_OP_BROADCAST ? P - 1 : (op == LP_OP_REDUCE ? 1 : P);
    }
    size_t n_work = n;  // elements the launch touches per rank
    if (layered) {
        n_work = 0;
        for (int s = 0; s < segl->n; ++s) n_work += segl->len[s];
    }
    // LP_VARIANT_AUTO: below ~384 MB of HBM traffic (192 MB for reduce, 64 MB for a copy to one or two ranks) the one-CTA-per-tile
    // register kernel is ahead (no per-CTA pipeline to fill: 1.3-3 us against 2-6 us for a 4 KB message); above,
    // the persistent TMA pipeline (profiles/r1_tuning.md section 6).  A confined grid always takes the pipeline.
    int variant = g_variant;
    if (variant == LP_VARIANT_AUTO) {
        const uint64_t traffic = lp_min_bytes(op, P, n_work);
        const uint64_t cut = (op == LP_OP_BROADCAST && P <= 3) ? (64ull << 20)
                             : (op == LP_OP_REDUCE ? (192ull << 20) : (384ull << 20));
        variant = (traffic < cut && g_tuning.v[LP_TUNE_GRID_LIMIT] == 0) ? LP_VARIANT_DIRECT : LP_VARIANT_PIPELINE;
    }
    uint32_t tile;
    switch (variant) {
        case LP_VARIANT_DIRECT: tile = lp_direct_tile(g_tuning, a.n_in, n_work); break;
        case LP_VARIANT_CLUSTER: tile = lp_cluster_tile(g_tuning); break;
        default: tile = lp_pipeline_tile(g_tuning, a, n_work, block); break;
    }
    a.part = lp_make_partition(n_work, block, tile);
    lp_seg_table table;
    if (layered) {  // a1 per slice; tiles numbered slice by slice
        table.n_seg = (uint32_t)segl->n;
        uint64_t tiles = 0, blocks = 0;
        for (int s = 0; s < segl->n; ++s) {
            const lp_partition ps = lp_make_partition(segl->len[s], block, tile);
            table.off[s] = segl->off[s];
            table.len[s] = segl->len[s];
            table.tile_start[s] = tiles;
            tiles += ps.n_tiles;
            blocks += ps.nb;
        }
        table.tile_start[segl->n] = tiles;
        a.part.block = block;  // per-slice partitions are rebuilt from (block, tile) in the kernel
        a.part.nb = blocks;
        a.part.n_tiles = tiles;
    }
    if (!dry_run && g_tuning.v[LP_TUNE_SCHED] == 0 && variant == LP_VARIANT_PIPELINE && a.part.n_tiles > 0) {
        cudaError_t es = lp_sched_acquire(&a.sched);
        if (es != cudaSuccess) return cuda_fail(es, "tile-claim counters");
    }
    // identity collectives: nothing to move (P == 1 broadcast/reduce/allreduce; n == 0)
    const bool noop = (n_work == 0) || (P == 1 && !is_sgd(op));
    const lp_seg_table *tp = layered ? &table : nullptr;
    cudaError_t e = cudaSuccess;
    if (variant == LP_VARIANT_COPY_ENGINE) {
        cfg.grid = cfg.threads = 0;
        if (!dry_run && !noop) {
            if (!layered) {
                e = lp_copy_engine_run(op, bufs, weights, velocity, P, n, block, root, lr, mu, g_tuning, sm_count, stream);
            } else {  // one chain of copies + adds per slice
                for (int s = 0; s < segl->n && e == cudaSuccess; ++s) {
                    float *sb[LP_MAX_P], *sw[LP_MAX_P];
                    for (int r = 0; r < P; ++r) {
                        sb[r] = bufs[r] + segl->off[s];
                        sw[r] = weights ? weights[r] + segl->off[s] : nullptr;
                    }
                    e = lp_copy_engine_run(op, sb, weights ? sw : nullptr, nullptr, P, segl->len[s], block, root, lr, mu,
                                           g_tuning, sm_count, stream);
                }
            }
        }
    } else if (variant == LP_VARIANT_DIRECT) {
        e = lp_direct_launch(a, tp, g_tuning, sm_count, &cfg, dry_run || noop, stream);
    } else if (variant == LP_VARIANT_CLUSTER) {
        e = layered ? cudaErrorNotSupported : lp_cluster_launch(a, P, root, g_tuning, sm_count, &cfg, dry_run || noop, stream);
        if (e == cudaErrorNotSupported) return LP_ERR_UNSUPPORTED;
    } else {
        e = lp_pipeline_launch(a, tp, g_tuning, sm_count, &cfg, dry_run || noop, stream);
    }
    if (info) {
        info->nb = a.part.nb;
        info->n_tiles = a.part.n_tiles;
        info->tile_elems = tile;
        info->grid = cfg.grid;
        info->threads = cfg.threads;
        info->smem_bytes = cfg.smem_bytes;
        info->stages = cfg.stages;
        info->out_stages = cfg.out_stages;
        info->variant = (uint32_t)variant;
        info->sm_count = (uint32_t)sm_count;
    }
    if (e != cudaSuccess) return cuda_fail(e, "LP launch");
    return LP_OK;
}

int run_device(int op, float *const *bufs, float *const *weights, float *velocity, int P, size_t n, size_t block, int root,
               float lr, float mu, void *cuda_stream) {
    int rc = validate(op, bufs, weights, velocity, P, n, block, root);
    if (rc != LP_OK) return rc;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    const int sms = sm_count_or_fail();
    if (sms <= 0) return no_device(sms);
    return plan_and_run(op, bufs, weights, velocity, P, n, block, root, lr, mu, sms, nullptr, false,
                        (cudaStream_t)cuda_stream);
}

// Alg. 2 (PAPER.md:140-168 as read in U9; prose PAPER.md:178): reduce the sub-gradients to the root, the root
// applies GradientUpdate, the new weights are broadcast.  Three launches over the same virtual ranks -- the
// two-synchronisation-point counterpart of the fused Alg. 3 step.
int run_alg2(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block, int root, float lr,
             float mu, void *cuda_stream) {
    int rc = validate(velocity ? LP_OP_BSP_SGD_MOM : LP_OP_BSP_SGD, grads, weights, velocity, P, n, block, root);
    if (rc != LP_OK) return rc;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    const int sms = sm_count_or_fail();
    if (sms <= 0) return no_device(sms);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rc = plan_and_run(LP_OP_REDUCE, grads, nullptr, nullptr, P, n, block, root, 0.f, 0.f, sms, nullptr, false, st);
    if (rc != LP_OK) return rc;
    cudaError_t e = lp_update_launch(weights[root], grads[root], velocity, n, lr, 1.0f / (float)P, mu, st);
    if (e != cudaSuccess) return cuda_fail(e, "Alg. 2 GradientUpdate");
    return plan_and_run(LP_OP_BROADCAST, weights, nullptr, nullptr, P, n, block, root, 0.f, 0.f, sms, nullptr, false, st);
}

// Layer-wise collective (Alg. 1): `op` on every slice [seg_off[s], seg_off[s] + seg_len[s]) of the rank vectors,
// each slice its own LP message, tiles handed out slice by slice in list order; LP_MAX_SEGS slices per launch.
int run_segments(int op, float *const *bufs, float *const *weights, int P, size_t n, const size_t *seg_off,
                 const size_t *seg_len, int n_seg, size_t block, int root, float lr, void *cuda_stream) {
    int rc = validate(op, bufs, weights, nullptr, P, n, block, root);
    if (rc != LP_OK) return rc;
    if (n_seg < 0 || n_seg > LP_MAX_SEGMENTS || (n_seg > 0 && (seg_off == nullptr || seg_len == nullptr)))
        return LP_ERR_INVALID_ARG;
    // slices inside [0, n) and pairwise disjoint (an in-place allreduce of overlapping slices would sum twice)
    std::vector<std::pair<size_t, size_t>> sorted;
    sorted.reserve((size_t)n_seg);
    for (int s = 0; s < n_seg; ++s) {
        if (seg_off[s] > n || seg_len[s] > n - seg_off[s]) return LP_ERR_INVALID_ARG;
        if (seg_len[s]) sorted.emplace_back(seg_off[s], seg_len[s]);
    }
    std::sort(sorted.begin(), sorted.end());
    for (size_t i = 1; i < sorted.size(); ++i)
        if (sorted[i - 1].first + sorted[i - 1].second > sorted[i].first) return LP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_variant == LP_VARIANT_CLUSTER) return LP_ERR_UNSUPPORTED;
    const int sms = sm_count_or_fail();
    if (sms <= 0) return no_device(sms);
    size_t off[LP_MAX_SEGS], len[LP_MAX_SEGS];
    int m = 0;
    for (int s = 0; s <= n_seg; ++s) {
        if (s < n_seg && seg_len[s] > 0) {  // list order is kept: earlier slices finish first
            off[m] = seg_off[s];
            len[m] = seg_len[s];
            ++m;
        }
        if (m == LP_MAX_SEGS || (s == n_seg && m > 0)) {
            const SegList sl{off, len, m};
            rc = plan_and_run(op, bufs, weights, nullptr, P, n, block, root, lr, 0.f, sms, nullptr, false,
                              (cudaStream_t)cuda_stream, &sl);
            if (rc != LP_OK) return rc;
            m = 0;
        }
    }
    return LP_OK;
}

int run_baseline(bool be, int op, float *const *bufs, int P, size_t n, int root, void *cuda_stream) {
    int rc = validate(op, bufs, nullptr, nullptr, P, n, 1, root);
    if (rc != LP_OK) return rc;
    if (be && (P & (P - 1)) != 0) return LP_ERR_UNSUPPORTED;  // U14
    std::lock_guard<std::mutex> lock(g_mu);
    const int sms = sm_count_or_fail();
    if (sms <= 0) return no_device(sms);
    cudaError_t e = be ? lp_be_run(op, bufs, P, n, root, sms, (cudaStream_t)cuda_stream)
                       : lp_mst_run(op, bufs, P, n, root, sms, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, be ? "BE baseline" : "MST baseline");
    return LP_OK;
}

}  // namespace

bool lp_pdl_enabled() { return g_tuning.v[LP_TUNE_NO_PDL] == 0; }

void lp_count_launch(uint64_t k) { g_launches.fetch_add(k, std::memory_order_relaxed); }

// Called with g_mu held.  The ring is allocated and zeroed once (synchronously: before any launch that uses it).
cudaError_t lp_sched_acquire(unsigned long long **pair) {
    if (g_sched == nullptr) {
        const size_t bytes = (size_t)kSchedPairs * kSchedStride * sizeof(unsigned long long);
        cudaError_t e = cudaMalloc((void **)&g_sched, bytes);
        if (e != cudaSuccess) return e;
        e = cudaMemset(g_sched, 0, bytes);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) {
            cudaFree(g_sched);
            g_sched = nullptr;
            return e;
        }
    }
    *pair = g_sched + (size_t)(g_sched_next++ % kSchedPairs) * kSchedStride;
    return cudaSuccess;
}

// Library scratch: grows on demand (cudaFree synchronises the device, so growing is safe against work in flight).
cudaError_t lp_scratch_get(int slot, size_t bytes, float **ptr) {
    if (slot < 0 || slot >= kScratchSlots) return cudaErrorInvalidValue;
    if (g_scratch_bytes[slot] < bytes) {
        if (g_scratch[slot]) cudaFree(g_scratch[slot]);
        g_scratch[slot] = nullptr;
        g_scratch_bytes[slot] = 0;
        cudaError_t e = cudaMalloc((void **)&g_scratch[slot], bytes);
        if (e != cudaSuccess) return e;
        g_scratch_bytes[slot] = bytes;
    }
    *ptr = g_scratch[slot];
    return cudaSuccess;
}

// ---- host-buffer (end-to-end) path ---------------------------------------------------------------------
// The LP idea applied to the host link as well: the message is cut into chunks that flow
// host -> device (stream up) -> LP kernel (stream mid) -> host (stream down); three chunk sets rotate, so
// the upload of chunk c+1, the kernel on chunk c and the download of chunk c-1 overlap (PCI-E is full duplex).
namespace {

constexpr size_t kChunkElems = 4u << 20;  // 16 MB per rank per chunk
constexpr int kSets = 3;
cudaStream_t g_up, g_mid, g_down;
cudaEvent_t g_ev_up[kSets], g_ev_done[kSets], g_ev_down[kSets];
bool g_host_ready = false;

#define LP_TRYC(x, where)                                  \
    do {                                                   \
        cudaError_t e__ = (x);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, where); \
    } while (0)

int host_init() {
    if (g_host_ready) return LP_OK;
    LP_TRYC(cudaStreamCreateWithFlags(&g_up, cudaStreamNonBlocking), "host path init");
    LP_TRYC(cudaStreamCreateWithFlags(&g_mid, cudaStreamNonBlocking), "host path init");
    LP_TRYC(cudaStreamCreateWithFlags(&g_down, cudaStreamNonBlocking), "host path init");
    for (int s = 0; s < kSets; ++s) {
        LP_TRYC(cudaEventCreateWithFlags(&g_ev_up[s], cudaEventDisableTiming), "host path init");
        LP_TRYC(cudaEventCreateWithFlags(&g_ev_done[s], cudaEventDisableTiming), "host path init");
        LP_TRYC(cudaEventCreateWithFlags(&g_ev_down[s], cudaEventDisableTiming), "host path init");
    }
    g_host_ready = true;
    return LP_OK;
}

int run_host(int op, float *const *hbufs, float *const *hweights, int P, size_t n, size_t block, int root, float lr) {
    // host pointers: same structural checks, but only 4-byte alignment is needed
    if (P < 1 || P > LP_MAX_P || hbufs == nullptr || block == 0 || root < 0 || root >= P) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_BSP_SGD && hweights == nullptr) return LP_ERR_INVALID_ARG;
    for (int r = 0; r < P; ++r) {
        if (hbufs[r] == nullptr || ((uintptr_t)hbufs[r] & 3u)) return LP_ERR_INVALID_ARG;
        if (op == LP_OP_BSP_SGD && (hweights[r] == nullptr || ((uintptr_t)hweights[r] & 3u))) return LP_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    const int sms = sm_count_or_fail();
    if (sms <= 0) return no_device(sms);
    if (n == 0) return LP_OK;
    int rc = host_init();
    if (rc != LP_OK) return rc;
    const bool sgd = (op == LP_OP_BSP_SGD);
    // chunk: a multiple of the LP block (so block boundaries fall where they would in the whole message)
    size_t chunk = kChunkElems;
    if (block < chunk) chunk = (chunk / block) * block;
    else chunk = block;
    if (chunk > n) chunk = n;
    const size_t stride = (chunk + 63) & ~(size_t)63;  // keeps every device vector 16-byte (256-byte) aligned
    const int per_set = sgd ? 2 * P : P;
    float *set_base[kSets];
    for (int s = 0; s < kSets; ++s)
        LP_TRYC(lp_scratch_get(2 * LP_MAX_P + s, (size_t)per_set * stride * sizeof(float), &set_base[s]), "host path scratch");

    const size_t n_chunks = (n + chunk - 1) / chunk;
    for (size_t c = 0; c < n_chunks; ++c) {
        const int s = (int)(c % kSets);
        const size_t off = c * chunk;
        const size_t len = off + chunk <= n ? chunk : n - off;
        float *dg[LP_MAX_P], *dw[LP_MAX_P];
        for (int r = 0; r < P; ++r) {
            dg[r] = set_base[s] + (size_t)r * stride;
            dw[r] = set_base[s] + (size_t)(P + r) * stride;
        }
        // upload (after the previous user of this set has been downloaded)
        if (c >= (size_t)kSets) LP_TRYC(cudaStreamWaitEvent(g_up, g_ev_down[s], 0), "host path");
        for (int r = 0; r < P; ++r)
            LP_TRYC(cudaMemcpyAsync(dg[r], hbufs[r] + off, len * sizeof(float), cudaMemcpyHostToDevice, g_up), "H2D");
        if (sgd)  // only the root's replica is read (U8)
            LP_TRYC(cudaMemcpyAsync(dw[root], hweights[root] + off, len * sizeof(float), cudaMemcpyHostToDevice, g_up), "H2D");
        lp_count_launch((uint64_t)P + (sgd ? 1 : 0));
        LP_TRYC(cudaEventRecord(g_ev_up[s], g_up), "host path");
        // LP kernel
        LP_TRYC(cudaStreamWaitEvent(g_mid, g_ev_up[s], 0), "host path");
        rc = plan_and_run(op, dg, sgd ? dw : nullptr, nullptr, P, len, block, root, lr, 0.f, sms, nullptr, false, g_mid);
        if (rc != LP_OK) return rc;
        LP_TRYC(cudaEventRecord(g_ev_done[s], g_mid), "host path");
        // download
        LP_TRYC(cudaStreamWaitEvent(g_down, g_ev_done[s], 0), "host path");
        for (int r = 0; r < P; ++r) {
            float *src = sgd ? dw[r] : dg[r];
            float *dst = sgd ? hweights[r] : hbufs[r];
            LP_TRYC(cudaMemcpyAsync(dst + off, src, len * sizeof(float), cudaMemcpyDeviceToHost, g_down), "D2H");
        }
        lp_count_launch((uint64_t)P);
        LP_TRYC(cudaEventRecord(g_ev_down[s], g_down), "host path");
    }
    LP_TRYC(cudaStreamSynchronize(g_down), "host path sync");
    return LP_OK;
}

}  // namespace

// ---- C ABI -----------------------------------------------------------------------------------------------
extern "C" {

int lp_broadcast(float *const *bufs, int P, size_t n, size_t block, int root, void *cuda_stream) {
    return run_device(LP_OP_BROADCAST, bufs, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
}
int lp_reduce(float *const *bufs, int P, size_t n, size_t block, int root, void *cuda_stream) {
    return run_device(LP_OP_REDUCE, bufs, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
}
int lp_allreduce(float *const *bufs, int P, size_t n, size_t block, void *cuda_stream) {
    return run_device(LP_OP_ALLREDUCE, bufs, nullptr, nullptr, P, n, block, 0, 0.f, 0.f, cuda_stream);
}
int lp_bsp_sgd_step(float *const *grads, float *const *weights, int P, size_t n, size_t block, int root, float lr,
                    void *cuda_stream) {
    return run_device(LP_OP_BSP_SGD, grads, weights, nullptr, P, n, block, root, lr, 0.f, cuda_stream);
}
int lp_bsp_sgd_momentum_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block,
                             int root, float lr, float mu, void *cuda_stream) {
    return run_device(LP_OP_BSP_SGD_MOM, grads, weights, velocity, P, n, block, root, lr, mu, cuda_stream);
}
int lp_bsp_sgd_alg2_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block,
                         int root, float lr, float mu, void *cuda_stream) {
    return run_alg2(grads, weights, velocity, P, n, block, root, lr, mu, cuda_stream);
}

int lp_broadcast_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                          size_t block, int root, void *cuda_stream) {
    return run_segments(LP_OP_BROADCAST, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, root, 0.f, cuda_stream);
}
int lp_reduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                       size_t block, int root, void *cuda_stream) {
    return run_segments(LP_OP_REDUCE, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, root, 0.f, cuda_stream);
}
int lp_allreduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                          size_t block, void *cuda_stream) {
    return run_segments(LP_OP_ALLREDUCE, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, 0, 0.f, cuda_stream);
}
int lp_bsp_sgd_step_segments(float *const *grads, float *const *weights, int P, size_t n, const size_t *seg_off,
                             const size_t *seg_len, int n_seg, size_t block, int root, float lr, void *cuda_stream) {
    if (weights == nullptr) return LP_ERR_INVALID_ARG;
    return run_segments(LP_OP_BSP_SGD, grads, weights, P, n, seg_off, seg_len, n_seg, block, root, lr, cuda_stream);
}

int lp_mst_broadcast(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(false, LP_OP_BROADCAST, bufs, P, n, root, s);
}
int lp_mst_reduce(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(false, LP_OP_REDUCE, bufs, P, n, root, s);
}
int lp_mst_allreduce(float *const *bufs, int P, size_t n, void *s) {
    return run_baseline(false, LP_OP_ALLREDUCE, bufs, P, n, 0, s);
}
int lp_be_broadcast(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(true, LP_OP_BROADCAST, bufs, P, n, root, s);
}
int lp_be_reduce(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(true, LP_OP_REDUCE, bufs, P, n, root, s);
}
int lp_be_allreduce(float *const *bufs, int P, size_t n, void *s) {
    return run_baseline(true, LP_OP_ALLREDUCE, bufs, P, n, 0, s);
}

int lp_allreduce_host(float *const *host_bufs, int P, size_t n, size_t block) {
    return run_host(LP_OP_ALLREDUCE, host_bufs, nullptr, P, n, block, 0, 0.f);
}
int lp_bsp_sgd_step_host(float *const *host_grads, float *const *host_weights, int P, size_t n, size_t block, int root,
                         float lr) {
    return run_host(LP_OP_BSP_SGD, host_grads, host_weights, P, n, block, root, lr);
}

// ---- lp_comm: the comm stream of Alg. 1's non-blocking collectives ----------------------------------------
struct lp_comm {
    cudaStream_t stream;
    cudaEvent_t after, done;
};

int lp_comm_create(lp_comm **comm) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    *comm = nullptr;
    std::lock_guard<std::mutex> lock(g_mu);
    {
        const int sms = sm_count_or_fail();
        if (sms <= 0) return no_device(sms);
    }
    int lo = 0, hi = 0;  // hi = numerically lowest = highest priority
    LP_TRYC(cudaDeviceGetStreamPriorityRange(&lo, &hi), "lp_comm_create");
    lp_comm *c = new lp_comm{nullptr, nullptr, nullptr};
    cudaError_t e = cudaStreamCreateWithPriority(&c->stream, cudaStreamNonBlocking, hi);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->after, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->done, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        if (c->done) cudaEventDestroy(c->done);
        if (c->after) cudaEventDestroy(c->after);
        if (c->stream) cudaStreamDestroy(c->stream);
        delete c;
        return cuda_fail(e, "lp_comm_create");
    }
    *comm = c;
    return LP_OK;
}

int lp_comm_destroy(lp_comm *comm) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    cudaStreamSynchronize(comm->stream);
    cudaEventDestroy(comm->after);
    cudaEventDestroy(comm->done);
    cudaStreamDestroy(comm->stream);
    cudaGetLastError();
    delete comm;
    return LP_OK;
}

void *lp_comm_stream(lp_comm *comm) { return comm ? (void *)comm->stream : nullptr; }

int lp_comm_after(lp_comm *comm, void *cuda_stream) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    LP_TRYC(cudaEventRecord(comm->after, (cudaStream_t)cuda_stream), "lp_comm_after");
    LP_TRYC(cudaStreamWaitEvent(comm->stream, comm->after, 0), "lp_comm_after");
    return LP_OK;
}

int lp_comm_wait(lp_comm *comm, void *cuda_stream) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    LP_TRYC(cudaEventRecord(comm->done, comm->stream), "lp_comm_wait");
    LP_TRYC(cudaStreamWaitEvent((cudaStream_t)cuda_stream, comm->done, 0), "lp_comm_wait");
    return LP_OK;
}

int lp_comm_test(lp_comm *comm, int *done) {
    if (comm == nullptr || done == nullptr) return LP_ERR_INVALID_ARG;
    const cudaError_t e = cudaStreamQuery(comm->stream);
    if (e == cudaSuccess) {
        *done = 1;
    } else if (e == cudaErrorNotReady) {
        cudaGetLastError();
        *done = 0;
    } else {
        return cuda_fail(e, "lp_comm_test");
    }
    return LP_OK;
}

int lp_plan_query(int op, int P, size_t n, size_t block, lp_plan_info *out) {
    if (out == nullptr || P < 1 || P > LP_MAX_P || block == 0) return LP_ERR_INVALID_ARG;
    if (op < LP_OP_BROADCAST || op > LP_OP_BSP_SGD_MOM) return LP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    int sms = sm_count_or_fail();
    if (sms <= 0) sms = 148;  // planning works without a device: a B200 has 148 SMs
    memset(out, 0, sizeof(*out));
    return plan_and_run(op, nullptr, nullptr, nullptr, P, n, block, 0, 0.f, 0.f, sms, out, true, nullptr);
}

uint64_t lp_min_bytes(int op, int P, size_t n) {
    const uint64_t v = (uint64_t)n * 4u;
    switch (op) {
        case LP_OP_BROADCAST: return (uint64_t)P * v;
        case LP_OP_REDUCE: return (uint64_t)(P + 1) * v;
        case LP_OP_ALLREDUCE: return 2u * (uint64_t)P * v;
        case LP_OP_BSP_SGD: return (2u * (uint64_t)P + 1u) * v;
        case LP_OP_BSP_SGD_MOM: return (2u * (uint64_t)P + 3u) * v;
        default: return 0;
    }
}

int lp_set_variant(int variant) {
    if (variant < LP_VARIANT_PIPELINE || variant > LP_VARIANT_AUTO) return LP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    g_variant = variant;
    return LP_OK;
}
int lp_get_variant(void) { return g_variant; }

int lp_set_tuning(int key, int value) {
    if (key < 0 || key >= LP_TUNE_COUNT || value < 0) return LP_ERR_INVALID_ARG;
    switch (key) {
        case LP_TUNE_TILE_ELEMS:
            if (value != 0 && value != 1024 && value != 2048 && value != 4096 && value != 8192) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_STAGES:
            if (value != 0 && (value < 2 || value > 32)) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_OUT_STAGES:
        case LP_TUNE_CTAS_PER_SM:
        case LP_TUNE_CE_STREAMS:
            if (value > 8) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_L2_HINT:
            if (value > 2) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_STORE_WAIT:
        case LP_TUNE_SCHED:
        case LP_TUNE_NO_PDL:
            if (value > 1) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_GRID_LIMIT:
            if (value > 65535) return LP_ERR_INVALID_ARG;
            break;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    g_tuning.v[key] = value;
    return LP_OK;
}
int lp_get_tuning(int key) { return (key < 0 || key >= LP_TUNE_COUNT) ? -1 : g_tuning.v[key]; }

uint64_t lp_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int lp_shutdown(void) {
    std::lock_guard<std::mutex> lock(g_mu);
    bool any = g_host_ready || g_sched != nullptr;
    for (int s = 0; s < kScratchSlots; ++s) any = any || g_scratch[s] != nullptr;
    if (any) cudaDeviceSynchronize();
    if (g_sched) cudaFree(g_sched);
    g_sched = nullptr;
    g_sched_next = 0;
    g_sm_count = 0;  // unbind: the next call binds to whatever device is current then
    g_device = -1;
    for (int s = 0; s < kScratchSlots; ++s) {
        if (g_scratch[s]) cudaFree(g_scratch[s]);
        g_scratch[s] = nullptr;
        g_scratch_bytes[s] = 0;
    }
    lp_copy_engine_shutdown();
    if (g_host_ready) {
        cudaStreamDestroy(g_up);
        cudaStreamDestroy(g_mid);
        cudaStreamDestroy(g_down);
        for (int s = 0; s < kSets; ++s) {
            cudaEventDestroy(g_ev_up[s]);
            cudaEventDestroy(g_ev_done[s]);
            cudaEventDestroy(g_ev_down[s]);
        }
        g_host_ready = false;
    }
    cudaGetLastError();
    return LP_OK;
}

const char *lp_status_string(int status) {
    switch (status) {
        case LP_OK: return "LP_OK";
        case LP_ERR_INVALID_ARG: return "LP_ERR_INVALID_ARG: bad P / pointer / block / root / alignment / overlap";
        case LP_ERR_UNSUPPORTED:
            return g_err[0] && strstr(g_err, "bound to CUDA device")
                       ? g_err
                       : "LP_ERR_UNSUPPORTED: BE needs a power-of-two P; cluster variant: P <= 16, no momentum, no slice lists";
        case LP_ERR_CUDA: return g_err[0] ? g_err : "LP_ERR_CUDA";
        default: return "unknown status";
    }
}

int lp_version(void) { return 100; }  // 0.1.0

}  // extern "C"
