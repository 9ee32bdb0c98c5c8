// lp_api.cu -- the C ABI of include/lp_collectives.h: argument validation, the planner that turns
// (op, P, n, block) into a kernel argument block + launch shape, variant dispatch, plans, library scratch and the
// host-buffer (end-to-end) entry points.  Every step of the path runs in the kernels of this library.
//
// Concurrency: a call reads its settings ONCE (the process defaults under g_mu, or its plan) into an LpCallCfg and
// carries them through; g_mu covers only the library's tables (defaults, device binding, tile-claim counters,
// scratch) and is never held across a launch, a copy or a synchronisation.  The host-buffer path has its own lock
// (it owns three streams and the staging chunks), the copy-engine variant its own (lp_copy_engine.cu).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <map>
#include <mutex>
#include <unordered_map>
#include <utility>
#include <vector>

#include "lp_common.cuh"

cudaError_t lp_mst_run(int op, int red_op, float *const *bufs, int P, size_t n, int root, int sm_count, bool pdl,
                       bool chain, cudaStream_t stream);
cudaError_t lp_be_run(int op, int red_op, float *const *bufs, int P, size_t n, int root, int sm_count, bool pdl,
                      bool chain, cudaStream_t stream);
cudaError_t lp_copy_engine_run(int op, int red_op, float *const *bufs, float *const *weights, float *velocity, int P,
                               size_t n, size_t block, int root, float lr, float mu, const LpTuning &t, int sm_count,
                               cudaStream_t stream, int dtype);
cudaError_t lp_tail16_launch(const LpArgs &a, uint64_t elem, cudaStream_t stream, bool pdl);
void lp_copy_engine_shutdown();
void lp_chain_shutdown();
cudaError_t lp_probe_launch(float *const *bufs, int n_read, int n_write, size_t n, cudaStream_t stream);

// The settings of one call: the process defaults at the time of the call, or a plan's own.
struct LpCallCfg {
    int variant;
    LpTuning tuning;
};

struct lp_plan {
    lp_plan_desc d;
    LpCallCfg cfg;
};

namespace {

std::mutex g_mu;
int g_variant = LP_VARIANT_AUTO;
LpTuning g_tuning = {{0}};
std::atomic<uint64_t> g_launches{0};
std::atomic<unsigned> g_attr_epoch{1};
thread_local char t_err[256] = "";
int g_sm_count = 0;  // 0 = not queried yet
int g_device = -1;

// ---- fitted cost-model constants: Eq. 1 of PAPER.md:81-85 for the copy-engine variant on B200.
// profiles/r2_cost_model_fit.md, fits at p = 2, 6, 16 (n = 61 M): the latency of one pipeline step is A = 2 alpha =
// 8.9 / 44.5 / 130.2 us = 8.8 us x (p - 1) -- the stream operations of a block (per hop one copy, one add launch, one
// copy back at ~2.9 us of submission each), and on one GPU the p - 1 hops of a block share two streams instead of
// each owning a link, so alpha grows with p - 1 where Eq. 1 takes it as constant.  The per-byte cost W = 2 beta + gamma
// = 0.65 / 1.47 / 0.83 ps/B follows no such law (the "pipeline fill" of p - 1 blocks that multiplies it does not exist
// when all hops run on the same device); 1.0 ps/B is within a factor 1.5 of all three and the optimal block moves
// only with its square root.
constexpr double kFitAlphaHop = 4.4e-6;  // s per block exchange and hop
constexpr double kFitBeta = 0.5e-12;     // s per byte

// ---- tile-claim counters (LpArgs::sched) ----------------------------------------------------------------------
// One self-resetting pair per STREAM (launches of a stream are ordered, and a kernel claims only after its
// predecessor's CTAs have all finished claiming and re-armed the pair: LpTileClaimer::finish precedes the trigger),
// handed out on a stream's first launch.  Launches recorded under CUDA-graph capture take the pair of their CAPTURE
// (capture id, stream): a graph may be replayed on any stream beside anything -- eager launches of the stream it was
// captured on, other graphs -- but never beside itself, and inside it the launches of one stream are ordered.  When a
// table is full the launch takes the static schedule instead: same results, a few per cent slower.
constexpr int kStreamPairs = 1024;
constexpr int kSchedStride = 4;  // unsigned long longs per pair (32 bytes: one L2 sector each)
unsigned long long *g_sched = nullptr;
std::unordered_map<cudaStream_t, int> g_stream_pair;
std::vector<int> g_free_pairs;  // given back by lp_comm_destroy
int g_stream_next = 0;
std::map<std::pair<unsigned long long, cudaStream_t>, int> g_capture_pair;
int g_capture_next = 0;

// ---- scratch: (stream, slot) -> device buffer ---------------------------------------------------------------------
struct Scratch {
    float *ptr;
    size_t bytes;
    bool captured;  // handed out while its stream was being captured: a graph holds the pointer, never free it early
};
std::map<std::pair<cudaStream_t, int>, Scratch> g_scratch;
std::vector<float *> g_scratch_retired;  // outgrown buffers a captured graph may still use: freed by lp_shutdown()

// ---- stream chains (lp_chain_admit, lp_common.cuh) ---------------------------------------------------------------
struct ChainEntry {
    std::vector<LpRange> r;
    uintptr_t lo, hi;  // bounding box
};
struct Chain {
    std::vector<ChainEntry> e;  // launches that may still be running when the next launch of the stream starts
    bool unknown = true;        // an untracked launch is among them
    uint64_t call_id = 0;       // the API call (begin_call) that enqueued the last tracked launch
};
// Which API call the calling thread is in, and whether its settings allow a launch to chain onto launches of EARLIER
// calls (LP_TUNE_CHAIN 1 / 3).  The table above knows only this library's launches: between two API calls the caller may
// have put anything on the stream (a GEMM that writes the next call's input and triggers programmatic completion
// early), so by default a launch may only skip its leading wait when the launch right ahead of it on the stream was
// enqueued by the SAME API call (tree levels of MST / BE, the launches of one Alg. 2 step, the slices of one list).
std::atomic<uint64_t> g_call_seq{0};
thread_local uint64_t t_call_id = 0;
thread_local bool t_chain_across_calls = false;
std::unordered_map<cudaStream_t, Chain> g_chains;
constexpr size_t kChainMax = 8;

// cudaMalloc with the calling thread's stream-capture mode relaxed for the duration (it is a legal call during a
// capture in another mode, but flagged "unsafe" in the default global mode because it may synchronise the device)
cudaError_t malloc_relaxed(void **p, size_t bytes) {
    cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
    cudaThreadExchangeStreamCaptureMode(&mode);
    const cudaError_t e = cudaMalloc(p, bytes);
    cudaThreadExchangeStreamCaptureMode(&mode);
    return e;
}

bool stream_capturing(cudaStream_t stream) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cap) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return cap != cudaStreamCaptureStatusNone;
}

int cuda_fail(cudaError_t e, const char *where) {
    snprintf(t_err, sizeof(t_err), "CUDA error in %s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
    return LP_ERR_CUDA;
}

// SM count of the current device; <= 0 when there is no usable device.  The library binds to the device that is
// current at its first call (its scratch, tile-claim counters and streams live there: one process per GPU); a call
// made with another device current is refused (-1) rather than allowed to touch the wrong device's memory.
// Called with g_mu held.
int sm_count_locked() {
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

// Message for a failed device check.
int no_device(int sms) {
    if (sms < 0) {
        snprintf(t_err, sizeof(t_err),
                 "liblp_b200 is bound to another CUDA device (one process per GPU); call lp_shutdown() before using this one");
        return LP_ERR_UNSUPPORTED;
    }
    snprintf(t_err, sizeof(t_err), "no CUDA device: liblp_b200 has no CPU fallback");
    return LP_ERR_CUDA;
}

// The call's settings and the device's SM count, read once.  cfg_in != NULL: a plan's settings.
int begin_call(const LpCallCfg *cfg_in, LpCallCfg &cfg, int &sms) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (cfg_in) {
        cfg = *cfg_in;
    } else {
        cfg.variant = g_variant;
        cfg.tuning = g_tuning;
    }
    sms = sm_count_locked();
    t_call_id = g_call_seq.fetch_add(1, std::memory_order_relaxed) + 1;
    t_chain_across_calls = cfg.tuning.v[LP_TUNE_CHAIN] == 1 || cfg.tuning.v[LP_TUNE_CHAIN] == 3;
    return sms <= 0 ? no_device(sms) : LP_OK;
}

bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

// NULL, alignment and pairwise-overlap checks over `count` buffers of `bytes` bytes.
int check_buffers(const float *const *ptrs, int count, size_t bytes) {
    for (int i = 0; i < count; ++i)
        if (ptrs[i] == nullptr || !aligned16(ptrs[i])) return LP_ERR_INVALID_ARG;
    if (bytes == 0) return LP_OK;
    for (int i = 0; i < count; ++i)
        for (int j = i + 1; j < count; ++j) {
            const uintptr_t a = (uintptr_t)ptrs[i], b = (uintptr_t)ptrs[j];
            if (a < b + bytes && b < a + bytes) return LP_ERR_INVALID_ARG;
        }
    return LP_OK;
}

bool is_sgd(int op) { return op == LP_OP_BSP_SGD || op == LP_OP_BSP_SGD_MOM; }
bool bad_red(int red_op) { return red_op != LP_REDUCE_SUM && red_op != LP_REDUCE_PROD; }

// What can be checked without looking at a buffer (shared by the calls and lp_plan_create).
int validate_shape(int op, int red_op, int P, int root) {
    if (op < LP_OP_BROADCAST || op > LP_OP_BSP_SGD_MOM) return LP_ERR_INVALID_ARG;
    if (P < 1 || P > LP_MAX_P || root < 0 || root >= P || bad_red(red_op)) return LP_ERR_INVALID_ARG;
    if (is_sgd(op) && red_op != LP_REDUCE_SUM) return LP_ERR_INVALID_ARG;  // the global gradient is the AVERAGE
    return LP_OK;
}

int validate(int op, int red_op, float *const *bufs, float *const *weights, const float *velocity, int P, size_t n,
             int root, size_t elem_bytes = sizeof(float)) {
    int rc = validate_shape(op, red_op, P, root);
    if (rc != LP_OK || bufs == nullptr) return LP_ERR_INVALID_ARG;
    if (is_sgd(op) && weights == nullptr) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_BSP_SGD_MOM && velocity == nullptr) return LP_ERR_INVALID_ARG;
    const float *all[2 * LP_MAX_P + 1];
    int m = 0;
    for (int r = 0; r < P; ++r) all[m++] = bufs[r];
    if (is_sgd(op))
        for (int r = 0; r < P; ++r) all[m++] = weights[r];
    if (velocity) all[m++] = velocity;
    return check_buffers(all, m, n * elem_bytes);
}

int validate_tuning(int key, int value) {
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
        case LP_TUNE_DIRECT_OCC:
            if (value > 8) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_L2_HINT:
        case LP_TUNE_PREFETCH:
            if (value > 2) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_CHAIN:
            if (value > 3) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_STORE_WAIT:
        case LP_TUNE_SCHED:
        case LP_TUNE_NO_PDL:
            if (value > 1) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_GRID_LIMIT:
            if (value > 65535) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_GRANULE_DIV:
            if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_CLAIM_SLOTS:
            if (value > 16) return LP_ERR_INVALID_ARG;
            break;
        case LP_TUNE_CLUSTER_TILE:
            if (value != 0 && value != 1024 && value != 2048 && value != 4096) return LP_ERR_INVALID_ARG;
            break;
    }
    return LP_OK;
}

// The kernel argument block of one collective (which vectors are folded, in which order; where the finished
// tile goes).  The fold order is ALWAYS rank 0 -> P-1 (U4); `root` only selects sources / destinations.
void fill_args(LpArgs &a, int op, int red_op, float *const *bufs, float *const *weights, float *velocity, int P, int root,
               float lr, float mu, const LpTuning &t, int dtype) {
    memset(&a, 0, sizeof(a));
    a.dtype = dtype;
    a.lr = lr;
    a.mu = mu;
    a.invP = 1.0f / (float)P;  // one RN division on the host (U7)
    a.red_op = red_op;
    a.l2_hint = t.v[LP_TUNE_L2_HINT];
    a.store_wait = t.v[LP_TUNE_STORE_WAIT];
    a.sched = nullptr;  // set by plan_and_run for a real launch
    switch (op) {
        case LP_OP_BROADCAST:
            a.epilogue = LP_EPI_COPY;
            a.n_sum = a.n_in = 1;
            a.n_out = P - 1;
            if (bufs) {
                a.in[0] = bufs[root];
                int q = 0;
                for (int r = 0; r < P; ++r)
                    if (r != root) a.out[q++] = bufs[r];
            }
            break;
        case LP_OP_REDUCE:
        case LP_OP_ALLREDUCE:
            a.epilogue = LP_EPI_SUM;
            a.n_sum = a.n_in = P;
            a.n_out = op == LP_OP_REDUCE ? 1 : P;
            if (bufs) {
                for (int r = 0; r < P; ++r) a.in[r] = bufs[r];
                if (op == LP_OP_REDUCE) {
                    a.out[0] = bufs[root];
                } else {
                    for (int r = 0; r < P; ++r) a.out[r] = bufs[r];
                }
            }
            break;
        default:  // LP_OP_BSP_SGD, LP_OP_BSP_SGD_MOM
            a.epilogue = op == LP_OP_BSP_SGD_MOM ? LP_EPI_SGD_MOM : LP_EPI_SGD;
            a.n_sum = P;
            a.n_in = op == LP_OP_BSP_SGD_MOM ? P + 2 : P + 1;
            a.n_out = P;
            if (bufs) {
                for (int r = 0; r < P; ++r) a.in[r] = bufs[r];
                a.in[P] = weights[root];
                if (op == LP_OP_BSP_SGD_MOM) {
                    a.in[P + 1] = velocity;  // read and rewritten in place, tile by tile
                    a.vel_out = velocity;
                }
                for (int r = 0; r < P; ++r) a.out[r] = weights[r];
            }
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

// LP_VARIANT_AUTO.  The one-CTA-per-tile register kernel has nothing to fill before its first store leaves and keeps
// ~128 KB of loads in flight per SM however few ranks there are, so it owns the latency regime and stays ahead of the
// persistent TMA pipeline up to ~2 GB of HBM traffic per call (by 8 % at 64 MB, 1 % at 256 MB); above, the pipeline's
// steadier request stream wins by 1-2 %, and for the read-dominated reduce from 4 ranks on already at ~640 MB
// (7.3 against 7.1 TB/s at P = 16, 512 MB).  A 2-rank reduce never crosses over.  Cut-offs measured on a 148-SM B200
// (profiles/r2_tuning.md section 3), kept as traffic per SM: what matters is how much each SM streams per launch.
// A confined grid always takes the pipeline (a CTA per SM with a deep ring moves the most per CTA).
int resolve_variant(const LpCallCfg &cfg, int op, int P, size_t n_work, int sm_count) {
    if (cfg.variant != LP_VARIANT_AUTO) return cfg.variant;
    if (cfg.tuning.v[LP_TUNE_GRID_LIMIT] > 0) return LP_VARIANT_PIPELINE;
    const uint64_t traffic = lp_min_bytes(op, P, n_work);
    const uint64_t mb_per_sm = (uint64_t)sm_count << 20;  // one MB of traffic per SM
    uint64_t cut;
    if (op == LP_OP_REDUCE)
        cut = P <= 2 ? ~0ull : (P == 3 ? mb_per_sm * 7 : mb_per_sm * 9 / 2);  // never / 1036 MB / 666 MB on 148 SMs
    else
        cut = mb_per_sm * 27 / 2;  // 1998 MB: a call of 2 GB (allreduce of 64 MB over 16 ranks) takes the pipeline
    return traffic < cut ? LP_VARIANT_DIRECT : LP_VARIANT_PIPELINE;
}

// block == 0: the library chooses (include/lp_collectives.h).
size_t resolve_block(size_t block, int op, int P, size_t n, int variant) {
    if (block != 0) return block;
    const size_t b = lp_auto_block(op, P, n, variant);
    return b ? b : LP_DEFAULT_BLOCK;
}

// Plans (and unless dry_run, enqueues) one LP collective on device buffers.
int plan_and_run(const LpCallCfg &cfg, int op, int red_op, float *const *bufs, float *const *weights, float *velocity,
                 int P, size_t n, size_t block, int root, float lr, float mu, int sm_count, lp_plan_info *info,
                 bool dry_run, cudaStream_t stream, const SegList *segl = nullptr, int dtype = LP_DT_F32,
                 LpArgs *args_out = nullptr) {
    const bool layered = segl != nullptr && segl->n > 0;
    const LpTuning &tun = cfg.tuning;
    LpArgs a;
    LpLaunch cfg_l = {0, 0, 0, 0, 0, false};
    fill_args(a, op, red_op, dry_run ? nullptr : bufs, weights, velocity, P, root, lr, mu, tun, dtype);
    size_t n_work = n;  // elements the launch touches per rank
    if (layered) {
        n_work = 0;
        for (int s = 0; s < segl->n; ++s) n_work += segl->len[s];
    }
    const int variant = resolve_variant(cfg, op, P, n_work, sm_count);
    block = resolve_block(block, op, P, layered ? n_work : n, variant);
    uint32_t tile, gran;
    switch (variant) {
        case LP_VARIANT_DIRECT: tile = gran = lp_direct_tile(tun, a, n_work, sm_count); break;
        case LP_VARIANT_CLUSTER: tile = gran = lp_cluster_tile(tun); break;
        case LP_VARIANT_PIPELINE:
            tile = lp_pipeline_tile(tun, a, n_work, block, sm_count);
            gran = lp_pipeline_granule(tun, tile);
            break;
        default: tile = gran = 2048u; break;  // copy engine: no tiles; the figure only fills lp_plan_info
    }
    a.slot_gran = tile / gran;
    a.claim_max = 1;
    a.span_elems = n;
    a.part = lp_make_partition(n_work, block, gran);
    lp_seg_table table;
    if (layered) {  // a1 per slice; tiles numbered slice by slice
        table.n_seg = (uint32_t)segl->n;
        uint64_t tiles = 0, blocks = 0;
        for (int s = 0; s < segl->n; ++s) {
            const lp_partition ps = lp_make_partition(segl->len[s], block, gran);
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
    if (!dry_run && tun.v[LP_TUNE_SCHED] == 0 && variant == LP_VARIANT_PIPELINE && a.part.n_tiles > 0) {
        cudaError_t es = lp_sched_acquire(stream, &a.sched);
        if (es != cudaSuccess) return cuda_fail(es, "tile-claim counters");
    }
    // identity collectives: nothing to move (P == 1 broadcast/reduce/allreduce; n == 0)
    const bool noop = (n_work == 0) || (P == 1 && !is_sgd(op));
    const lp_seg_table *tp = layered ? &table : nullptr;
    cudaError_t e = cudaSuccess;
    if (!dry_run && !noop && (variant == LP_VARIANT_COPY_ENGINE || variant == LP_VARIANT_CLUSTER)) lp_chain_reset(stream);
    if (variant == LP_VARIANT_COPY_ENGINE) {
        cfg_l.grid = cfg_l.threads = 0;
        if (!dry_run && !noop) {
            if (!layered) {
                e = lp_copy_engine_run(op, red_op, bufs, weights, velocity, P, n, block, root, lr, mu, tun, sm_count, stream,
                                       dtype);
            } else {  // one chain of copies + adds per slice
                for (int s = 0; s < segl->n && e == cudaSuccess; ++s) {
                    float *sb[LP_MAX_P], *sw[LP_MAX_P];
                    for (int r = 0; r < P; ++r) {
                        sb[r] = bufs[r] + segl->off[s];
                        sw[r] = weights ? weights[r] + segl->off[s] : nullptr;
                    }
                    e = lp_copy_engine_run(op, red_op, sb, weights ? sw : nullptr, nullptr, P, segl->len[s], block, root, lr,
                                           mu, tun, sm_count, stream, dtype);
                }
            }
        }
    } else if (variant == LP_VARIANT_DIRECT) {
        e = lp_direct_launch(a, tp, tun, sm_count, &cfg_l, dry_run || noop, stream);
    } else if (variant == LP_VARIANT_CLUSTER) {
        if (!layered) {
            e = lp_cluster_launch(a, P, root, 0, tun, sm_count, &cfg_l, dry_run || noop, stream);
        } else {  // one launch per slice: the cluster kernel's tile list is one message
            for (int s = 0; s < segl->n && e == cudaSuccess; ++s) {
                LpArgs as = a;
                as.part = lp_make_partition(segl->len[s], block, gran);
                e = lp_cluster_launch(as, P, root, segl->off[s], tun, sm_count, &cfg_l, dry_run || noop, stream);
            }
        }
        if (e == cudaErrorNotSupported) return LP_ERR_UNSUPPORTED;
    } else {
        e = lp_pipeline_launch(a, tp, tun, sm_count, &cfg_l, dry_run || noop, stream);
    }
    if (info) {
        info->nb = a.part.nb;
        info->n_tiles = a.part.n_tiles;
        info->tile_elems = tile;
        info->grid = cfg_l.grid;
        info->threads = cfg_l.threads;
        info->smem_bytes = cfg_l.smem_bytes;
        info->stages = cfg_l.stages;
        info->out_stages = cfg_l.out_stages;
        info->variant = (uint32_t)variant;
        info->sm_count = (uint32_t)sm_count;
        info->block = a.part.block;
        info->granule_elems = gran;
        info->claim_granules = cfg_l.claim;
    }
    if (args_out) *args_out = a;
    if (e != cudaSuccess) return cuda_fail(e, "LP launch");
    return LP_OK;
}

int run_device(const LpCallCfg *cfg_in, int op, int red_op, float *const *bufs, float *const *weights, float *velocity,
               int P, size_t n, size_t block, int root, float lr, float mu, void *cuda_stream) {
    int rc = validate(op, red_op, bufs, weights, velocity, P, n, root);
    if (rc != LP_OK) return rc;
    LpCallCfg cfg;
    int sms;
    rc = begin_call(cfg_in, cfg, sms);
    if (rc != LP_OK) return rc;
    if (cfg.variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    return plan_and_run(cfg, op, red_op, bufs, weights, velocity, P, n, block, root, lr, mu, sms, nullptr, false,
                        (cudaStream_t)cuda_stream);
}

size_t dtype_bytes(int dtype) { return dtype == LP_DT_F64 ? 8 : (dtype == LP_DT_F32 ? 4 : 2); }

// Collectives on vectors of element type `dtype` (U21).  The kernels address memory in 4-byte words (LpArgs::dtype):
// an f64 element is two words, two f16 / bf16 elements share one.  n and block arrive in ELEMENTS; 16-bit blocks are
// rounded up to whole words (results never depend on the block), and the odd last element of a 16-bit vector, which
// fills only half a word, is folded by a one-thread kernel behind the main launch.
// n and block of a typed call in 4-byte words (block == 0, "the library chooses", stays 0); *odd: a 16-bit vector
// ends in half a word.
void typed_words(int dtype, size_t n, size_t block, size_t &n_words, size_t &block_words, bool &odd) {
    odd = false;
    if (dtype == LP_DT_F64) {
        n_words = 2 * n;
        block_words = block > (~(size_t)0) / 2 ? ~(size_t)1 : 2 * block;
    } else if (dtype == LP_DT_F32) {
        n_words = n;
        block_words = block;
    } else {
        n_words = n / 2;
        odd = (n & 1u) != 0;
        block_words = block / 2 + (block & 1u);
    }
}

int run_device_dt(const LpCallCfg *cfg_in, int op, int red_op, int dtype, void *const *bufs, int P, size_t n, size_t block,
                  int root, void *cuda_stream) {
    if (dtype < LP_DT_F32 || dtype > LP_DT_F64) return LP_ERR_INVALID_ARG;
    float *const *fb = reinterpret_cast<float *const *>(bufs);
    if (dtype == LP_DT_F32)
        return run_device(cfg_in, op, red_op, fb, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
    if (is_sgd(op)) return LP_ERR_INVALID_ARG;  // the SGD steps are the paper's fp32 solver
    int rc = validate(op, red_op, fb, nullptr, nullptr, P, n, root, dtype_bytes(dtype));
    if (rc != LP_OK) return rc;
    if (n > (~(size_t)0) / 8) return LP_ERR_INVALID_ARG;
    LpCallCfg cfg;
    int sms;
    rc = begin_call(cfg_in, cfg, sms);
    if (rc != LP_OK) return rc;
    if (cfg.variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    size_t n_words, block_words;
    bool odd;
    typed_words(dtype, n, block, n_words, block_words, odd);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LpArgs a;
    rc = plan_and_run(cfg, op, red_op, fb, nullptr, nullptr, P, n_words, block_words, root, 0.f, 0.f, sms, nullptr, false, st,
                      nullptr, dtype, &a);
    if (rc != LP_OK || !odd || (P == 1)) return rc;
    const cudaError_t e = lp_tail16_launch(a, (uint64_t)n - 1, st, cfg.tuning.v[LP_TUNE_NO_PDL] == 0);
    if (e != cudaSuccess) return cuda_fail(e, "16-bit tail element");
    return LP_OK;
}

// Alg. 2 (PAPER.md:140-168 as read in U9; prose PAPER.md:178): reduce the sub-gradients to the root, the root
// applies GradientUpdate, the new weights are broadcast.  Three launches over the same virtual ranks -- the
// two-synchronisation-point counterpart of the fused Alg. 3 step.
int run_alg2(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block, int root, float lr,
             float mu, void *cuda_stream) {
    int rc = validate(velocity ? LP_OP_BSP_SGD_MOM : LP_OP_BSP_SGD, LP_REDUCE_SUM, grads, weights, velocity, P, n, root);
    if (rc != LP_OK) return rc;
    LpCallCfg cfg;
    int sms;
    rc = begin_call(nullptr, cfg, sms);
    if (rc != LP_OK) return rc;
    if (cfg.variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rc = plan_and_run(cfg, LP_OP_REDUCE, LP_REDUCE_SUM, grads, nullptr, nullptr, P, n, block, root, 0.f, 0.f, sms, nullptr,
                      false, st);
    if (rc != LP_OK) return rc;
    cudaError_t e = lp_update_launch(weights[root], grads[root], velocity, n, lr, 1.0f / (float)P, mu, st,
                                     cfg.tuning.v[LP_TUNE_NO_PDL] == 0);
    if (e != cudaSuccess) return cuda_fail(e, "Alg. 2 GradientUpdate");
    return plan_and_run(cfg, LP_OP_BROADCAST, LP_REDUCE_SUM, weights, nullptr, nullptr, P, n, block, root, 0.f, 0.f, sms,
                        nullptr, false, st);
}

// Layer-wise collective (Alg. 1): `op` on every slice [seg_off[s], seg_off[s] + seg_len[s]) of the rank vectors,
// each slice its own LP message, tiles handed out slice by slice in list order; LP_MAX_SEGS slices per launch.
int run_segments(const LpCallCfg *cfg_in, int op, int red_op, float *const *bufs, float *const *weights, int P, size_t n,
                 const size_t *seg_off, const size_t *seg_len, int n_seg, size_t block, int root, float lr,
                 void *cuda_stream, int dtype = LP_DT_F32) {
    if (op == LP_OP_BSP_SGD_MOM) return LP_ERR_INVALID_ARG;
    if (dtype < LP_DT_F32 || dtype > LP_DT_F64 || (dtype != LP_DT_F32 && is_sgd(op))) return LP_ERR_INVALID_ARG;
    int rc = validate(op, red_op, bufs, weights, nullptr, P, n, root, dtype_bytes(dtype));
    if (rc != LP_OK) return rc;
    const bool half = dtype == LP_DT_F16 || dtype == LP_DT_BF16;
    if (n_seg < 0 || n_seg > LP_MAX_SEGMENTS || (n_seg > 0 && (seg_off == nullptr || seg_len == nullptr)))
        return LP_ERR_INVALID_ARG;
    // slices inside [0, n) and pairwise disjoint (an in-place allreduce of overlapping slices would sum twice)
    std::vector<std::pair<size_t, size_t>> sorted;
    sorted.reserve((size_t)n_seg);
    for (int s = 0; s < n_seg; ++s) {
        if (seg_off[s] > n || seg_len[s] > n - seg_off[s]) return LP_ERR_INVALID_ARG;
        if (half && seg_len[s] && (seg_off[s] & 1u)) return LP_ERR_INVALID_ARG;  // a 16-bit slice starts on a 4-byte word
        if (seg_len[s]) sorted.emplace_back(seg_off[s], seg_len[s]);
    }
    std::sort(sorted.begin(), sorted.end());
    for (size_t i = 1; i < sorted.size(); ++i)
        if (sorted[i - 1].first + sorted[i - 1].second > sorted[i].first) return LP_ERR_INVALID_ARG;
    LpCallCfg cfg;
    int sms;
    rc = begin_call(cfg_in, cfg, sms);
    if (rc != LP_OK) return rc;
    if (cfg.variant == LP_VARIANT_CLUSTER && P > 16) return LP_ERR_UNSUPPORTED;
    // typed slices: offsets and lengths in 4-byte words (LpArgs::dtype); the odd last element of a 16-bit slice is
    // folded by the one-thread tail kernel behind the launch that carries the slice
    size_t n_words, block_words;
    bool odd_n;
    typed_words(dtype, n, block, n_words, block_words, odd_n);
    if (odd_n) ++n_words;  // the span of the vectors, for the stream-chaining ranges
    const size_t wmul = dtype == LP_DT_F64 ? 2 : 1, wdiv = half ? 2 : 1;
    size_t off[LP_MAX_SEGS], len[LP_MAX_SEGS];
    std::vector<uint64_t> tails;
    int m = 0;
    for (int s = 0; s <= n_seg; ++s) {
        if (s < n_seg && seg_len[s] > 0) {  // list order is kept: earlier slices finish first
            if (half && (seg_len[s] & 1u)) tails.push_back((uint64_t)(seg_off[s] + seg_len[s] - 1));
            if (seg_len[s] / wdiv > 0) {
                off[m] = seg_off[s] * wmul / wdiv;
                len[m] = seg_len[s] * wmul / wdiv;
                ++m;
            }
        }
        if (m == LP_MAX_SEGS || (s == n_seg && m > 0)) {
            const SegList sl{off, len, m};
            rc = plan_and_run(cfg, op, red_op, bufs, weights, nullptr, P, n_words, block_words, root, lr, 0.f, sms, nullptr,
                              false, (cudaStream_t)cuda_stream, &sl, dtype);
            if (rc != LP_OK) return rc;
            m = 0;
        }
    }
    if (!tails.empty() && P > 1) {
        LpArgs a;
        fill_args(a, op, red_op, bufs, nullptr, nullptr, P, root, 0.f, 0.f, cfg.tuning, dtype);
        for (uint64_t e : tails) {
            const cudaError_t ce = lp_tail16_launch(a, e, (cudaStream_t)cuda_stream, cfg.tuning.v[LP_TUNE_NO_PDL] == 0);
            if (ce != cudaSuccess) return cuda_fail(ce, "16-bit tail element");
        }
    }
    return LP_OK;
}

int run_baseline(bool be, int op, int red_op, float *const *bufs, int P, size_t n, int root, void *cuda_stream) {
    int rc = validate(op, red_op, bufs, nullptr, nullptr, P, n, root);
    if (rc != LP_OK) return rc;
    if (be && (P & (P - 1)) != 0) return LP_ERR_UNSUPPORTED;  // U14
    LpCallCfg cfg;
    int sms;
    rc = begin_call(nullptr, cfg, sms);
    if (rc != LP_OK) return rc;
    const bool pdl = cfg.tuning.v[LP_TUNE_NO_PDL] == 0;
    const bool chain = cfg.tuning.v[LP_TUNE_CHAIN] != 2;
    cudaError_t e = be ? lp_be_run(op, red_op, bufs, P, n, root, sms, pdl, chain, (cudaStream_t)cuda_stream)
                       : lp_mst_run(op, red_op, bufs, P, n, root, sms, pdl, chain, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, be ? "BE baseline" : "MST baseline");
    return LP_OK;
}

}  // namespace

unsigned lp_attr_epoch() { return g_attr_epoch.load(std::memory_order_relaxed); }

void lp_count_launch(uint64_t k) { g_launches.fetch_add(k, std::memory_order_relaxed); }

cudaError_t lp_sched_acquire(cudaStream_t stream, unsigned long long **pair) {
    *pair = nullptr;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    unsigned long long capture_id = 0;
    if (cudaStreamGetCaptureInfo(stream, &cap, &capture_id) != cudaSuccess) {
        cudaGetLastError();
        cap = cudaStreamCaptureStatusNone;
    }
    const bool capturing = cap != cudaStreamCaptureStatusNone;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_sched == nullptr) {
        if (capturing) return cudaSuccess;  // no allocation under capture: static schedule for this launch
        // allocated and zeroed once, synchronously: before any launch that uses it
        const size_t bytes = (size_t)(kStreamPairs + LP_CAPTURE_PAIRS) * kSchedStride * sizeof(unsigned long long);
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
    int idx;
    if (capturing) {
        auto key = std::make_pair(capture_id, stream);
        auto it = g_capture_pair.find(key);
        if (it == g_capture_pair.end()) {
            if (g_capture_next >= LP_CAPTURE_PAIRS) return cudaSuccess;
            it = g_capture_pair.emplace(key, kStreamPairs + g_capture_next++).first;
        }
        idx = it->second;
    } else {
        auto it = g_stream_pair.find(stream);
        if (it == g_stream_pair.end()) {
            int fresh;
            if (!g_free_pairs.empty()) {
                fresh = g_free_pairs.back();
                g_free_pairs.pop_back();
            } else if (g_stream_next < kStreamPairs) {
                fresh = g_stream_next++;
            } else {
                return cudaSuccess;
            }
            it = g_stream_pair.emplace(stream, fresh).first;
        }
        idx = it->second;
    }
    *pair = g_sched + (size_t)idx * kSchedStride;
    return cudaSuccess;
}

// Library scratch: grows on demand.  cudaFree synchronises the device, so growing is safe against work in flight; a
// buffer that was handed out under stream capture is retired instead of freed (a graph may replay with it).
cudaError_t lp_scratch_get(cudaStream_t stream, int slot, size_t bytes, float **ptr) {
    const bool capturing = stream != LP_SCRATCH_SHARED && stream_capturing(stream);
    std::lock_guard<std::mutex> lock(g_mu);
    Scratch &s = g_scratch[std::make_pair(stream, slot)];
    if (s.bytes < bytes) {
        if (s.ptr) {
            if (s.captured || capturing)
                g_scratch_retired.push_back(s.ptr);
            else
                cudaFree(s.ptr);
        }
        s.ptr = nullptr;
        s.bytes = 0;
        s.captured = false;
        cudaError_t e = malloc_relaxed((void **)&s.ptr, bytes);
        if (e != cudaSuccess) return e;
        s.bytes = bytes;
    }
    s.captured = s.captured || capturing;
    *ptr = s.ptr;
    return cudaSuccess;
}

bool lp_chain_admit(cudaStream_t stream, const LpRange *ranges, int n, bool pdl, bool allowed) {
    ChainEntry ent;
    ent.lo = ~(uintptr_t)0;
    ent.hi = 0;
    ent.r.reserve((size_t)n);
    for (int i = 0; i < n; ++i) {
        if (ranges[i].hi <= ranges[i].lo) continue;
        ent.r.push_back(ranges[i]);
        if (ranges[i].lo < ent.lo) ent.lo = ranges[i].lo;
        if (ranges[i].hi > ent.hi) ent.hi = ranges[i].hi;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    Chain &c = g_chains[stream];
    bool late = allowed && pdl && !c.unknown && c.e.size() < kChainMax && (t_chain_across_calls || c.call_id == t_call_id);
    c.call_id = t_call_id;
    for (size_t k = 0; late && k < c.e.size(); ++k) {
        const ChainEntry &o = c.e[k];
        if (ent.hi <= o.lo || o.hi <= ent.lo) continue;  // bounding boxes apart
        for (size_t i = 0; late && i < ent.r.size(); ++i)
            for (size_t j = 0; j < o.r.size(); ++j)
                if (ent.r[i].lo < o.r[j].hi && o.r[j].lo < ent.r[i].hi) {
                    late = false;
                    break;
                }
    }
    if (!late) {  // this launch waits first: when ITS successor starts, everything ahead of it has completed
        c.e.clear();
        c.unknown = false;
    }
    c.e.push_back(std::move(ent));
    return late;
}

void lp_chain_reset(cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g_mu);
    Chain &c = g_chains[stream];
    c.e.clear();
    c.unknown = true;
}

// ---- host-buffer (end-to-end) path ---------------------------------------------------------------------
// The LP idea applied to the host link as well: the message is cut into chunks that flow
// host -> device (stream up) -> LP kernel (stream mid) -> host (stream down); kSets chunk sets rotate, so
// the upload of chunk c+1, the kernel on chunk c and the download of chunk c-1 overlap (PCI-E is full duplex).
// The first and the last chunks are short (a quarter, a half, then full size; mirrored at the end): the upload of the
// first chunk and the download of the last one are the only transfers nothing overlaps with.
namespace {

std::mutex g_host_mu;  // the three streams, their events and the staging sets: one host-buffer call at a time
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
    if (P < 1 || P > LP_MAX_P || hbufs == nullptr || root < 0 || root >= P) return LP_ERR_INVALID_ARG;
    if (op == LP_OP_BSP_SGD && hweights == nullptr) return LP_ERR_INVALID_ARG;
    for (int r = 0; r < P; ++r) {
        if (hbufs[r] == nullptr || ((uintptr_t)hbufs[r] & 3u)) return LP_ERR_INVALID_ARG;
        if (op == LP_OP_BSP_SGD && (hweights[r] == nullptr || ((uintptr_t)hweights[r] & 3u))) return LP_ERR_INVALID_ARG;
    }
    LpCallCfg cfg;
    int sms;
    int rc = begin_call(nullptr, cfg, sms);
    if (rc != LP_OK) return rc;
    if (n == 0) return LP_OK;
    std::lock_guard<std::mutex> host_lock(g_host_mu);
    rc = host_init();
    if (rc != LP_OK) return rc;
    const bool sgd = (op == LP_OP_BSP_SGD);
    block = resolve_block(block, op, P, n, resolve_variant(cfg, op, P, n, sms));
    // chunk: a multiple of the LP block (so block boundaries fall where they would in the whole message)
    size_t chunk = kChunkElems;
    if (block < chunk) chunk = (chunk / block) * block;
    else chunk = block;
    if (chunk > n) chunk = n;
    const size_t stride = (chunk + 63) & ~(size_t)63;  // keeps every device vector 16-byte (256-byte) aligned
    const int per_set = sgd ? 2 * P : P;
    float *set_base[kSets];
    for (int s = 0; s < kSets; ++s)
        LP_TRYC(lp_scratch_get(LP_SCRATCH_SHARED, 2 * LP_MAX_P + s, (size_t)per_set * stride * sizeof(float), &set_base[s]),
                "host path scratch");

    // chunk boundaries: short chunks (multiples of the block) at both ends, full ones in between
    std::vector<size_t> cuts;  // start offsets
    {
        auto short_len = [&](int k) {  // k = 0: a quarter, k = 1: a half
            size_t l = chunk >> (2 - k);
            l = l / block * block;
            return l;
        };
        size_t lo = 0, hi = n;
        std::vector<size_t> tail;
        for (int k = 0; k < 2; ++k) {
            const size_t l = short_len(k);
            if (l == 0 || hi - lo < 4 * chunk) break;
            cuts.push_back(lo);
            lo += l;
            // the tail cut must fall on a block boundary of the whole message
            size_t t = hi - l;
            t = t / block * block;
            if (t <= lo) break;
            tail.push_back(t);
            hi = t;
        }
        for (size_t o = lo; o < hi; o += chunk) cuts.push_back(o);
        for (size_t k = tail.size(); k-- > 0;) cuts.push_back(tail[k]);
        cuts.push_back(n);
    }
    const size_t n_chunks = cuts.size() - 1;
    for (size_t c = 0; c < n_chunks; ++c) {
        const int s = (int)(c % kSets);
        const size_t off = cuts[c];
        const size_t len = cuts[c + 1] - off;
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
        rc = plan_and_run(cfg, op, LP_REDUCE_SUM, dg, sgd ? dw : nullptr, nullptr, P, len, block, root, lr, 0.f, sms, nullptr,
                          false, g_mid);
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
    return run_device(nullptr, LP_OP_BROADCAST, LP_REDUCE_SUM, bufs, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
}
int lp_reduce(float *const *bufs, int P, size_t n, size_t block, int root, void *cuda_stream) {
    return run_device(nullptr, LP_OP_REDUCE, LP_REDUCE_SUM, bufs, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
}
int lp_allreduce(float *const *bufs, int P, size_t n, size_t block, void *cuda_stream) {
    return run_device(nullptr, LP_OP_ALLREDUCE, LP_REDUCE_SUM, bufs, nullptr, nullptr, P, n, block, 0, 0.f, 0.f, cuda_stream);
}
int lp_reduce_op(float *const *bufs, int P, size_t n, size_t block, int root, int reduce_op, void *cuda_stream) {
    return run_device(nullptr, LP_OP_REDUCE, reduce_op, bufs, nullptr, nullptr, P, n, block, root, 0.f, 0.f, cuda_stream);
}
int lp_allreduce_op(float *const *bufs, int P, size_t n, size_t block, int reduce_op, void *cuda_stream) {
    return run_device(nullptr, LP_OP_ALLREDUCE, reduce_op, bufs, nullptr, nullptr, P, n, block, 0, 0.f, 0.f, cuda_stream);
}
int lp_broadcast_dt(void *const *bufs, int P, size_t n, size_t block, int root, int dtype, void *cuda_stream) {
    return run_device_dt(nullptr, LP_OP_BROADCAST, LP_REDUCE_SUM, dtype, bufs, P, n, block, root, cuda_stream);
}
int lp_reduce_dt(void *const *bufs, int P, size_t n, size_t block, int root, int dtype, int reduce_op, void *cuda_stream) {
    return run_device_dt(nullptr, LP_OP_REDUCE, reduce_op, dtype, bufs, P, n, block, root, cuda_stream);
}
int lp_allreduce_dt(void *const *bufs, int P, size_t n, size_t block, int dtype, int reduce_op, void *cuda_stream) {
    return run_device_dt(nullptr, LP_OP_ALLREDUCE, reduce_op, dtype, bufs, P, n, block, 0, cuda_stream);
}
int lp_broadcast_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                             size_t block, int root, int dtype, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_BROADCAST, LP_REDUCE_SUM, reinterpret_cast<float *const *>(bufs), nullptr, P, n, seg_off,
                        seg_len, n_seg, block, root, 0.f, cuda_stream, dtype);
}
int lp_reduce_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                          size_t block, int root, int dtype, int reduce_op, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_REDUCE, reduce_op, reinterpret_cast<float *const *>(bufs), nullptr, P, n, seg_off,
                        seg_len, n_seg, block, root, 0.f, cuda_stream, dtype);
}
int lp_allreduce_segments_dt(void *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                             size_t block, int dtype, int reduce_op, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_ALLREDUCE, reduce_op, reinterpret_cast<float *const *>(bufs), nullptr, P, n, seg_off,
                        seg_len, n_seg, block, 0, 0.f, cuda_stream, dtype);
}
size_t lp_dtype_size(int dtype) { return dtype < LP_DT_F32 || dtype > LP_DT_F64 ? 0 : dtype_bytes(dtype); }
int lp_bsp_sgd_step(float *const *grads, float *const *weights, int P, size_t n, size_t block, int root, float lr,
                    void *cuda_stream) {
    return run_device(nullptr, LP_OP_BSP_SGD, LP_REDUCE_SUM, grads, weights, nullptr, P, n, block, root, lr, 0.f, cuda_stream);
}
int lp_bsp_sgd_momentum_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block,
                             int root, float lr, float mu, void *cuda_stream) {
    return run_device(nullptr, LP_OP_BSP_SGD_MOM, LP_REDUCE_SUM, grads, weights, velocity, P, n, block, root, lr, mu,
                      cuda_stream);
}
int lp_bsp_sgd_alg2_step(float *const *grads, float *const *weights, float *velocity, int P, size_t n, size_t block,
                         int root, float lr, float mu, void *cuda_stream) {
    return run_alg2(grads, weights, velocity, P, n, block, root, lr, mu, cuda_stream);
}

int lp_broadcast_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                          size_t block, int root, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_BROADCAST, LP_REDUCE_SUM, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, root,
                        0.f, cuda_stream);
}
int lp_reduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                       size_t block, int root, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_REDUCE, LP_REDUCE_SUM, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, root, 0.f,
                        cuda_stream);
}
int lp_allreduce_segments(float *const *bufs, int P, size_t n, const size_t *seg_off, const size_t *seg_len, int n_seg,
                          size_t block, void *cuda_stream) {
    return run_segments(nullptr, LP_OP_ALLREDUCE, LP_REDUCE_SUM, bufs, nullptr, P, n, seg_off, seg_len, n_seg, block, 0, 0.f,
                        cuda_stream);
}
int lp_bsp_sgd_step_segments(float *const *grads, float *const *weights, int P, size_t n, const size_t *seg_off,
                             const size_t *seg_len, int n_seg, size_t block, int root, float lr, void *cuda_stream) {
    if (weights == nullptr) return LP_ERR_INVALID_ARG;
    return run_segments(nullptr, LP_OP_BSP_SGD, LP_REDUCE_SUM, grads, weights, P, n, seg_off, seg_len, n_seg, block, root, lr,
                        cuda_stream);
}

int lp_mst_broadcast(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(false, LP_OP_BROADCAST, LP_REDUCE_SUM, bufs, P, n, root, s);
}
int lp_mst_reduce(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(false, LP_OP_REDUCE, LP_REDUCE_SUM, bufs, P, n, root, s);
}
int lp_mst_allreduce(float *const *bufs, int P, size_t n, void *s) {
    return run_baseline(false, LP_OP_ALLREDUCE, LP_REDUCE_SUM, bufs, P, n, 0, s);
}
int lp_be_broadcast(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(true, LP_OP_BROADCAST, LP_REDUCE_SUM, bufs, P, n, root, s);
}
int lp_be_reduce(float *const *bufs, int P, size_t n, int root, void *s) {
    return run_baseline(true, LP_OP_REDUCE, LP_REDUCE_SUM, bufs, P, n, root, s);
}
int lp_be_allreduce(float *const *bufs, int P, size_t n, void *s) {
    return run_baseline(true, LP_OP_ALLREDUCE, LP_REDUCE_SUM, bufs, P, n, 0, s);
}
int lp_mst_reduce_op(float *const *bufs, int P, size_t n, int root, int reduce_op, void *s) {
    return run_baseline(false, LP_OP_REDUCE, reduce_op, bufs, P, n, root, s);
}
int lp_mst_allreduce_op(float *const *bufs, int P, size_t n, int reduce_op, void *s) {
    return run_baseline(false, LP_OP_ALLREDUCE, reduce_op, bufs, P, n, 0, s);
}
int lp_be_reduce_op(float *const *bufs, int P, size_t n, int root, int reduce_op, void *s) {
    return run_baseline(true, LP_OP_REDUCE, reduce_op, bufs, P, n, root, s);
}
int lp_be_allreduce_op(float *const *bufs, int P, size_t n, int reduce_op, void *s) {
    return run_baseline(true, LP_OP_ALLREDUCE, reduce_op, bufs, P, n, 0, s);
}

int lp_allreduce_host(float *const *host_bufs, int P, size_t n, size_t block) {
    return run_host(LP_OP_ALLREDUCE, host_bufs, nullptr, P, n, block, 0, 0.f);
}
int lp_bsp_sgd_step_host(float *const *host_grads, float *const *host_weights, int P, size_t n, size_t block, int root,
                         float lr) {
    return run_host(LP_OP_BSP_SGD, host_grads, host_weights, P, n, block, root, lr);
}

// ---- plans ---------------------------------------------------------------------------------------------------
int lp_plan_desc_init(lp_plan_desc *desc) {
    if (desc == nullptr) return LP_ERR_INVALID_ARG;
    memset(desc, 0, sizeof(*desc));
    desc->op = LP_OP_ALLREDUCE;
    desc->reduce_op = LP_REDUCE_SUM;
    desc->variant = LP_VARIANT_AUTO;
    desc->dtype = LP_DT_F32;
    return LP_OK;
}

int lp_plan_create(const lp_plan_desc *desc, lp_plan **plan) {
    if (plan == nullptr) return LP_ERR_INVALID_ARG;
    *plan = nullptr;
    if (desc == nullptr) return LP_ERR_INVALID_ARG;
    const int root = desc->op == LP_OP_ALLREDUCE ? 0 : desc->root;
    int rc = validate_shape(desc->op, desc->reduce_op, desc->P, root);
    if (rc != LP_OK) return rc;
    if (desc->variant < LP_VARIANT_PIPELINE || desc->variant > LP_VARIANT_AUTO) return LP_ERR_INVALID_ARG;
    if (desc->dtype < LP_DT_F32 || desc->dtype > LP_DT_F64 || (desc->dtype != LP_DT_F32 && is_sgd(desc->op)))
        return LP_ERR_INVALID_ARG;
    for (int k = 0; k < 16; ++k) {
        if (k >= LP_TUNE_COUNT) {
            if (desc->tuning[k] != 0) return LP_ERR_INVALID_ARG;
            continue;
        }
        rc = validate_tuning(k, desc->tuning[k]);
        if (rc != LP_OK) return rc;
    }
    if (desc->variant == LP_VARIANT_CLUSTER && desc->P > 16) return LP_ERR_UNSUPPORTED;
    lp_plan *p = new lp_plan;
    p->d = *desc;
    p->d.root = root;
    p->cfg.variant = desc->variant;
    for (int k = 0; k < LP_TUNE_COUNT; ++k) p->cfg.tuning.v[k] = desc->tuning[k];
    *plan = p;
    return LP_OK;
}

int lp_plan_destroy(lp_plan *plan) {
    if (plan == nullptr) return LP_ERR_INVALID_ARG;
    delete plan;
    return LP_OK;
}

int lp_plan_run(const lp_plan *plan, float *const *bufs, float *const *weights, float *velocity, float lr, float mu,
                void *cuda_stream) {
    if (plan == nullptr) return LP_ERR_INVALID_ARG;
    const lp_plan_desc &d = plan->d;
    if (!is_sgd(d.op) && (weights != nullptr || velocity != nullptr)) return LP_ERR_INVALID_ARG;
    if (d.op == LP_OP_BSP_SGD && velocity != nullptr) return LP_ERR_INVALID_ARG;
    if (d.dtype != LP_DT_F32)  // bufs then point at elements of the plan's type
        return run_device_dt(&plan->cfg, d.op, d.reduce_op, d.dtype, reinterpret_cast<void *const *>(bufs), d.P, d.n, d.block,
                             d.root, cuda_stream);
    return run_device(&plan->cfg, d.op, d.reduce_op, bufs, weights, velocity, d.P, d.n, d.block, d.root, lr, mu, cuda_stream);
}

int lp_plan_run_segments(const lp_plan *plan, float *const *bufs, float *const *weights, const size_t *seg_off,
                         const size_t *seg_len, int n_seg, float lr, void *cuda_stream) {
    if (plan == nullptr) return LP_ERR_INVALID_ARG;
    const lp_plan_desc &d = plan->d;
    if (d.op == LP_OP_BSP_SGD ? weights == nullptr : weights != nullptr) return LP_ERR_INVALID_ARG;
    return run_segments(&plan->cfg, d.op, d.reduce_op, bufs, weights, d.P, d.n, seg_off, seg_len, n_seg, d.block, d.root, lr,
                        cuda_stream, d.dtype);
}

int lp_plan_get_info(const lp_plan *plan, lp_plan_info *out) {
    if (plan == nullptr || out == nullptr) return LP_ERR_INVALID_ARG;
    int sms;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        sms = sm_count_locked();
    }
    if (sms <= 0) sms = 148;  // planning works without a device: a B200 has 148 SMs
    memset(out, 0, sizeof(*out));
    const lp_plan_desc &d = plan->d;
    size_t n_words, block_words;  // a typed plan is laid out in 4-byte words (tile_elems, block then count words)
    bool odd;
    typed_words(d.dtype, d.n, d.block, n_words, block_words, odd);
    return plan_and_run(plan->cfg, d.op, d.reduce_op, nullptr, nullptr, nullptr, d.P, n_words, block_words, d.root, 0.f, 0.f,
                        sms, out, true, nullptr, nullptr, d.dtype);
}

int lp_hbm_probe(float *const *bufs, int n_read, int n_write, size_t n, void *cuda_stream) {
    if (bufs == nullptr || n_read < 0 || n_write < 0 || n_read + n_write < 1 || n_read > 2 * LP_MAX_P ||
        n_write > 2 * LP_MAX_P)
        return LP_ERR_INVALID_ARG;
    for (int i = 0; i < n_read + n_write; ++i)  // outputs may alias inputs (an in-place mix), so no overlap check
        if (bufs[i] == nullptr || !aligned16(bufs[i])) return LP_ERR_INVALID_ARG;
    LpCallCfg cfg;
    int sms;
    int rc = begin_call(nullptr, cfg, sms);
    if (rc != LP_OK) return rc;
    cudaError_t e = lp_probe_launch(bufs, n_read, n_write, n, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "lp_hbm_probe");
    return LP_OK;
}

// ---- lp_comm: the comm stream of Alg. 1's non-blocking collectives ----------------------------------------
struct lp_comm {
    cudaStream_t stream;
    cudaEvent_t after, done;
};

// Device check of the lp_comm calls: the comm stream lives on the device the library is bound to.
static int comm_device_check() {
    int sms;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        sms = sm_count_locked();
    }
    return sms <= 0 ? no_device(sms) : LP_OK;
}

int lp_comm_create(lp_comm **comm) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    *comm = nullptr;
    int rc = comm_device_check();
    if (rc != LP_OK) return rc;
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
    {
        std::lock_guard<std::mutex> lock(g_mu);
        g_chains.erase(comm->stream);
        auto it = g_stream_pair.find(comm->stream);  // the stream is idle, so its pair is re-armed: reusable
        if (it != g_stream_pair.end()) {
            g_free_pairs.push_back(it->second);
            g_stream_pair.erase(it);
        }
    }
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
    int rc = comm_device_check();
    if (rc != LP_OK) return rc;
    LP_TRYC(cudaEventRecord(comm->after, (cudaStream_t)cuda_stream), "lp_comm_after");
    LP_TRYC(cudaStreamWaitEvent(comm->stream, comm->after, 0), "lp_comm_after");
    return LP_OK;
}

int lp_comm_wait(lp_comm *comm, void *cuda_stream) {
    if (comm == nullptr) return LP_ERR_INVALID_ARG;
    int rc = comm_device_check();
    if (rc != LP_OK) return rc;
    LP_TRYC(cudaEventRecord(comm->done, comm->stream), "lp_comm_wait");
    LP_TRYC(cudaStreamWaitEvent((cudaStream_t)cuda_stream, comm->done, 0), "lp_comm_wait");
    return LP_OK;
}

int lp_comm_test(lp_comm *comm, int *done) {
    if (comm == nullptr || done == nullptr) return LP_ERR_INVALID_ARG;
    int rc = comm_device_check();
    if (rc != LP_OK) return rc;
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
    if (out == nullptr || P < 1 || P > LP_MAX_P) return LP_ERR_INVALID_ARG;
    if (op < LP_OP_BROADCAST || op > LP_OP_BSP_SGD_MOM) return LP_ERR_INVALID_ARG;
    LpCallCfg cfg;
    int sms;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        cfg.variant = g_variant;
        cfg.tuning = g_tuning;
        sms = sm_count_locked();
    }
    if (sms <= 0) sms = 148;  // planning works without a device: a B200 has 148 SMs
    memset(out, 0, sizeof(*out));
    return plan_and_run(cfg, op, LP_REDUCE_SUM, nullptr, nullptr, nullptr, P, n, block, 0, 0.f, 0.f, sms, out, true, nullptr);
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

size_t lp_auto_block(int op, int P, size_t n, int variant) {
    if (op < LP_OP_BROADCAST || op > LP_OP_BSP_SGD_MOM || P < 1 || P > LP_MAX_P) return 0;
    if (variant < LP_VARIANT_PIPELINE || variant > LP_VARIANT_AUTO) return 0;
    size_t b = LP_DEFAULT_BLOCK;
    if (variant == LP_VARIANT_COPY_ENGINE && n > 0) {
        const int model_op = op == LP_OP_BROADCAST ? LP_OP_BROADCAST : (op == LP_OP_REDUCE ? LP_OP_REDUCE : LP_OP_ALLREDUCE);
        double alpha, beta;
        lp_fitted_constants(P, &alpha, &beta);
        const double bytes = lp_optimal_block(model_op, (double)P, (double)n * 4.0, alpha, beta, 0.0);
        b = bytes > 0.0 ? (size_t)(bytes / 4.0) : n;
        b = (b + 3) & ~(size_t)3;
    }
    if (n > 0 && b > n) b = n;
    if (b < 4) b = n > 0 && n < 4 ? n : 4;
    return b;
}

void lp_fitted_constants(int P, double *alpha, double *beta) {
    const double hops = P > 1 ? (double)(P - 1) : 1.0;
    if (alpha) *alpha = kFitAlphaHop * hops;
    if (beta) *beta = kFitBeta;
}

int lp_set_variant(int variant) {
    if (variant < LP_VARIANT_PIPELINE || variant > LP_VARIANT_AUTO) return LP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    g_variant = variant;
    return LP_OK;
}
int lp_get_variant(void) {
    std::lock_guard<std::mutex> lock(g_mu);
    return g_variant;
}

int lp_set_tuning(int key, int value) {
    int rc = validate_tuning(key, value);
    if (rc != LP_OK) return rc;
    std::lock_guard<std::mutex> lock(g_mu);
    g_tuning.v[key] = value;
    return LP_OK;
}
int lp_get_tuning(int key) {
    if (key < 0 || key >= LP_TUNE_COUNT) return -1;
    std::lock_guard<std::mutex> lock(g_mu);
    return g_tuning.v[key];
}

uint64_t lp_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int lp_shutdown(void) {
    std::lock_guard<std::mutex> host_lock(g_host_mu);
    lp_copy_engine_shutdown();
    std::lock_guard<std::mutex> lock(g_mu);
    lp_chain_shutdown();
    if (g_host_ready || g_sched != nullptr || !g_scratch.empty()) cudaDeviceSynchronize();
    if (g_sched) cudaFree(g_sched);
    g_sched = nullptr;
    g_stream_pair.clear();
    g_free_pairs.clear();
    g_stream_next = 0;
    g_capture_pair.clear();
    g_capture_next = 0;
    g_sm_count = 0;  // unbind: the next call binds to whatever device is current then
    g_device = -1;
    g_attr_epoch.fetch_add(1);  // function attributes are per device: every launcher sets them again
    for (auto &kv : g_scratch)
        if (kv.second.ptr) cudaFree(kv.second.ptr);
    g_scratch.clear();
    for (float *p : g_scratch_retired) cudaFree(p);
    g_scratch_retired.clear();
    g_chains.clear();
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
        case LP_ERR_INVALID_ARG: return "LP_ERR_INVALID_ARG: bad P / pointer / root / alignment / overlap / enum value";
        case LP_ERR_UNSUPPORTED:
            return t_err[0] && strstr(t_err, "bound to another CUDA device")
                       ? t_err
                       : "LP_ERR_UNSUPPORTED: BE needs a power-of-two P; cluster variant: P <= 16; chain: more CTAs than the device "
                         "holds at once, a call from another device, or a first emulation call under stream capture";
        case LP_ERR_CUDA: return t_err[0] ? t_err : "LP_ERR_CUDA";
        default: return "unknown status";
    }
}

int lp_stream_fence(void *cuda_stream) {
    lp_chain_reset((cudaStream_t)cuda_stream);
    return LP_OK;
}

int lp_version(void) { return 300; }  // 0.3.0

}  // extern "C"
