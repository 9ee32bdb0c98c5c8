// lp_chain_api.cu -- host side of the chain over real GPUs (lp_chain.cu holds the kernels): the roles of a rank
// (lp_chain_plan: host only), endpoints and their exchange (CUDA IPC), the per-rank launch, and the one-GPU emulation
// that runs all P ranks in one cooperative launch.
#include <string.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "lp_chain.cuh"

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

std::atomic<int> g_chain_kernel{LP_CHAIN_KERNEL_DEFAULT};
bool use_tma() { return g_chain_kernel.load() != LP_CHAIN_KERNEL_REGISTER; }
cudaError_t resident(int *ctas) { return lp_chain_resident(use_tma(), ctas); }
cudaError_t launch(const LpChainLaunch &L, bool cooperative, cudaStream_t stream) {
    return lp_chain_launch_kernel(L, use_tma(), cooperative, stream);
}

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

// a1 for the chain: blocks of `block` elements rounded up to a multiple of 4 (every tile then starts on a 16-byte
// boundary; results never depend on the block), cut into tiles of at most one ring slot.  block == 0, "the library
// chooses": the block that minimises the paper's own cost model (Table 1: an allreduce of a
// channel's share n_c of the message takes (p - 1 + n_c / b) (2 alpha + b (2 beta + gamma))), lp_optimal_block with the
// constants fitted to this kernel (profiles/r2_chain_cost_model.md): 2 alpha = 5.9 us per block exchange, the same at
// p = 2, 4, 8 as Eq. 1 assumes, and 2 beta + gamma = 48 ps per byte and channel -- rounded to a power of two between 4096
// elements and the slot.  Small blocks fill the chain sooner ((p - 1) b), large ones pay fewer flag exchanges (n_c / b).
constexpr double kChainFitAlpha = 2.95e-6;  // s per block exchange and direction (2 alpha = 5.9 us)
constexpr double kChainFitBeta = 24e-12;    // s per byte and channel (2 beta + gamma = 48 ps/B, gamma folded in)

size_t chain_auto_block(size_t n, int P, int tile, int channels) {
    const double n_c = (double)n * 4.0 / (double)channels;
    const double b_bytes = lp_optimal_block(LP_OP_ALLREDUCE, (double)(P > 1 ? P : 2), n_c > 1.0 ? n_c : 1.0, kChainFitAlpha,
                                            kChainFitBeta, 0.0);
    size_t b = 4096;
    while (b < (size_t)tile && (double)b * 4.0 * 1.41421356 < b_bytes) b *= 2;  // nearest power of two (geometric)
    return b;
}

lp_partition chain_partition(size_t n, size_t block, int tile, int channels, int P) {
    if (block == 0) block = chain_auto_block(n, P, tile, channels);
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
    int device;  // the device the endpoints were allocated on: another device (or a stream handle reused there) gets its own
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

size_t lp_chain_auto_block(size_t n, int P, int channels, int tile) {
    if (channels == 0) channels = LP_CHAIN_DEFAULT_CHANNELS;
    if (tile == 0) tile = LP_CHAIN_DEFAULT_TILE;
    if (P < 1 || P > LP_MAX_P || !valid_geometry(channels, 1, tile)) return 0;
    return chain_auto_block(n, P, tile, channels);
}

void lp_chain_fitted_constants(double *alpha, double *beta) {
    if (alpha) *alpha = kChainFitAlpha;
    if (beta) *beta = kChainFitBeta;
}

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

// Unmaps the neighbours' endpoints (after this rank's kernels have drained).  Tear-down across ranks is three steps with a
// host barrier between them: every rank synchronises its device (no kernel anywhere can still push data or a credit into
// a neighbour), every rank disconnects (no mapping of an exported endpoint is left), every rank destroys.
int lp_chain_disconnect(lp_chain *ch) {
    if (ch == nullptr) return LP_ERR_INVALID_ARG;
    cudaDeviceSynchronize();
    if (ch->connected) {
        if (ch->up_ipc) cudaIpcCloseMemHandle(ch->peer_up);
        if (ch->down_ipc) cudaIpcCloseMemHandle(ch->peer_down);
        ch->up_ipc = ch->down_ipc = false;
        ch->peer_up = ch->peer_down = nullptr;
        ch->connected = false;
    }
    cudaGetLastError();
    return LP_OK;
}

int lp_chain_destroy(lp_chain *ch) {
    if (ch == nullptr) return LP_ERR_INVALID_ARG;
    lp_chain_disconnect(ch);
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
    L.part = chain_partition(n, block, ch->tile, ch->C, ch->P);
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
        int device = -1;
        if (cudaGetDevice(&device) != cudaSuccess) return chain_fail(cudaGetLastError());
        for (auto &e : g_emul)
            if (e.P == P && e.C == channels && e.S == slots && e.tile == tile && e.device == device &&
                e.stream == (cudaStream_t)cuda_stream)
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
            g_emul.push_back(EmulEndpoints{P, channels, slots, tile, device, (cudaStream_t)cuda_stream, base});
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
    L.part = chain_partition(n, block, tile, channels, P);
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
        int device = -1;
        cudaGetDevice(&device);
        for (auto &e : g_emul)
            if (e.P == P && e.C == channels && e.S == slots && e.tile == tile && e.device == device) bases.push_back(e.base);
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
