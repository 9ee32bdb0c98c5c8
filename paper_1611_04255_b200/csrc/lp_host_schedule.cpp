// lp_host_schedule.cpp -- host-only part of the LP schedule engine (a1, a2): block partition, the stage-model
// tick -> (rank, block) map and the step counts of the stage and link models.  No CUDA here.
//
// Stage model ("the length of pipeline is p - 1 + n/b blocks"; U2): the P ranks are the stages,
// rank r handles block k = t - r at tick t ("GPU n ... duplicates the same pattern of GPU 1").
// Link model (Fig. 2): one step moves one block over one link; per step a rank sends at
// most one block (outbound DMA) and receives at most one (inbound DMA); reduction costs no time
// ("we assume no latency on it").  Allreduce sends every finished block out again, either back
// down the chain (LP_MODEL_LINK, U3-A) or round the ring P-1 -> 0 -> 1 ... (LP_MODEL_LINK_RING, U3-B);
// reduce traffic has priority over redistribution traffic, lower blocks first.
#include <stdint.h>

#include <math.h>

#include <vector>

#include "../../include/lp_collectives.h"

extern "C" uint64_t lp_num_blocks(size_t n, size_t block) {
    if (block == 0) return 0;
    return (uint64_t)(n / block) + (n % block ? 1u : 0u);
}

extern "C" int64_t lp_stage_block(int P, uint64_t nb, uint64_t t, int r) {
    if (r < 0 || r >= P || t < (uint64_t)r) return -1;
    const uint64_t k = t - (uint64_t)r;
    return k < nb ? (int64_t)k : -1;
}

extern "C" int lp_mst_levels(int P) {
    int levels = 0;
    while ((1 << levels) < P) ++levels;
    return levels;
}

namespace {

// Route of a block in the link model: hop h moves it from src(h) to dst(h).
struct Route {
    int P, op, model;
    int hops() const {
        if (op != LP_OP_ALLREDUCE) return P - 1;
        return model == LP_MODEL_LINK ? 2 * (P - 1) : 2 * P - 1;
    }
    void hop(int h, int &src, int &dst) const {
        if (h < P - 1) {  // the chain 0 -> 1 -> ... -> P-1
            src = h;
            dst = h + 1;
        } else if (model == LP_MODEL_LINK) {  // reverse flow P-1 -> ... -> 0
            src = 2 * (P - 1) - h;
            dst = src - 1;
        } else if (h == P - 1) {  // ring closure
            src = P - 1;
            dst = 0;
        } else {
            src = h - P;
            dst = src + 1;
        }
    }
};

uint64_t link_steps(int P, uint64_t nb, int op, int model) {
    if (P <= 1 || nb == 0) return 0;
    const Route route{P, op, model};
    const int H = route.hops();
    std::vector<int> done_hops;      // per block in the window: hops finished so far
    std::vector<uint64_t> last_step; // step of its last hop
    uint64_t first = 0;              // first block not yet fully delivered
    std::vector<char> out_busy(P), in_busy(P);
    uint64_t step = 0;
    // blocks [first, first + window) are those that have started or are next to start
    while (first < nb) {
        ++step;
        std::fill(out_busy.begin(), out_busy.end(), 0);
        std::fill(in_busy.begin(), in_busy.end(), 0);
        for (int pass = 0; pass < 2; ++pass) {  // pass 0: chain (reduce) hops, pass 1: redistribution hops
            for (uint64_t k = first; k < nb; ++k) {
                const size_t w = (size_t)(k - first);
                if (w >= done_hops.size()) {
                    if (pass == 1) break;
                    done_hops.push_back(0);
                    last_step.push_back(0);
                }
                const int h = done_hops[w];
                if (h >= H || (h < P - 1) != (pass == 0)) continue;
                if (last_step[w] >= step) continue;  // its previous hop ran in this very step
                int src, dst;
                route.hop(h, src, dst);
                const bool fire = !out_busy[src] && !in_busy[dst];
                if (fire) {
                    out_busy[src] = in_busy[dst] = 1;
                    done_hops[w] = h + 1;
                    last_step[w] = step;
                }
                // hop 0 needs rank 0's outbound engine: whether this block took it or found it taken, no
                // later block can leave rank 0 in this step
                if (pass == 0 && h == 0) break;
            }
        }
        size_t drop = 0;
        while (drop < done_hops.size() && done_hops[drop] >= H) ++drop;
        if (drop) {
            done_hops.erase(done_hops.begin(), done_hops.begin() + drop);
            last_step.erase(last_step.begin(), last_step.begin() + drop);
            first += drop;
        }
    }
    return step;
}

}  // namespace

extern "C" int lp_schedule_steps(int P, size_t n, size_t block, int op, int model, uint64_t *steps_out) {
    if (P < 1 || P > LP_MAX_P || block == 0 || steps_out == nullptr) return LP_ERR_INVALID_ARG;
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return LP_ERR_INVALID_ARG;
    if (model != LP_MODEL_STAGE && model != LP_MODEL_LINK && model != LP_MODEL_LINK_RING) return LP_ERR_INVALID_ARG;
    const uint64_t nb = lp_num_blocks(n, block);
    if (model == LP_MODEL_STAGE)
        *steps_out = nb == 0 ? 0 : (uint64_t)P - 1 + nb;  // PAPER.md:89; the last stage stores to all ranks
    else
        *steps_out = link_steps(P, nb, op, model);
    return LP_OK;
}

// ---- cost model of Sec. 3.2 (Eq. 1, Table 1) -----------------------------------------
// A block exchange costs alpha + beta b (+ gamma b with a reduce); LP pays it over a pipeline of p - 1 + n/b
// blocks, MST pays a whole-message exchange per tree level (log2 p, ceiling omitted as in PAPER.md:93), BE pays
// the scatter / reduce-scatter + gather / allgather sums of PAPER.md:95.  Table 1 read as in DESIGN.md U10/U11.
extern "C" double lp_cost_model(int algo, int op, double p, double n_bytes, double b_bytes, double alpha, double beta,
                                double gamma) {
    if (p < 1.0 || n_bytes < 0.0 || alpha < 0.0 || beta < 0.0 || gamma < 0.0) return -1.0;
    if (op != LP_OP_BROADCAST && op != LP_OP_REDUCE && op != LP_OP_ALLREDUCE) return -1.0;
    const double levels = log2(p);
    const double share = (p - 1.0) / p;
    switch (algo) {
        case LP_ALGO_LP: {
            if (b_bytes <= 0.0) return -1.0;
            const double exchanges = p - 1.0 + n_bytes / b_bytes;
            const double per_exchange_bw = op == LP_OP_BROADCAST ? beta : (op == LP_OP_REDUCE ? beta + gamma : 2.0 * beta + gamma);
            const double per_exchange_lat = op == LP_OP_ALLREDUCE ? 2.0 * alpha : alpha;
            return exchanges * (per_exchange_lat + b_bytes * per_exchange_bw);
        }
        case LP_ALGO_MST: {
            const double per_level = op == LP_OP_BROADCAST ? alpha + n_bytes * beta
                                     : (op == LP_OP_REDUCE ? alpha + n_bytes * (beta + gamma)
                                                           : 2.0 * alpha + n_bytes * (2.0 * beta + gamma));
            return levels * per_level;
        }
        case LP_ALGO_BE: {
            const double moved = share * n_bytes;
            if (op == LP_OP_BROADCAST) return (levels + p - 1.0) * alpha + 2.0 * moved * beta;
            return 2.0 * levels * alpha + 2.0 * moved * beta + moved * gamma;
        }
        default: return -1.0;
    }
}

// Block size that minimises the LP cost above: d/db [(p - 1 + n/b)(a + b w)] = (p - 1) w - n a / b^2 = 0, with a the
// latency and w the bandwidth cost of one exchange  =>  b* = sqrt(n a / ((p - 1) w)).  (The paper picks "around
// 64 KB" by hand; this is the closed form its own model implies.)  p <= 1 or a == 0: any block does,
// returns n.
extern "C" double lp_optimal_block(int op, double p, double n_bytes, double alpha, double beta, double gamma) {
    if (p < 1.0 || n_bytes <= 0.0 || alpha < 0.0 || beta < 0.0 || gamma < 0.0) return -1.0;
    const double w = op == LP_OP_BROADCAST ? beta : (op == LP_OP_REDUCE ? beta + gamma : 2.0 * beta + gamma);
    const double a = op == LP_OP_ALLREDUCE ? 2.0 * alpha : alpha;
    if (p <= 1.0 || a == 0.0 || w == 0.0) return n_bytes;
    const double b = sqrt(n_bytes * a / ((p - 1.0) * w));
    return b < n_bytes ? b : n_bytes;
}
