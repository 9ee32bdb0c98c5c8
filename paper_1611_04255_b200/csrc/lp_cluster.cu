// lp_cluster.cu -- LP_VARIANT_CLUSTER (stage-per-rank over distributed shared memory).  Placeholder until the
// kernel lands: reports "not supported" so the API returns LP_ERR_UNSUPPORTED.
#include "lp_common.cuh"

uint32_t lp_cluster_tile(const LpTuning &) { return 2048u; }

cudaError_t lp_cluster_launch(const LpArgs &, const LpTuning &, int, LpLaunch *cfg, bool, cudaStream_t) {
    cfg->grid = cfg->threads = cfg->smem_bytes = cfg->stages = cfg->out_stages = 0;
    return cudaErrorNotSupported;
}
