// lp_baselines.cu -- MST (binomial tree) and BE (recursive halving / doubling) collectives over the same
// P virtual ranks: the comparison algorithms of PAPER.md:93-95 and Table 1, built from
// whole-segment launches of lp_seg_kernel (one launch per tree level / exchange step).
//
// MST: virtual rank v = (r - root) mod P.  Reduce: for d = 1, 2, 4, ... < P every v with
// v % 2d == 0 and v + d < P does x_v = x_v + x_{v+d} on the whole message.  Broadcast: the same pairs with d
// descending, copies.  ceil(log2 P) levels (1,2,2,3,3 for 2..6 GPUs).
// BE: reduce-scatter by recursive halving (d = P/2 .. 1: r and r^d split their segment, each
// keeps one half and adds the partner's copy of it), allgather by recursive doubling (d = 1 .. P/2, copies);
// reduce = reduce-scatter + gather to root; broadcast = binomial scatter + allgather.  P power of two (U14).
// Reduce leaves the non-root buffers unchanged (U5): partial results of non-root ranks live in library scratch.
#include "lp_common.cuh"


namespace {

inline float *rank_buf(float *const *bufs, int v, int root, int P) { return bufs[(v + root) % P]; }

#define LP_TRY(x)                         \
    do {                                  \
        cudaError_t e__ = (x);            \
        if (e__ != cudaSuccess) return e__; \
    } while (0)

}  // namespace

cudaError_t lp_mst_run(int op, int red_op, float *const *bufs, int P, size_t n, int root, int sm_count, bool pdl,
                       bool chain, cudaStream_t stream) {
    if (P == 1 || n == 0) return cudaSuccess;
    LpSegJob jobs[LP_MAX_JOBS];
    float *cur[LP_MAX_P];
    if (op == LP_OP_ALLREDUCE) root = 0;  // "allreduce is a combination of broadcast and reduce", tree root = rank 0
    for (int v = 0; v < P; ++v) cur[v] = rank_buf(bufs, v, root, P);
    if (op == LP_OP_REDUCE || op == LP_OP_ALLREDUCE) {
        const bool keep_others = (op == LP_OP_REDUCE);
        if (keep_others)  // reserve every working copy before anything is enqueued
            for (int d = 1; d < P; d *= 2)
                for (int v = 2 * d; v + d < P; v += 2 * d) {
                    float *s;
                    LP_TRY(lp_scratch_get(stream, v, n * sizeof(float), &s));
                }
        for (int d = 1; d < P; d *= 2) {
            int m = 0;
            for (int v = 0; v + d < P; v += 2 * d) {
                float *out = cur[v];
                if (keep_others && v != 0) LP_TRY(lp_scratch_get(stream, v, n * sizeof(float), &out));
                jobs[m++] = LpSegJob{out, cur[v], cur[v + d], n};
                cur[v] = out;
            }
            LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        }
    }
    if (op == LP_OP_BROADCAST || op == LP_OP_ALLREDUCE) {
        int dmax = 1;
        while (dmax * 2 < P) dmax *= 2;
        for (int d = dmax; d >= 1; d /= 2) {
            int m = 0;
            for (int v = 0; v + d < P; v += 2 * d) jobs[m++] = LpSegJob{cur[v + d], cur[v], nullptr, n};
            LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        }
    }
    return cudaSuccess;
}

cudaError_t lp_be_run(int op, int red_op, float *const *bufs, int P, size_t n, int root, int sm_count, bool pdl,
                      bool chain, cudaStream_t stream) {
    if (P == 1 || n == 0) return cudaSuccess;
    LpSegJob jobs[LP_MAX_JOBS];
    size_t lo[LP_MAX_P], hi[LP_MAX_P];
    float *cur[LP_MAX_P];  // where rank r's current values live (indexed by absolute element index)

    if (op == LP_OP_BROADCAST) {
        // scatter on virtual ranks v = r ^ root, then allgather: copies only, in place
        float *work[LP_MAX_P];
        for (int v = 0; v < P; ++v) work[v] = bufs[v ^ root];
        lo[0] = 0;
        hi[0] = n;
        for (int d = P / 2; d >= 1; d /= 2) {
            int m = 0;
            for (int v = 0; v < P; v += 2 * d) {
                size_t mid = lo[v] + (hi[v] - lo[v]) / 2;
                jobs[m++] = LpSegJob{work[v + d] + mid, work[v] + mid, nullptr, hi[v] - mid};
                lo[v + d] = mid;
                hi[v + d] = hi[v];
                hi[v] = mid;
            }
            LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        }
        for (int d = 1; d < P; d *= 2) {
            int m = 0;
            for (int v = 0; v < P; ++v) {
                int q = v ^ d;
                jobs[m++] = LpSegJob{work[v] + lo[q], work[q] + lo[q], nullptr, hi[q] - lo[q]};
            }
            LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
            for (int v = 0; v < P; ++v) {
                int q = v ^ d;
                if (q < v) continue;
                size_t l = lo[v] < lo[q] ? lo[v] : lo[q];
                size_t h = hi[v] > hi[q] ? hi[v] : hi[q];
                lo[v] = lo[q] = l;
                hi[v] = hi[q] = h;
            }
        }
        return cudaSuccess;
    }

    const bool keep_others = (op == LP_OP_REDUCE);
    float *outp[LP_MAX_P];  // where rank r writes its kept halves
    for (int r = 0; r < P; ++r) {
        lo[r] = 0;
        hi[r] = n;
        cur[r] = bufs[r];
        outp[r] = bufs[r];
    }
    if (keep_others) {
        // a non-root rank keeps only one half of the message after the first step: its scratch holds that half,
        // addressed by absolute element index (the +(k & 3) keeps the 16-byte phase of the real buffers)
        const int d0 = P / 2;
        const size_t mid = n / 2;
        for (int r = 0; r < P; ++r) {
            if (r == root) continue;
            size_t klo = (r & d0) ? mid : 0, khi = (r & d0) ? n : mid;
            float *s;
            LP_TRY(lp_scratch_get(stream, r, (khi - klo + 4) * sizeof(float), &s));
            outp[r] = s + (klo & 3) - klo;
        }
    }
    for (int d = P / 2; d >= 1; d /= 2) {
        int m = 0;
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            size_t mid = lo[r] + (hi[r] - lo[r]) / 2;
            size_t klo = (r & d) ? mid : lo[r];
            size_t khi = (r & d) ? hi[r] : mid;
            jobs[m++] = LpSegJob{outp[r] + klo, cur[r] + klo, cur[q] + klo, khi - klo};
        }
        LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        for (int r = 0; r < P; ++r) {
            size_t mid = lo[r] + (hi[r] - lo[r]) / 2;
            if (r & d)
                lo[r] = mid;
            else
                hi[r] = mid;
            cur[r] = outp[r];
        }
    }
    if (op == LP_OP_REDUCE) {  // gather every final segment to the root
        int m = 0;
        for (int r = 0; r < P; ++r)
            if (r != root) jobs[m++] = LpSegJob{bufs[root] + lo[r], cur[r] + lo[r], nullptr, hi[r] - lo[r]};
        LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        return cudaSuccess;
    }
    for (int d = 1; d < P; d *= 2) {  // allgather by recursive doubling
        int m = 0;
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            jobs[m++] = LpSegJob{cur[r] + lo[q], cur[q] + lo[q], nullptr, hi[q] - lo[q]};
        }
        LP_TRY(lp_seg_launch(jobs, m, sm_count, stream, pdl, red_op, chain));
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            if (q < r) continue;
            size_t l = lo[r] < lo[q] ? lo[r] : lo[q];
            size_t h = hi[r] > hi[q] ? hi[r] : hi[q];
            lo[r] = lo[q] = l;
            hi[r] = hi[q] = h;
        }
    }
    return cudaSuccess;
}
