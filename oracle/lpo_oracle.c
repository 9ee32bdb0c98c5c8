/*
 * lpo_oracle.c -- CPU ORACLE for the Linear Pipeline (LP) collectives of
 * arXiv 1611.04255 ("Efficient Communications in Training Large Scale Neural
 * Networks").  Citations are PAPER.md:<line> (section / figure / equation).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check
 * in __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * load it.  It shares no code, header, table or helper with the CUDA path in
 * paper_1611_04255_b200/csrc/, and neither side includes the other.
 *
 * Plain C11, slow, meant to be checked against the paper by eye.  Build with
 *   gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -fPIC -shared
 * (-ffp-contract=off: no FMA contraction; every fp32 op below is one IEEE-754
 * round-to-nearest-even operation, no flush-to-zero.)
 *
 * Precision: the paper's messages are fp32 (Caffe) and north_star fixes
 * "bit-exact when summation follows the LP chain order (rank 0 -> P-1)", so
 * the value functions compute in fp32, in exactly that order.  Nothing is
 * blocked, fused or reordered beyond what the cited passage states.
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): every function below is
 * pinned to something other than itself; none is "parity unpinned".  Absolute
 * performance is the only thing the paper leaves unpinned (it prints no GB/s).
 *
 * Conventions: bufs is an array of P host pointers, each to n floats; ranks are
 * 0..P-1; all functions return 0 on success, a negative value on bad arguments.
 */
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#define LPO_OK 0
#define LPO_EINVAL (-1)
#define LPO_EUNSUPPORTED (-2)
#define LPO_ENOMEM (-3)

/* ------------------------------------------------------------------------ */
/* 1. Result definitions (what the method reaches exactly)                    */
/* ------------------------------------------------------------------------ */

/* S[i] = (((x_0[i] + x_1[i]) + x_2[i]) + ...) + x_{P-1}[i]
 * PAPER.md:59 (Sec. 3, Fig. 2b): GPU0's block a0 goes to GPU1, "GPU1 reduces the
 * received block a0 with a1 to yield a'", then a' goes to GPU2 "to reduce to
 * a''": a left fold along the chain, rank 0 first.  out may not alias inputs. */
void lpo_chain_sum(const float *const *in, int P, size_t n, float *out)
{
    for (size_t i = 0; i < n; ++i) {
        float s = in[0][i];
        for (int r = 1; r < P; ++r)
            s = s + in[r][i];
        out[i] = s;
    }
}

static int bad_args(float *const *bufs, int P, int root)
{
    if (bufs == NULL || P < 1 || root < 0 || root >= P)
        return 1;
    for (int r = 0; r < P; ++r)
        if (bufs[r] == NULL)
            return 1;
    return 0;
}

/* Broadcast: "It copies the source vector to every GPUs." PAPER.md:57. */
int lpo_broadcast(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    for (int r = 0; r < P; ++r) {
        if (r == root)
            continue;
        for (size_t i = 0; i < n; ++i)
            bufs[r][i] = bufs[root][i];
    }
    return LPO_OK;
}

/* Reduce: "combines the elements provided in the vector of each GPU, and
 * returns the combined value in the receive vector to a specific GPU."
 * PAPER.md:59.  Sum order is always rank 0 -> P-1 (reading U4);
 * non-root vectors are left as they were (reading U5: a0 is written "to a
 * buffer on GPU1", not over a1). */
int lpo_reduce(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        float s = bufs[0][i];
        for (int r = 1; r < P; ++r)
            s = s + bufs[r][i];
        bufs[root][i] = s;
    }
    return LPO_OK;
}

/* Allreduce: "combines vectors from all GPUs and distributes the result back
 * to them. Mathematically, it is equivalent to a reduce followed by a
 * broadcast." PAPER.md:61,71.  The reduced block is forwarded, never
 * recomputed, so every rank holds the same bits. */
int lpo_allreduce(float *const *bufs, int P, size_t n)
{
    if (bad_args(bufs, P, 0))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        float s = bufs[0][i];
        for (int r = 1; r < P; ++r)
            s = s + bufs[r][i];
        for (int r = 0; r < P; ++r)
            bufs[r][i] = s;
    }
    return LPO_OK;
}

/* BSP-SGD step, Alg. 3 communication + update:
 *   grad = allreduce(grad_sub)                       (chain order sum S)
 *   "The global gradient is equivalent to the average of sub-gradients."
 *                                                    PAPER.md:174  g = S * (1/P)
 *   w^t = w^{t-1} - eta * grad                       PAPER.md:172, Eq. 5
 *   "w^t is synchronized to all GPUs"
 * Reading U7: three separately rounded fp32 ops, invP = fl(1.0f / P) computed
 * once; no FMA.  Reading U8: the replica read is weights[root]; the one new w
 * is written to every replica, so replicas never diverge.  grads are unchanged. */
int lpo_bsp_sgd_step(float *const *grads, float *const *weights, int P,
                     size_t n, int root, float lr)
{
    if (bad_args(grads, P, root) || bad_args(weights, P, root))
        return LPO_EINVAL;
    const float invP = 1.0f / (float)P;
    for (size_t i = 0; i < n; ++i) {
        float s = grads[0][i];
        for (int r = 1; r < P; ++r)
            s = s + grads[r][i];
        float g = s * invP;
        float t = lr * g;
        float w = weights[root][i] - t;
        for (int r = 0; r < P; ++r)
            weights[r][i] = w;
    }
    return LPO_OK;
}

/* BSP-SGD step with momentum.  PAPER.md:216: "The solver is
 * SGD + momentum"; the paper prints no formula.  Reading U18: the solver of
 * the system the paper modifies (Caffe's SGD solver):
 *   v' = mu * v + eta * grad ;  w' = w - v'
 * with grad = S * (1/P) as in lpo_bsp_sgd_step.  Five separately
 * rounded fp32 ops per element, in this order, no FMA:
 *   g = S * invP ; t = lr * g ; m = mu * v ; v' = m + t ; w' = w_root - v'.
 * The velocity is ONE vector of n floats: it lives where the update is
 * computed (in Alg. 3 every replica of it would hold the same bits).  The new
 * w' goes to every weight replica (U8); grads are unchanged.  mu = 0 with
 * v = 0 is lpo_bsp_sgd_step. */
int lpo_bsp_sgd_momentum_step(float *const *grads, float *const *weights,
                              float *velocity, int P, size_t n, int root,
                              float lr, float mu)
{
    if (bad_args(grads, P, root) || bad_args(weights, P, root) || velocity == NULL)
        return LPO_EINVAL;
    const float invP = 1.0f / (float)P;
    for (size_t i = 0; i < n; ++i) {
        float s = grads[0][i];
        for (int r = 1; r < P; ++r)
            s = s + grads[r][i];
        float g = s * invP;
        float t = lr * g;
        float m = mu * velocity[i];
        float v = m + t;
        float w = weights[root][i] - v;
        velocity[i] = v;
        for (int r = 0; r < P; ++r)
            weights[r][i] = w;
    }
    return LPO_OK;
}

/* BSP-SGD step the Alg. 2 way (PAPER.md:140-168 as reconstructed in reading
 * U9, prose PAPER.md:178): "The master GPU reconstructs grad by reducing all
 * grad_sub.  Then, GPUs synchronize latest weight w by broadcasting."
 *   1. grad = reduce(grad_sub) to the root       -> grads[root] holds S (in place, MPI style)
 *   2. if root: w = GradientUpdate()             -> weights[root] updated from grads[root]
 *   3. broadcast(w) from the root                -> every replica = weights[root]
 * Written as those three steps, each calling the definition above it.  The
 * update arithmetic is that of lpo_bsp_sgd_step (velocity == NULL) or of
 * lpo_bsp_sgd_momentum_step, so the weights agree bit for bit with Alg. 3's
 * fused step (tests pin that); the difference is the side effect on
 * grads[root] and the number of passes over memory. */
int lpo_bsp_sgd_alg2_step(float *const *grads, float *const *weights,
                          float *velocity, int P, size_t n, int root,
                          float lr, float mu)
{
    if (bad_args(grads, P, root) || bad_args(weights, P, root))
        return LPO_EINVAL;
    int rc = lpo_reduce(grads, P, n, root);                 /* step 1 */
    if (rc != LPO_OK)
        return rc;
    const float invP = 1.0f / (float)P;
    float *w = weights[root];
    const float *S = grads[root];
    for (size_t i = 0; i < n; ++i) {                        /* step 2, root only */
        float g = S[i] * invP;
        float t = lr * g;
        if (velocity != NULL) {
            float m = mu * velocity[i];
            float v = m + t;
            velocity[i] = v;
            w[i] = w[i] - v;
        } else {
            w[i] = w[i] - t;
        }
    }
    return lpo_broadcast(weights, P, n, root);              /* step 3 */
}

/* Layer-wise collectives.  Alg. 1 (prose
 * PAPER.md:182): "GPUs broadcast network parameters of layer t+1 amid forward
 * computations at layer t ... all-reduce or reduce sub-gradients of layer t+1
 * amidst backward computations at layer t": one collective PER LAYER, i.e. per
 * slice [seg_off[s], seg_off[s] + seg_len[s]) of the flat rank vectors.  The
 * definition is just that: the whole-message definition above applied to each
 * slice in list order; elements outside every slice are not touched.
 * op: 0 broadcast, 1 reduce, 2 allreduce.  Slices must lie inside [0, n). */
int lpo_collective_segments(int op, float *const *bufs, int P, size_t n,
                            const size_t *seg_off, const size_t *seg_len,
                            int n_seg, int root)
{
    if (bad_args(bufs, P, root) || n_seg < 0 || (n_seg > 0 && (!seg_off || !seg_len)))
        return LPO_EINVAL;
    if (P > 64)
        return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s)
        if (seg_off[s] > n || seg_len[s] > n - seg_off[s])
            return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s) {
        float *slice[64];
        for (int r = 0; r < P; ++r)
            slice[r] = bufs[r] + seg_off[s];
        int rc;
        if (op == 0)
            rc = lpo_broadcast(slice, P, seg_len[s], root);
        else if (op == 1)
            rc = lpo_reduce(slice, P, seg_len[s], root);
        else if (op == 2)
            rc = lpo_allreduce(slice, P, seg_len[s]);
        else
            rc = LPO_EINVAL;
        if (rc != LPO_OK)
            return rc;
    }
    return LPO_OK;
}

/* Layer-wise fused BSP-SGD step: Alg. 1's per-layer communication with Alg. 3's update
 * applied to each layer as soon as its gradient has been allreduced: lpo_bsp_sgd_step on
 * every slice, in list order; elements outside every slice keep their weights. */
int lpo_bsp_sgd_step_segments(float *const *grads, float *const *weights, int P, size_t n,
                              const size_t *seg_off, const size_t *seg_len, int n_seg,
                              int root, float lr)
{
    if (bad_args(grads, P, root) || bad_args(weights, P, root) || P > 64 ||
        n_seg < 0 || (n_seg > 0 && (!seg_off || !seg_len)))
        return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s)
        if (seg_off[s] > n || seg_len[s] > n - seg_off[s])
            return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s) {
        float *g[64], *w[64];
        for (int r = 0; r < P; ++r) {
            g[r] = grads[r] + seg_off[s];
            w[r] = weights[r] + seg_off[s];
        }
        int rc = lpo_bsp_sgd_step(g, w, P, seg_len[s], root, lr);
        if (rc != LPO_OK)
            return rc;
    }
    return LPO_OK;
}

/* The same two definitions with the element loop spread over host threads.
 * Element i never depends on element j != i, so the bits are those of the
 * serial loops above (tests assert it).  These are the versions bench.py times
 * as cpu_baseline; they are not tuned. */
int lpo_allreduce_omp(float *const *bufs, int P, size_t n)
{
    if (bad_args(bufs, P, 0))
        return LPO_EINVAL;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        float s = bufs[0][i];
        for (int r = 1; r < P; ++r)
            s = s + bufs[r][i];
        for (int r = 0; r < P; ++r)
            bufs[r][i] = s;
    }
    return LPO_OK;
}

int lpo_bsp_sgd_step_omp(float *const *grads, float *const *weights, int P,
                         size_t n, int root, float lr)
{
    if (bad_args(grads, P, root) || bad_args(weights, P, root))
        return LPO_EINVAL;
    const float invP = 1.0f / (float)P;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        float s = grads[0][i];
        for (int r = 1; r < P; ++r)
            s = s + grads[r][i];
        float g = s * invP;
        float t = lr * g;
        float w = weights[root][i] - t;
        for (int r = 0; r < P; ++r)
            weights[r][i] = w;
    }
    return LPO_OK;
}

#ifdef _OPENMP
#include <omp.h>
int lpo_num_threads(void) { return omp_get_max_threads(); }
#else
int lpo_num_threads(void) { return 1; }
#endif

/* ------------------------------------------------------------------------ */
/* 2. The same results computed the way the paper describes the pipeline      */
/*    (stage model: the P ranks are the P stages)       */
/* ------------------------------------------------------------------------ */

/* a1: "we dissect a long message into fine-grained blocks" PAPER.md:55.
 * Reading U6: nb = ceil(n / block), the last block is short. */
uint64_t lpo_num_blocks(size_t n, size_t block)
{
    if (block == 0)
        return 0;
    return (uint64_t)((n + block - 1) / block);
}

/* a2: which block rank r handles at tick t (stage model).  Rank r handles
 * block k = t - r at tick t, for 0 <= k < nb: rank 0 starts block k at tick k
 * and "GPU n, 0 < n < k-1, duplicates the same pattern of GPU 1"
 * one tick later per hop.  Returns -1 when rank r is idle at tick t. */
int64_t lpo_stage_block(int P, uint64_t nb, uint64_t t, int r)
{
    if (r < 0 || r >= P)
        return -1;
    if (t < (uint64_t)r)
        return -1;
    uint64_t k = t - (uint64_t)r;
    return k < nb ? (int64_t)k : -1;
}

/* Pipeline length "p - 1 + n/b" blocks, PAPER.md:89 (stage model, U2). */
uint64_t lpo_stage_ticks(int P, uint64_t nb)
{
    return nb == 0 ? 0 : (uint64_t)P - 1 + nb;
}

/* LP reduce / allreduce / broadcast, tick by tick, with an explicit receive
 * buffer per rank ("writing block a0 to a buffer on GPU1. Then,
 * GPU1 reduces the received block a0 with a1 to yield a'").
 *
 * Per tick t (t = 0 .. P+nb-2) every rank r with a block k = t - r:
 *   r == 0 : exposes its local block k as the partial            (load stage)
 *   r  > 0 : copies the partial exposed by r-1 at tick t-1 into its receive
 *            buffer, adds its local block, exposes the sum
 * The last rank's partial is the finished block; it is written to root
 * (reduce) or to every rank (allreduce: "a'' is broadcast").
 * op: 0 broadcast, 1 reduce, 2 allreduce.  *ticks_out receives the tick count.
 *
 * Finished blocks are written only after the tick loop has read every local
 * block it needs, so in-place operation is safe: outputs are staged in `done`.
 */
int lpo_lp_blocked(float *const *bufs, int P, size_t n, size_t block, int root,
                   int op, uint64_t *ticks_out)
{
    if (bad_args(bufs, P, root) || block == 0 || op < 0 || op > 2)
        return LPO_EINVAL;
    const uint64_t nb = lpo_num_blocks(n, block);
    const uint64_t ticks = lpo_stage_ticks(P, nb);
    if (ticks_out)
        *ticks_out = ticks;
    if (n == 0)
        return LPO_OK;

    /* exposed[r]: the partial rank r exposed at the previous tick; recvbuf[r]:
     * rank r's receive buffer.  One block each. */
    float **exposed = (float **)calloc((size_t)P, sizeof(float *));
    float **recvbuf = (float **)calloc((size_t)P, sizeof(float *));
    float **next = (float **)calloc((size_t)P, sizeof(float *));
    float *done = (float *)malloc(n * sizeof(float));
    if (!exposed || !recvbuf || !next || !done)
        return LPO_ENOMEM;
    for (int r = 0; r < P; ++r) {
        exposed[r] = (float *)malloc(block * sizeof(float));
        recvbuf[r] = (float *)malloc(block * sizeof(float));
        next[r] = (float *)malloc(block * sizeof(float));
        if (!exposed[r] || !recvbuf[r] || !next[r])
            return LPO_ENOMEM;
    }

    for (uint64_t t = 0; t < ticks; ++t) {
        /* all ranks act "simultaneously": read exposed[] of tick t-1, write
         * next[], then swap. */
        for (int r = 0; r < P; ++r) {
            int64_t k = lpo_stage_block(P, nb, t, r);
            if (k < 0)
                continue;
            size_t off = (size_t)k * block;
            size_t len = (off + block <= n) ? block : n - off;
            if (op == 0) {
                /* broadcast chain: stage 0 is the root's load; every later
                 * stage forwards what it received unchanged. */
                if (r == 0)
                    memcpy(next[0], bufs[root] + off, len * sizeof(float));
                else {
                    memcpy(recvbuf[r], exposed[r - 1], len * sizeof(float));
                    memcpy(next[r], recvbuf[r], len * sizeof(float));
                }
            } else {
                if (r == 0)
                    memcpy(next[0], bufs[0] + off, len * sizeof(float));
                else {
                    memcpy(recvbuf[r], exposed[r - 1], len * sizeof(float));
                    for (size_t j = 0; j < len; ++j)
                        next[r][j] = recvbuf[r][j] + bufs[r][off + j];
                }
            }
            if (r == P - 1)
                memcpy(done + off, next[r], len * sizeof(float));
        }
        for (int r = 0; r < P; ++r) {
            float *tmp = exposed[r];
            exposed[r] = next[r];
            next[r] = tmp;
        }
    }

    for (int r = 0; r < P; ++r) {
        int writes = (op == 1) ? (r == root) : (op == 0 ? (r != root) : 1);
        if (writes)
            memcpy(bufs[r], done, n * sizeof(float));
    }
    for (int r = 0; r < P; ++r) {
        free(exposed[r]);
        free(recvbuf[r]);
        free(next[r]);
    }
    free(exposed);
    free(recvbuf);
    free(next);
    free(done);
    return LPO_OK;
}

/* ------------------------------------------------------------------------ */
/* 3. Link-model schedule simulation (what Fig. 2 draws)   */
/* ------------------------------------------------------------------------ */

/* One transfer = one block moving over one link in one time step.  "a GPU
 * receives a block from the prior GPU via DMA1 while sending a block to the
 * next one via DMA2": per step each rank may send at most one
 * block and receive at most one block.  A transfer may start once the data it
 * carries is at its source (its dependency finished in an earlier step);
 * reduction is free ("we assume no latency on it").
 *
 * Chain as in Fig. 2: rank 0 -> 1 -> ... -> P-1, reduce root = rank P-1,
 * broadcast root = rank 0.
 *
 * op: 0 broadcast, 1 reduce, 2 allreduce.
 * reading (allreduce only, reading U3):
 *   0 = A, reverse flow: finished block k flows back P-1 -> P-2 -> ... -> 0
 *   1 = B, ring closure: P-1 -> 0, then 0 -> 1 -> ... -> P-1 (the text's
 *       literal "a'' is broadcast to GPU1 and GPU2 at the timestep 5, 6")
 * Greedy: steps are simulated one by one; in each step transfers are
 * considered in order (reduce traffic before redistribution traffic, lower
 * block first) and started when their dependency is met and both engines are
 * free.  done_step (optional, nb entries) receives, per block, the step at
 * which the block's last transfer finished.  Returns the number of steps. */
typedef struct {
    int src, dst;
    int64_t dep;      /* index of the transfer that must finish first, or -1 */
    uint64_t blk;
    uint64_t fin;     /* step at which it ran, 0 = not yet */
} lpo_xfer;

int lpo_link_sim(int P, uint64_t nb, int op, int reading, uint64_t *steps_out,
                 uint64_t *done_step)
{
    if (P < 1 || op < 0 || op > 2 || reading < 0 || reading > 1 || !steps_out)
        return LPO_EINVAL;
    *steps_out = 0;
    if (P == 1 || nb == 0)
        return LPO_OK;

    const uint64_t hops_fwd = (uint64_t)(P - 1);
    uint64_t per_block = hops_fwd;              /* broadcast or reduce */
    if (op == 2)
        per_block += (reading == 0) ? hops_fwd : (uint64_t)P;
    const uint64_t nx = per_block * nb;
    lpo_xfer *x = (lpo_xfer *)calloc((size_t)nx, sizeof(lpo_xfer));
    if (!x)
        return LPO_ENOMEM;

    /* Build the list: first all chain transfers (phase 1), then all
     * redistribution transfers (phase 2); lower block first in each. */
    uint64_t m = 0;
    for (uint64_t k = 0; k < nb; ++k)
        for (int h = 0; h < P - 1; ++h) {
            x[m].src = h;
            x[m].dst = h + 1;
            x[m].blk = k;
            x[m].dep = (h == 0) ? -1 : (int64_t)(m - 1);
            ++m;
        }
    if (op == 2) {
        for (uint64_t k = 0; k < nb; ++k) {
            int64_t last_reduce = (int64_t)(k * hops_fwd + hops_fwd - 1);
            if (reading == 0) {
                for (int h = P - 1; h > 0; --h) {
                    x[m].src = h;
                    x[m].dst = h - 1;
                    x[m].blk = k;
                    x[m].dep = (h == P - 1) ? last_reduce : (int64_t)(m - 1);
                    ++m;
                }
            } else {
                x[m].src = P - 1;
                x[m].dst = 0;
                x[m].blk = k;
                x[m].dep = last_reduce;
                ++m;
                for (int h = 0; h < P - 1; ++h) {
                    x[m].src = h;
                    x[m].dst = h + 1;
                    x[m].blk = k;
                    x[m].dep = (int64_t)(m - 1);
                    ++m;
                }
            }
        }
    }

    unsigned char *out_busy = (unsigned char *)malloc((size_t)P);
    unsigned char *in_busy = (unsigned char *)malloc((size_t)P);
    if (!out_busy || !in_busy)
        return LPO_ENOMEM;
    uint64_t remaining = nx, step = 0, first_open = 0;
    while (remaining > 0) {
        ++step;
        memset(out_busy, 0, (size_t)P);
        memset(in_busy, 0, (size_t)P);
        /* Phase-1 transfers come first in x[], so one pass in index order gives
         * them priority; phase 2 is scanned after.  To keep reduce traffic
         * ahead of redistribution traffic on shared engines, scan phase 1
         * fully, then phase 2. */
        for (uint64_t i = first_open; i < nx; ++i) {
            if (x[i].fin)
                continue;
            if (x[i].dep >= 0 && (x[x[i].dep].fin == 0 || x[x[i].dep].fin >= step))
                continue;
            if (out_busy[x[i].src] || in_busy[x[i].dst])
                continue;
            out_busy[x[i].src] = 1;
            in_busy[x[i].dst] = 1;
            x[i].fin = step;
            --remaining;
        }
        while (first_open < nx && x[first_open].fin)
            ++first_open;
    }
    *steps_out = step;
    if (done_step) {
        for (uint64_t k = 0; k < nb; ++k)
            done_step[k] = 0;
        for (uint64_t i = 0; i < nx; ++i)
            if (x[i].fin > done_step[x[i].blk])
                done_step[x[i].blk] = x[i].fin;
    }
    free(x);
    free(out_busy);
    free(in_busy);
    return LPO_OK;
}

/* Step at which block k's chain (phase 1) finished, i.e. when "a'', b'', ..."
 * exist at the last rank (a'' at step 2, b'',c'',d'' at 3,4,5 for
 * 3 GPUs).  Separate entry so the test can pin exactly that sentence. */
int lpo_link_sim_reduce_ready(int P, uint64_t nb, uint64_t *ready_step)
{
    uint64_t steps;
    return lpo_link_sim(P, nb, 1, 0, &steps, ready_step);
}

/* ------------------------------------------------------------------------ */
/* 4. MST (binomial tree) baseline values                    */
/* ------------------------------------------------------------------------ */

/* "organizes p GPUs into a balanced tree of height ceil(log p)" PAPER.md:93. */
int lpo_mst_levels(int P)
{
    int levels = 0;
    for (int d = 1; d < P; d *= 2)
        ++levels;
    return levels;
}

static int vrank_to_rank(int v, int root, int P) { return (v + root) % P; }

/* MST reduce on working copies work[v] (virtual ranks, v = 0 is the root):
 * for d = 1, 2, 4, ... < P: every v with v % 2d == 0 and v + d < P does
 * x_v = x_v + x_{v+d} on the whole message ("GPUs reduce the incoming data
 * only after the entire data is available"). */
static void mst_reduce_virtual(float **work, int P, size_t n)
{
    for (int d = 1; d < P; d *= 2)
        for (int v = 0; v + d < P; v += 2 * d)
            for (size_t i = 0; i < n; ++i)
                work[v][i] = work[v][i] + work[v + d][i];
}

/* MST broadcast on virtual ranks: for d from the largest power of two < P
 * down to 1: every v with v % 2d == 0 and v + d < P copies to v + d. */
static void mst_broadcast_virtual(float **work, int P, size_t n)
{
    int dmax = 1;
    while (dmax * 2 < P)
        dmax *= 2;
    for (int d = dmax; d >= 1; d /= 2)
        for (int v = 0; v + d < P; v += 2 * d)
            memcpy(work[v + d], work[v], n * sizeof(float));
}

int lpo_mst_broadcast(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!work)
        return LPO_ENOMEM;
    for (int v = 0; v < P; ++v)
        work[v] = bufs[vrank_to_rank(v, root, P)];
    if (P > 1)
        mst_broadcast_virtual(work, P, n);
    free(work);
    return LPO_OK;
}

/* Reduce leaves non-root vectors unchanged (U5): the tree runs on copies. */
int lpo_mst_reduce(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!work)
        return LPO_ENOMEM;
    for (int v = 0; v < P; ++v) {
        work[v] = (float *)malloc((n ? n : 1) * sizeof(float));
        if (!work[v])
            return LPO_ENOMEM;
        memcpy(work[v], bufs[vrank_to_rank(v, root, P)], n * sizeof(float));
    }
    mst_reduce_virtual(work, P, n);
    memcpy(bufs[root], work[0], n * sizeof(float));
    for (int v = 0; v < P; ++v)
        free(work[v]);
    free(work);
    return LPO_OK;
}

/* "allreduce is a combination of broadcast and reduce" PAPER.md:93; the tree
 * root is rank 0. */
int lpo_mst_allreduce(float *const *bufs, int P, size_t n)
{
    int rc = lpo_mst_reduce(bufs, P, n, 0);
    if (rc != LPO_OK)
        return rc;
    return lpo_mst_broadcast(bufs, P, n, 0);
}

/* ------------------------------------------------------------------------ */
/* 5. BE (bidirectional exchange) baseline values                 */
/* ------------------------------------------------------------------------ */

static int is_pow2(int P) { return P >= 1 && (P & (P - 1)) == 0; }

/* Segment boundaries: recursive halving of [lo, hi) splits at lo + (hi-lo)/2. */

/* Reduce-scatter by recursive halving on working copies: for d = P/2, P/4,
 * ..., 1: rank r and partner r^d split their current segment in half; r keeps
 * the lower half if (r & d) == 0 else the upper, and adds the partner's copy
 * of that half into its own.  seg_lo/seg_hi return each rank's final segment. */
static void be_reduce_scatter(float **work, int P, size_t n, size_t *seg_lo,
                              size_t *seg_hi)
{
    for (int r = 0; r < P; ++r) {
        seg_lo[r] = 0;
        seg_hi[r] = n;
    }
    for (int d = P / 2; d >= 1; d /= 2) {
        /* all ranks exchange "simultaneously": each rank only writes the half
         * it keeps and only reads the partner's copy of that same half, which
         * the partner does not write in this step. */
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            size_t lo = seg_lo[r], hi = seg_hi[r];
            size_t mid = lo + (hi - lo) / 2;
            size_t klo = (r & d) ? mid : lo;
            size_t khi = (r & d) ? hi : mid;
            for (size_t i = klo; i < khi; ++i)
                work[r][i] = work[r][i] + work[q][i];
        }
        for (int r = 0; r < P; ++r) {
            size_t lo = seg_lo[r], hi = seg_hi[r];
            size_t mid = lo + (hi - lo) / 2;
            if (r & d)
                seg_lo[r] = mid;
            else
                seg_hi[r] = mid;
        }
    }
}

/* Allgather by recursive doubling, the halving steps in reverse: for d = 1, 2,
 * ..., P/2: rank r and partner r^d copy each other's current segment. */
static void be_allgather(float **work, int P, size_t *seg_lo, size_t *seg_hi)
{
    for (int d = 1; d < P; d *= 2) {
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            memcpy(work[r] + seg_lo[q], work[q] + seg_lo[q],
                   (seg_hi[q] - seg_lo[q]) * sizeof(float));
        }
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            if (q < r)
                continue;
            size_t lo = seg_lo[r] < seg_lo[q] ? seg_lo[r] : seg_lo[q];
            size_t hi = seg_hi[r] > seg_hi[q] ? seg_hi[r] : seg_hi[q];
            seg_lo[r] = seg_lo[q] = lo;
            seg_hi[r] = seg_hi[q] = hi;
        }
    }
}

/* "allreduce consists of a reducescatter and a allgather" PAPER.md:95. */
int lpo_be_allreduce(float *const *bufs, int P, size_t n)
{
    if (bad_args(bufs, P, 0))
        return LPO_EINVAL;
    if (!is_pow2(P))
        return LPO_EUNSUPPORTED; /* reading U14 */
    size_t *lo = (size_t *)malloc((size_t)P * sizeof(size_t));
    size_t *hi = (size_t *)malloc((size_t)P * sizeof(size_t));
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!lo || !hi || !work)
        return LPO_ENOMEM;
    for (int r = 0; r < P; ++r)
        work[r] = bufs[r];
    be_reduce_scatter(work, P, n, lo, hi);
    be_allgather(work, P, lo, hi);
    free(lo);
    free(hi);
    free(work);
    return LPO_OK;
}

/* "The MPI long message reduce consists of a reducescatter plus a gather"
 * PAPER.md:95.  Runs on copies so non-root vectors stay unchanged (U5). */
int lpo_be_reduce(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    if (!is_pow2(P))
        return LPO_EUNSUPPORTED;
    size_t *lo = (size_t *)malloc((size_t)P * sizeof(size_t));
    size_t *hi = (size_t *)malloc((size_t)P * sizeof(size_t));
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!lo || !hi || !work)
        return LPO_ENOMEM;
    for (int r = 0; r < P; ++r) {
        work[r] = (float *)malloc((n ? n : 1) * sizeof(float));
        if (!work[r])
            return LPO_ENOMEM;
        memcpy(work[r], bufs[r], n * sizeof(float));
    }
    be_reduce_scatter(work, P, n, lo, hi);
    for (int r = 0; r < P; ++r) /* gather every final segment to the root */
        memcpy(bufs[root] + lo[r], work[r] + lo[r], (hi[r] - lo[r]) * sizeof(float));
    for (int r = 0; r < P; ++r)
        free(work[r]);
    free(lo);
    free(hi);
    free(work);
    return LPO_OK;
}

/* "MPI broadcast handles long messages with a MST based scatter followed by a
 * BE allgather" PAPER.md:95.  Scatter on virtual ranks v = r XOR root (so that
 * the exchange partner is v ^ d in both phases): for d = P/2, ..., 1: every v
 * that holds a segment (v % 2d == 0) sends the upper half of its segment to
 * v + d.  Then the allgather above. */
int lpo_be_broadcast(float *const *bufs, int P, size_t n, int root)
{
    if (bad_args(bufs, P, root))
        return LPO_EINVAL;
    if (!is_pow2(P))
        return LPO_EUNSUPPORTED;
    size_t *lo = (size_t *)malloc((size_t)P * sizeof(size_t));
    size_t *hi = (size_t *)malloc((size_t)P * sizeof(size_t));
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!lo || !hi || !work)
        return LPO_ENOMEM;
    for (int v = 0; v < P; ++v)
        work[v] = bufs[v ^ root];
    lo[0] = 0;
    hi[0] = n;
    for (int d = P / 2; d >= 1; d /= 2)
        for (int v = 0; v < P; v += 2 * d) {
            size_t mid = lo[v] + (hi[v] - lo[v]) / 2;
            memcpy(work[v + d] + mid, work[v] + mid, (hi[v] - mid) * sizeof(float));
            lo[v + d] = mid;
            hi[v + d] = hi[v];
            hi[v] = mid;
        }
    be_allgather(work, P, lo, hi);
    free(lo);
    free(hi);
    free(work);
    return LPO_OK;
}

/* ------------------------------------------------------------------------ */
/* 5b. Reduce / allreduce with an operator                        */
/* ------------------------------------------------------------------------ */

/* PAPER.md:59 (Sec. 3, Reduce): "It supports basic arithmetic operations such
 * as summations and multiplications."  red: 0 = sum, 1 = product.  Everything
 * else is as in sections 1, 4 and 5: the LP result is the left fold in rank
 * order 0 -> P-1 (a0, a' = a0 (op) a1, a'' = a' (op) a2), MST and BE combine
 * along their own trees; one fp32 RN operation per combine, no FMA. */
#define LPO_RED_SUM 0
#define LPO_RED_PROD 1

static float combine(float a, float b, int red)
{
    return red == LPO_RED_PROD ? a * b : a + b;
}

static int bad_red(int red) { return red != LPO_RED_SUM && red != LPO_RED_PROD; }

/* F[i] = (((x_0[i] op x_1[i]) op x_2[i]) op ...) op x_{P-1}[i].  out may not alias inputs. */
int lpo_chain_fold(const float *const *in, int P, size_t n, int red, float *out)
{
    if (in == NULL || out == NULL || P < 1 || bad_red(red))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        float s = in[0][i];
        for (int r = 1; r < P; ++r)
            s = combine(s, in[r][i], red);
        out[i] = s;
    }
    return LPO_OK;
}

/* Reduce with operator: root <- F, the other vectors unchanged (U5). */
int lpo_reduce_op(float *const *bufs, int P, size_t n, int root, int red)
{
    if (bad_args(bufs, P, root) || bad_red(red))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        float s = bufs[0][i];
        for (int r = 1; r < P; ++r)
            s = combine(s, bufs[r][i], red);
        bufs[root][i] = s;
    }
    return LPO_OK;
}

/* Allreduce with operator: every rank <- F, the same bits everywhere. */
int lpo_allreduce_op(float *const *bufs, int P, size_t n, int red)
{
    if (bad_args(bufs, P, 0) || bad_red(red))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        float s = bufs[0][i];
        for (int r = 1; r < P; ++r)
            s = combine(s, bufs[r][i], red);
        for (int r = 0; r < P; ++r)
            bufs[r][i] = s;
    }
    return LPO_OK;
}

/* MST tree (section 4) with operator: x_v = x_v op x_{v+d}, d = 1, 2, 4, ... */
static void mst_reduce_virtual_op(float **work, int P, size_t n, int red)
{
    for (int d = 1; d < P; d *= 2)
        for (int v = 0; v + d < P; v += 2 * d)
            for (size_t i = 0; i < n; ++i)
                work[v][i] = combine(work[v][i], work[v + d][i], red);
}

int lpo_mst_reduce_op(float *const *bufs, int P, size_t n, int root, int red)
{
    if (bad_args(bufs, P, root) || bad_red(red))
        return LPO_EINVAL;
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!work)
        return LPO_ENOMEM;
    for (int v = 0; v < P; ++v) {
        work[v] = (float *)malloc((n ? n : 1) * sizeof(float));
        if (!work[v])
            return LPO_ENOMEM;
        memcpy(work[v], bufs[vrank_to_rank(v, root, P)], n * sizeof(float));
    }
    mst_reduce_virtual_op(work, P, n, red);
    memcpy(bufs[root], work[0], n * sizeof(float));
    for (int v = 0; v < P; ++v)
        free(work[v]);
    free(work);
    return LPO_OK;
}

int lpo_mst_allreduce_op(float *const *bufs, int P, size_t n, int red)
{
    int rc = lpo_mst_reduce_op(bufs, P, n, 0, red);
    if (rc != LPO_OK)
        return rc;
    return lpo_mst_broadcast(bufs, P, n, 0);
}

/* BE reduce-scatter (section 5) with operator: own_half = own_half op partner's copy of that half. */
static void be_reduce_scatter_op(float **work, int P, size_t n, size_t *seg_lo,
                                 size_t *seg_hi, int red)
{
    for (int r = 0; r < P; ++r) {
        seg_lo[r] = 0;
        seg_hi[r] = n;
    }
    for (int d = P / 2; d >= 1; d /= 2) {
        for (int r = 0; r < P; ++r) {
            int q = r ^ d;
            size_t lo = seg_lo[r], hi = seg_hi[r];
            size_t mid = lo + (hi - lo) / 2;
            size_t klo = (r & d) ? mid : lo;
            size_t khi = (r & d) ? hi : mid;
            for (size_t i = klo; i < khi; ++i)
                work[r][i] = combine(work[r][i], work[q][i], red);
        }
        for (int r = 0; r < P; ++r) {
            size_t lo = seg_lo[r], hi = seg_hi[r];
            size_t mid = lo + (hi - lo) / 2;
            if (r & d)
                seg_lo[r] = mid;
            else
                seg_hi[r] = mid;
        }
    }
}

int lpo_be_allreduce_op(float *const *bufs, int P, size_t n, int red)
{
    if (bad_args(bufs, P, 0) || bad_red(red))
        return LPO_EINVAL;
    if (!is_pow2(P))
        return LPO_EUNSUPPORTED;
    size_t *lo = (size_t *)malloc((size_t)P * sizeof(size_t));
    size_t *hi = (size_t *)malloc((size_t)P * sizeof(size_t));
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!lo || !hi || !work)
        return LPO_ENOMEM;
    for (int r = 0; r < P; ++r)
        work[r] = bufs[r];
    be_reduce_scatter_op(work, P, n, lo, hi, red);
    be_allgather(work, P, lo, hi);
    free(lo);
    free(hi);
    free(work);
    return LPO_OK;
}

int lpo_be_reduce_op(float *const *bufs, int P, size_t n, int root, int red)
{
    if (bad_args(bufs, P, root) || bad_red(red))
        return LPO_EINVAL;
    if (!is_pow2(P))
        return LPO_EUNSUPPORTED;
    size_t *lo = (size_t *)malloc((size_t)P * sizeof(size_t));
    size_t *hi = (size_t *)malloc((size_t)P * sizeof(size_t));
    float **work = (float **)malloc((size_t)P * sizeof(float *));
    if (!lo || !hi || !work)
        return LPO_ENOMEM;
    for (int r = 0; r < P; ++r) {
        work[r] = (float *)malloc((n ? n : 1) * sizeof(float));
        if (!work[r])
            return LPO_ENOMEM;
        memcpy(work[r], bufs[r], n * sizeof(float));
    }
    be_reduce_scatter_op(work, P, n, lo, hi, red);
    for (int r = 0; r < P; ++r)
        memcpy(bufs[root] + lo[r], work[r] + lo[r], (hi[r] - lo[r]) * sizeof(float));
    for (int r = 0; r < P; ++r)
        free(work[r]);
    free(lo);
    free(hi);
    free(work);
    return LPO_OK;
}

/* Layer-wise reduce / allreduce with operator: the definitions above on every
 * slice, in list order (Alg. 1).  op: 1 reduce, 2 allreduce. */
int lpo_collective_segments_op(int op, int red, float *const *bufs, int P, size_t n,
                               const size_t *seg_off, const size_t *seg_len,
                               int n_seg, int root)
{
    if (bad_args(bufs, P, root) || bad_red(red) || n_seg < 0 ||
        (n_seg > 0 && (!seg_off || !seg_len)) || P > 64 || (op != 1 && op != 2))
        return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s)
        if (seg_off[s] > n || seg_len[s] > n - seg_off[s])
            return LPO_EINVAL;
    for (int s = 0; s < n_seg; ++s) {
        float *slice[64];
        for (int r = 0; r < P; ++r)
            slice[r] = bufs[r] + seg_off[s];
        int rc = op == 1 ? lpo_reduce_op(slice, P, seg_len[s], root, red)
                         : lpo_allreduce_op(slice, P, seg_len[s], red);
        if (rc != LPO_OK)
            return rc;
    }
    return LPO_OK;
}

/* ------------------------------------------------------------------------ */
/* 6. Cost model, Table 1, fp64                        */
/* ------------------------------------------------------------------------ */

/* algo: 0 LP, 1 MST, 2 BE.  op: 0 broadcast, 1 reduce, 2 allreduce.
 * p ranks, n message bytes, b block bytes; alpha latency, beta s/byte
 * transfer, gamma s/byte reduce (Eq. 1).  log p is log2 p, not rounded up
 * ("we omit the ceiling for simplicity").  Table 1 as read in
 * DESIGN.md U10/U11. */
double lpo_cost(int algo, int op, double p, double n, double b, double alpha,
                double beta, double gamma)
{
    const double lg = log2(p);
    const double f = (p - 1.0) / p;
    if (algo == 0) {
        const double len = p - 1.0 + n / b;       /* pipeline length */
        const double vol = b * (p - 1.0) + n;     /* = b * len */
        if (op == 0)
            return len * alpha + vol * beta;
        if (op == 1)
            return len * alpha + vol * (beta + gamma);
        return 2.0 * len * alpha + vol * (2.0 * beta + gamma);
    }
    if (algo == 1) {
        if (op == 0)
            return lg * (alpha + n * beta);
        if (op == 1)
            return lg * (alpha + n * beta + n * gamma);
        return lg * (2.0 * alpha + 2.0 * n * beta + n * gamma);
    }
    if (op == 0)
        return (lg + p - 1.0) * alpha + 2.0 * f * n * beta;
    return 2.0 * lg * alpha + 2.0 * f * n * beta + f * n * gamma;
}

/* ------------------------------------------------------------------------ */
/* 7. Element types other than fp32 (SURVEY 8(f)-4 "other reduce ops /        */
/*    dtypes"; reading U21)                                         */
/* ------------------------------------------------------------------------ */

/* The paper's messages are fp32 (Caffe).  This section extends the result
 * definitions of sections 1 and 5b to vectors of IEEE binary16 (f16), bfloat16
 * (bf16: 1 sign, 8 exponent, 7 fraction bits) and binary64 (f64).  Reading U21:
 * the chain forwards the running partial as a block of the message itself
 * ("GPU1 reduces the received block a0 with a1 to yield a'", and
 * a' then travels to GPU2 like any block), so the partial HAS the message's
 * element type: every combine is ONE round-to-nearest-even operation in that
 * type,
 *     F[i] = (((x_0[i] op x_1[i]) op x_2[i]) op ...) op x_{P-1}[i],
 * op = + or *, no wider accumulator, no flush-to-zero.  f16 and bf16 values are
 * passed as their 16-bit patterns (uint16_t).
 *
 * How one RN operation in a 16-bit type is computed here: both operands are
 * converted to double (exact), the operation is done in double, and the result
 * is rounded ONCE more to the narrow type by round_to_narrow() below.
 *  - products: 11 x 11 (f16) or 8 x 8 (bf16) significand bits -> exact in double;
 *  - sums: exact in double whenever the operands' exponents differ by less
 *    than 53 - p bits (p = 11 / 8 significand bits); beyond that the smaller
 *    operand is below 2^-40 ulp of the larger and neither rounding moves the
 *    result off the larger operand.  (In general a second rounding from a
 *    format with at least 2p + 2 significand bits is innocuous for + and *.)
 * So the value is the correctly rounded result of the exact operation.       */

#define LPO_DT_F32 0
#define LPO_DT_F16 1
#define LPO_DT_BF16 2
#define LPO_DT_F64 3

/* Round a double to the nearest value of a binary format with `p` significand
 * bits (hidden bit included), minimum normal exponent emin (value 2^emin) and
 * largest finite value (2 - 2^(1-p)) * 2^emax; ties to even; overflow to
 * infinity; gradual underflow.  Returns sign, biased exponent field and
 * fraction field packed as (sign << (ebits + p - 1)) | (E << (p - 1)) | frac.
 * NaN -> quiet NaN with the top fraction bit set.                            */
static uint32_t round_to_narrow(double x, int p, int ebits)
{
    const int bias = (1 << (ebits - 1)) - 1;
    const int emin = 1 - bias;            /* exponent of the smallest normal */
    const int emax = bias;                /* exponent of the largest binade  */
    const uint32_t sign = signbit(x) ? 1u << (ebits + p - 1) : 0u;
    const uint32_t inf = ((1u << ebits) - 1u) << (p - 1);
    if (isnan(x))
        return sign | inf | (1u << (p - 2));
    double ax = fabs(x);
    if (isinf(ax))
        return sign | inf;
    if (ax == 0.0)
        return sign;
    if (ax < ldexp(1.0, emin)) {
        /* subnormal range: spacing 2^(emin - (p-1)); the scaling is exact     */
        double q = nearbyint(ldexp(ax, (p - 1) - emin));   /* ties to even     */
        return sign | (uint32_t)q;       /* q == 2^(p-1) is the smallest normal */
    }
    int e;
    double m = frexp(ax, &e);            /* ax = m * 2^e, 0.5 <= m < 1         */
    double q = nearbyint(ldexp(m, p));   /* p-bit integer significand, RNE    */
    if (q == ldexp(1.0, p)) {            /* rounded up into the next binade   */
        q = ldexp(1.0, p - 1);
        e += 1;
    }
    int E = (e - 1) + bias;              /* ax = (q / 2^(p-1)) * 2^(e-1)       */
    if (e - 1 > emax)
        return sign | inf;               /* overflow: RN gives infinity       */
    return sign | ((uint32_t)E << (p - 1)) | ((uint32_t)q - (1u << (p - 1)));
}

/* Exact widening of a narrow pattern (p significand bits, ebits exponent bits). */
static double widen_narrow(uint32_t bits, int p, int ebits)
{
    const int bias = (1 << (ebits - 1)) - 1;
    const uint32_t frac = bits & ((1u << (p - 1)) - 1u);
    const uint32_t E = (bits >> (p - 1)) & ((1u << ebits) - 1u);
    const int neg = (bits >> (ebits + p - 1)) & 1u;
    double v;
    if (E == (1u << ebits) - 1u)
        v = frac ? NAN : INFINITY;
    else if (E == 0)
        v = ldexp((double)frac, (1 - bias) - (p - 1));
    else
        v = ldexp((double)(frac | (1u << (p - 1))), (int)E - bias - (p - 1));
    return neg ? -v : v;
}

uint16_t lpo_f16_from_f64(double x) { return (uint16_t)round_to_narrow(x, 11, 5); }
uint16_t lpo_bf16_from_f64(double x) { return (uint16_t)round_to_narrow(x, 8, 8); }
double lpo_f16_to_f64(uint16_t h) { return widen_narrow(h, 11, 5); }
double lpo_bf16_to_f64(uint16_t h) { return widen_narrow(h, 8, 8); }

static size_t dt_size(int dt)
{
    return dt == LPO_DT_F64 ? 8 : (dt == LPO_DT_F32 ? 4 : 2);
}
static int bad_dt(int dt) { return dt < LPO_DT_F32 || dt > LPO_DT_F64; }

/* element i of a vector of type dt, as a double (exact for every dt) */
static double dt_load(const void *v, size_t i, int dt)
{
    switch (dt) {
    case LPO_DT_F16: return lpo_f16_to_f64(((const uint16_t *)v)[i]);
    case LPO_DT_BF16: return lpo_bf16_to_f64(((const uint16_t *)v)[i]);
    case LPO_DT_F64: return ((const double *)v)[i];
    default: return (double)((const float *)v)[i];
    }
}

/* one RN operation in type dt on two values of type dt (held exactly in doubles) */
static double dt_combine(double a, double b, int dt, int red)
{
    switch (dt) {
    case LPO_DT_F16: {
        double r = red == LPO_RED_PROD ? a * b : a + b;
        return lpo_f16_to_f64(lpo_f16_from_f64(r));
    }
    case LPO_DT_BF16: {
        double r = red == LPO_RED_PROD ? a * b : a + b;
        return lpo_bf16_to_f64(lpo_bf16_from_f64(r));
    }
    case LPO_DT_F64:
        return red == LPO_RED_PROD ? a * b : a + b;
    default: {
        float fa = (float)a, fb = (float)b;      /* exact: a, b are fp32 values */
        return (double)(red == LPO_RED_PROD ? fa * fb : fa + fb);
    }
    }
}

static void dt_store(void *v, size_t i, int dt, double x)
{
    switch (dt) {
    case LPO_DT_F16: ((uint16_t *)v)[i] = lpo_f16_from_f64(x); break;   /* x is already an f16 value: exact */
    case LPO_DT_BF16: ((uint16_t *)v)[i] = lpo_bf16_from_f64(x); break;
    case LPO_DT_F64: ((double *)v)[i] = x; break;
    default: ((float *)v)[i] = (float)x; break;
    }
}

/* F = left fold in rank order of P vectors of n elements of type dt; out may not alias inputs. */
int lpo_chain_fold_dt(const void *const *in, int P, size_t n, int dt, int red, void *out)
{
    if (in == NULL || out == NULL || P < 1 || bad_red(red) || bad_dt(dt))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        double s = dt_load(in[0], i, dt);
        for (int r = 1; r < P; ++r)
            s = dt_combine(s, dt_load(in[r], i, dt), dt, red);
        dt_store(out, i, dt, s);
    }
    return LPO_OK;
}

/* Broadcast: every rank's vector <- the root's, byte for byte. */
int lpo_broadcast_dt(void *const *bufs, int P, size_t n, int dt, int root)
{
    if (bufs == NULL || P < 1 || root < 0 || root >= P || bad_dt(dt))
        return LPO_EINVAL;
    for (int r = 0; r < P; ++r)
        if (r != root)
            memcpy(bufs[r], bufs[root], n * dt_size(dt));
    return LPO_OK;
}

/* Reduce: root <- F, the other vectors unchanged (U5). */
int lpo_reduce_dt(void *const *bufs, int P, size_t n, int dt, int root, int red)
{
    if (bufs == NULL || P < 1 || root < 0 || root >= P || bad_red(red) || bad_dt(dt))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        double s = dt_load(bufs[0], i, dt);
        for (int r = 1; r < P; ++r)
            s = dt_combine(s, dt_load(bufs[r], i, dt), dt, red);
        dt_store(bufs[root], i, dt, s);
    }
    return LPO_OK;
}

/* Allreduce: every rank <- F, the same bits everywhere. */
int lpo_allreduce_dt(void *const *bufs, int P, size_t n, int dt, int red)
{
    if (bufs == NULL || P < 1 || bad_red(red) || bad_dt(dt))
        return LPO_EINVAL;
    for (size_t i = 0; i < n; ++i) {
        double s = dt_load(bufs[0], i, dt);
        for (int r = 1; r < P; ++r)
            s = dt_combine(s, dt_load(bufs[r], i, dt), dt, red);
        for (int r = 0; r < P; ++r)
            dt_store(bufs[r], i, dt, s);
    }
    return LPO_OK;
}
