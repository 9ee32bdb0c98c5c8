"""Pins for the oracle's LP schedule (stage model + link model), the MST level
count, the Table 1 cost functions and the fused BSP-SGD step.  CPU only.
Citations are PAPER.md:<line>; U<k> are the readings listed in DESIGN.md.
"""
import math

import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from tests.conftest import read_golden

LP, MST, BE = 0, 1, 2
BCAST, REDUCE, ALLREDUCE = 0, 1, 2


def _copy(bufs):
    return [b.copy() for b in bufs]


# ----------------------------------------------------------------------------
# link model: the paper's worked example, tests/golden
# ----------------------------------------------------------------------------

def test_link_sim_matches_paper_worked_example(oracle):
    g = {(int(P), int(nb), q): int(v) for P, nb, q, v in read_golden("paper_fig2_link_steps.txt")}
    P, nb = 3, 4
    ready = oracle.link_sim_reduce_ready(P, nb)
    for k in range(nb):
        assert ready[k] == g[(P, nb, f"reduce_ready_block{k}")]
    assert oracle.link_sim(P, nb, REDUCE) == g[(P, nb, "reduce_steps")]
    assert oracle.link_sim(P, nb, BCAST) == g[(P, nb, "broadcast_steps")]
    for reading in (0, 1):  # U3: both readings must reproduce the printed 9 and "5, 6"
        steps, done = oracle.link_sim(P, nb, ALLREDUCE, reading, per_block=True)
        assert steps == g[(P, nb, "allreduce_steps")]
        assert done[0] == g[(P, nb, "allreduce_block0_done")]
    assert (oracle.link_sim(P, nb, REDUCE) + oracle.link_sim(P, nb, BCAST)
            == g[(P, nb, "reduce_plus_broadcast_steps")])


@pytest.mark.parametrize("P", [2, 3, 4, 6, 8, 16])
@pytest.mark.parametrize("nb", [1, 2, 4, 16, 59])
def test_link_model_closed_form_and_allreduce_bounds(oracle, P, nb):
    # one block crosses P-1 links, one new block enters per step: P-2+nb (U2)
    assert oracle.link_sim(P, nb, BCAST) == P - 2 + nb
    assert oracle.link_sim(P, nb, REDUCE) == P - 2 + nb
    # PAPER.md:71 "only needs to fill the pipeline once": strictly cheaper than
    # the two separate calls whenever there is a pipeline to fill (P >= 3),
    # never more than Table 1's 2(p-1+n/b).
    for reading in (0, 1):
        ar = oracle.link_sim(P, nb, ALLREDUCE, reading)
        assert P - 2 + nb < ar <= 2 * (P - 1 + nb)
    # reading A (U3) never does a redundant hop, so it beats reduce + broadcast
    # as soon as there is a second block to overlap with.
    if nb >= 2:
        assert oracle.link_sim(P, nb, ALLREDUCE, 0) < 2 * (P - 2 + nb)


def test_link_sim_trivial(oracle):
    assert oracle.link_sim(1, 7, ALLREDUCE) == 0
    assert oracle.link_sim(4, 0, REDUCE) == 0
    assert oracle.link_sim(2, 1, BCAST) == 1


# ----------------------------------------------------------------------------
# stage model: pipeline length p - 1 + n/b, schedule validity
# ----------------------------------------------------------------------------

@pytest.mark.parametrize("P,nb", [(1, 1), (2, 5), (3, 4), (4, 16), (6, 931), (16, 527)])
def test_stage_schedule_properties(oracle, P, nb):
    T = oracle.stage_ticks(P, nb)
    assert T == P + nb - 1                       # PAPER.md:89 / north_star fixed point
    seen = {}
    for t in range(T):
        blocks = [oracle.stage_block(P, nb, t, r) for r in range(P)]
        busy = [(r, k) for r, k in enumerate(blocks) if k >= 0]
        assert len({k for _, k in busy}) == len(busy)     # a block is at one stage per tick
        for r, k in busy:
            assert (r, k) not in seen                     # every (rank, block) once
            seen[(r, k)] = t
            if r > 0:
                assert seen[(r - 1, k)] == t - 1          # hop order along the chain
        if P - 1 <= t < nb:                               # PAPER.md:55 "fully utilized once
            assert len(busy) == P                         #  the pipeline is filled"
    assert len(seen) == P * nb
    assert oracle.stage_block(P, nb, T, P - 1) == -1


def test_num_blocks_configs(oracle):
    # U6: ceil; BASELINE.json configs
    assert oracle.num_blocks(1_048_576, 65_536) == 16
    assert oracle.num_blocks(61_000_000, 65_536) == 931
    assert 61_000_000 - 930 * 65_536 == 51_520
    assert oracle.num_blocks(138_000_000, 262_144) == 527
    assert oracle.num_blocks(7_000_000, 65_536) == 107
    assert oracle.num_blocks(5, 100) == 1
    assert oracle.num_blocks(0, 8) == 0


@pytest.mark.parametrize("op", [BCAST, REDUCE, ALLREDUCE])
@pytest.mark.parametrize("P,n,block,root", [(1, 10, 3, 0), (3, 100, 7, 2), (4, 64, 16, 0),
                                            (5, 33, 64, 1), (6, 1000, 9, 5)])
def test_tick_by_tick_pipeline_reaches_the_definition(oracle, op, P, n, block, root):
    # The blocked, receive-buffer, tick-by-tick pipeline must give
    # the plain definitions' bits for every block size, and take P+nb-1 ticks.
    src = inputs.rank_vectors(51, P, n)
    a, b = _copy(src), _copy(src)
    ticks = oracle.lp_blocked(a, block, op, root=root)
    assert ticks == P + math.ceil(n / block) - 1
    if op == BCAST:
        oracle.broadcast(b, root=root)
    elif op == REDUCE:
        oracle.reduce(b, root=root)
    else:
        oracle.allreduce(b)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(a, b))


def test_mst_levels_match_paper(oracle):
    for P, steps in read_golden("paper_mst_steps.txt"):
        assert oracle.mst_levels(int(P)) == int(steps)
    for P in range(1, 40):
        assert oracle.mst_levels(P) == (math.ceil(math.log2(P)) if P > 1 else 0)


# ----------------------------------------------------------------------------
# Table 1 cost functions
# ----------------------------------------------------------------------------

def test_cost_table1_hand_values(oracle):
    # p=4, n=1000, b=10, alpha=1, beta=2, gamma=3; expanded by hand from Table 1.
    p, n, b, al, be, ga = 4, 1000, 10, 1.0, 2.0, 3.0
    c = lambda algo, op: oracle.cost(algo, op, p, n, b, al, be, ga)
    assert c(LP, BCAST) == 103 * 1 + 1030 * 2                       # (p-1+n/b)a+(b(p-1)+n)B
    assert c(LP, REDUCE) == 103 * 1 + 1030 * 5                      # ... (B+g)
    assert c(LP, ALLREDUCE) == 2 * 103 * 1 + 1030 * 7               # 2(..)a + (..)(2B+g)
    assert c(MST, BCAST) == 2 * (1 + 2000)                          # log p (a + nB)
    assert c(MST, REDUCE) == 2 * (1 + 2000 + 3000)                  # U10
    assert c(MST, ALLREDUCE) == 2 * (2 + 4000 + 3000)
    assert c(BE, BCAST) == (2 + 3) * 1 + 2 * 750 * 2                # (log p+p-1)a + 2((p-1)/p n)B
    assert c(BE, REDUCE) == 4 * 1 + 2 * 750 * 2 + 750 * 3
    assert c(BE, ALLREDUCE) == c(BE, REDUCE)                        # Table 1: same row


@pytest.mark.parametrize("p", [2, 3, 4, 6, 8, 16, 64])
def test_cost_proposition1(oracle, p):
    # alpha -> 0: Eq. 2  T_BE/T_LP < 2 ; Eq. 3  T_MST/T_LP < log p 
    for n, b in ((2 ** 26, 2 ** 16), (2 ** 20, 2 ** 16), (2 ** 16, 2 ** 16)):
        for op, ga in ((BCAST, 0.0), (REDUCE, 0.0), (ALLREDUCE, 0.0)):
            lp = oracle.cost(LP, op, p, n, b, 0.0, 1e-9, ga)
            be = oracle.cost(BE, op, p, n, b, 0.0, 1e-9, ga)
            mst = oracle.cost(MST, op, p, n, b, 0.0, 1e-9, ga)
            assert be / lp < 2.0
            assert mst / lp < math.log2(p) or p == 2 and mst / lp < 1.0 + 1e-12
        # Eq. 2's closed form
        lp = oracle.cost(LP, BCAST, p, n, b, 0.0, 1e-9, 0.0)
        be = oracle.cost(BE, BCAST, p, n, b, 0.0, 1e-9, 0.0)
        assert be / lp == pytest.approx(2 * (1 - 1 / p) / (1 + b / n * (p - 1)), rel=1e-12)


def test_cost_lp_invariant_to_p(oracle):
    # with b(p-1) << n the bandwidth term is n*beta for every p.
    n, b = 61_000_000 * 4, 65_536
    base = oracle.cost(LP, BCAST, 2, n, b, 0.0, 1e-9, 0.0)
    for p in (2, 4, 8, 16):
        c = oracle.cost(LP, BCAST, p, n, b, 0.0, 1e-9, 0.0)
        assert c / (n * 1e-9) == pytest.approx(1 + b * (p - 1) / n, rel=1e-12)
        assert abs(c / base - 1) < 0.005
        assert oracle.cost(MST, BCAST, p, n, b, 0.0, 1e-9, 0.0) == pytest.approx(
            math.log2(p) * n * 1e-9)


# ----------------------------------------------------------------------------
# fused BSP-SGD step (U7, U8)
# ----------------------------------------------------------------------------

def test_sgd_step_is_allreduce_scale_update(oracle):
    # composition written with numpy float32 ops (each one RN op, no FMA):
    # S by chain order, g = S * fl(1/P), t = lr * g, w' = w_root - t.
    P, n, lr, root = 6, 5003, np.float32(0.01), 2
    grads, weights = inputs.sgd_inputs(61, P, n)
    for r in range(P):       # make replicas differ so that "reads weights[root]" is tested
        weights[r] = weights[r] + np.float32(r)
    g0 = _copy(grads)
    S = grads[0].copy()
    for r in range(1, P):
        S = S + grads[r]
    invP = np.float32(1.0) / np.float32(P)
    want = weights[root] - lr * (S * invP)
    assert want.dtype == np.float32
    oracle.bsp_sgd_step(grads, weights, root=root, lr=float(lr))
    for r in range(P):
        assert weights[r].tobytes() == want.tobytes()       # U8: replicas identical
        assert grads[r].tobytes() == g0[r].tobytes()        # grads unchanged
    # and via the oracle's own allreduce ("allreduce(grad_sub)")
    ar = _copy(g0)
    oracle.allreduce(ar)
    assert ar[0].tobytes() == S.tobytes()


def test_sgd_step_closed_forms(oracle):
    n = 64
    # lr = 0: w unchanged (w - 0 exact)
    grads, weights = inputs.sgd_inputs(62, 4, n)
    w0 = weights[0].copy()
    oracle.bsp_sgd_step(grads, weights, root=0, lr=0.0)
    assert all(w.tobytes() == w0.tobytes() for w in weights)
    # identical small-integer gradients on P = 2^k ranks: the average is the
    # gradient itself, lr = 0.5 exact => w' = w - g/2 exactly.
    for P in (2, 4, 8):
        g = inputs.small_integers(63, 0, n)
        grads = [g.copy() for _ in range(P)]
        w = inputs.small_integers(63, 1, n, -100, 100)
        weights = [w.copy() for _ in range(P)]
        oracle.bsp_sgd_step(grads, weights, root=P - 1, lr=0.5)
        want = (w.astype(np.float64) - 0.5 * g.astype(np.float64)).astype(np.float32)
        assert all(x.tolist() == want.tolist() for x in weights)
    # sign: a positive gradient must DEcrease w (Eq. 5)
    grads = [np.ones(4, np.float32) for _ in range(2)]
    weights = [np.zeros(4, np.float32) for _ in range(2)]
    oracle.bsp_sgd_step(grads, weights, root=0, lr=0.25)
    assert weights[0].tolist() == [-0.25] * 4


def test_sgd_step_fp64_bound_and_iterations(oracle):
    # 20 iterations with the same gradients (config 3's recipe, smaller): the
    # result tracks the fp64 recurrence w - k*lr*mean(g) within rounding, and
    # replicas stay bitwise equal after every iteration (U8).
    P, n, lr = 8, 2048, 0.01
    grads, weights = inputs.sgd_inputs(2, P, n)
    w64 = weights[0].astype(np.float64)
    gbar = np.stack([g.astype(np.float64) for g in grads]).mean(axis=0)
    for it in range(1, 21):
        oracle.bsp_sgd_step(grads, weights, root=0, lr=lr)
        assert all(w.tobytes() == weights[0].tobytes() for w in weights)
        ref = w64 - it * lr * gbar
        assert np.max(np.abs(weights[0] - ref)) <= it * (2.0 ** -23) * 0.3


# ----------------------------------------------------------------------------
# SGD + momentum (reading U18) and the Alg. 2 step (U9)
# ----------------------------------------------------------------------------

def test_momentum_step_is_the_five_op_composition(oracle):
    # written out with numpy float32 ops, one RN op each: g = S*invP, t = lr*g, m = mu*v, v' = m+t, w' = w_root-v'
    P, n, lr, mu, root = 5, 4099, np.float32(0.015), np.float32(0.9), 3
    grads, weights = inputs.sgd_inputs(71, P, n)
    for r in range(P):
        weights[r] = weights[r] + np.float32(r)
    vel = inputs.normal(71, 99, n, 0.01)
    g0 = _copy(grads)
    S = grads[0].copy()
    for r in range(1, P):
        S = S + grads[r]
    invP = np.float32(1.0) / np.float32(P)
    t = lr * (S * invP)
    m = mu * vel
    v_want = m + t
    w_want = weights[root] - v_want
    assert v_want.dtype == np.float32 and w_want.dtype == np.float32
    oracle.bsp_sgd_momentum_step(grads, weights, vel, root=root, lr=float(lr), mu=float(mu))
    assert vel.tobytes() == v_want.tobytes()
    for r in range(P):
        assert weights[r].tobytes() == w_want.tobytes()
        assert grads[r].tobytes() == g0[r].tobytes()


def test_momentum_closed_forms(oracle):
    n = 96
    # mu = 0, v = 0: exactly the plain step (m = 0*0 = 0, v' = 0 + t = t)
    grads, weights = inputs.sgd_inputs(72, 4, n)
    w_plain = _copy(weights)
    oracle.bsp_sgd_step(grads, w_plain, root=1, lr=0.01)
    vel = np.zeros(n, np.float32)
    oracle.bsp_sgd_momentum_step(grads, weights, vel, root=1, lr=0.01, mu=0.0)
    assert all(a.tobytes() == b.tobytes() for a, b in zip(weights, w_plain))
    # lr = 0: v' = mu*v, w' = w - mu*v  (dyadic values: exact)
    P = 2
    grads = [inputs.small_integers(73, r, n) for r in range(P)]
    w = inputs.small_integers(73, 7, n, -100, 100)
    weights = [w.copy() for _ in range(P)]
    v = inputs.small_integers(73, 8, n, -64, 64)
    vel = v.copy()
    oracle.bsp_sgd_momentum_step(grads, weights, vel, root=0, lr=0.0, mu=0.5)
    assert vel.tolist() == (0.5 * v.astype(np.float64)).tolist()
    assert weights[1].tolist() == (w.astype(np.float64) - 0.5 * v.astype(np.float64)).tolist()
    # constant small-integer gradient g on P = 4 ranks, lr = 0.25, mu = 0.5, v0 = 0: everything stays dyadic, so
    # the geometric recurrence holds EXACTLY:  v_k = lr*g*(1 - mu^k)/(1 - mu),  w_k = w_0 - sum_{j<=k} v_j
    P, lr, mu = 4, 0.25, 0.5
    g = inputs.small_integers(74, 0, n, -8, 8)
    grads = [g.copy() for _ in range(P)]
    w0 = inputs.small_integers(74, 1, n, -100, 100)
    weights = [w0.copy() for _ in range(P)]
    vel = np.zeros(n, np.float32)
    g64, w64, acc = g.astype(np.float64), w0.astype(np.float64), np.zeros(n)
    for k in range(1, 9):
        oracle.bsp_sgd_momentum_step(grads, weights, vel, root=k % P, lr=lr, mu=mu)
        vk = lr * g64 * (1.0 - mu ** k) / (1.0 - mu)
        acc = acc + vk
        assert vel.tolist() == vk.tolist(), k
        assert all(x.tolist() == (w64 - acc).tolist() for x in weights), k
    # sign: positive gradient, positive velocity both decrease w
    grads = [np.ones(4, np.float32) for _ in range(2)]
    weights = [np.zeros(4, np.float32) for _ in range(2)]
    vel = np.full(4, 2.0, np.float32)
    oracle.bsp_sgd_momentum_step(grads, weights, vel, root=0, lr=0.25, mu=0.5)
    assert vel.tolist() == [1.25] * 4 and weights[1].tolist() == [-1.25] * 4


def test_momentum_tracks_fp64_recurrence(oracle):
    P, n, lr, mu = 8, 2048, 0.01, 0.9
    grads, weights = inputs.sgd_inputs(2, P, n)
    vel = np.zeros(n, np.float32)
    w64, v64 = weights[0].astype(np.float64), np.zeros(n)
    gbar = np.stack([g.astype(np.float64) for g in grads]).mean(axis=0)
    for it in range(1, 21):
        oracle.bsp_sgd_momentum_step(grads, weights, vel, root=0, lr=lr, mu=mu)
        v64 = mu * v64 + lr * gbar
        w64 = w64 - v64
        assert all(w.tobytes() == weights[0].tobytes() for w in weights)
        assert np.max(np.abs(vel - v64)) <= it * 2.0 ** -23 * 0.02
        assert np.max(np.abs(weights[0] - w64)) <= it * 2.0 ** -23 * 0.5


@pytest.mark.parametrize("with_momentum", [False, True])
def test_alg2_step_is_reduce_update_broadcast(oracle, with_momentum):
    # Alg. 2 written with the oracle's OTHER entry points and numpy: reduce (grads[root] <- S), numpy update of
    # the root replica, broadcast.  Its weights equal the fused Alg. 3 step bit for bit (same arithmetic on the same S).
    P, n, lr, mu, root = 6, 3001, np.float32(0.02), np.float32(0.9), 4
    grads, weights = inputs.sgd_inputs(75, P, n)
    for r in range(P):
        weights[r] = weights[r] + np.float32(r)
    vel = inputs.normal(75, 99, n, 0.01) if with_momentum else None
    g_a, w_a, v_a = _copy(grads), _copy(weights), (vel.copy() if with_momentum else None)
    g_b, w_b, v_b = _copy(grads), _copy(weights), (vel.copy() if with_momentum else None)
    # (a) by hand
    oracle.reduce(g_a, root=root)
    S = g_a[root]
    t = lr * (S * (np.float32(1.0) / np.float32(P)))
    if with_momentum:
        v_a = mu * v_a + t
        w_a[root] = w_a[root] - v_a
    else:
        w_a[root] = w_a[root] - t
    oracle.broadcast(w_a, root=root)
    # (b) the oracle's Alg. 2 step
    oracle.bsp_sgd_alg2_step(g_b, w_b, v_b, root=root, lr=float(lr), mu=float(mu))
    for r in range(P):
        assert w_b[r].tobytes() == w_a[r].tobytes()
        assert g_b[r].tobytes() == g_a[r].tobytes()       # grads[root] = S, others untouched
    assert g_b[root].tobytes() == oracle.chain_sum(grads).tobytes()
    if with_momentum:
        assert v_b.tobytes() == v_a.tobytes()
    # (c) Alg. 3's fused step gives the same weights (the two differ in synchronisation points only)
    w_c, v_c = _copy(weights), (vel.copy() if with_momentum else None)
    if with_momentum:
        oracle.bsp_sgd_momentum_step(grads, w_c, v_c, root=root, lr=float(lr), mu=float(mu))
        assert v_c.tobytes() == v_b.tobytes()
    else:
        oracle.bsp_sgd_step(grads, w_c, root=root, lr=float(lr))
    assert all(a.tobytes() == b.tobytes() for a, b in zip(w_c, w_b))
