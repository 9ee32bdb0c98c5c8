"""Pins for the operator-parameterised oracle functions (oracle/lpo_oracle.c section 5b): reduce / allreduce with
`sum` or `product` (Sec. 3 Reduce: "It supports basic arithmetic operations such as summations and
multiplications").  Every check ties the oracle to something other than itself: exact integer arithmetic in Python
ints, hand-computed overflow / underflow orderings that give a different value under every wrong fold order or tree,
numpy's own fp32 `*` as an independent left fold, an fp64 bound, and -- for red = sum -- the already pinned
functions of sections 1, 4, 5.  CPU only.
"""
import math

import numpy as np
import pytest

from paper_1611_04255_b200 import inputs

LP, MST, BE = 0, 1, 2
SUM, PROD = 0, 1
INF = float("inf")


def _copy(bufs):
    return [b.copy() for b in bufs]


def _algos(P):
    return [LP, MST] + ([BE] if P & (P - 1) == 0 else [])


@pytest.mark.parametrize("P", [1, 2, 3, 4, 6, 8])
@pytest.mark.parametrize("n", [1, 5, 9])
def test_product_brute_force_small_integers(oracle, P, n):
    # factors in {-2, -1, 1, 2}: every partial product is an integer of magnitude <= 2^P, exact in fp32, so chain,
    # MST and BE trees must all equal the product computed in Python ints
    rng = np.random.default_rng([31, P, n])
    bufs = [rng.choice(np.array([-2, -1, 1, 2], dtype=np.float32), size=n) for _ in range(P)]
    exact = [math.prod(int(bufs[r][i]) for r in range(P)) for i in range(n)]
    want = np.array(exact, dtype=np.float32)
    assert oracle.chain_fold(bufs, PROD).tolist() == want.tolist()
    for algo in _algos(P):
        for root in range(P):
            b = _copy(bufs)
            oracle.reduce_op(b, PROD, root=root, algo=algo)
            assert b[root].tolist() == want.tolist()
            for r in range(P):  # U5: the other vectors are untouched
                if r != root:
                    assert b[r].tobytes() == bufs[r].tobytes()
        b = _copy(bufs)
        oracle.allreduce_op(b, PROD, algo=algo)
        assert all(x.tolist() == want.tolist() for x in b)


def test_product_chain_order_separator(oracle):
    # fp32 multiplication is not associative across overflow / underflow.  Worked by hand (fp32 max 3.4e38, smallest
    # denormal 1.4e-45):
    #   ranks [1e30, 1e30, 1e-30]: (1e30 * 1e30) = inf, inf * 1e-30 = inf;  1e30 * (1e30 * 1e-30) would be ~1e30
    #   ranks [1e30, 1e-30, 1e30]: (1e30 * 1e-30) ~ 1, * 1e30 ~ 1e30
    #   ranks [1e-30, 1e-30, 1e30]: (1e-30 * 1e-30) = 0 (underflow), 0 * 1e30 = 0;  right-to-left would give ~1e-30
    f = np.float32
    col = lambda *v: [np.array([x], dtype=f) for x in v]  # noqa: E731
    assert oracle.chain_fold(col(1e30, 1e30, 1e-30), PROD)[0] == INF
    got = oracle.chain_fold(col(1e30, 1e-30, 1e30), PROD)[0]
    assert abs(got / f(1e30) - 1) < 1e-6
    assert oracle.chain_fold(col(1e-30, 1e-30, 1e30), PROD)[0] == 0.0
    # and the sum separator of the sum pins still holds through the operator entry point
    assert oracle.chain_fold(col(1e8, -1e8, 1), SUM)[0] == 1.0
    assert oracle.chain_fold(col(1, 1e8, -1e8), SUM)[0] == 0.0


def test_product_tree_separator_chain_mst_be(oracle):
    # x = [1e30, 1e30, 1e-30, 1e-30]:
    #   chain ((x0 x1) x2) x3 = (inf * 1e-30) * 1e-30 = inf
    #   MST   (x0 x1)(x2 x3) = inf * 0 = NaN          (1e-60 underflows to 0)
    #   BE    (x0 x2)(x1 x3) ~ 1 * 1 ~ 1
    x = [np.array([v], dtype=np.float32) for v in (1e30, 1e30, 1e-30, 1e-30)]
    b = _copy(x)
    oracle.allreduce_op(b, PROD, algo=LP)
    assert all(v[0] == INF for v in b)
    b = _copy(x)
    oracle.allreduce_op(b, PROD, algo=MST)
    assert all(math.isnan(v[0]) for v in b)
    b = _copy(x)
    oracle.allreduce_op(b, PROD, algo=BE)
    assert all(abs(v[0] - 1.0) < 1e-6 for v in b)
    for algo, check in ((LP, lambda v: v == INF), (MST, math.isnan), (BE, lambda v: abs(v - 1.0) < 1e-6)):
        for root in range(4):  # the LP fold and the BE butterfly do not depend on the root; MST's tree is rotated with it
            b = _copy(x)
            oracle.reduce_op(b, PROD, root=root, algo=algo)
            if algo == MST and root != 0:
                continue
            assert check(b[root][0]), (algo, root, b[root][0])


@pytest.mark.parametrize("P", [2, 3, 6, 8, 16])
def test_product_equals_numpy_left_fold_and_fp64_bound(oracle, P):
    # independent left fold: numpy's own float32 multiply, one rounding per step
    n = 4099
    rng = np.random.default_rng([32, P])
    bufs = [(rng.random(n, dtype=np.float32) + np.float32(0.5)) * rng.choice(np.array([-1, 1], dtype=np.float32), n)
            for _ in range(P)]  # |x| in [0.5, 1.5): no overflow / underflow within 16 factors
    want = bufs[0].copy()
    for r in range(1, P):
        want = (want * bufs[r]).astype(np.float32)
    got = oracle.chain_fold(bufs, PROD)
    assert got.tobytes() == want.tobytes()
    # exact product in fp64 (53 bits hold 16 factors' worth of rounding slack): each of the P-1 multiplications
    # contributes a relative error <= 2^-24, so |got - exact| <= ((1 + u)^(P-1) - 1) |exact| (+ fp64 noise)
    exact = np.ones(n, dtype=np.float64)
    for r in range(P):
        exact *= bufs[r].astype(np.float64)
    u = 2.0 ** -24
    bound = ((1 + u) ** (P - 1) - 1) * np.abs(exact) * (1 + 1e-9)
    assert np.all(np.abs(got.astype(np.float64) - exact) <= bound)
    for algo in _algos(P):  # the reordered trees obey the same bound (they do P-1 multiplications too)
        b = _copy(bufs)
        oracle.allreduce_op(b, PROD, algo=algo)
        assert all(x.tobytes() == b[0].tobytes() for x in b)
        assert np.all(np.abs(b[0].astype(np.float64) - exact) <= bound)
        if algo == LP:
            assert b[0].tobytes() == want.tobytes()


@pytest.mark.parametrize("algo", [LP, MST, BE])
@pytest.mark.parametrize("P", [1, 2, 4, 5, 8])
def test_sum_operator_is_the_pinned_sum(oracle, algo, P):
    # red = sum must be the functions of sections 1, 4, 5 (pinned in test_oracle_pins.py), bit for bit
    if algo == BE and P & (P - 1):
        return
    n = 1001
    src = inputs.rank_vectors(33, P, n)
    for root in range(P):
        a, b = _copy(src), _copy(src)
        oracle.reduce(a, root=root, algo=algo)
        oracle.reduce_op(b, SUM, root=root, algo=algo)
        assert all(x.tobytes() == y.tobytes() for x, y in zip(a, b))
    a, b = _copy(src), _copy(src)
    oracle.allreduce(a, algo=algo)
    oracle.allreduce_op(b, SUM, algo=algo)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(a, b))
    if algo == LP:
        assert oracle.chain_fold(src, SUM).tobytes() == oracle.chain_sum(src).tobytes()


@pytest.mark.parametrize("red", [SUM, PROD])
def test_operator_special_cases(oracle, red):
    n = 257
    rng = np.random.default_rng([34, red])
    x = (rng.random(n, dtype=np.float32) + np.float32(0.25))
    ident = np.float32(0.0 if red == SUM else 1.0)
    # P = 1: identity
    b = [x.copy()]
    oracle.allreduce_op(b, red)
    assert b[0].tobytes() == x.tobytes()
    # P = 2: one operation -- chain, MST and BE coincide and equal numpy's
    y = (rng.random(n, dtype=np.float32) + np.float32(0.25))
    want = (x + y if red == SUM else x * y).astype(np.float32)
    for algo in (LP, MST, BE):
        b = [x.copy(), y.copy()]
        oracle.allreduce_op(b, red, algo=algo)
        assert b[0].tobytes() == want.tobytes() and b[1].tobytes() == want.tobytes()
    # one-hot: every rank but one holds the operator's identity -> the result is that rank's vector, exactly
    for P in (3, 4, 8):
        for hot in range(P):
            for algo in _algos(P):
                b = [np.full(n, ident, dtype=np.float32) for _ in range(P)]
                b[hot] = x.copy()
                oracle.allreduce_op(b, red, algo=algo)
                assert all(v.tobytes() == x.tobytes() for v in b)
    # an absorbing zero for the product: one rank all zeros -> all zeros (finite inputs)
    if red == PROD:
        b = [x.copy(), np.zeros(n, dtype=np.float32), y.copy()]
        oracle.allreduce_op(b, red)
        assert all(not v.any() for v in b)


@pytest.mark.parametrize("red", [SUM, PROD])
def test_operator_root_invariance_and_allreduce_is_broadcast_of_reduce(oracle, red):
    # U4: the LP fold is rank 0 -> P-1 whatever the root; allreduce == reduce followed by broadcast
    P, n = 6, 515
    rng = np.random.default_rng([35, red])
    src = [(rng.random(n, dtype=np.float32) + np.float32(0.5)) for _ in range(P)]
    fold = oracle.chain_fold(src, red)
    for root in range(P):
        b = _copy(src)
        oracle.reduce_op(b, red, root=root)
        assert b[root].tobytes() == fold.tobytes()
        oracle.broadcast(b, root=root)
        assert all(v.tobytes() == fold.tobytes() for v in b)
    b = _copy(src)
    oracle.allreduce_op(b, red)
    assert all(v.tobytes() == fold.tobytes() for v in b)


@pytest.mark.parametrize("red", [SUM, PROD])
@pytest.mark.parametrize("op", [1, 2])
def test_segments_with_operator(oracle, red, op):
    # Alg. 1 slices: each slice is the whole-message definition on that slice; everything else untouched
    P, n = 4, 1000
    rng = np.random.default_rng([36, red, op])
    src = [(rng.random(n, dtype=np.float32) + np.float32(0.5)) for _ in range(P)]
    segs = [(3, 100), (500, 1), (200, 77), (999, 1), (600, 0)]
    got = _copy(src)
    oracle.collective_segments_op(op, red, got, segs, root=2)
    want = _copy(src)
    for off, ln in segs:
        sl = [w[off:off + ln].copy() for w in want]
        if op == 1:
            oracle.reduce_op(sl, red, root=2)
        else:
            oracle.allreduce_op(sl, red)
        for w, s in zip(want, sl):
            w[off:off + ln] = s
    assert all(g.tobytes() == w.tobytes() for g, w in zip(got, want))
    # brute force on the union in exact arithmetic for small integers
    ints = [rng.choice(np.array([-2, -1, 1, 2], dtype=np.float32), size=n) for _ in range(P)]
    got = _copy(ints)
    oracle.collective_segments_op(2, red, got, segs)
    for off, ln in segs:
        for i in range(off, off + ln):
            vals = [int(ints[r][i]) for r in range(P)]
            exact = sum(vals) if red == SUM else math.prod(vals)
            assert all(g[i] == exact for g in got)


def test_operator_bad_arguments(oracle):
    b = [np.ones(4, dtype=np.float32) for _ in range(2)]
    with pytest.raises(RuntimeError):
        oracle.allreduce_op(b, 2)
    with pytest.raises(RuntimeError):
        oracle.reduce_op(b, -1)
    with pytest.raises(RuntimeError):
        oracle.allreduce_op([np.ones(4, dtype=np.float32) for _ in range(3)], PROD, algo=BE)  # U14
