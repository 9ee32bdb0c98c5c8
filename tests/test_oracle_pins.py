"""Pins for the CPU oracle (oracle/lpo_oracle.c): each check ties an oracle
function to something OTHER than the oracle -- values the paper prints
(tests/golden/), closed forms, brute force in exact integer arithmetic,
constructed non-associative inputs whose result under each summation tree is
known by hand, and an fp64 error bound.  CPU only.

Citations are PAPER.md:<line>; U<k> are the readings listed in DESIGN.md.
"""
import itertools
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
# values: broadcast / reduce / allreduce definitions
# ----------------------------------------------------------------------------

@pytest.mark.parametrize("algo", [LP, MST, BE])
@pytest.mark.parametrize("P,root", [(1, 0), (2, 1), (4, 0), (4, 3), (8, 5)])
def test_broadcast_is_identity_of_root(oracle, algo, P, root):
    # PAPER.md:57 "It copies the source vector to every GPUs."
    n = 37
    bufs = inputs.rank_vectors(11, P, n)
    want = bufs[root].copy()
    oracle.broadcast(bufs, root=root, algo=algo)
    for r in range(P):
        assert bufs[r].tobytes() == want.tobytes()


@pytest.mark.parametrize("P", [3, 5, 6])
def test_mst_broadcast_non_pow2(oracle, P):
    for root in range(P):
        bufs = inputs.rank_vectors(12, P, 9)
        want = bufs[root].copy()
        oracle.broadcast(bufs, root=root, algo=MST)
        assert all(b.tobytes() == want.tobytes() for b in bufs)


@pytest.mark.parametrize("P", [1, 2, 3, 4])
@pytest.mark.parametrize("n", [1, 5, 8])
def test_sum_brute_force_small_integers(oracle, P, n):
    # Small integers: every association order is exact, so chain / MST / BE
    # must all equal the integer sum computed in Python ints.
    bufs = [inputs.small_integers(21, r, n) for r in range(P)]
    exact = [sum(int(bufs[r][i]) for r in range(P)) for i in range(n)]
    want = np.array(exact, dtype=np.float32)
    assert oracle.chain_sum(bufs).tolist() == want.tolist()
    algos = [LP, MST] + ([BE] if P & (P - 1) == 0 else [])
    for algo in algos:
        b = _copy(bufs)
        oracle.allreduce(b, algo=algo)
        for r in range(P):
            assert b[r].tolist() == want.tolist(), (algo, r)
        for root in range(P):
            b = _copy(bufs)
            oracle.reduce(b, root=root, algo=algo)
            assert b[root].tolist() == want.tolist()
            for r in range(P):
                if r != root:  # U5: non-root vectors unchanged
                    assert b[r].tobytes() == bufs[r].tobytes()


def test_chain_order_pinned_by_non_associative_triple(oracle):
    # fp32: (1e8 + -1e8) + 1 = 1 but (1 + 1e8) + -1e8 = 0 (1 is below half an
    # ulp of 1e8 = 8).  A fold that starts anywhere but rank 0, or runs
    # backwards, gives a different element somewhere below.
    vals = [1e8, -1e8, 1.0]
    hand = {(0, 1, 2): 1.0, (0, 2, 1): 0.0, (1, 0, 2): 1.0, (1, 2, 0): 0.0,
            (2, 0, 1): 0.0, (2, 1, 0): 0.0}
    for perm, want in hand.items():
        bufs = [np.array([vals[p]], dtype=np.float32) for p in perm]
        assert oracle.chain_sum(bufs)[0] == np.float32(want), perm
        b = _copy(bufs)
        oracle.allreduce(b)
        assert all(x[0] == np.float32(want) for x in b)


def test_trees_distinguished_at_P4(oracle):
    # x = [1e8, 1, -1e8, 1]
    # chain ((x0+x1)+x2)+x3 = ((1e8)+-1e8)+1 = 1
    # MST   (x0+x1)+(x2+x3) = 1e8 + -1e8     = 0          PAPER.md:93 (U: binomial)
    # BE    (x0+x2)+(x1+x3) = 0 + 2          = 2          PAPER.md:95 (halving)
    x = [1e8, 1.0, -1e8, 1.0]
    n = 16  # BE: every element, whichever rank owns its segment, has the same tree
    bufs = [np.full(n, v, dtype=np.float32) for v in x]
    for algo, want in ((LP, 1.0), (MST, 0.0), (BE, 2.0)):
        b = _copy(bufs)
        oracle.allreduce(b, algo=algo)
        for r in range(4):
            assert b[r].tolist() == [want] * n, (algo, r)
        b = _copy(bufs)
        oracle.reduce(b, root=0, algo=algo)
        assert b[0].tolist() == [want] * n


def test_trees_distinguished_at_P8(oracle):
    # fp32 near 1e8 has a spacing of 8 (1e8 = 12,500,000 * 8, an even multiple: ties go to it), so |s| <= 4 vanishes in
    # 1e8 + s and the three association trees of eight ranks give three different sums.  Worked by hand:
    #   chain  ((((((x0+x1)+x2)+x3)+x4)+x5)+x6)+x7
    #   MST    ((x0+x1)+(x2+x3)) + ((x4+x5)+(x6+x7))
    #   BE     ((x0+x4)+(x2+x6)) + ((x1+x5)+(x3+x7))    halving: distance 4, then 2, then 1
    # A = [4, 3, -1e8, 5, 1, 5, 1e8, 2]
    #   chain: 7; 7-1e8 = -99999993 -> -99999992; +5 = -99999987 -> -99999984; +1 -> -99999984; +5 = -99999979 ->
    #          -99999976; +1e8 = 24; +2 = 26
    #   MST:   (7 + (-1e8+5 -> -99999992)) = -99999985 -> -99999984;  (6 + (1e8+2 -> 1e8)) = 100000006 -> 100000008;  24
    #   BE:    ((4+1) + (-1e8+1e8)) = 5;  ((3+5) + (5+2)) = 15;  20
    #   (a halving that takes distance 2 before distance 4 would give ((4-1e8 -> -1e8) + (1+1e8 -> 1e8)) + (8+7) = 15)
    # B = [1, 1, 3, 2, -1e8, 1e8, 4, 1]
    #   chain: 2; 5; 7; 7-1e8 -> -99999992; +1e8 = 8; +4 = 12; +1 = 13
    #   MST:   (2+5) + ((-1e8+1e8) + (4+1)) = 7 + 5 = 12
    #   BE:    ((1-1e8 -> -1e8) + (3+4)) = -99999993 -> -99999992;  ((1+1e8 -> 1e8) + (2+1)) = 1e8;  8
    #   (a halving that takes distance 1 before distance 2 would give (-1e8+1e8) + (7+3) = 10)
    n = 24  # BE: every element has the same tree whichever rank ends up owning its segment
    for x, chain, mst, be in (([4.0, 3.0, -1e8, 5.0, 1.0, 5.0, 1e8, 2.0], 26.0, 24.0, 20.0),
                              ([1.0, 1.0, 3.0, 2.0, -1e8, 1e8, 4.0, 1.0], 13.0, 12.0, 8.0)):
        bufs = [np.full(n, v, dtype=np.float32) for v in x]
        for algo, want in ((LP, chain), (MST, mst), (BE, be)):
            b = _copy(bufs)
            oracle.allreduce(b, algo=algo)
            for r in range(8):
                assert b[r].tolist() == [want] * n, (algo, r)
            b = _copy(bufs)
            oracle.reduce(b, root=0, algo=algo)
            assert b[0].tolist() == [want] * n, algo
        b = _copy(bufs)                       # BE's tree does not move with the root (only the gather does)
        oracle.reduce(b, root=5, algo=BE)
        assert b[5].tolist() == [be] * n


def test_mst_tree_rotates_with_root(oracle):
    # virtual rank v = (r - root) mod P: with root=1 the tree is
    # (x1+x2)+(x3+x0).  x = [1, 1e8, 1, -1e8]: (1e8+1)+(-1e8+1) = 0;
    # root=0 tree (x0+x1)+(x2+x3) = 1e8 + -1e8 = 0 too, so use x=[1e8,-1e8,1,1]:
    # root 0: (1e8-1e8)+(1+1) = 2 ; root 1: (-1e8+1)+(1+1e8) = 0.
    x = [1e8, -1e8, 1.0, 1.0]
    for root, want in ((0, 2.0), (1, 0.0)):
        b = [np.array([v], dtype=np.float32) for v in x]
        oracle.reduce(b, root=root, algo=MST)
        assert b[root][0] == np.float32(want)


def test_special_cases(oracle):
    n = 33
    # P = 1: identity
    b = inputs.rank_vectors(31, 1, n)
    w = b[0].copy()
    oracle.allreduce(b)
    assert b[0].tobytes() == w.tobytes()
    # P = 2: one add -- chain, MST and BE coincide bit for bit and equal numpy's
    # single fp32 add
    src = inputs.rank_vectors(32, 2, n)
    want = src[0] + src[1]
    for algo in (LP, MST, BE):
        b = _copy(src)
        oracle.allreduce(b, algo=algo)
        assert b[0].tobytes() == want.tobytes() and b[1].tobytes() == want.tobytes()
    # all zeros; one-hot rank (the sum is that rank's vector: x + 0 is exact)
    for P in (3, 4, 8):
        z = [np.zeros(n, np.float32) for _ in range(P)]
        oracle.allreduce(z)
        assert not any(x.any() for x in z)
        for hot in range(P):
            v = inputs.uniform(33, hot, n)
            for algo in (LP, MST) + ((BE,) if P & (P - 1) == 0 else ()):
                b = [v.copy() if r == hot else np.zeros(n, np.float32) for r in range(P)]
                oracle.allreduce(b, algo=algo)
                assert all(x.tobytes() == v.tobytes() for x in b)


@pytest.mark.parametrize("P", [2, 4, 6, 8, 16])
def test_fp64_bound(oracle, P):
    # |fl-chain-sum - exact| <= (P-1) u sum|x| (1+O(u)), u = 2^-24 (first-order
    # bound of recursive summation); the same bound holds for any tree.  U15.
    n = 4099
    bufs = inputs.rank_vectors(41, P, n)
    x64 = np.stack([b.astype(np.float64) for b in bufs])
    exact = x64.sum(axis=0)
    bound = (P - 1) * 2.0 ** -24 * np.abs(x64).sum(axis=0) * 1.0001 + 1e-45
    got = oracle.chain_sum(bufs).astype(np.float64)
    assert np.all(np.abs(got - exact) <= bound)
    for algo in (MST,) + ((BE,) if P & (P - 1) == 0 else ()):
        b = _copy(bufs)
        oracle.allreduce(b, algo=algo)
        assert np.all(np.abs(b[0].astype(np.float64) - exact) <= bound)
        # north_star: reordered variants within 1e-6 (relative to sum|x|, U15)
        assert np.all(np.abs(b[0].astype(np.float64) - got) <= 1e-6 * np.abs(x64).sum(axis=0))


@pytest.mark.parametrize("P", [2, 3, 4, 6, 8])
def test_chain_sum_matches_numpy_left_fold(oracle, P):
    # numpy float32 '+' is one IEEE RN add per element: an independent
    # evaluation of S = ((x0+x1)+x2)+... in rank order.
    bufs = inputs.rank_vectors(42, P, 1000)
    s = bufs[0].copy()
    for r in range(1, P):
        s = s + bufs[r]
    assert oracle.chain_sum(bufs).tobytes() == s.tobytes()


def test_root_invariance_and_allreduce_equals_reduce_then_broadcast(oracle):
    # U4: sum order is rank 0 -> P-1 for every root; "equivalent to
    # a reduce followed by a broadcast".
    P, n = 5, 257
    src = inputs.rank_vectors(43, P, n)
    ar = _copy(src)
    oracle.allreduce(ar)
    assert all(a.tobytes() == ar[0].tobytes() for a in ar)
    for root in range(P):
        b = _copy(src)
        oracle.reduce(b, root=root)
        assert b[root].tobytes() == ar[0].tobytes()
        oracle.broadcast(b, root=root)
        assert all(x.tobytes() == ar[0].tobytes() for x in b)


def test_omp_versions_bit_identical(oracle):
    P, n = 6, 100_003
    src = inputs.rank_vectors(44, P, n, "normal", 1e-3)
    a, b = _copy(src), _copy(src)
    oracle.allreduce(a)
    oracle.allreduce(b, omp=True)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(a, b))
    g, w = inputs.sgd_inputs(45, P, n)
    w2 = _copy(w)
    oracle.bsp_sgd_step(g, w, root=2, lr=0.01)
    oracle.bsp_sgd_step(g, w2, root=2, lr=0.01, omp=True)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(w, w2))


# ----------------------------------------------------------------------------
# layer-wise collectives (Alg. 1): one collective per slice
# ----------------------------------------------------------------------------

@pytest.mark.parametrize("op", [BCAST, REDUCE, ALLREDUCE])
def test_segments_equal_whole_message_on_their_union(oracle, op):
    # element-wise ops: a collective per slice touches exactly the slices' elements and gives them the values
    # the whole-message collective gives; everything else keeps its bytes.  Slices unordered, ragged, some empty.
    P, n, root = 5, 10_007, 3
    segs = [(9000, 1007), (0, 1), (5, 3), (100, 0), (4096, 2048), (1001, 999), (8999, 1)]
    src = inputs.rank_vectors(81, P, n, "uniform")
    whole = _copy(src)
    {BCAST: oracle.broadcast, REDUCE: oracle.reduce}.get(op, None)(whole, root=root) if op != ALLREDUCE \
        else oracle.allreduce(whole)
    got = _copy(src)
    oracle.collective_segments(op, got, segs, root=root)
    mask = np.zeros(n, bool)
    for o, l in segs:
        mask[o:o + l] = True
    for r in range(P):
        assert got[r][mask].tobytes() == whole[r][mask].tobytes()
        assert got[r][~mask].tobytes() == src[r][~mask].tobytes()


def test_segments_brute_force_small_integers(oracle):
    P, n = 4, 64
    src = [inputs.small_integers(82, r, n) for r in range(P)]
    segs = [(60, 4), (0, 7), (31, 2)]
    got = _copy(src)
    oracle.collective_segments(ALLREDUCE, got, segs)
    total = np.sum(np.stack(src).astype(np.int64), axis=0)
    for r in range(P):
        for i in range(n):
            inside = any(o <= i < o + l for o, l in segs)
            assert got[r][i] == (total[i] if inside else src[r][i])
    with pytest.raises(RuntimeError):
        oracle.collective_segments(ALLREDUCE, got, [(60, 5)])      # runs past n


def test_sgd_segments_equal_whole_step_on_their_union(oracle):
    # the update is element-wise: per-slice steps give the whole-vector step's weights inside the slices and leave
    # every other weight (and every gradient) alone; written against the numpy composition, not the oracle's own step
    P, n, root, lr = 4, 5003, 2, np.float32(0.05)
    segs = [(4000, 1003), (0, 2), (17, 900), (2000, 0)]
    grads, weights = inputs.sgd_inputs(83, P, n)
    for r in range(P):
        weights[r] = weights[r] + np.float32(r)
    S = grads[0].copy()
    for r in range(1, P):
        S = S + grads[r]
    w_new = weights[root] - lr * (S * (np.float32(1.0) / np.float32(P)))
    g0, w0 = _copy(grads), _copy(weights)
    oracle.bsp_sgd_step_segments(grads, weights, segs, root=root, lr=float(lr))
    mask = np.zeros(n, bool)
    for o, l in segs:
        mask[o:o + l] = True
    for r in range(P):
        assert weights[r][mask].tobytes() == w_new[mask].tobytes()
        assert weights[r][~mask].tobytes() == w0[r][~mask].tobytes()
        assert grads[r].tobytes() == g0[r].tobytes()
