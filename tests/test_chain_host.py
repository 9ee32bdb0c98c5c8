"""Host logic of the multi-GPU chain (lp_chain_plan; csrc/lp_chain.cu), no GPU: what every rank does in a collective
must fit what its neighbours do.  A symbolic one-tile simulation of the message passing (queues for the rings, strings
for the values) checks that every push has its receiver, every rank ends with the right expression -- the LEFT FOLD in
rank order 0 -> P-1 whatever the root (Fig. 2b, U4) -- and that no message is left in a ring (the
sequence counters of both ends of a ring stay equal, which is what lets the counters grow for ever)."""
from collections import deque

import pytest

from paper_1611_04255_b200 import binding as lp

OPS = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}


def roles_of(op, P, root):
    return [lp.lp_chain_plan(OPS[op], P, root, r) for r in range(P)]


def simulate(op, P, root):
    """One tile through the chain.  Returns (final buffers, messages left in the rings, pushes per ring)."""
    roles = roles_of(op, P, root)
    buf = [f"x{r}" for r in range(P)]
    fwd = [deque() for _ in range(P)]   # rank r's forward receive ring
    bwd = [deque() for _ in range(P)]   # rank r's backward receive ring
    done_f = [not roles[r]["f_active"] for r in range(P)]
    done_r = [not roles[r]["r_active"] for r in range(P)]
    pushes = {"fwd": [0] * P, "bwd": [0] * P}
    for _ in range(4 * P + 4):
        progressed = False
        for r, ro in enumerate(roles):
            if not done_f[r] and (not ro["f_recv"] or fwd[r]):
                v = buf[r] if ro["f_load"] else None
                if ro["f_recv"]:
                    partial = fwd[r].popleft()
                    v = f"({partial}+{v})" if ro["f_load"] else partial   # partial op mine, in that order
                if ro["f_send_up"]:
                    fwd[ro["up"]].append(v)
                    pushes["fwd"][ro["up"]] += 1
                if ro["f_store"]:
                    buf[r] = v
                if ro["f_send_down"]:
                    bwd[ro["down"]].append(v)
                    pushes["bwd"][ro["down"]] += 1
                done_f[r] = progressed = True
            if not done_r[r] and bwd[r]:
                v = bwd[r].popleft()
                if ro["r_store"]:
                    buf[r] = v
                if ro["r_send_down"]:
                    bwd[ro["down"]].append(v)
                    pushes["bwd"][ro["down"]] += 1
                done_r[r] = progressed = True
        if not progressed:
            break
    assert all(done_f) and all(done_r), ("a CTA never got its message", op, P, root)
    left = sum(len(q) for q in fwd) + sum(len(q) for q in bwd)
    return buf, left, pushes


def left_fold(P):
    s = "x0"
    for r in range(1, P):
        s = f"({s}+x{r})"
    return s


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5, 6, 8, 16, 32])
def test_chain_roles_give_the_collectives(P):
    S = left_fold(P)
    buf, left, _ = simulate("allreduce", P, 0)
    assert buf == [S] * P and left == 0
    for root in range(P):
        buf, left, _ = simulate("reduce", P, root)
        assert buf == [S if r == root else f"x{r}" for r in range(P)] and left == 0      # U5: the others unchanged
        buf, left, _ = simulate("broadcast", P, root)
        assert buf == [f"x{root}"] * P and left == 0


@pytest.mark.parametrize("P", [2, 3, 6, 16])
def test_chain_ring_neighbours_never_change(P):
    """Rank r's forward ring is only ever written by rank r-1 (mod P), its backward ring by rank r+1 (mod P): that is
    what allows per-ring sequence numbers that are never reset."""
    for op in OPS:
        for root in range(P):
            for r, ro in enumerate(roles_of(op, P, root)):
                assert ro["up"] == (r + 1) % P and ro["down"] == (r - 1) % P
                up, down = roles_of(op, P, root)[ro["up"]], roles_of(op, P, root)[ro["down"]]
                assert bool(ro["f_send_up"]) == bool(up["f_recv"]), (op, root, r)
                assert bool(ro["f_recv"]) == bool(down["f_send_up"]), (op, root, r)
                assert bool(ro["r_active"]) == bool(up["f_send_down"] or up["r_send_down"]), (op, root, r)
                assert bool(ro["f_send_down"] or ro["r_send_down"]) == bool(down["r_active"]), (op, root, r)


def test_chain_sgd_step_roles():
    """The fused step is an allreduce whose end applies the update: same roles, plus f_update on the last rank only."""
    for P in (1, 2, 6, 16):
        for r in range(P):
            a = lp.lp_chain_plan(lp.OP_ALLREDUCE, P, 0, r)
            g = lp.lp_chain_plan(lp.OP_BSP_SGD, P, 0, r)
            assert lp.lp_chain_plan(lp.OP_BSP_SGD_MOM, P, 0, r) == g          # momentum: the same roles
            assert g["f_update"] == (1 if r == P - 1 else 0) and a["f_update"] == 0
            if P > 1:
                assert {k: v for k, v in g.items() if k != "f_update"} == {k: v for k, v in a.items() if k != "f_update"}
    one = lp.lp_chain_plan(lp.OP_BSP_SGD, 1, 0, 0)
    assert one["f_active"] and one["f_load"] and one["f_store"] and not one["f_send_up"] and not one["f_send_down"]


def test_chain_link_traffic_is_invariant_to_p():
    """PAPER.md:106 "the cost of Linear Pipeline is invariant to GPU count p": per tile every rank pushes at most one
    block up and one block down, whatever P -- the busiest link of an allreduce carries 1 block per tile and direction."""
    for P in (2, 3, 6, 16, 32):
        _, _, pushes = simulate("allreduce", P, 0)
        assert max(pushes["fwd"]) == 1 and max(pushes["bwd"]) == 1
        assert sum(pushes["fwd"]) == P - 1 and sum(pushes["bwd"]) == P - 1


def test_chain_plan_argument_errors():
    L = lp.lib()
    role = lp.ChainRole()
    ref = lp.ctypes.byref(role)
    assert L.lp_chain_plan(lp.OP_ALLREDUCE, 0, 0, 0, ref) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_plan(lp.OP_ALLREDUCE, 33, 0, 0, ref) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_plan(lp.OP_ALLREDUCE, 4, 0, 4, ref) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_plan(lp.OP_REDUCE, 4, 4, 0, ref) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_plan(5, 4, 0, 0, ref) == lp.LP_ERR_INVALID_ARG and L.lp_chain_plan(-1, 4, 0, 0, ref) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_plan(lp.OP_ALLREDUCE, 4, 99, 0, ref) == lp.LP_OK          # allreduce ignores the root
    assert L.lp_chain_endpoint_bytes(32, 8, 16384) == 32 * 64 * 8 + 32 * 4 * 8 + 256 + 2 * 32 * 8 * 16384 * 4 \
        or L.lp_chain_endpoint_bytes(32, 8, 16384) > 2 * 32 * 8 * 16384 * 4
    assert L.lp_chain_endpoint_bytes(0, 8, 16384) == 0 and L.lp_chain_endpoint_bytes(4, 8, 1000) == 0


def test_chain_auto_block_is_the_papers_optimum():
    """block = 0 over the chain: the power of two nearest to the minimiser of Table 1's LP allreduce cost for one channel's
    share of the message, with the constants fitted to the chain kernel."""
    import math
    alpha, beta = lp.lp_chain_fitted_constants()
    assert 1e-6 < alpha < 1e-5 and 1e-12 < beta < 1e-10
    tile = 262_144
    for P in (2, 4, 8, 16):
        last = 0
        for mb in (1, 4, 16, 64, 256, 1024):
            n = (mb << 20) // 4
            for C in (8, 16, 40):
                b = lp.lp_chain_auto_block(n, P, C, tile)
                assert 4096 <= b <= tile and b & (b - 1) == 0
                n_c = n * 4 / C
                opt = lp.lp_optimal_block(lp.OP_ALLREDUCE, P, n_c, alpha, beta)        # bytes
                # the minimiser is what Table 1's cost says it is: no other power of two in range is cheaper by > 1 %
                cost = lambda bb: lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, n_c, bb * 4, alpha, beta)
                best = min(cost(bb) for bb in (4096 << k for k in range(7)) if bb * 4 <= max(n_c, 4096 * 4))
                if b * 4 <= n_c:
                    assert cost(b) <= 1.06 * best, (P, mb, C, b, opt)
                assert 0.7 <= (b * 4) / min(max(opt, 4096 * 4), tile * 4) <= 1.42 or b in (4096, tile), (P, mb, C, b, opt)
            b16 = lp.lp_chain_auto_block(n, P, 16, tile)
            assert b16 >= last                     # longer messages never get smaller blocks
            last = b16
    # more ranks: a longer fill, so never a larger block
    assert lp.lp_chain_auto_block(1 << 26, 16, 16, tile) <= lp.lp_chain_auto_block(1 << 26, 2, 16, tile)
    assert lp.lp_chain_auto_block(1 << 20, 0, 16, tile) == 0 and lp.lp_chain_auto_block(1 << 20, 4, 16, 1000) == 0


def test_chain_create_needs_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CPU-box check")
    h = lp.ctypes.c_void_p()
    assert lp.lib().lp_chain_create(0, 2, 0, 0, 0, lp.ctypes.byref(h)) == lp.LP_ERR_CUDA
