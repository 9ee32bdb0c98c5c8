"""A model of the chain's flow control (csrc/lp_chain.cu), run under RANDOM schedules on the CPU.

What the GPU tests cannot vary is the order in which the CTAs of different ranks make progress; on a real multi-GPU
machine every order is possible.  This model keeps exactly the state the kernels keep -- per rank and channel a forward
and a backward receive ring of S slots, the four counters (ring tails in the receiver's memory, credits in the sender's),
the private sequence numbers that are never reset -- and lets a random scheduler interleave the steps of all forward and
return CTAs of all ranks, over several collectives in a row with changing roots (a rank's CTAs of the next call may start
while a neighbour is still in the previous one, as on real hardware; calls of one rank run in order, as launches of one
stream do).  Checked on every step: a slot is only overwritten after its previous content was consumed, a slot that is read
holds the message with the expected sequence number; at the end: nobody is stuck (no deadlock), every rank holds the left
fold in rank order / the root's block (U4, U5), all counters of the two ends of a ring agree.
The roles come from the library (lp_chain_plan); the slot-reuse rule is the kernels' slot_free_at."""
import random

import pytest

from paper_1611_04255_b200 import binding as lp

OPS = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}


def slot_free_at(sent, S):
    """Credit the sender needs before send number sent + 1 may overwrite the slot of send sent + 1 - S (lp_chain.cu)."""
    return sent + 1 - S if sent + 1 > S else 0


class Endpoint:
    def __init__(self, S):
        self.S = S
        self.fwd_ring = [None] * S          # (sequence number, value, consumed)
        self.bwd_ring = [None] * S
        self.fwd_tail = self.bwd_tail = 0   # written by the senders (ranks r-1 / r+1), polled here
        self.up_credit = self.down_credit = 0   # written by the receivers of MY pushes (ranks r+1 / r-1), polled here
        self.recv_fwd = self.sent_up = self.recv_bwd = self.sent_down = 0   # private, never reset


def push(ring, S, seq, val):
    old = ring[(seq - 1) % S]
    assert old is None or old[2], f"slot overwritten before it was consumed (send {seq} over {old})"
    ring[(seq - 1) % S] = [seq, val, False]


def take(ring, S, seq):
    slot = ring[(seq - 1) % S]
    assert slot is not None and slot[0] == seq and not slot[2], f"expected message {seq}, found {slot}"
    slot[2] = True
    return slot[1]


def forward_cta(E, r, role, buf, out, tiles):
    """Generator: yields the condition it waits for (None = runnable); everything between two yields is one step."""
    me, up, down = E[r], E[role["up"]], E[role["down"]]
    for i in range(tiles):
        yield lambda: ((not role["f_recv"] or me.fwd_tail >= me.recv_fwd + 1)
                       and (not role["f_send_up"] or me.up_credit >= slot_free_at(me.sent_up, me.S))
                       and (not role["f_send_down"] or me.down_credit >= slot_free_at(me.sent_down, me.S)))
        v = buf[r][i] if role["f_load"] else None
        if role["f_recv"]:
            partial = take(me.fwd_ring, me.S, me.recv_fwd + 1)
            v = f"({partial}+{v})" if role["f_load"] else partial
        if role["f_send_up"]:
            push(up.fwd_ring, me.S, me.sent_up + 1, v)
        if role["f_store"]:
            out[r][i] = v
        if role["f_send_down"]:
            push(down.bwd_ring, me.S, me.sent_down + 1, v)
        yield None                                        # the data is on its way; the counters follow in a later step
        if role["f_send_up"]:
            me.sent_up += 1
            up.fwd_tail = me.sent_up
        if role["f_send_down"]:
            me.sent_down += 1
            down.bwd_tail = me.sent_down
        if role["f_recv"]:
            me.recv_fwd += 1
            down.up_credit = me.recv_fwd


def return_cta(E, r, role, out, tiles):
    me, up, down = E[r], E[role["up"]], E[role["down"]]
    for i in range(tiles):
        yield lambda: (me.bwd_tail >= me.recv_bwd + 1
                       and (not role["r_send_down"] or me.down_credit >= slot_free_at(me.sent_down, me.S)))
        v = take(me.bwd_ring, me.S, me.recv_bwd + 1)
        if role["r_store"]:
            out[r][i] = v
        if role["r_send_down"]:
            push(down.bwd_ring, me.S, me.sent_down + 1, v)
        yield None
        if role["r_send_down"]:
            me.sent_down += 1
            down.bwd_tail = me.sent_down
        me.recv_bwd += 1
        up.down_credit = me.recv_bwd


def expected(op, P, root, buf, tiles):
    want = [list(b) for b in buf]
    for i in range(tiles):
        fold = buf[0][i]
        for r in range(1, P):
            fold = f"({fold}+{buf[r][i]})"
        for r in range(P):
            if op == "allreduce" or (op == "reduce" and r == root):
                want[r][i] = fold
            elif op == "broadcast":
                want[r][i] = buf[root][i]
    return want


def run_sequence(P, S, calls, rng):
    """calls: list of (op, root, tiles).  One channel; every rank runs its calls in order, ranks run independently."""
    E = [Endpoint(S) for _ in range(P)]
    buf = [[f"x{r}.0.{i}" for i in range(8)] for r in range(P)]
    per_rank = [[] for _ in range(P)]           # rank -> list of (call index, [generators])
    wants = []
    for k, (op, root, tiles) in enumerate(calls):
        # every call works on fresh symbolic inputs so that a message of the wrong call cannot pass for the right one
        inputs = [[f"x{r}.{k}.{i}" for i in range(tiles)] for r in range(P)]
        out = [list(b) for b in inputs]
        wants.append((expected(op, P, root, inputs, tiles), out))
        for r in range(P):
            role = lp.lp_chain_plan(OPS[op], P, root, r)
            gens = []
            if role["f_active"]:
                gens.append(forward_cta(E, r, role, inputs, out, tiles))
            if role["r_active"]:
                gens.append(return_cta(E, r, role, out, tiles))
            per_rank[r].append(gens)
    # scheduler: a rank's CTAs of call k + 1 become runnable when all its CTAs of call k have finished (stream order)
    cur = [0] * P
    live = [[] for _ in range(P)]               # rank -> [generator, pending condition]
    for r in range(P):
        live[r] = [[g, next(g)] for g in per_rank[r][0]] if per_rank[r] else []
    steps = 0
    while True:
        for r in range(P):
            while not live[r] and cur[r] + 1 < len(calls):
                cur[r] += 1
                live[r] = [[g, c] for g in per_rank[r][cur[r]] for c in [next(g, "done")] if c != "done"]
        runnable = [(r, j) for r in range(P) for j, (g, c) in enumerate(live[r]) if c is None or c()]
        if not runnable:
            break
        r, j = rng.choice(runnable)
        g = live[r][j][0]
        try:
            live[r][j][1] = next(g)
        except StopIteration:
            live[r].pop(j)
        steps += 1
        assert steps < 200_000
    stuck = [(r, cur[r]) for r in range(P) if live[r] or cur[r] + 1 < len(calls)]
    assert not stuck, f"deadlock: ranks {stuck} never finished (P={P}, S={S}, calls={calls})"
    for k, (want, out) in enumerate(wants):
        assert out == want, (k, calls[k])
    for r in range(P):                          # both ends of every ring count the same sequence
        up = E[(r + 1) % P]
        assert E[r].sent_up == up.recv_fwd == up.fwd_tail == E[r].up_credit
        down = E[(r - 1) % P]
        assert E[r].sent_down == down.recv_bwd == down.bwd_tail == E[r].down_credit


@pytest.mark.parametrize("seed", range(12))
def test_chain_protocol_under_random_schedules(seed):
    rng = random.Random(1611_04255 + seed)
    for _ in range(25):
        P = rng.choice([2, 3, 4, 5, 6])
        S = rng.choice([1, 1, 2, 3])
        calls = [(rng.choice(["allreduce", "reduce", "broadcast"]), rng.randrange(P), rng.choice([1, 2, 3, 5, 7]))
                 for _ in range(rng.choice([1, 3, 5]))]
        run_sequence(P, S, calls, rng)


def test_model_catches_a_wrong_credit_rule(monkeypatch):
    """The model is only worth something if a plausible mistake fails it: reuse a slot one send too early."""
    import tests.test_chain_protocol_model as m
    monkeypatch.setattr(m, "slot_free_at", lambda sent, S: sent - S if sent > S else 0)
    caught = 0
    for seed in range(20):
        rng = random.Random(seed)
        try:
            run_sequence(3, 1, [("allreduce", 0, 5), ("broadcast", 1, 5)], rng)
        except AssertionError:
            caught += 1
    assert caught >= 15
