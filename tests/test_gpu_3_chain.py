"""GPU parity of the multi-GPU chain's device code (csrc/lp_chain.cu) against the oracle.  The box
has one GPU and kernels that wait on each other may not run there as separate launches, so the P ranks run as ONE
cooperative launch (lp_chain_emulate: the same per-rank code, P endpoints in one device's memory).  Bit-exact: the
chain folds in rank order 0 -> P-1 whatever the root (U4), one RN operation per combine.  Every test is marked gpu.
"""
import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from paper_1611_04255_b200 import binding as lp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

OPS = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}


@pytest.fixture(autouse=True, params=[lp.CHAIN_KERNEL_TMA, lp.CHAIN_KERNEL_REGISTER], ids=["tma", "register"])
def _device(request):
    """Every test runs with both realisations of a rank's CTAs (the protocol between ranks is the same)."""
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    lp.lib()
    lp.lp_chain_set_kernel(request.param)
    yield
    torch.cuda.synchronize()
    lp.lp_chain_set_kernel(lp.CHAIN_KERNEL_DEFAULT)


def up(arrs):
    return [torch.from_numpy(a).cuda() for a in arrs]


def down(tensors):
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in tensors]


def run_oracle(oracle, op, host, root, red):
    if op == "allreduce":
        oracle.allreduce_op(host, red)
    elif op == "reduce":
        oracle.reduce_op(host, red, root=root)
    else:
        oracle.broadcast(host, root=root)


def check(oracle, P, n, block, op, root=0, red=lp.REDUCE_SUM, kind="uniform", **geom):
    src = inputs.rank_vectors([31, n, P], P, n, kind)
    want = [a.copy() for a in src]
    run_oracle(oracle, op, want, root, red)
    dev = up(src)
    lp.lp_chain_emulate(OPS[op], dev, block=block, root=root, reduce_op=red, **geom)
    got = down(dev)
    assert lp.lp_chain_emulate_error(P, **geom) == 0, "a wait of the chain gave up"
    for r in range(P):
        assert got[r].tobytes() == want[r].tobytes(), (op, P, n, block, root, red, geom, r)


SHAPES = [
    # P, n, block
    (1, 1000, 64), (2, 1, 1), (2, 3, 64), (2, 5, 4), (3, 1001, 100), (3, 4097, 1000), (4, 70_001, 4096),
    (5, 300_003, 65_536), (6, 70_001, 1001), (7, 12_345, 333), (8, 262_147, 16_384), (16, 100_003, 8192),
    (32, 20_001, 5000), (4, 16384 * 3 + 5, 16384), (6, 1 << 20, 1 << 22),
]


@pytest.mark.parametrize("op", ["allreduce", "reduce", "broadcast"])
@pytest.mark.parametrize("P,n,block", SHAPES)
def test_chain_ragged_shapes_bit_exact(oracle, op, P, n, block):
    check(oracle, P, n, block, op, root=P // 2)


@pytest.mark.parametrize("op", ["reduce", "broadcast"])
def test_chain_every_root(oracle, op):
    for P in (2, 3, 5):
        for root in range(P):
            check(oracle, P, 50_001, 4096, op, root=root)


@pytest.mark.parametrize("tile", [4096, 16384, 65536, 262144])
@pytest.mark.parametrize("slots", [1, 2, 8])
def test_chain_ring_geometry_and_back_pressure(oracle, tile, slots):
    """Few channels and shallow rings: every slot is reused hundreds of times, so credits and sequence numbers wrap
    the ring over and over (a one-slot ring is pure stop-and-wait)."""
    for op in ("allreduce", "reduce", "broadcast"):
        check(oracle, 6, 1_500_003, 65_536, op, root=2, channels=2, slots=slots, tile=tile)


def test_chain_product(oracle):
    src = inputs.typed_rank_vectors([32, 0], 6, 200_001, inputs.DT_F32, "prod")
    want = [a.copy() for a in src]
    oracle.allreduce_op(want, oracle.RED_PROD)
    dev = up(src)
    lp.lp_chain_emulate(lp.OP_ALLREDUCE, dev, block=8192, reduce_op=lp.REDUCE_PROD)
    got = down(dev)
    assert all(g.tobytes() == w.tobytes() for g, w in zip(got, want))


def test_chain_back_to_back_collectives_share_the_rings(oracle):
    """Counters only grow: a sequence of different collectives (different roots, so different senders into the same
    rings) on one stream, no reset in between."""
    P, n = 4, 300_007
    src = inputs.rank_vectors([33, 0], P, n, "uniform")
    host = [a.copy() for a in src]
    dev = up(src)
    seq = [("allreduce", 0), ("broadcast", 2), ("reduce", 1), ("broadcast", 0), ("allreduce", 0), ("reduce", 3),
           ("broadcast", 3), ("reduce", 0)] * 3
    for op, root in seq:
        run_oracle(oracle, op, host, root, oracle.RED_SUM)
        lp.lp_chain_emulate(OPS[op], dev, block=16_384, root=root)
    got = down(dev)
    assert lp.lp_chain_emulate_error(P) == 0
    for r in range(P):
        assert got[r].tobytes() == host[r].tobytes(), r


def test_chain_large_message(oracle):
    P, n = 4, (64 << 20) // 4 + 3          # 64 MB per rank: ~1000 tiles per rank, 8 channels
    src = inputs.rank_vectors([34, 0], P, n, "normal", 1e-3)
    want = [a.copy() for a in src]
    oracle.allreduce(want, omp=True)
    dev = up(src)
    lp.lp_chain_emulate(lp.OP_ALLREDUCE, dev, block=65_536)
    got = down(dev)
    assert lp.lp_chain_emulate_error(P) == 0
    for r in range(P):
        assert got[r].tobytes() == want[r].tobytes(), r


@pytest.mark.parametrize("P,n,block", [(1, 5_001, 1024), (2, 70_001, 4096), (6, 300_003, 65_536), (8, 1_000_003, 65_536),
                                       (16, 100_003, 8192)])
def test_chain_fused_bsp_sgd_step(oracle, P, n, block):
    """Alg. 3 over the chain: the chain's end applies the update from its own replica and the new
    weights travel back down -- the oracle's fused step with root = P - 1, three RN operations, bit for bit; the
    gradients are only read.  Replicas are made DIFFERENT on purpose so that reading any other one would show."""
    grads, weights = inputs.sgd_inputs([35, n], P, n)
    weights = [w + np.float32(r) for r, w in enumerate(weights)]
    hw = [w.copy() for w in weights]
    oracle.bsp_sgd_step(grads, hw, root=P - 1, lr=0.01)
    dg, dw = up(grads), up(weights)
    for it in range(3):                       # three steps back to back over the same rings
        lp.lp_chain_emulate_bsp_sgd_step(dg, dw, block=block, lr=0.01)
        if it < 2:
            oracle.bsp_sgd_step(grads, hw, root=P - 1, lr=0.01)
    got_w, got_g = down(dw), down(dg)
    assert lp.lp_chain_emulate_error(P) == 0
    for r in range(P):
        assert got_w[r].tobytes() == hw[r].tobytes(), ("weights", r)
        assert got_g[r].tobytes() == grads[r].tobytes(), ("grads must be untouched", r)


@pytest.mark.parametrize("P,n,block", [(1, 5_001, 1024), (3, 70_001, 4096), (6, 300_003, 65_536), (16, 100_003, 0)])
def test_chain_fused_bsp_sgd_momentum_step(oracle, P, n, block):
    """The paper's solver (U18) over the chain: five RN operations at the chain's end, the velocity lives
    there; four steps back to back (the velocity feeds back), against the oracle's momentum step with root = P - 1."""
    grads, weights = inputs.sgd_inputs([39, n], P, n)
    weights = [w + np.float32(r) for r, w in enumerate(weights)]
    hw = [w.copy() for w in weights]
    hv = np.zeros(n, dtype=np.float32)
    dg, dw = up(grads), up(weights)
    dv = torch.zeros(n, device="cuda")
    for _ in range(4):
        oracle.bsp_sgd_momentum_step(grads, hw, hv, root=P - 1, lr=0.01, mu=0.9)
        lp.lp_chain_emulate_bsp_sgd_momentum_step(dg, dw, dv, block=block, lr=0.01, mu=0.9)
    got_w = down(dw)
    assert lp.lp_chain_emulate_error(P) == 0
    assert dv.cpu().numpy().tobytes() == hv.tobytes(), "velocity"
    for r in range(P):
        assert got_w[r].tobytes() == hw[r].tobytes(), ("weights", r)


@pytest.mark.parametrize("root", [0, 2, 4])
def test_chain_alg2_step(oracle, root):
    """Alg. 2 over the chain (reduce to root, root update, broadcast): the oracle's Alg. 2 step, bit for bit -- the
    reduced gradient lands in the root's gradient vector (U20), weights and velocity equal the fused step's."""
    P, n = 5, 200_003
    grads, weights = inputs.sgd_inputs([40, root], P, n)
    hg, hw = [g.copy() for g in grads], [w.copy() for w in weights]
    hv = np.zeros(n, dtype=np.float32)
    dg, dw = up(grads), up(weights)
    dv = torch.zeros(n, device="cuda")
    for _ in range(2):
        oracle.bsp_sgd_alg2_step(hg, hw, hv, root=root, lr=0.01, mu=0.9)
        lp.lp_chain_emulate_bsp_sgd_alg2_step(dg, dw, dv, block=8192, root=root, lr=0.01, mu=0.9)
    got_w, got_g = down(dw), down(dg)
    assert lp.lp_chain_emulate_error(P) == 0
    assert dv.cpu().numpy().tobytes() == hv.tobytes()
    for r in range(P):
        assert got_w[r].tobytes() == hw[r].tobytes(), ("weights", r)
        assert got_g[r].tobytes() == hg[r].tobytes(), ("grads", r)


@pytest.mark.parametrize("dt", [inputs.DT_F16, inputs.DT_BF16, inputs.DT_F64])
def test_chain_element_types(oracle, dt):
    P, n = 5, 200_002
    for red, kind in ((lp.REDUCE_SUM, "sum"), (lp.REDUCE_PROD, "prod")):
        src = inputs.typed_rank_vectors([36, dt], P, n, dt, kind)
        for op in ("allreduce", "reduce", "broadcast"):
            want = [a.copy() for a in src]
            if op == "allreduce":
                oracle.allreduce_dt(want, dt, red=red)
            elif op == "reduce":
                oracle.reduce_dt(want, dt, red=red, root=2)
            else:
                oracle.broadcast_dt(want, dt, root=2)
            dev = [torch.from_numpy(a.view(np.int16) if dt == inputs.DT_BF16 else a).cuda() for a in src]
            lp.lp_chain_emulate_dt(OPS[op], dev, block=8192, root=2, dtype=dt, reduce_op=red)
            torch.cuda.synchronize()
            assert lp.lp_chain_emulate_error(P) == 0
            for r in range(P):
                assert dev[r].cpu().numpy().tobytes() == want[r].view(np.int16 if dt == inputs.DT_BF16 else want[r].dtype).tobytes(), \
                    (op, dt, red, r)


@pytest.mark.parametrize("n", [1, 3, 4097, 200_001, 200_003])
def test_chain_f64_odd_lengths(oracle, n):
    """An f64 vector of odd length is 2 n = 2 (mod 4) words: the last element lies outside the 16-byte body and is folded
    by the tile's scalar tail, which has to treat its two words as ONE double (round 2's TMA kernel folded them as two
    bf16 pairs).  Allreduce, and reduce to a middle root, sum and product, both kernels (the fixture)."""
    P, dt = 5, inputs.DT_F64
    for red, kind in ((lp.REDUCE_SUM, "sum"), (lp.REDUCE_PROD, "prod")):
        src = inputs.typed_rank_vectors([39, n], P, n, dt, kind)
        for op, root in (("allreduce", 0), ("reduce", 2), ("broadcast", 3)):
            want = [a.copy() for a in src]
            if op == "allreduce":
                oracle.allreduce_dt(want, dt, red=red)
            elif op == "reduce":
                oracle.reduce_dt(want, dt, red=red, root=root)
            else:
                oracle.broadcast_dt(want, dt, root=root)
            dev = [torch.from_numpy(a).cuda() for a in src]
            lp.lp_chain_emulate_dt(OPS[op], dev, block=4096, root=root, dtype=dt, reduce_op=red)
            torch.cuda.synchronize()
            assert lp.lp_chain_emulate_error(P) == 0
            for r in range(P):
                assert dev[r].cpu().numpy().tobytes() == want[r].tobytes(), (op, n, red, r)


def test_chain_seeded_fuzz(oracle):
    """200 seeded random collectives (op, P, n, block, root, operator) back to back on one stream, ring geometries drawn
    per P from a small set so that rings are shared by consecutive calls: shakes out ordering bugs that a fixed list of
    shapes would miss (a slot handed back before its loads returned shows up as one wrong tile in a few of many runs)."""
    rng = np.random.default_rng(20161104)
    geoms = {}
    checked = 0
    for case in range(200):
        P = int(rng.choice([2, 3, 4, 5, 7, 8, 12, 16]))
        n = int(rng.choice([1, 7, 4095, 4097, 20_000, 70_001, 300_007, 1_000_003]))
        block = int(rng.choice([0, 4, 1000, 4096, 16_384, 65_536, 1 << 22]))
        op = str(rng.choice(["allreduce", "reduce", "broadcast"]))
        root = int(rng.integers(0, P))
        red = int(rng.choice([lp.REDUCE_SUM, lp.REDUCE_PROD]))
        if P not in geoms:
            geoms[P] = dict(channels=int(rng.choice([1, 2, 3])), slots=int(rng.choice([1, 2, 3, 8])),
                            tile=int(rng.choice([4096, 16_384, 65_536])))
        g = geoms[P]
        src = inputs.typed_rank_vectors([38, case], P, n, inputs.DT_F32, "prod" if red == lp.REDUCE_PROD else "sum")
        want = [a.copy() for a in src]
        run_oracle(oracle, op, want, root, red)
        dev = up(src)
        lp.lp_chain_emulate(OPS[op], dev, block=block, root=root, reduce_op=red, **g)
        if case % 8 == 7 or n >= 300_000:      # mostly no host sync between calls: the next one queues behind
            got = down(dev)
            for r in range(P):
                assert got[r].tobytes() == want[r].tobytes(), (case, op, P, n, block, root, red, g, r)
            checked += 1
    torch.cuda.synchronize()
    assert checked > 40 and all(lp.lp_chain_emulate_error(P, **g) == 0 for P, g in geoms.items())


def test_chain_two_streams_do_not_share_rings(oracle):
    """Emulated endpoints belong to (P, geometry, stream): two chains of the same shape running at the same time on two
    streams must not see each other's blocks."""
    P, n = 3, 400_003
    srcs = [inputs.rank_vectors([42, k], P, n, "uniform") for k in range(2)]
    wants = []
    for src in srcs:
        w = [a.copy() for a in src]
        oracle.allreduce(w)
        wants.append(w)
    devs = [up(src) for src in srcs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for rep in range(3):
        for k in range(2):
            for d, a in zip(devs[k], srcs[k]):
                d.copy_(torch.from_numpy(a))
        torch.cuda.synchronize()
        for k in range(2):
            lp.lp_chain_emulate(lp.OP_ALLREDUCE, devs[k], block=8192, channels=4, slots=2, tile=4096, stream=streams[k])
        torch.cuda.synchronize()
        for k in range(2):
            for r in range(P):
                assert devs[k][r].cpu().numpy().tobytes() == wants[k][r].tobytes(), (rep, k, r)
    assert lp.lp_chain_emulate_error(P, 4, 2, 4096) == 0


def test_chain_argument_errors():
    dev = [torch.zeros(64, device="cuda") for _ in range(2)]
    arr, n = lp._dev_ptrs(dev)
    L = lp.lib()
    s = lp._stream_ptr(None)
    assert L.lp_chain_emulate(lp.OP_ALLREDUCE, arr, 2, n, 16, 0, 7, 0, 0, 0, s) == lp.LP_ERR_INVALID_ARG   # operator
    assert L.lp_chain_emulate(lp.OP_REDUCE, arr, 2, n, 16, 2, 0, 0, 0, 0, s) == lp.LP_ERR_INVALID_ARG      # root
    assert L.lp_chain_emulate(lp.OP_BSP_SGD, arr, 2, n, 16, 0, 0, 0, 0, 0, s) == lp.LP_ERR_INVALID_ARG     # collective
    assert L.lp_chain_emulate(lp.OP_ALLREDUCE, arr, 2, n, 16, 0, 0, 0, 0, 1000, s) == lp.LP_ERR_INVALID_ARG  # tile
    dev4 = [torch.zeros(64, device="cuda") for _ in range(4)]
    arr4, _ = lp._dev_ptrs(dev4)
    assert L.lp_chain_emulate(lp.OP_ALLREDUCE, arr4, 4, n, 16, 0, 0, 64, 0, 0, s) == lp.LP_ERR_UNSUPPORTED  # 512 CTAs at once
    assert L.lp_chain_set_kernel(7) == lp.LP_ERR_INVALID_ARG
    assert L.lp_chain_emulate(lp.OP_ALLREDUCE, arr, 2, 0, 16, 0, 0, 0, 0, 0, s) == lp.LP_OK                 # n == 0


def test_chain_real_entry_points_rank_after_rank(oracle):
    """The REAL per-rank entry points (lp_chain_create / connect_ptrs / run: the launch a rank of a multi-GPU job makes,
    not the cooperative emulation) on P endpoints of this one GPU.  Kernels that wait for each other may not run here as
    separate launches, so only collectives whose data flows one way are run, rank after rank in chain order, with rings
    that never wrap within a call (tiles per channel <= slots): every wait of a kernel is then already satisfied when
    it starts, and the counters -- which are never reset -- carry over from call to call."""
    P, C, S, tile = 4, 2, 8, 4096
    n = 50_001                                            # 13 tiles over 2 channels: 7 <= 8 slots
    chains = [lp.Chain(r, P, channels=C, slots=S, tile=tile) for r in range(P)]
    for r, ch in enumerate(chains):
        ch.set_timeout(1 << 22)
        ch.connect_ptrs(chains[(r + 1) % P].endpoint(), chains[(r - 1) % P].endpoint())
    src = inputs.rank_vectors([37, 0], P, n, "uniform")
    host = [a.copy() for a in src]
    dev = up(src)
    calls = [("broadcast", 0), ("reduce", P - 1), ("broadcast", 2), ("reduce", P - 1), ("broadcast", 3), ("broadcast", 1)]
    for op, root in calls:
        run_oracle(oracle, op, host, root, oracle.RED_SUM)
        order = [(root + j) % P for j in range(P)] if op == "broadcast" else list(range(P))
        for r in order:
            chains[r].run(OPS[op], dev[r], block=tile, root=root)
            torch.cuda.synchronize()                      # rank after rank: nothing runs beside anything
    got = down(dev)
    assert all(ch.error() == 0 for ch in chains)
    for r in range(P):
        assert got[r].tobytes() == host[r].tobytes(), r
    for ch in chains:
        ch.destroy()


def test_chain_endpoint_of_one_rank(oracle):
    """The real entry points on the one GPU there is: create / handle / connect-to-self / run with P = 1 (a no-op by
    definition), and a P = 2 endpoint refuses to run before it is connected."""
    ch = lp.Chain(0, 1)
    assert len(ch.handle()) == lp.CHAIN_HANDLE_BYTES and ch.endpoint() != 0
    ch.connect([ch.handle()])
    x = torch.arange(1000, dtype=torch.float32, device="cuda")
    ch.run(lp.OP_ALLREDUCE, x)
    assert ch.error() == 0 and torch.equal(x.cpu(), torch.arange(1000, dtype=torch.float32))
    ch.destroy()
    ch2 = lp.Chain(1, 2, channels=2, slots=2, tile=4096)
    with pytest.raises(lp.LpError):
        ch2.run(lp.OP_ALLREDUCE, x)
    ch2.destroy()
