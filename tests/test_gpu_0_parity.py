"""GPU parity: the CUDA library (through its C ABI / thin binding) against the CPU oracle, element by element on
the same seeded inputs.  Bit-exact in chain order (north_star); MST / BE bit-exact against the same-tree oracle
and within 1e-6 * sum|x| of the chain order (U15).  Needs a B200: every test is marked gpu.
"""
import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from paper_1611_04255_b200 import binding as lp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

LP, MST, BE = 0, 1, 2
VARIANTS = [lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_COPY_ENGINE, lp.VARIANT_AUTO]


@pytest.fixture(autouse=True)
def _device_and_defaults():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    lp.lib()
    lp.lp_set_variant(lp.VARIANT_AUTO)
    for k in range(lp.TUNE_COUNT):
        lp.lp_set_tuning(k, 0)
    yield
    torch.cuda.synchronize()
    lp.lp_set_variant(lp.VARIANT_AUTO)


def up(arrs):
    return [torch.from_numpy(a).cuda() for a in arrs]


def down(tensors):
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in tensors]


def same(a, b):
    return a.shape == b.shape and a.tobytes() == b.tobytes()


def copies(arrs):
    return [a.copy() for a in arrs]


def same_but_nan_payload(a, b):
    """Bit-exact except that a NaN may carry any payload (IEEE-754 leaves it open; x86 keeps an operand's, the GPU
    returns the canonical quiet NaN): NaNs in the same places, every other element the same bytes."""
    na, nb = np.isnan(a), np.isnan(b)
    return a.shape == b.shape and np.array_equal(na, nb) and a[~na].tobytes() == b[~nb].tobytes()


def run_lp(op, dev, block, root=0, stream=None):
    if op == "allreduce":
        lp.lp_allreduce(dev, block, stream=stream)
    elif op == "reduce":
        lp.lp_reduce(dev, block, root=root, stream=stream)
    else:
        lp.lp_broadcast(dev, block, root=root, stream=stream)


def run_oracle(oracle, op, host, root=0, algo=LP):
    if op == "allreduce":
        oracle.allreduce(host, algo=algo)
    elif op == "reduce":
        oracle.reduce(host, root=root, algo=algo)
    else:
        oracle.broadcast(host, root=root, algo=algo)


# ---------------------------------------------------------------------------------------------------
# BASELINE.json configs[0]: P=4, n=1Mi, b=65536, U[-1,1] seed 0; allreduce, reduce(0), broadcast(0)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("op", ["allreduce", "reduce", "broadcast"])
def test_config0_bit_exact(oracle, variant, op):
    c = inputs.CONFIGS[0]
    src = inputs.rank_vectors(0, c["P"], c["n"], "uniform")
    want = copies(src)
    run_oracle(oracle, op, want, root=0)
    lp.lp_set_variant(variant)
    dev = up(src)
    run_lp(op, dev, c["block"], root=0)
    got = down(dev)
    for r in range(c["P"]):
        assert same(got[r], want[r]), (op, variant, r)
    # the stage-model tick count of this shape: P + nb - 1 = 19
    assert lp.lp_schedule_steps(c["P"], c["n"], c["block"], 2) == 19


# ---------------------------------------------------------------------------------------------------
# ragged shapes: several tiles + tails, unaligned blocks, every root, all variants
# ---------------------------------------------------------------------------------------------------
SHAPES = [
    # P, n, block
    (1, 1000, 64), (2, 1, 1), (2, 3, 64), (2, 5, 4), (3, 1001, 100), (3, 4097, 1000), (4, 70_001, 4096),
    (5, 300_003, 65_536), (6, 70_001, 1001), (7, 12_345, 333), (8, 262_147, 16_384), (16, 100_003, 8192),
    (32, 20_001, 5000), (4, 8192 * 3 + 5, 8192), (6, 1 << 20, 1 << 22),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("P,n,block", SHAPES)
def test_ragged_shapes_bit_exact(oracle, variant, P, n, block):
    if variant == lp.VARIANT_COPY_ENGINE and n // block > 400:
        pytest.skip("copy-engine variant: thousands of tiny copies, covered by smaller shapes")
    lp.lp_set_variant(variant)
    src = inputs.rank_vectors([7, n], P, n, "uniform")
    for op in ("allreduce", "reduce", "broadcast"):
        for root in sorted({0, P - 1, P // 2}):
            if op == "allreduce" and root != 0:
                continue
            want = copies(src)
            run_oracle(oracle, op, want, root=root)
            dev = up(src)
            run_lp(op, dev, block, root=root)
            got = down(dev)
            for r in range(P):
                assert same(got[r], want[r]), (op, root, r)


def test_tuning_space_bit_exact(oracle):
    # every tile size / ring depth / CTA count / cache hint gives the same bits
    P, n, block = 5, 400_003, 32_768
    src = inputs.rank_vectors(8, P, n, "normal", 1e-3)
    want = copies(src)
    oracle.allreduce(want)
    for tile in (1024, 2048, 4096, 8192):
        for stages, out_stages, ctas, hint, sched in ((2, 1, 1, 0, 0), (3, 2, 2, 1, 1), (8, 3, 1, 2, 0), (4, 4, 3, 0, 1)):
            lp.lp_set_tuning(lp.TUNE_SCHED, sched)
            lp.lp_set_tuning(lp.TUNE_TILE_ELEMS, tile)
            lp.lp_set_tuning(lp.TUNE_STAGES, stages)
            lp.lp_set_tuning(lp.TUNE_OUT_STAGES, out_stages)
            lp.lp_set_tuning(lp.TUNE_CTAS_PER_SM, ctas)
            lp.lp_set_tuning(lp.TUNE_L2_HINT, hint)
            dev = up(src)
            lp.lp_allreduce(dev, block)
            got = down(dev)
            assert all(same(g, w) for g, w in zip(got, want)), (tile, stages, out_stages, ctas, hint)
            dev = up(src)
            lp.lp_broadcast(dev, block, root=3)
            got = down(dev)
            assert all(same(g, src[3]) for g in got), ("bcast", tile, stages)
    for tile in (1024, 2048, 4096):
        for sched in (0, 1):
            lp.lp_set_variant(lp.VARIANT_DIRECT)
            lp.lp_set_tuning(lp.TUNE_TILE_ELEMS, tile)
            lp.lp_set_tuning(lp.TUNE_SCHED, sched)
            dev = up(src)
            lp.lp_allreduce(dev, block)
            assert all(same(g, w) for g, w in zip(down(dev), want)), ("direct", tile, sched)


def test_tile_claim_counters_rearm_and_streams(oracle):
    # a2 with dynamic tile claims: every launch takes a self-resetting counter pair from a ring of 1024.  More
    # launches than pairs (each pair reused), back to back on one stream and interleaved on two streams, must
    # all give the oracle's bits: a pair that was not re-armed would skip or repeat tiles.
    P, n, block = 3, 150_001, 8_192
    src = inputs.rank_vectors(21, P, n, "uniform")
    want = oracle.chain_sum(src)
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT):
        lp.lp_set_variant(variant)
        pristine = up(src)
        work = [torch.empty_like(t) for t in pristine]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        sets = []
        for s in streams:
            with torch.cuda.stream(s):
                sets.append(([torch.empty_like(t) for t in pristine], s))
        torch.cuda.synchronize()
        for it in range(1300):
            for w, p in zip(work, pristine):
                w.copy_(p)
            lp.lp_reduce(work, block, root=it % P)
            if it % 97 == 0 or it == 1299:
                torch.cuda.synchronize()
                assert same(work[it % P].cpu().numpy(), want), (variant, it)
        for it in range(40):
            for bufs, s in sets:
                with torch.cuda.stream(s):
                    for w, p in zip(bufs, pristine):
                        w.copy_(p)
                    lp.lp_allreduce(bufs, block, stream=s)
            torch.cuda.synchronize()
            for bufs, _ in sets:
                assert all(same(b.cpu().numpy(), want) for b in bufs), (variant, "streams", it)


def test_chain_order_and_invariances(oracle):
    # the non-associative triple of the oracle pin: a wrong fold order shows up in one element
    vals = [1e8, -1e8, 1.0]
    for variant in VARIANTS:
        lp.lp_set_variant(variant)
        for perm, want in (((0, 1, 2), 1.0), ((2, 0, 1), 0.0), ((1, 2, 0), 0.0), ((1, 0, 2), 1.0)):
            dev = up([np.full(4100, vals[p], np.float32) for p in perm])
            lp.lp_allreduce(dev, 1024)
            got = down(dev)
            assert all((g == np.float32(want)).all() for g in got), (variant, perm)
    # result independent of block, root, stream; allreduce == broadcast(reduce)
    lp.lp_set_variant(lp.VARIANT_PIPELINE)
    P, n = 6, 123_457
    src = inputs.rank_vectors(9, P, n, "uniform")
    want = oracle.chain_sum(src)
    side = torch.cuda.Stream()
    for block in (4, 256, 4096, 40_000, n, 10 * n):
        dev = up(src)
        torch.cuda.synchronize()
        lp.lp_allreduce(dev, block, stream=side)
        side.synchronize()
        assert all(same(g, want) for g in down(dev)), block
    for root in range(P):
        dev = up(src)
        lp.lp_reduce(dev, 4096, root=root)
        got = down(dev)
        assert same(got[root], want)
        assert all(same(got[r], src[r]) for r in range(P) if r != root)  # U5
        lp.lp_broadcast(dev, 4096, root=root)
        assert all(same(g, want) for g in down(dev))


def test_noops_and_device_side_validation():
    dev = up([np.arange(10, dtype=np.float32)])
    lp.lp_allreduce(dev, 4)          # P == 1: identity
    lp.lp_reduce(dev, 4, root=0)
    lp.lp_broadcast(dev, 4, root=0)
    assert same(down(dev)[0], np.arange(10, dtype=np.float32))
    empty = [torch.empty(0, dtype=torch.float32, device="cuda") for _ in range(3)]
    big = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(lp.LpError) as e:   # overlapping device buffers
        lp.lp_allreduce([big[:32], big[16:48]], 8)
    assert e.value.status == lp.LP_ERR_INVALID_ARG
    with pytest.raises(lp.LpError) as e:   # misaligned device buffer
        lp.lp_allreduce([big[1:17], big[32:48]], 8)
    assert e.value.status == lp.LP_ERR_INVALID_ARG
    with pytest.raises(lp.LpError) as e:
        lp.lp_be_allreduce([big[0:16], big[16:32], big[32:48]])
    assert e.value.status == lp.LP_ERR_UNSUPPORTED
    assert not big.any().item()
    before = lp.lp_launch_count()
    dev = up([np.ones(5000, np.float32) for _ in range(3)])
    lp.lp_allreduce(dev, 1024)
    assert lp.lp_launch_count() == before + 1   # the whole pipeline is ONE launch
    assert (down(dev)[2] == 3).all()
    del empty


# ---------------------------------------------------------------------------------------------------
# fused BSP-SGD step (a6)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("P,n,block,root", [(1, 1000, 256, 0), (2, 4099, 1024, 1), (6, 70_001, 1001, 2),
                                            (8, 150_003, 16_384, 0), (16, 33_333, 4096, 15)])
def test_sgd_step_bit_exact(oracle, variant, P, n, block, root):
    lp.lp_set_variant(variant)
    grads, weights = inputs.sgd_inputs([5, n], P, n)
    weights[root] += np.float32(0.125)  # replicas differ: only weights[root] may be read (U8)
    hg, hw = copies(grads), copies(weights)
    dg, dw = up(grads), up(weights)
    for it in range(3):
        oracle.bsp_sgd_step(hg, hw, root=root, lr=0.01)
        lp.lp_bsp_sgd_step(dg, dw, block, root=root, lr=0.01)
        gw = down(dw)
        for r in range(P):
            assert same(gw[r], hw[r]), (it, r)
    assert all(same(g, s) for g, s in zip(down(dg), grads))  # grads only read


def test_config2_sgd_100_iterations(oracle):
    # BASELINE.json configs[2]: P=8, n=7,000,000, grads N(0,1e-2), w N(0,0.05), lr=0.01, 100 iterations
    c = inputs.CONFIGS[2]
    P, n = c["P"], c["n"]
    grads, weights = inputs.sgd_inputs(2, P, n, c["sigma"], c["w_sigma"])
    hw = copies(weights)
    dg, dw = up(grads), up(weights)
    for it in range(1, c["iters"] + 1):
        oracle.bsp_sgd_step(grads, hw, root=0, lr=c["lr"], omp=True)
        lp.lp_bsp_sgd_step(dg, dw, c["block"], root=0, lr=c["lr"])
        if it in (1, 5, 100):
            gw = down(dw)
            assert all(same(gw[r], hw[r]) for r in range(P)), it


# ---------------------------------------------------------------------------------------------------
# SGD + momentum (U18) and the Alg. 2 step (U9)  -- SURVEY 8(f)-1
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("P,n,block,root", [(1, 1000, 256, 0), (2, 4099, 1024, 1), (6, 70_001, 1001, 2),
                                            (8, 150_003, 16_384, 0), (16, 33_333, 4096, 15)])
def test_momentum_step_bit_exact(oracle, variant, P, n, block, root):
    lp.lp_set_variant(variant)
    grads, weights = inputs.sgd_inputs([6, n], P, n)
    weights[root] += np.float32(0.125)
    vel = inputs.normal([6, n], 99, n, 0.01)
    hg, hw, hv = copies(grads), copies(weights), vel.copy()
    dg, dw, dv = up(grads), up(weights), torch.from_numpy(vel).cuda()
    for it in range(4):
        oracle.bsp_sgd_momentum_step(hg, hw, hv, root=root, lr=0.01, mu=0.9)
        lp.lp_bsp_sgd_momentum_step(dg, dw, dv, block, root=root, lr=0.01, mu=0.9)
        gw = down(dw)
        for r in range(P):
            assert same(gw[r], hw[r]), (it, r)
        assert same(dv.cpu().numpy(), hv), it
    assert all(same(g, s) for g, s in zip(down(dg), grads))  # grads only read


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("with_momentum", [False, True])
@pytest.mark.parametrize("P,n,block,root", [(1, 1000, 256, 0), (3, 4099, 1024, 1), (6, 70_003, 1001, 5),
                                            (8, 150_001, 16_384, 2)])
def test_alg2_step_bit_exact_and_equals_alg3(oracle, variant, with_momentum, P, n, block, root):
    lp.lp_set_variant(variant)
    grads, weights = inputs.sgd_inputs([7, n], P, n)
    weights[root] += np.float32(0.25)
    vel = inputs.normal([7, n], 99, n, 0.01) if with_momentum else None
    hg, hw, hv = copies(grads), copies(weights), (vel.copy() if with_momentum else None)
    dg, dw = up(grads), up(weights)
    dv = torch.from_numpy(vel).cuda() if with_momentum else None
    oracle.bsp_sgd_alg2_step(hg, hw, hv, root=root, lr=0.02, mu=0.9)
    lp.lp_bsp_sgd_alg2_step(dg, dw, block, velocity=dv, root=root, lr=0.02, mu=0.9)
    gw, gg = down(dw), down(dg)
    for r in range(P):
        assert same(gw[r], hw[r]), ("w", r)
        assert same(gg[r], hg[r]), ("g", r)  # grads[root] = S, the others untouched
    if with_momentum:
        assert same(dv.cpu().numpy(), hv)
    # the fused Alg. 3 step on the same inputs leaves the same weights (and velocity)
    dg3, dw3 = up(grads), up(weights)
    if with_momentum:
        dv3 = torch.from_numpy(vel).cuda()
        lp.lp_bsp_sgd_momentum_step(dg3, dw3, dv3, block, root=root, lr=0.02, mu=0.9)
        assert same(dv3.cpu().numpy(), hv)
    else:
        lp.lp_bsp_sgd_step(dg3, dw3, block, root=root, lr=0.02)
    assert all(same(a, b) for a, b in zip(down(dw3), hw))


def test_config2_momentum_20_iterations_all_tiles(oracle):
    # configs[2]'s vectors (P=8, n=7,000,000) through the momentum step, every tile size of the pipeline
    c = inputs.CONFIGS[2]
    P, n = c["P"], c["n"]
    grads, weights = inputs.sgd_inputs(2, P, n, c["sigma"], c["w_sigma"])
    hw, hv = copies(weights), np.zeros(n, np.float32)
    dg, dw, dv = up(grads), up(weights), torch.zeros(n, device="cuda")
    tiles = (0, 1024, 2048, 4096, 8192)
    for it in range(1, 21):
        lp.lp_set_tuning(lp.TUNE_TILE_ELEMS, tiles[it % len(tiles)])
        oracle.bsp_sgd_momentum_step(grads, hw, hv, root=it % P, lr=c["lr"], mu=0.9)
        lp.lp_bsp_sgd_momentum_step(dg, dw, dv, c["block"], root=it % P, lr=c["lr"], mu=0.9)
        if it in (1, 2, 5, 20):
            gw = down(dw)
            assert all(same(gw[r], hw[r]) for r in range(P)), it
            assert same(dv.cpu().numpy(), hv), it


# ---------------------------------------------------------------------------------------------------
# layer-wise collectives (Alg. 1): a list of slices in one launch  -- SURVEY 8(f)-2
# ---------------------------------------------------------------------------------------------------
def _layer_slices(n, rng, k):
    """k ragged, unordered, non-overlapping slices of [0, n) with gaps; offsets deliberately off 16-byte boundaries."""
    cuts = np.sort(rng.choice(np.arange(1, n), size=2 * k - 1, replace=False))
    bounds = np.concatenate([[0], cuts, [n]])
    segs = [(int(bounds[2 * i]), int(bounds[2 * i + 1] - bounds[2 * i])) for i in range(k)]   # every other gap is a hole
    order = rng.permutation(k)
    return [segs[i] for i in order]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("op", ["broadcast", "reduce", "allreduce"])
@pytest.mark.parametrize("P,n,k,block", [(4, 300_007, 9, 16_384), (6, 1_000_003, 40, 65_536), (3, 5_000, 17, 100),
                                         (16, 200_001, 5, 4096)])
def test_segments_bit_exact(oracle, variant, op, P, n, k, block):
    if variant == lp.VARIANT_COPY_ENGINE and k > 20:
        pytest.skip("copy-engine variant: thousands of tiny copies, covered by the smaller cases")
    lp.lp_set_variant(variant)
    rng = np.random.default_rng([91, P, n])
    segs = _layer_slices(n, rng, k) + [(n // 2, 0)]          # plus an empty slice
    src = inputs.rank_vectors([9, n], P, n, "uniform")
    root = P - 1
    want = copies(src)
    oracle.collective_segments({"broadcast": 0, "reduce": 1, "allreduce": 2}[op], want, segs, root=root)
    dev = up(src)
    if op == "allreduce":
        lp.lp_allreduce_segments(dev, segs, block)
    elif op == "reduce":
        lp.lp_reduce_segments(dev, segs, block, root=root)
    else:
        lp.lp_broadcast_segments(dev, segs, block, root=root)
    got = down(dev)
    for r in range(P):
        assert same(got[r], want[r]), (op, r)


def test_segments_many_layers_and_all_tiles(oracle):
    # more slices than one launch carries (96), every pipeline tile size, 1-element and 3-element slices included
    P, n, block = 5, 2_000_003, 32_768
    rng = np.random.default_rng(92)
    segs = _layer_slices(n, rng, 230) + [(n - 1, 1)]
    src = inputs.rank_vectors(93, P, n, "normal", 1e-3)
    want = copies(src)
    oracle.collective_segments(2, want, segs)
    for tile in (0, 1024, 2048, 4096, 8192):
        lp.lp_set_tuning(lp.TUNE_TILE_ELEMS, tile)
        dev = up(src)
        lp.lp_allreduce_segments(dev, segs, block)
        assert all(same(g, w) for g, w in zip(down(dev), want)), tile


@pytest.mark.parametrize("variant", VARIANTS)
def test_sgd_step_segments_bit_exact(oracle, variant):
    lp.lp_set_variant(variant)
    P, n, block, root = 6, 500_009, 16_384, 4
    rng = np.random.default_rng(98)
    segs = _layer_slices(n, rng, 12) + [(7, 0)]
    grads, weights = inputs.sgd_inputs([16, n], P, n)
    weights[root] += np.float32(0.125)
    hw = copies(weights)
    dg, dw = up(grads), up(weights)
    for it in range(2):
        oracle.bsp_sgd_step_segments(grads, hw, segs, root=root, lr=0.01)
        lp.lp_bsp_sgd_step_segments(dg, dw, segs, block, root=root, lr=0.01)
        gw = down(dw)
        for r in range(P):
            assert same(gw[r], hw[r]), (it, r)
    assert all(same(g, s) for g, s in zip(down(dg), grads))


def test_segments_validation():
    dev = [torch.zeros(1000, device="cuda") for _ in range(3)]
    for bad in ([(990, 11)], [(0, 10), (9, 5)], [(5, 10), (0, 6)]):     # past n; overlapping (either order)
        with pytest.raises(lp.LpError) as e:
            lp.lp_allreduce_segments(dev, bad, 64)
        assert e.value.status == lp.LP_ERR_INVALID_ARG
    lp.lp_allreduce_segments(dev, [], 64)                                # empty list: a no-op
    lp.lp_allreduce_segments(dev, [(0, 0), (1000, 0)], 64)               # empty slices too


def test_comm_nonblocking_alg1_backward_pass(oracle):
    # Alg. 1's backward loop: nonblocking_reduce(layer i+1) on the comm stream while
    # "Backward(i)" (here: a kernel that WRITES layer i's gradient on the compute stream) runs; sync_reduce() at
    # the end.  The gradient of a layer only exists once its Backward has run, so a collective that did not wait
    # for lp_comm_after would sum stale zeros.
    P, block = 4, 16_384
    layers = [(0, 70_001), (70_001, 300_000), (370_001, 13), (370_014, 1_000_003)]   # (offset, length), flat layout
    n = layers[-1][0] + layers[-1][1]
    src = inputs.rank_vectors(95, P, n, "normal", 1e-2)
    want = copies(src)
    oracle.collective_segments(2, want, layers)
    staged = up(src)
    grads = [torch.zeros(n, device="cuda") for _ in range(P)]
    comm = lp.Comm()
    compute = torch.cuda.Stream()
    for limit in (0, 24):
        lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, limit)
        for g in grads:
            g.zero_()
        torch.cuda.synchronize()
        with torch.cuda.stream(compute):
            for i in reversed(range(len(layers))):
                o, l = layers[i]
                torch.cuda._sleep(200_000)                    # Backward(i) takes a while ...
                for g, s in zip(grads, staged):
                    g[o:o + l].copy_(s[o:o + l])              # ... and produces layer i's sub-gradients
                comm.after(compute)                           # nonblocking_allreduce(grad of layer i)
                lp.lp_allreduce_segments(grads, [layers[i]], block, stream=comm.stream)
            comm.wait(compute)                                # sync_reduce()
            check = [g.clone() for g in grads]                # on the compute stream: must see the reduced values
        torch.cuda.synchronize()
        assert comm.test()
        for r in range(P):
            assert same(check[r].cpu().numpy(), want[r]), (limit, r)
    comm.close()


def test_grid_limit_bit_exact(oracle):
    P, n, block = 6, 900_001, 65_536
    src = inputs.rank_vectors(96, P, n, "uniform")
    want = oracle.chain_sum(src)
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT):
        lp.lp_set_variant(variant)
        for limit in (1, 7, 148):
            lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, limit)
            dev = up(src)
            lp.lp_allreduce(dev, block)
            assert all(same(g, want) for g in down(dev)), (variant, limit)
            assert lp.lp_plan_query(lp.OP_ALLREDUCE, P, n, block)["grid"] <= limit


# ---------------------------------------------------------------------------------------------------
# stage-per-rank cluster variant: CTA r of a thread-block cluster plays GPU r of Fig. 2
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P,n,block", [(2, 100_003, 16_384), (3, 70_001, 4096), (4, 1 << 20, 65_536), (6, 300_007, 1001),
                                       (8, 150_003, 16_384), (16, 200_001, 65_536), (5, 7, 64), (6, 2_000_003, 65_536)])
def test_cluster_variant_bit_exact(oracle, P, n, block):
    lp.lp_set_variant(lp.VARIANT_CLUSTER)
    src = inputs.rank_vectors([13, n], P, n, "uniform")
    chain = oracle.chain_sum(src)
    dev = up(src)
    lp.lp_allreduce(dev, block)
    assert all(same(g, chain) for g in down(dev)), "allreduce"
    for root in sorted({0, P // 2, P - 1}):
        dev = up(src)
        lp.lp_reduce(dev, block, root=root)
        got = down(dev)
        for r in range(P):
            assert same(got[r], chain if r == root else src[r]), ("reduce", root, r)
        dev = up(src)
        lp.lp_broadcast(dev, block, root=root)
        assert all(same(g, src[root]) for g in down(dev)), ("broadcast", root)
    grads, weights = inputs.sgd_inputs([14, n], P, n)
    root = P - 1
    weights[root] += np.float32(0.5)
    hw = copies(weights)
    dg, dw = up(grads), up(weights)
    for it in range(2):
        oracle.bsp_sgd_step(grads, hw, root=root, lr=0.01)
        lp.lp_bsp_sgd_step(dg, dw, block, root=root, lr=0.01)
        assert all(same(a, b) for a, b in zip(down(dw), hw)), ("sgd", it)


@pytest.mark.parametrize("P,n", [(3, 3_000_003), (6, 2_000_003), (16, 1_000_003)])
def test_cluster_variant_under_backpressure(oracle, P, n):
    # many tiles per cluster: the rings wrap dozens of times and the middle CTAs of the chain run back-pressured by
    # both halves of the allreduce.  This is the case that exposed a slot handed back before its shared-memory
    # reads had returned (one warp row of one tile wrong in ~1 of 10 runs): repeat it.
    lp.lp_set_variant(lp.VARIANT_CLUSTER)
    src = inputs.rank_vectors([15, n], P, n, "uniform")
    want = oracle.chain_sum(src)
    pristine = up(src)
    for it in range(15):
        dev = [p.clone() for p in pristine]
        lp.lp_allreduce(dev, 65_536)
        for r, g in enumerate(down(dev)):
            assert same(g, want), (it, r, int(np.count_nonzero(g != want)))


def test_cluster_variant_limits():
    lp.lp_set_variant(lp.VARIANT_CLUSTER)
    dev = [torch.zeros(4096, device="cuda") for _ in range(17)]
    with pytest.raises(lp.LpError) as e:
        lp.lp_allreduce(dev, 1024)                           # P > 16: no cluster that large
    assert e.value.status == lp.LP_ERR_UNSUPPORTED


@pytest.mark.parametrize("tile,stages,out_stages", [(0, 0, 0), (1024, 0, 0), (4096, 0, 0), (2048, 3, 2), (2048, 8, 6), (4096, 5, 4)])
def test_cluster_variant_tiles_rings_momentum_slices(oracle, tile, stages, out_stages):
    # tile size and ring depths of the stage-per-rank kernel are launch parameters; momentum and slice lists run in
    # it too (one launch per slice)
    lp.lp_set_variant(lp.VARIANT_CLUSTER)
    lp.lp_set_tuning(lp.TUNE_CLUSTER_TILE, tile)
    lp.lp_set_tuning(lp.TUNE_STAGES, stages)
    lp.lp_set_tuning(lp.TUNE_OUT_STAGES, out_stages)
    P, n, block = 6, 700_003, 65_536
    src = inputs.rank_vectors([16, n], P, n, "uniform")
    chain = oracle.chain_sum(src)
    dev = up(src)
    lp.lp_allreduce(dev, block)
    assert all(same(g, chain) for g in down(dev))
    dev = up(src)
    lp.lp_broadcast(dev, block, root=4)
    assert all(same(g, src[4]) for g in down(dev))
    # momentum (U18): 3 iterations, weights and velocity bit-exact
    grads, weights = inputs.sgd_inputs([17, n], P, n)
    hw, hv = copies(weights), np.zeros(n, np.float32)
    dg, dw, dv = up(grads), up(weights), torch.zeros(n, device="cuda")
    for it in range(3):
        oracle.bsp_sgd_momentum_step(grads, hw, hv, root=2, lr=0.01, mu=0.9)
        lp.lp_bsp_sgd_momentum_step(dg, dw, dv, block, root=2, lr=0.01, mu=0.9)
        assert all(same(a, b) for a, b in zip(down(dw), hw)), ("momentum w", it)
        assert same(down([dv])[0], hv), ("momentum v", it)
    # slices that start off the 16-byte grid
    segs = [(5, 1000), (70_001, 123_457), (200_000, 3), (300_002, 250_001)]
    for op, opid in (("broadcast", 0), ("reduce", 1), ("allreduce", 2)):
        want = copies(src)
        oracle.collective_segments(opid, want, segs, root=1)
        dev = up(src)
        if op == "allreduce":
            lp.lp_allreduce_segments(dev, segs, block)
        elif op == "reduce":
            lp.lp_reduce_segments(dev, segs, block, root=1)
        else:
            lp.lp_broadcast_segments(dev, segs, block, root=1)
        assert all(same(a, b) for a, b in zip(down(dev), want)), op


# ---------------------------------------------------------------------------------------------------
# reduce operator ("summations and multiplications"): every LP variant and the MST / BE trees
# ---------------------------------------------------------------------------------------------------
OP_SHAPES = [(1, 1000, 256), (2, 4099, 1024), (3, 70_001, 1001), (4, 1 << 20, 65_536), (6, 300_007, 16_384), (8, 100_001, 4096),
             (16, 250_003, 65_536), (5, 3, 64)]


def product_inputs(seed, P, n):
    # factors around 1 (|x| in [0.5, 1.5), random sign): 16 of them stay far from overflow / underflow
    out = []
    for r in range(P):
        rng = np.random.default_rng([seed, r])
        out.append((rng.random(n, dtype=np.float32) + np.float32(0.5)) * rng.choice(np.array([-1, 1], np.float32), n))
    return out


@pytest.mark.parametrize("variant", VARIANTS + [lp.VARIANT_CLUSTER])
@pytest.mark.parametrize("P,n,block", OP_SHAPES)
def test_product_bit_exact(oracle, variant, P, n, block):
    if variant == lp.VARIANT_COPY_ENGINE and (n // block) * P > 400:
        pytest.skip("copy-engine variant: thousands of tiny operations")
    lp.lp_set_variant(variant)
    src = product_inputs([18, n], P, n)
    fold = oracle.chain_fold(src, oracle.RED_PROD)
    dev = up(src)
    lp.lp_allreduce_op(dev, block, lp.REDUCE_PROD)
    assert all(same(g, fold) for g in down(dev)), "allreduce prod"
    for root in sorted({0, P - 1}):
        dev = up(src)
        lp.lp_reduce_op(dev, block, lp.REDUCE_PROD, root=root)
        got = down(dev)
        for r in range(P):
            assert same(got[r], fold if r == root else src[r]), ("reduce prod", root, r)
    dev = up(src)   # red = sum through the operator entry point is lp_allreduce
    lp.lp_allreduce_op(dev, block, lp.REDUCE_SUM)
    assert all(same(g, oracle.chain_sum(src)) for g in down(dev))


def test_product_overflow_order_and_specials(oracle):
    # (1e30 * 1e30) * 1e-30 = inf in chain order, ~1e30 in any other; NaN / inf / denormal factors as the oracle's
    P, n = 4, 5000
    src = [np.full(n, v, np.float32) for v in (1e30, 1e30, 1e-30, 1e-30)]
    src[0][::7] = np.float32("nan")
    src[1][1::7] = np.float32("-inf")
    src[2][2::7] = np.float32(1e-42)
    src[3][3::7] = 0.0
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER):
        lp.lp_set_variant(variant)
        want = oracle.chain_fold(src, oracle.RED_PROD)
        dev = up(src)
        lp.lp_allreduce_op(dev, 1024, lp.REDUCE_PROD)
        for g in down(dev):
            assert same_but_nan_payload(g, want), variant
    assert np.isinf(want[4]) and np.isnan(want[0])
    for algo, fn in ((MST, lp.lp_mst_allreduce_op), (BE, lp.lp_be_allreduce_op)):
        h = copies(src)
        oracle.allreduce_op(h, oracle.RED_PROD, algo=algo)
        dev = up(src)
        fn(dev, lp.REDUCE_PROD)
        assert all(same_but_nan_payload(a, b) for a, b in zip(down(dev), h)), algo


@pytest.mark.parametrize("P,n", [(2, 1001), (3, 70_001), (4, 65_536), (5, 4099), (6, 300_003), (8, 100_001), (16, 50_001)])
def test_mst_be_product_against_same_tree_oracle(oracle, P, n):
    src = product_inputs([19, n], P, n)
    for algo, red_fn, all_fn in ((MST, lp.lp_mst_reduce_op, lp.lp_mst_allreduce_op), (BE, lp.lp_be_reduce_op, lp.lp_be_allreduce_op)):
        if algo == BE and P & (P - 1):
            continue
        h = copies(src)
        oracle.allreduce_op(h, oracle.RED_PROD, algo=algo)
        dev = up(src)
        all_fn(dev, lp.REDUCE_PROD)
        assert all(same(a, b) for a, b in zip(down(dev), h)), ("allreduce", algo)
        root = P - 1
        h = copies(src)
        oracle.reduce_op(h, oracle.RED_PROD, root=root, algo=algo)
        dev = up(src)
        red_fn(dev, lp.REDUCE_PROD, root=root)
        assert all(same(a, b) for a, b in zip(down(dev), h)), ("reduce", algo)


def test_product_segments_through_a_plan(oracle):
    P, n, block = 4, 300_007, 16_384
    src = product_inputs([20, n], P, n)
    segs = [(5, 1000), (70_001, 123_457), (200_000, 3)]
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER):
        for op, opid in ((lp.OP_REDUCE, 1), (lp.OP_ALLREDUCE, 2)):
            want = copies(src)
            oracle.collective_segments_op(opid, oracle.RED_PROD, want, segs, root=3)
            dev = up(src)
            plan = lp.Plan(op, P, n, block=block, root=3, reduce_op=lp.REDUCE_PROD, variant=variant)
            plan.run_segments(dev, segs)
            assert all(same(a, b) for a, b in zip(down(dev), want)), (variant, op)
            plan.close()


# ---------------------------------------------------------------------------------------------------
# plans: per-call settings; two threads / streams with different settings at once
# ---------------------------------------------------------------------------------------------------
def test_plans_bit_exact_every_op(oracle):
    P, n, block = 6, 500_003, 65_536
    src = inputs.rank_vectors([21, n], P, n, "uniform")
    chain = oracle.chain_sum(src)
    for variant in (lp.VARIANT_AUTO, lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER):
        for tuning in ({}, {lp.TUNE_GRID_LIMIT: 24}, {lp.TUNE_GRANULE_DIV: 8, lp.TUNE_CLAIM_SLOTS: 1}):
            dev = up(src)
            lp.Plan(lp.OP_ALLREDUCE, P, n, block=block, variant=variant, tuning=tuning).run(dev)
            assert all(same(g, chain) for g in down(dev)), (variant, tuning)
            dev = up(src)
            lp.Plan(lp.OP_REDUCE, P, n, root=4, variant=variant, tuning=tuning).run(dev)     # block 0: library chooses
            got = down(dev)
            assert all(same(got[r], chain if r == 4 else src[r]) for r in range(P))
            dev = up(src)
            lp.Plan(lp.OP_BROADCAST, P, n, block=block, root=5, variant=variant, tuning=tuning).run(dev)
            assert all(same(g, src[5]) for g in down(dev))
    grads, weights = inputs.sgd_inputs([22, n], P, n)
    hw, hv = copies(weights), np.zeros(n, np.float32)
    oracle.bsp_sgd_momentum_step(grads, hw, hv, root=1, lr=0.02, mu=0.8)
    dg, dw, dv = up(grads), up(weights), torch.zeros(n, device="cuda")
    lp.Plan(lp.OP_BSP_SGD_MOM, P, n, block=block, root=1).run(dg, weights=dw, velocity=dv, lr=0.02, mu=0.8)
    assert all(same(a, b) for a, b in zip(down(dw), hw)) and same(down([dv])[0], hv)
    hw = copies(weights)
    oracle.bsp_sgd_step(grads, hw, root=1, lr=0.02)
    dw = up(weights)
    lp.Plan(lp.OP_BSP_SGD, P, n, block=block, root=1, tuning={lp.TUNE_GRID_LIMIT: 64}).run(dg, weights=dw, lr=0.02)
    assert all(same(a, b) for a, b in zip(down(dw), hw))
    # the process-wide defaults were never touched
    assert lp.lp_get_variant() == lp.VARIANT_AUTO and all(lp.lp_get_tuning(k) == 0 for k in range(lp.TUNE_COUNT))


def test_two_threads_two_streams_different_grid_limits(oracle):
    # a confined comm-stream collective must not confine anyone else.  Two host threads, two
    # streams, two plans (64 CTAs / unconfined), 40 launches each, running concurrently; both bit-exact every time.
    import threading
    P, n, block = 6, 4_000_003, 65_536
    src_a = inputs.rank_vectors([23, 0], P, n, "uniform")
    src_b = inputs.rank_vectors([23, 1], P, n, "uniform")
    want_a, want_b = oracle.chain_sum(src_a), oracle.chain_sum(src_b)
    plan_a = lp.Plan(lp.OP_ALLREDUCE, P, n, block=block, variant=lp.VARIANT_PIPELINE, tuning={lp.TUNE_GRID_LIMIT: 64})
    plan_b = lp.Plan(lp.OP_ALLREDUCE, P, n, block=block, variant=lp.VARIANT_PIPELINE)
    assert plan_a.info()["grid"] == 64 and plan_b.info()["grid"] > 64
    pa, pb = up(src_a), up(src_b)
    bad = []

    def worker(plan, pristine, want, tag):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for it in range(40):
                    dev = [p.clone() for p in pristine]
                    plan.run(dev, stream=st)
                    st.synchronize()
                    for r, d in enumerate(dev):
                        if not same(d.cpu().numpy(), want):
                            bad.append((tag, it, r))
        except Exception as ex:  # noqa: BLE001
            bad.append((tag, repr(ex)))

    ts = [threading.Thread(target=worker, args=(plan_a, pa, want_a, "a")),
          threading.Thread(target=worker, args=(plan_b, pb, want_b, "b"))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not bad, bad[:5]


def test_many_launches_in_flight_on_many_streams(oracle):
    # tile-claim counters belong to the stream (the old ring of 1024 pairs was shared by launch k
    # and launch k + 1024): 2100 pipeline launches spread over 3 streams without a host sync in between, then 40
    # captured in one CUDA graph replayed twice beside eager launches on another stream
    P, n, block = 4, 600_003, 65_536
    lp.lp_set_variant(lp.VARIANT_PIPELINE)
    src = inputs.rank_vectors([24, n], P, n, "uniform")
    streams = [torch.cuda.Stream() for _ in range(3)]
    pristine = up(src)
    work = [[p.clone() for p in pristine] for _ in streams]
    torch.cuda.synchronize()
    for it in range(700):
        for st, w in zip(streams, work):
            lp.lp_broadcast(w, block, root=it % P, stream=st)    # idempotent after the first: every rank = src[0]
    torch.cuda.synchronize()
    for w in work:
        assert all(same(g, src[0]) for g in down(w))
    chain = oracle.chain_sum(src)
    gsets = [[p.clone() for p in pristine] for _ in range(40)]
    side = [p.clone() for p in pristine]
    lp.lp_allreduce(gsets[0], block)
    torch.cuda.synchronize()
    for d, p_ in zip(gsets[0], pristine):
        d.copy_(p_)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for d in gsets:
            lp.lp_allreduce(d, block)
    for rep in range(2):
        for d in gsets:
            for x, p_ in zip(d, pristine):
                x.copy_(p_)
        torch.cuda.synchronize()
        g.replay()
        for it in range(20):
            for x, p_ in zip(side, pristine):
                x.copy_(p_, non_blocking=True)
            lp.lp_allreduce(side, block, stream=streams[0])
        torch.cuda.synchronize()
        for d in gsets:
            assert all(same(x, chain) for x in down(d)), rep
        assert all(same(x, chain) for x in down(side))


@pytest.mark.parametrize("chain_mode", [0, 1, 3])
def test_stream_chaining_keeps_stream_order(oracle, chain_mode):
    # LP_TUNE_CHAIN: a launch that touches none of the buffers of the launches still in flight ahead of it starts without
    # waiting for them -- by default only inside one API call (0), across calls when the caller opts in (1, 3) and
    # fences work of its own with lp_stream_fence.  Everything that DOES depend on an earlier call -- same buffers, a
    # sub-range of them, a foreign kernel in between -- must still see stream order.  No host sync inside a sequence.
    P, n, block = 4, 1_500_012, 65_536    # a multiple of 4 (the views below must start 16-byte aligned), not of a tile
    rng = np.random.default_rng(27)
    base = [rng.integers(-3, 4, 3 * n).astype(np.float32) for _ in range(P)]   # small integers: sums stay exact, no overflow
    lp.lp_set_tuning(lp.TUNE_CHAIN, chain_mode)
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_AUTO):
        lp.lp_set_variant(variant)
        for rep in range(6):
            big = up(base)                                    # each rank: one tensor of 3n, used through views
            A = [b[0:n] for b in big]
            B = [b[n:2 * n] for b in big]
            C = [b[2 * n:3 * n] for b in big]
            off = (n // 2) & ~3                               # a 16-byte aligned start
            AB = [b[off:off + n] for b in big]                # straddles A and B
            h = copies(base)
            hA, hB, hC = [x[0:n] for x in h], [x[n:2 * n] for x in h], [x[2 * n:3 * n] for x in h]
            hAB = [x[off:off + n] for x in h]
            lp.lp_allreduce(A, block)          # 1
            lp.lp_allreduce(B, block)          # 2: disjoint from 1 -> may start early
            lp.lp_broadcast(C, block, root=1)  # 3: disjoint from 1, 2
            lp.lp_reduce(A, block, root=2)     # 4: depends on 1
            big[0].mul_(2.0)                   # a foreign kernel on the stream, touching everything of rank 0
            if chain_mode:
                lp.lp_stream_fence()           # the opt-in modes' contract; the default needs nothing
            lp.lp_allreduce(AB, block)         # 5: depends on 1, 2, 4 and on the foreign kernel
            lp.lp_broadcast(B, block, root=0)  # 6: depends on 2, 5
            lp.lp_allreduce(C, block)          # 7: depends on 3
            lp.lp_mst_allreduce(A)             # 8: the baselines are chained too
            lp.lp_be_allreduce(C)              # 9
            # the last library call touched C only; a foreign kernel now writes B (a backward GEMM producing the
            # next gradient), then the library reads B.  The default mode must order this by itself.
            for b_ in B:
                b_.add_(1.0)
            if chain_mode:
                lp.lp_stream_fence()
            lp.lp_allreduce(B, block)          # 10
            for fn, args in ((oracle.allreduce, (hA,)), (oracle.allreduce, (hB,))):
                fn(*args)
            oracle.broadcast(hC, root=1)
            oracle.reduce(hA, root=2)
            h[0] *= np.float32(2.0)
            oracle.allreduce(hAB)
            oracle.broadcast(hB, root=0)
            oracle.allreduce(hC)
            oracle.allreduce(hA, algo=MST)
            oracle.allreduce(hC, algo=BE)
            for x in hB:
                x += np.float32(1.0)
            oracle.allreduce(hB)
            got = down(big)
            for r in range(P):
                assert same(got[r], h[r]), (variant, rep, r, int(np.count_nonzero(got[r] != h[r])))
    # the same with chaining off gives the same bits
    lp.lp_set_tuning(lp.TUNE_CHAIN, 2)
    lp.lp_set_variant(lp.VARIANT_PIPELINE)
    big = up(base)
    A, B = [b[0:n] for b in big], [b[n:2 * n] for b in big]
    lp.lp_allreduce(A, block)
    lp.lp_allreduce(B, block)
    lp.lp_reduce(A, block, root=2)
    h = copies(base)
    hA, hB = [x[0:n] for x in h], [x[n:2 * n] for x in h]
    oracle.allreduce(hA)
    oracle.allreduce(hB)
    oracle.reduce(hA, root=2)
    assert all(same(g, w) for g, w in zip(down(big), h))


def test_stream_chaining_long_runs_and_graphs(oracle):
    # many independent calls back to back (rotating buffer sets, as bench.py times them), eagerly and as a CUDA graph:
    # every set must hold the chain sum; then a dependent tail (an SGD loop on ONE set, which may never be chained)
    P, n, block = 6, 800_003, 65_536
    src = inputs.rank_vectors([28, n], P, n, "uniform")
    chain = oracle.chain_sum(src)
    pristine = up(src)
    n_sets = 12
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT):
        lp.lp_set_variant(variant)
        sets = [lp.Ranks([p.clone() for p in pristine]) for _ in range(n_sets)]
        torch.cuda.synchronize()
        for s_ in sets:
            lp.lp_allreduce(s_, block)
        torch.cuda.synchronize()
        for k, s_ in enumerate(sets):
            assert all(same(g, chain) for g in down(s_.bufs)), (variant, "eager", k)
        for s_ in sets:
            for d, p in zip(s_.bufs, pristine):
                d.copy_(p)
        lp.lp_allreduce(sets[0], block)
        torch.cuda.synchronize()
        for d, p in zip(sets[0].bufs, pristine):
            d.copy_(p)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for s_ in sets:
                lp.lp_reduce(s_, block, root=3)
            for s_ in sets:
                lp.lp_broadcast(s_, block, root=3)
        for rep in range(3):
            for s_ in sets:
                for d, p in zip(s_.bufs, pristine):
                    d.copy_(p)
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            for k, s_ in enumerate(sets):
                assert all(same(x, chain) for x in down(s_.bufs)), (variant, "graph", rep, k)
        del g
    grads, weights = inputs.sgd_inputs([29, n], P, n)
    hw = copies(weights)
    dg, dw = up(grads), up(weights)
    for it in range(25):   # step k + 1 reads the weights step k wrote: never chained
        lp.lp_bsp_sgd_step(dg, dw, block, root=it % P, lr=0.01)
    for it in range(25):
        oracle.bsp_sgd_step(grads, hw, root=it % P, lr=0.01)
    assert all(same(a, b) for a, b in zip(down(dw), hw))


def test_shutdown_and_rebind(oracle):
    # function attributes are per device; lp_shutdown() unbinds the library, and the launchers
    # must set them again afterwards (the pipeline's 49 KB and the cluster kernel's ring need the opt-in limit)
    P, n, block = 4, 300_003, 65_536
    src = inputs.rank_vectors([25, n], P, n, "uniform")
    chain = oracle.chain_sum(src)
    for rounds in range(2):
        for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_CLUSTER, lp.VARIANT_DIRECT):
            lp.lp_set_variant(variant)
            dev = up(src)
            lp.lp_allreduce(dev, block)
            assert all(same(g, chain) for g in down(dev)), (rounds, variant)
            dev = up(src)
            lp.lp_broadcast(dev, block, root=1)
            assert all(same(g, src[1]) for g in down(dev))
        h = [torch.from_numpy(s.copy()).pin_memory() for s in src]
        lp.lp_allreduce_host(h, block)
        assert all(same(x.numpy(), chain) for x in h)
        torch.cuda.synchronize()
        lp.lp_shutdown()


def test_guided_claims_cover_every_element_once(oracle):
    # the shrinking claims (LpTileClaimer): every granule exactly once for any granule / claim size, odd block sizes
    # (runs that end at block boundaries), and a message short for the grid
    lp.lp_set_variant(lp.VARIANT_PIPELINE)
    for P, n, block in ((3, 5_000_011, 65_536), (2, 3_000_001, 1001), (5, 40_003, 4099), (4, 2_500_000, 300_000)):
        src = inputs.rank_vectors([26, n], P, n, "uniform")
        chain = oracle.chain_sum(src)
        for div, claim, tile in ((0, 0, 0), (1, 1, 0), (8, 16, 0), (2, 3, 4096), (4, 2, 1024), (8, 8, 8192)):
            lp.lp_set_tuning(lp.TUNE_GRANULE_DIV, div)
            lp.lp_set_tuning(lp.TUNE_CLAIM_SLOTS, claim)
            lp.lp_set_tuning(lp.TUNE_TILE_ELEMS, tile)
            for sched in (0, 1):
                lp.lp_set_tuning(lp.TUNE_SCHED, sched)
                dev = up(src)
                lp.lp_allreduce(dev, block)
                assert all(same(g, chain) for g in down(dev)), (P, n, block, div, claim, tile, sched)
                dev = up(src)
                lp.lp_broadcast(dev, block, root=P - 1)
                assert all(same(g, src[P - 1]) for g in down(dev)), (P, n, block, div, claim, tile, sched)


# ---------------------------------------------------------------------------------------------------
# IEEE corner values (U16): no flush-to-zero, inf and NaN propagate
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [lp.VARIANT_AUTO, lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER])
def test_denormals_inf_nan(oracle, variant):
    # subnormal inputs and subnormal sums must survive bit for bit (nvcc default -ftz=false, oracle without DAZ/FTZ);
    # +-inf propagate exactly; NaN propagates as NaN (payload bits are not compared: x86 keeps the operand's
    # payload, the GPU returns the canonical NaN)
    lp.lp_set_variant(variant)
    P, n = 4, 40_003
    rng = np.random.default_rng(97)
    tiny = np.float32(1e-45)                                   # smallest subnormal
    src = [(rng.integers(-2000, 2000, n).astype(np.float32) * tiny) for _ in range(P)]   # all subnormal or zero
    src[1][::7] = np.float32(1.17549435e-38)                   # smallest normal: sums cross the normal boundary
    src[2][::7] = np.float32(-1.17549435e-38)
    src[0][5::101] = np.inf
    src[3][6::101] = -np.inf
    src[0][7::101] = np.inf
    src[3][7::101] = -np.inf                                   # inf + -inf = NaN
    src[2][8::101] = np.nan
    want = oracle.chain_sum(src)
    assert np.any((want != 0) & (np.abs(want) < np.float32(1.17549435e-38)))      # subnormal results exist
    dev = up(src)
    lp.lp_allreduce(dev, 4096)
    got = down(dev)
    nan = np.isnan(want)
    assert nan.any() and np.isinf(want).any()
    for r in range(P):
        assert np.array_equal(np.isnan(got[r]), nan), r
        assert got[r][~nan].tobytes() == want[~nan].tobytes(), r
    # SGD epilogue on subnormal sums: products that underflow must round the same way
    weights = [np.full(n, np.float32(3e-39)) for _ in range(P)]
    grads = [s.copy() for s in src]
    for g in grads:
        g[~np.isfinite(g)] = 0
    hw = copies(weights)
    oracle.bsp_sgd_step(grads, hw, root=0, lr=0.5)
    dg, dw = up(grads), up(weights)
    lp.lp_bsp_sgd_step(dg, dw, 4096, root=0, lr=0.5)
    assert all(same(a, b) for a, b in zip(down(dw), hw))


# ---------------------------------------------------------------------------------------------------
# MST / BE baselines (a7, a8)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P,n", [(2, 1001), (3, 70_001), (4, 65_536), (5, 4099), (6, 300_003), (8, 100_001),
                                 (16, 50_005), (7, 3)])
def test_mst_be_against_same_tree_oracle(oracle, P, n):
    src = inputs.rank_vectors([3, n], P, n, "uniform")
    chain = oracle.chain_sum(src).astype(np.float64)
    sabs = np.abs(np.stack(src).astype(np.float64)).sum(axis=0)
    algos = [(MST, "mst")] + ([(BE, "be")] if P & (P - 1) == 0 else [])
    for algo, name in algos:
        for op in ("allreduce", "reduce", "broadcast"):
            for root in sorted({0, P - 1}):
                if op == "allreduce" and root != 0:
                    continue
                want = copies(src)
                run_oracle(oracle, op, want, root=root, algo=algo)
                dev = up(src)
                f = getattr(lp, f"lp_{name}_{op}")
                f(dev) if op == "allreduce" else f(dev, root=root)
                got = down(dev)
                for r in range(P):
                    assert same(got[r], want[r]), (name, op, root, r)
                if op != "broadcast":   # reordered sum vs chain order: north_star 1e-6, relative to sum|x| (U15)
                    assert np.all(np.abs(got[root].astype(np.float64) - chain) <= 1e-6 * sabs)


# ---------------------------------------------------------------------------------------------------
# host-buffer entry points (the e2e path bench.py times)
# ---------------------------------------------------------------------------------------------------
def test_host_entry_points(oracle):
    P, n, block = 3, 9_000_001, 65_536   # three 16 MB chunks per rank
    src = inputs.rank_vectors(10, P, n, "normal", 1e-3)
    want = copies(src)
    oracle.allreduce(want, omp=True)
    pinned = [torch.from_numpy(s.copy()).pin_memory() for s in src]
    lp.lp_allreduce_host(pinned, block)
    assert all(same(p.numpy(), w) for p, w in zip(pinned, want))
    pageable = copies(src)
    lp.lp_allreduce_host(pageable, block)
    assert all(same(p, w) for p, w in zip(pageable, want))
    grads, weights = inputs.sgd_inputs(11, 4, 5_000_003)
    hw = copies(weights)
    oracle.bsp_sgd_step(grads, hw, root=1, lr=0.05, omp=True)
    lp.lp_bsp_sgd_step_host(grads, weights, 65_536, root=1, lr=0.05)
    assert all(same(a, b) for a, b in zip(weights, hw))


# ---------------------------------------------------------------------------------------------------
# block = 0 (the cost model's optimum).  What the model predicts against the clock is a measurement, not a
# property of the result: those checks live in tests/test_timing_cost_model.py (marker `timing`, outside the gpu gate).
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P", [2, 6, 16])
def test_auto_block_result_is_the_oracles(oracle, P):
    n = 61_000_000 if P == 6 else 8_000_003
    src = inputs.rank_vectors([30, P], P, n, "normal", 1e-3)
    want = oracle.chain_sum(src)
    for variant in (lp.VARIANT_COPY_ENGINE, lp.VARIANT_AUTO):
        lp.lp_set_variant(variant)
        auto_block = lp.lp_auto_block(lp.OP_ALLREDUCE, P, n, variant)
        assert 1 <= auto_block <= max(n, lp.DEFAULT_BLOCK)
        dev = up(src)
        lp.lp_allreduce(dev, 0)
        assert all(same(g, want) for g in down(dev)), (P, variant)
