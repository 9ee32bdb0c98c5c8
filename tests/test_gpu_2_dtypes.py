"""GPU parity of the typed collectives (lp_*_dt: f16, bf16, f64, reading U21) against the oracle's
lpo_*_dt, element by element on the same seeded bit patterns.  Bit-exact: every combine is one RN operation in the
element type on both sides, chain order rank 0 -> P-1.  A NaN may carry any payload (IEEE-754 leaves it open: the
oracle returns a quiet NaN with the sign of the exact result, the GPU its canonical NaN), so NaNs are compared by
position.  Needs a B200: every test is marked gpu.
"""
import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from paper_1611_04255_b200 import binding as lp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

DTS = [inputs.DT_F16, inputs.DT_BF16, inputs.DT_F64]
VARIANTS = [lp.VARIANT_AUTO, lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER, lp.VARIANT_COPY_ENGINE]
SUM, PROD = lp.REDUCE_SUM, lp.REDUCE_PROD


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


def up(arrs, dt):
    """numpy vectors of element type dt -> CUDA tensors that carry the same bytes (bf16 travels as int16 patterns)."""
    out = []
    for a in arrs:
        if dt == inputs.DT_BF16:
            out.append(torch.from_numpy(a.view(np.int16)).cuda())
        else:
            out.append(torch.from_numpy(a).cuda())
    return out


def down(tensors, dt):
    torch.cuda.synchronize()
    res = [t.cpu().numpy() for t in tensors]
    return [r.view(np.uint16) for r in res] if dt == inputs.DT_BF16 else res


def is_nan(a, dt):
    if dt == inputs.DT_BF16:
        return ((a & 0x7F80) == 0x7F80) & ((a & 0x007F) != 0)
    return np.isnan(a)


def same_typed(got, want, dt):
    ng, nw = is_nan(got, dt), is_nan(want, dt)
    return got.shape == want.shape and np.array_equal(ng, nw) and got[~ng].tobytes() == want[~nw].tobytes()


def run_lp(op, dev, block, dt, red=SUM, root=0):
    if op == "allreduce":
        lp.lp_allreduce_dt(dev, block, dtype=dt, reduce_op=red)
    elif op == "reduce":
        lp.lp_reduce_dt(dev, block, root=root, dtype=dt, reduce_op=red)
    else:
        lp.lp_broadcast_dt(dev, block, root=root, dtype=dt)


def run_oracle(oracle, op, host, dt, red=SUM, root=0):
    if op == "allreduce":
        oracle.allreduce_dt(host, dt, red=red)
    elif op == "reduce":
        oracle.reduce_dt(host, dt, red=red, root=root)
    else:
        oracle.broadcast_dt(host, dt, root=root)


def check(oracle, P, n, block, dt, kind, red, variant, ops=("allreduce", "reduce", "broadcast"), root=None):
    lp.lp_set_variant(variant)
    src = inputs.typed_rank_vectors([21, n, P], P, n, dt, kind)
    for op in ops:
        r0 = (P - 1 if op == "reduce" else P // 2) if root is None else root
        want = [a.copy() for a in src]
        run_oracle(oracle, op, want, dt, red=red, root=r0)
        dev = up(src, dt)
        run_lp(op, dev, block, dt, red=red, root=r0)
        got = down(dev, dt)
        for r in range(P):
            assert same_typed(got[r], want[r], dt), (op, inputs.DT_NAMES[dt], kind, red, variant, P, n, block, r)


# several tiles + ragged tails, odd lengths (a 16-bit vector then ends in half a word), odd blocks, every variant
SHAPES = [
    # P, n, block
    (1, 1001, 64), (2, 1, 1), (2, 2, 1), (2, 3, 64), (2, 7, 3), (3, 1001, 100), (3, 4097, 1000), (4, 70_001, 4096),
    (5, 300_003, 65_536), (6, 70_002, 1001), (8, 262_147, 16_384), (16, 100_003, 8192), (32, 20_001, 5000),
    (4, 8192 * 3 + 5, 8192), (6, 1 << 19, 1 << 22),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dt", DTS)
@pytest.mark.parametrize("P,n,block", SHAPES)
def test_typed_ragged_shapes_sum_bit_exact(oracle, variant, dt, P, n, block):
    if variant == lp.VARIANT_COPY_ENGINE and n // block > 300:
        pytest.skip("copy-engine variant: thousands of tiny copies, covered by smaller shapes")
    if variant == lp.VARIANT_CLUSTER and P > 16:
        pytest.skip("cluster variant: P <= 16")
    check(oracle, P, n, block, dt, "sum", SUM, variant)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dt", DTS)
@pytest.mark.parametrize("P,n,block", [(2, 4099, 512), (6, 70_001, 4096), (16, 33_333, 8192)])
def test_typed_product_bit_exact(oracle, variant, dt, P, n, block):
    check(oracle, P, n, block, dt, "prod", PROD, variant, ops=("allreduce", "reduce"))


@pytest.mark.parametrize("variant", [lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER])
@pytest.mark.parametrize("dt", [inputs.DT_F16, inputs.DT_BF16])
@pytest.mark.parametrize("red", [SUM, PROD])
def test_typed_full_exponent_range(oracle, variant, dt, red):
    """'wide' inputs: every finite exponent, subnormals included -- overflow to infinity, inf - inf = NaN, gradual
    underflow and subnormal results must all come out as one RN operation per combine gives them (no flush-to-zero)."""
    check(oracle, 6, 50_001, 4096, dt, "wide", red, variant, ops=("allreduce",))
    check(oracle, 3, 9_999, 1024, dt, "wide", red, variant, ops=("reduce",))


@pytest.mark.parametrize("dt", DTS)
def test_typed_every_root_and_block_invariance(oracle, dt):
    P, n = 5, 40_003
    src = inputs.typed_rank_vectors([22, 0], P, n, dt, "sum")
    want = [a.copy() for a in src]
    oracle.allreduce_dt(want, dt)
    for root in range(P):
        for block in (1001, 4096, 1 << 20):
            dev = up(src, dt)
            lp.lp_reduce_dt(dev, block, root=root, dtype=dt)
            got = down(dev, dt)
            assert same_typed(got[root], want[0], dt), (root, block)          # U4: the fold does not depend on the root
            for r in range(P):
                if r != root:
                    assert got[r].tobytes() == src[r].tobytes(), (root, block, r)   # U5: non-root vectors unchanged
            dev = up(src, dt)
            lp.lp_broadcast_dt(dev, block, root=root, dtype=dt)
            got = down(dev, dt)
            assert all(g.tobytes() == src[root].tobytes() for g in got), (root, block)


@pytest.mark.parametrize("dt", DTS)
def test_typed_large_message_pipeline_and_direct(oracle, dt):
    """A message of several grid-fulls of tiles (32 MB per rank) through both persistent kernels."""
    P = 4
    n = (32 << 20) // lp.lp_dtype_size(dt) + 3
    src = inputs.typed_rank_vectors([23, 0], P, n, dt, "sum")
    want = [a.copy() for a in src]
    oracle.allreduce_dt(want, dt)
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT):
        lp.lp_set_variant(variant)
        dev = up(src, dt)
        lp.lp_allreduce_dt(dev, 65_536, dtype=dt)
        got = down(dev, dt)
        for r in range(P):
            assert same_typed(got[r], want[r], dt), (variant, r)


def _oracle_slices(oracle, op, host, segs, dt, red, root):
    """The definition of a layer-wise call: the whole-message collective on every slice (Alg. 1), nothing elsewhere."""
    for off, ln in segs:
        if ln == 0:
            continue
        views = [h[off:off + ln] for h in host]           # contiguous views: the oracle works in place on them
        run_oracle(oracle, op, views, dt, red=red, root=root)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dt", DTS)
def test_typed_slice_lists(oracle, variant, dt):
    """Layer-wise collectives (Alg. 1) on typed vectors: slices of any length (odd ones end in half a word for the
    16-bit types), empty slices, a slice of one element, gaps that must stay untouched."""
    P, n = 4, 120_011
    segs = [(10, 1001), (2000, 0), (5000, 1), (7002, 30_000), (40_000, 4097), (60_000, 2), (100_000, 20_011)]
    lp.lp_set_variant(variant)
    src = inputs.typed_rank_vectors([25, dt], P, n, dt, "sum")
    for op, red in (("allreduce", SUM), ("reduce", PROD), ("broadcast", SUM)):
        want = [a.copy() for a in src]
        _oracle_slices(oracle, op, want, segs, dt, red, root=1)
        dev = up(src, dt)
        if op == "allreduce":
            lp.lp_allreduce_segments_dt(dev, segs, 4096, dtype=dt, reduce_op=red)
        elif op == "reduce":
            lp.lp_reduce_segments_dt(dev, segs, 4096, root=1, dtype=dt, reduce_op=red)
        else:
            lp.lp_broadcast_segments_dt(dev, segs, 4096, root=1, dtype=dt)
        got = down(dev, dt)
        for r in range(P):
            assert same_typed(got[r], want[r], dt), (op, variant, inputs.DT_NAMES[dt], r)


def test_typed_slices_must_start_on_a_word():
    dev = [torch.zeros(64, dtype=torch.float16, device="cuda") for _ in range(2)]
    with pytest.raises(lp.LpError) as e:
        lp.lp_allreduce_segments_dt(dev, [(3, 8)], 16)
    assert e.value.status == lp.LP_ERR_INVALID_ARG
    lp.lp_allreduce_segments_dt(dev, [(4, 7)], 16)                               # even offset, odd length: fine
    dev64 = [torch.zeros(64, dtype=torch.float64, device="cuda") for _ in range(2)]
    lp.lp_allreduce_segments_dt(dev64, [(3, 8)], 16)                             # f64: any offset


@pytest.mark.parametrize("dt", DTS)
def test_typed_plans(oracle, dt):
    """A plan fixes the element type too: two typed plans with different variants and tunings, one confined to 32 CTAs."""
    P, n = 6, 300_003
    src = inputs.typed_rank_vectors([26, dt], P, n, dt, "sum")
    want = [a.copy() for a in src]
    oracle.allreduce_dt(want, dt)
    plans = [lp.Plan(lp.OP_ALLREDUCE, P, n, block=8192, variant=lp.VARIANT_PIPELINE, dtype=dt,
                     tuning={lp.TUNE_GRID_LIMIT: 32}),
             lp.Plan(lp.OP_ALLREDUCE, P, n, block=0, variant=lp.VARIANT_DIRECT, dtype=dt)]
    for plan in plans:
        dev = up(src, dt)
        plan.run(dev)
        got = down(dev, dt)
        for r in range(P):
            assert same_typed(got[r], want[r], dt), (inputs.DT_NAMES[dt], r)
        assert plan.info()["n_tiles"] > 0
        plan.close()
    with pytest.raises(lp.LpError):
        lp.Plan(lp.OP_BSP_SGD, P, n, dtype=dt)                                    # the SGD steps are fp32
    segs = [(0, 1001), (2000, 50_001)]
    plan = lp.Plan(lp.OP_REDUCE, P, n, block=4096, root=2, reduce_op=PROD, dtype=dt)
    psrc = inputs.typed_rank_vectors([27, dt], P, n, dt, "prod")
    want = [a.copy() for a in psrc]
    _oracle_slices(oracle, "reduce", want, segs, dt, PROD, root=2)
    dev = up(psrc, dt)
    plan.run_segments(dev, segs)
    got = down(dev, dt)
    for r in range(P):
        assert same_typed(got[r], want[r], dt), (inputs.DT_NAMES[dt], r)
    plan.close()


def test_typed_f32_is_the_plain_call(oracle):
    P, n = 6, 70_001
    src = inputs.rank_vectors([24, 0], P, n, "uniform")
    want = [a.copy() for a in src]
    oracle.allreduce(want)
    dev = [torch.from_numpy(a).cuda() for a in src]
    lp.lp_allreduce_dt(dev, 4096)
    torch.cuda.synchronize()
    assert all(d.cpu().numpy().tobytes() == w.tobytes() for d, w in zip(dev, want))


def test_typed_argument_errors():
    dev = [torch.zeros(64, dtype=torch.float16, device="cuda") for _ in range(2)]
    arr, n, dt = lp._dev_ptrs_dt(dev)
    L = lp.lib()
    s = lp._stream_ptr(None)
    assert L.lp_allreduce_dt(arr, 2, n, 16, 7, lp.REDUCE_SUM, s) == lp.LP_ERR_INVALID_ARG       # unknown dtype
    assert L.lp_allreduce_dt(arr, 2, n, 16, dt, 5, s) == lp.LP_ERR_INVALID_ARG                  # unknown operator
    assert L.lp_reduce_dt(arr, 2, n, 16, 2, dt, lp.REDUCE_SUM, s) == lp.LP_ERR_INVALID_ARG      # root out of range
    view = [dev[0], dev[0][8:]]                                                                 # overlapping buffers
    arr2 = (lp.ctypes.c_void_p * 2)(*[v.data_ptr() for v in view])
    assert L.lp_allreduce_dt(arr2, 2, 32, 16, dt, lp.REDUCE_SUM, s) == lp.LP_ERR_INVALID_ARG
    assert L.lp_allreduce_dt(arr, 2, 0, 16, dt, lp.REDUCE_SUM, s) == lp.LP_OK                   # n == 0: a no-op
    assert lp.lp_dtype_size(lp.DT_F16) == 2 and lp.lp_dtype_size(lp.DT_F64) == 8 and lp.lp_dtype_size(9) == 0
