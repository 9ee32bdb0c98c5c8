"""SURVEY 8(f)-3 evidence, NOT part of the parity gate: the fitted alpha-beta cost model against the
clock.  Marker `timing` only -- `pytest -m gpu` (the driver's gate) never collects these; run them by hand on a GPU box with
`pytest -m timing`.  A wall-clock window around constants fitted on one pod says something about that pod, not about the
values the collectives return (round 2: the driver's box ran a latency-bound cell 1.9x faster than the model).
"""
import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from paper_1611_04255_b200 import binding as lp

torch = pytest.importorskip("torch")
pytestmark = [pytest.mark.timing,
              pytest.mark.skipif(not torch.cuda.is_available(), reason="timing checks need a CUDA device")]


@pytest.fixture(autouse=True)
def _defaults():
    lp.lib()
    lp.lp_set_variant(lp.VARIANT_AUTO)
    for k in range(lp.TUNE_COUNT):
        lp.lp_set_tuning(k, 0)
    yield
    torch.cuda.synchronize()
    lp.lp_set_variant(lp.VARIANT_AUTO)
    lp.lp_chain_set_kernel(lp.CHAIN_KERNEL_DEFAULT)


def up(arrs):
    return [torch.from_numpy(a).cuda() for a in arrs]


def down(tensors):
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in tensors]


def same(a, b):
    return a.shape == b.shape and a.tobytes() == b.tobytes()


def test_chain_cost_model_predicts_the_emulation():
    """Sec. 3.2's model with the committed constants (lp_chain_fitted_constants; profiles/r2_chain_cost_model.md) against
    the clock: a 64 MB allreduce over 4 emulated ranks at a latency-bound, a near-optimal and a fill-bound block, and
    block = 0 may not be slower than the fixed 64 K-element block by more than measurement noise."""
    if lp.lib().lp_chain_set_kernel(lp.CHAIN_KERNEL_TMA) != lp.LP_OK:
        pytest.skip("no TMA kernel")
    P, C, n = 4, 16, (64 << 20) // 4
    alpha, beta = lp.lp_chain_fitted_constants()
    bufs = lp.Ranks([torch.full((n,), 0.001 * (r + 1), device="cuda") for r in range(P)])

    def clock(block, tile):
        for _ in range(2):
            lp.lp_chain_emulate(lp.OP_ALLREDUCE, bufs, block=block, channels=C, slots=8, tile=tile)
        torch.cuda.synchronize()
        best = 1e9
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(4):
                lp.lp_chain_emulate(lp.OP_ALLREDUCE, bufs, block=block, channels=C, slots=8, tile=tile)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) / 4 * 1e-3)
        return best

    for b in (8192, 65_536, 262_144):
        t = clock(b, b)
        model = lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, n * 4 / C, b * 4, alpha, beta)
        assert 0.6 < t / model < 1.6, (b, t, model)
    assert clock(0, 131_072) < 1.15 * clock(65_536, 131_072)
    assert lp.lp_chain_emulate_error(P, C, 8, 131_072) == 0


def _time_allreduce(dev, pristine, block, reps=3):
    ms = []
    for it in range(reps + 1):
        for d, p in zip(dev, pristine):
            d.copy_(p)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        lp.lp_allreduce(dev, block)
        e1.record()
        torch.cuda.synchronize()
        if it:
            ms.append(e0.elapsed_time(e1))
    return float(np.median(ms)) * 1e-3


@pytest.mark.parametrize("P", [2, 6, 16])
def test_fitted_cost_model_and_auto_block(oracle, P):
    # The copy-engine variant (the paper's own design) is the realisation Eq. 1 / Table 1 describes.
    # (i) lp_cost_model with the constants committed in the library (lp_fitted_constants: profiles/r2_cost_model_fit.md)
    # predicts the measured time of the configs[1]-sized allreduce (244 MB per rank) at four block sizes within 45 %
    # (the fit's own error is 12-16 %, the constants' simple p-law adds up to 27 % more; for messages much shorter
    # than (p-1) blocks the model's pipeline-fill term, which has no counterpart on one GPU, overestimates further);
    # (ii) block = 0 -- the model's optimum -- is within 20 % of the best block of the scan, where the paper's 64 KB
    # (16 K elements) is 100x slower; (iii) the result with block = 0 is the oracle's, bit for bit.
    n = 61_000_000
    src = inputs.rank_vectors([30, P], P, n, "normal", 1e-3)
    pristine = up(src)
    dev = [p.clone() for p in pristine]
    lp.lp_set_variant(lp.VARIANT_COPY_ENGINE)
    alpha, beta = lp.lp_fitted_constants(P)
    times = {}
    for block in (1 << 18, 1 << 20, 1 << 22, 1 << 23, 1 << 24):
        times[block] = _time_allreduce(dev, pristine, block)
    for block in (1 << 18, 1 << 20, 1 << 22, 1 << 23):
        pred = lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, n * 4.0, block * 4.0, alpha, beta, 0.0)
        if block >= 1 << 22:   # bandwidth-dominated blocks: a property of the GPU
            assert abs(pred - times[block]) / times[block] < 0.45, (P, block, pred, times[block])
        else:                  # latency-dominated blocks: alpha is the HOST's cost of submitting a stream operation
            assert 0.4 < pred / times[block] < 2.5, (P, block, pred, times[block])   # (2.4 - 4.3 ms seen for the same call)
    t_auto = _time_allreduce(dev, pristine, 0)
    auto_block = lp.lp_auto_block(lp.OP_ALLREDUCE, P, n, lp.VARIANT_COPY_ENGINE)
    assert (1 << 21) <= auto_block <= n
    assert t_auto <= 1.2 * min(times.values()), (P, t_auto, times)
    t_paper = _time_allreduce(dev, pristine, 16_384, reps=1)
    assert t_paper > 20 * t_auto, (t_paper, t_auto)
    for d, p in zip(dev, pristine):
        d.copy_(p)
    lp.lp_allreduce(dev, 0)
    want = oracle.chain_sum(src)
    assert all(same(g, want) for g in down(dev))
    # the persistent kernels are flat in the block size: block = 0 is as good as any
    lp.lp_set_variant(lp.VARIANT_AUTO)
    t0 = _time_allreduce(dev, pristine, 0)
    t1 = _time_allreduce(dev, pristine, 16_384)
    t2 = _time_allreduce(dev, pristine, 1 << 22)
    assert max(t0, t1, t2) < 1.15 * min(t0, t1, t2), (t0, t1, t2)
