"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default variant and
tuning).  configs[1] (P=6, 61 M floats) is compared in full; configs[4] (P=16, 138 M floats, 8.8 GB) on sampled
slices -- the path is element-wise, so the oracle evaluated on a slice is exact for that slice -- plus the
properties that hold at any size (all ranks bit-identical)."""
import numpy as np
import pytest

from paper_1611_04255_b200 import inputs
from paper_1611_04255_b200 import binding as lp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(autouse=True)
def _defaults():
    assert torch.cuda.is_available()
    lp.lp_set_variant(lp.VARIANT_AUTO)
    for k in range(lp.TUNE_COUNT):
        lp.lp_set_tuning(k, 0)
    yield
    torch.cuda.synchronize()


def test_config1_alexnet_allreduce_full_compare(oracle):
    c = inputs.CONFIGS[1]
    P, n = c["P"], c["n"]
    src = inputs.rank_vectors(1, P, n, "normal", c["sigma"])
    dev = [torch.from_numpy(s).cuda() for s in src]
    pristine = [d.clone() for d in dev]
    want = oracle.chain_sum(src)
    for block in c["block_sweep"]:   # 64K .. 1M elements, plus the paper's 64 KB = 16K elements (U1)
        for d, p in zip(dev, pristine):
            d.copy_(p)
        lp.lp_allreduce(dev, block)
        torch.cuda.synchronize()
        for r in range(P):
            assert dev[r].cpu().numpy().tobytes() == want.tobytes(), (block, r)
    # reduce and broadcast at the same size
    for d, p in zip(dev, pristine):
        d.copy_(p)
    lp.lp_reduce(dev, 65_536, root=4)
    torch.cuda.synchronize()
    assert dev[4].cpu().numpy().tobytes() == want.tobytes()
    assert all(torch.equal(dev[r], pristine[r]) for r in range(P) if r != 4)
    lp.lp_broadcast(dev, 65_536, root=4)
    torch.cuda.synchronize()
    assert all(torch.equal(dev[r], dev[4]) for r in range(P))


def test_config4_vgg16_allreduce_sampled(oracle):
    c = inputs.CONFIGS[4]
    P, n, block = c["P"], c["n"], c["block"]
    # sampled slices: message head, a block boundary, a window in the middle, the ragged tail of the last block
    last_block = (n // block) * block
    windows = [(0, 200_000), (block - 4100, block + 4100), (n // 2 - 50_000, n // 2 + 50_000),
               (last_block - 5000, n)]
    dev, slices = [], []
    for r in range(P):
        x = inputs.normal(4, r, n, c["sigma"])
        slices.append([x[a:b].copy() for a, b in windows])
        dev.append(torch.from_numpy(x).cuda())
        del x
    lp.lp_allreduce(dev, block)
    torch.cuda.synchronize()
    for w, (a, b) in enumerate(windows):
        want = oracle.chain_sum([slices[r][w] for r in range(P)])
        for r in (0, 7, 15):
            assert dev[r][a:b].cpu().numpy().tobytes() == want.tobytes(), (w, r)
    for r in range(1, P):   # every rank holds the same bits (the reduced block is forwarded)
        assert torch.equal(dev[r], dev[0]), r
