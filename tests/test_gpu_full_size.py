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


@pytest.mark.parametrize("P", [2, 4, 8, 16])
def test_config3_sweep_cells(oracle, P):
    # BASELINE.json configs[3]: uniform[-1,1] from seed [3, r], n = 2^10 .. 2^27, LP vs MST vs BE.  Cells up to 2^20
    # are compared in full for every op and algorithm; 2^24 (the 64 MB message of the bar: AUTO takes the pipeline
    # there, the register kernel below) on sampled windows, the path being element-wise.
    for e in (10, 13, 16, 20):
        n = 1 << e
        src = [inputs.uniform(3, r, n) for r in range(P)]
        chain = oracle.chain_sum(src)
        sabs = np.abs(np.stack(src).astype(np.float64)).sum(axis=0)
        for algo, name in ((0, "lp"), (1, "mst"), (2, "be")):
            want = [s.copy() for s in src]
            oracle.allreduce(want, algo=algo)
            dev = [torch.from_numpy(s).cuda() for s in src]
            if name == "lp":
                lp.lp_allreduce(dev, 65_536)
            else:
                getattr(lp, f"lp_{name}_allreduce")(dev)
            torch.cuda.synchronize()
            got = [d.cpu().numpy() for d in dev]
            for r in range(P):
                assert got[r].tobytes() == want[r].tobytes(), (e, name, r)        # same-tree oracle: bit-exact
            if name != "lp":                                                       # reordered trees vs chain order (U15)
                assert np.all(np.abs(got[0].astype(np.float64) - chain) <= 1e-6 * sabs + 1e-30), (e, name)
            for op in ("reduce", "broadcast"):
                want = [s.copy() for s in src]
                getattr(oracle, op)(want, root=P - 1, algo=algo)
                dev = [torch.from_numpy(s).cuda() for s in src]
                if name == "lp":
                    getattr(lp, f"lp_{op}")(dev, 65_536, root=P - 1)
                else:
                    getattr(lp, f"lp_{name}_{op}")(dev, root=P - 1)
                torch.cuda.synchronize()
                for r in range(P):
                    assert dev[r].cpu().numpy().tobytes() == want[r].tobytes(), (e, name, op, r)
    n = 1 << 24
    windows = [(0, 70_000), (65_536 - 3000, 65_536 + 3000), (n // 2, n // 2 + 100_000), (n - 50_000, n)]
    src = [inputs.uniform(3, r, n) for r in range(P)]
    dev = [torch.from_numpy(s).cuda() for s in src]
    lp.lp_allreduce(dev, 65_536)
    torch.cuda.synchronize()
    for a, b in windows:
        want = oracle.chain_sum([s[a:b].copy() for s in src])
        for r in (0, P - 1):
            assert dev[r][a:b].cpu().numpy().tobytes() == want.tobytes(), (a, r)
    for r in range(1, P):
        assert torch.equal(dev[r], dev[0]), r
