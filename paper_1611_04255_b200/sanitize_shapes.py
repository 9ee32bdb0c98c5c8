"""Small-shape tour of every kernel of the library, meant to be run under compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|synccheck python -m paper_1611_04255_b200.sanitize_shapes

Every LP variant with every epilogue (sum / product, SGD, momentum, copy), slice lists, the typed folds, the cluster
variant at P = 4, MST / BE, the static MST reduce, the chain emulation with one-slot rings (both kernels), and a pair of
launches chained across calls (LP_TUNE_CHAIN 1).  It checks nothing but that the variants agree with each other byte for
byte (the parity tests compare with the oracle); the sanitizer's ERROR SUMMARY is the result (profiles/r3_sanitizer.md).
"""
import sys

import torch

from . import binding as lp
from . import inputs


def main():
    assert torch.cuda.is_available(), "needs a CUDA device"
    P, n, block = 4, 20_011, 4096
    src = inputs.rank_vectors(7, P, n, "uniform")
    up = lambda arrs: [torch.from_numpy(a).cuda() for a in arrs]  # noqa: E731
    ref = None
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER, lp.VARIANT_COPY_ENGINE):
        lp.lp_set_variant(variant)
        outs = []
        for red in (lp.REDUCE_SUM, lp.REDUCE_PROD):
            d = up(src)
            lp.lp_allreduce_op(d, block, red)
            outs.append(d)
            d = up(src)
            lp.lp_reduce_op(d, block, red, root=2)
            outs.append(d)
        d = up(src)
        lp.lp_broadcast(d, block, root=1)
        outs.append(d)
        g, w = inputs.sgd_inputs(8, P, n)
        dg, dw = up(g), up(w)
        lp.lp_bsp_sgd_step(dg, dw, block, root=1, lr=0.01)
        outs.append(dw)
        dg, dw, vel = up(g), up(w), torch.zeros(n, device="cuda")
        lp.lp_bsp_sgd_momentum_step(dg, dw, vel, block, root=0, lr=0.01, mu=0.9)
        outs.append(dw + [vel])
        if variant != lp.VARIANT_CLUSTER:
            d = up(src)
            lp.lp_allreduce_segments(d, [(5, 1000), (7001, 9000), (19_000, 3)], block)
            outs.append(d)
        torch.cuda.synchronize()
        got = [[t.cpu().numpy().tobytes() for t in o] for o in outs]
        if ref is None:
            ref = got
        else:
            assert got[:7] == ref[:7], ("variants disagree", variant)
    lp.lp_set_variant(lp.VARIANT_AUTO)
    for dt, kind in ((inputs.DT_F16, "sum"), (inputs.DT_BF16, "sum"), (inputs.DT_F64, "prod")):
        t = inputs.typed_rank_vectors([9, dt], P, 7001, dt, kind)
        import numpy as np
        d = [torch.from_numpy(a.view(np.int16) if dt == inputs.DT_BF16 else a).cuda() for a in t]
        lp.lp_allreduce_dt(d, block, dtype=dt, reduce_op=lp.REDUCE_PROD if kind == "prod" else lp.REDUCE_SUM)
    d = up(src)
    lp.lp_mst_allreduce(d)
    lp.lp_be_allreduce(d)
    lp.lp_mst_reduce(d, root=3)
    lp.lp_be_reduce(d, root=1)
    lp.lp_mst_reduce_static(d, root=2)
    g, w = inputs.sgd_inputs(8, P, n)
    lp.lp_bsp_sgd_alg2_step(up(g), up(w), block, root=1, lr=0.01)
    # launches chained across calls (opt-in): disjoint buffer sets back to back, then a dependent call
    lp.lp_set_tuning(lp.TUNE_CHAIN, 1)
    a, b = up(src), up(src)
    for variant in (lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT):
        lp.lp_set_variant(variant)
        lp.lp_allreduce(a, block)
        lp.lp_allreduce(b, block)
        lp.lp_reduce(a, block, root=1)
    lp.lp_set_tuning(lp.TUNE_CHAIN, 0)
    lp.lp_set_variant(lp.VARIANT_AUTO)
    torch.cuda.synchronize()
    # the chain's per-rank code, three ranks, one-slot rings (every slot reused at once), both kernels
    for kernel in (lp.CHAIN_KERNEL_TMA, lp.CHAIN_KERNEL_REGISTER):
        lp.lp_chain_set_kernel(kernel)
        for op in (lp.OP_ALLREDUCE, lp.OP_REDUCE, lp.OP_BROADCAST):
            d = up(inputs.rank_vectors(10, 3, 30_001, "uniform"))
            lp.lp_chain_emulate(op, d, block=4096, root=1, channels=2, slots=1, tile=4096)
        torch.cuda.synchronize()
        assert lp.lp_chain_emulate_error(3, 2, 1, 4096) == 0
    lp.lp_chain_set_kernel(lp.CHAIN_KERNEL_DEFAULT)
    torch.cuda.synchronize()
    print("sanitize_shapes: done, launches", lp.lp_launch_count())


if __name__ == "__main__":
    sys.exit(main())
