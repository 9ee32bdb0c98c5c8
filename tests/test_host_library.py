"""CPU-side checks of the CUDA library: it loads, exports every symbol include/lp_collectives.h declares, and
its host-only schedule engine / planner / argument validation behave (no compute call needs a GPU here).

The product's schedule engine (csrc/lp_host_schedule.cpp, csrc/lp_schedule.h) and the oracle's
(oracle/lpo_oracle.c) are separate implementations; here they are compared with each other AND with the
paper's printed values / closed forms.
"""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1611_04255_b200 import binding as lp
from tests.conftest import ROOT, read_golden

BCAST, REDUCE, ALLREDUCE, SGD = 0, 1, 2, 3


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "lp_collectives.h")).read()
    names = re.findall(r"^LP_API [^;(]*?\b(lp_[a-z_0-9]+)\(", header, flags=re.M)
    assert len(names) >= 25 and len(set(names)) == len(names)
    L = lp.lib()
    for name in names:
        assert hasattr(L, name), name
    assert lp.lp_version() >= 100
    assert "LP_OK" in lp.status_string(0)


def test_num_blocks_and_stage_block_closed_forms():
    # a1 (U6) and a2
    assert lp.lp_num_blocks(61_000_000, 65_536) == 931
    assert lp.lp_num_blocks(138_000_000, 262_144) == 527
    assert lp.lp_num_blocks(10, 0) == 0 and lp.lp_num_blocks(0, 7) == 0 and lp.lp_num_blocks(7, 100) == 1
    P, nb = 5, 7
    seen = set()
    for t in range(P + nb - 1):
        busy = 0
        for r in range(P):
            k = lp.lp_stage_block(P, nb, t, r)
            if k >= 0:
                assert k == t - r and (r, k) not in seen
                seen.add((r, k))
                busy += 1
        if P - 1 <= t < nb:
            assert busy == P  # "the entire network is fully utilized once the pipeline is filled"
    assert len(seen) == P * nb
    assert lp.lp_stage_block(P, nb, P + nb - 1, 0) == -1


def test_stage_model_steps_closed_form():
    # pipeline length p - 1 + n/b
    for P in (1, 2, 3, 6, 16):
        for n, b in ((1 << 20, 65_536), (61_000_000, 65_536), (5, 2), (0, 3)):
            nb = -(-n // b)
            for op in (BCAST, REDUCE, ALLREDUCE):
                want = 0 if nb == 0 else P - 1 + nb
                assert lp.lp_schedule_steps(P, n, b, op, lp.MODEL_STAGE) == want


def test_link_model_matches_paper_worked_example():
    # tests/golden/paper_fig2_link_steps.txt: PAPER.md:59,71 (3 GPUs, 4 blocks)
    rows = {(int(P), int(nb), q): int(v) for P, nb, q, v in read_golden("paper_fig2_link_steps.txt")}
    for model in (lp.MODEL_LINK, lp.MODEL_LINK_RING):
        assert lp.lp_schedule_steps(3, 4, 1, REDUCE, model) == rows[(3, 4, "reduce_steps")]
        assert lp.lp_schedule_steps(3, 4, 1, BCAST, model) == rows[(3, 4, "broadcast_steps")]
        assert lp.lp_schedule_steps(3, 4, 1, ALLREDUCE, model) == rows[(3, 4, "allreduce_steps")]


def test_link_model_matches_oracle_simulation(oracle):
    # two independent implementations of the same greedy Fig. 2 schedule
    for P in (2, 3, 4, 6, 8):
        for nb in (1, 2, 4, 8, 16, 33):
            for op in (BCAST, REDUCE, ALLREDUCE):
                assert lp.lp_schedule_steps(P, nb, 1, op, lp.MODEL_LINK) == oracle.link_sim(P, nb, op, 0), (P, nb, op)
                assert lp.lp_schedule_steps(P, nb, 1, op, lp.MODEL_LINK_RING) == oracle.link_sim(P, nb, op, 1), (P, nb, op)
            assert lp.lp_schedule_steps(P, nb, 1, REDUCE, lp.MODEL_LINK) == P + nb - 2  # U2
    assert lp.lp_schedule_steps(1, 100, 1, REDUCE, lp.MODEL_LINK) == 0


def test_mst_levels_match_paper():
    for P, steps in read_golden("paper_mst_steps.txt"):
        assert lp.lp_mst_levels(int(P)) == int(steps)


def test_min_bytes():
    n = 1000
    assert lp.lp_min_bytes(BCAST, 4, n) == 4 * n * 4
    assert lp.lp_min_bytes(REDUCE, 4, n) == 5 * n * 4
    assert lp.lp_min_bytes(ALLREDUCE, 6, n) == 2 * 6 * n * 4
    assert lp.lp_min_bytes(SGD, 8, n) == 17 * n * 4
    assert lp.lp_min_bytes(lp.OP_BSP_SGD_MOM, 8, n) == 19 * n * 4


@pytest.mark.parametrize("variant", [lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT])
@pytest.mark.parametrize("P,n,block", [(4, 1 << 20, 65_536), (6, 61_000_000, 65_536), (6, 61_000_000, 1 << 20),
                                        (16, 138_000_000, 262_144), (3, 1001, 100), (2, 5, 64), (8, 7_000_000, 3000)])
def test_plan_partition_covers_message_exactly(variant, P, n, block):
    # the tile list of the persistent kernel: tiles never straddle a block, cover [0, n) once
    lp.lp_set_variant(variant)
    try:
        info = lp.lp_plan_query(ALLREDUCE, P, n, block)
    finally:
        lp.lp_set_variant(lp.VARIANT_AUTO)
    nb = -(-n // block)
    assert info["nb"] == nb and info["block"] == min(block, n)
    # the pipeline variant counts GRANULES (the unit of a claim; a ring slot holds a run of tile / granule of them)
    tile = info["granule_elems"]
    assert info["tile_elems"] % tile == 0 and info["tile_elems"] // tile in (1, 2, 4, 8)
    if variant == lp.VARIANT_DIRECT:
        assert tile == info["tile_elems"]
    blk = min(block, n)
    tpb = -(-blk // tile)
    last = n - (nb - 1) * blk
    assert info["n_tiles"] == (nb - 1) * tpb + -(-last // tile)
    assert 1 <= info["grid"] <= info["n_tiles"]
    assert 1 <= info["claim_granules"] and info["grid"] * info["claim_granules"] < info["n_tiles"] + info["claim_granules"]
    if variant == lp.VARIANT_PIPELINE:
        assert info["grid"] <= info["sm_count"] * 8     # persistent CTAs
    else:
        assert info["grid"] == info["n_tiles"]           # register variant: one CTA per tile
    assert info["variant"] == variant
    if variant == lp.VARIANT_PIPELINE:  # any block size: tiles that start off a 16-byte boundary get a scalar head / tail
        assert info["smem_bytes"] <= 227 * 1024 and info["stages"] >= 2 and info["out_stages"] >= 1


def test_argument_validation_needs_no_device():
    L = lp.lib()
    n = 64
    raw = [np.zeros(n + 8, np.float32) for _ in range(4)]

    def aligned(a, phase=0):
        off = ((-a.ctypes.data) % 16) // 4
        return a.ctypes.data + 4 * off + phase

    ptrs = (ctypes.c_void_p * 4)(*[aligned(a) for a in raw])
    null_stream = ctypes.c_void_p(0)
    assert L.lp_allreduce(ptrs, 0, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG          # P < 1
    assert L.lp_allreduce(ptrs, 33, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG         # P > LP_MAX_P
    # block == 0 is valid since 0.2.0 ("library chooses"): with good arguments and no device the call gets as far as
    # the device check (test_compute_entry_fails_loudly_without_device); with bad ones it is still refused first
    assert L.lp_allreduce(ptrs, 0, n, 0, null_stream) == lp.LP_ERR_INVALID_ARG
    assert L.lp_reduce_op(ptrs, 4, n, 16, 0, 2, null_stream) == lp.LP_ERR_INVALID_ARG    # unknown reduce operator
    assert L.lp_allreduce_op(ptrs, 4, n, 16, -1, null_stream) == lp.LP_ERR_INVALID_ARG
    assert L.lp_mst_allreduce_op(ptrs, 4, n, 7, null_stream) == lp.LP_ERR_INVALID_ARG
    assert L.lp_be_reduce_op(ptrs, 3, n, 0, 1, null_stream) == lp.LP_ERR_UNSUPPORTED     # U14 holds for every operator
    assert L.lp_reduce(ptrs, 4, n, 16, 4, null_stream) == lp.LP_ERR_INVALID_ARG          # root out of range
    assert L.lp_broadcast(ptrs, 4, n, 16, -1, null_stream) == lp.LP_ERR_INVALID_ARG
    assert L.lp_allreduce(None, 4, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG          # NULL array
    bad = (ctypes.c_void_p * 4)(ptrs[0], None, ptrs[2], ptrs[3])
    assert L.lp_allreduce(bad, 4, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG           # NULL buffer
    mis = (ctypes.c_void_p * 4)(ptrs[0], aligned(raw[1], 4), ptrs[2], ptrs[3])
    assert L.lp_allreduce(mis, 4, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG           # not 16-byte aligned
    ovl = (ctypes.c_void_p * 4)(ptrs[0], ptrs[0] + 16, ptrs[2], ptrs[3])
    assert L.lp_allreduce(ovl, 4, n, 16, null_stream) == lp.LP_ERR_INVALID_ARG           # overlapping
    assert L.lp_be_allreduce(ptrs, 3, n, null_stream) == lp.LP_ERR_UNSUPPORTED           # U14
    assert L.lp_bsp_sgd_step(ptrs, None, 4, n, 16, 0, ctypes.c_float(0.1), null_stream) == lp.LP_ERR_INVALID_ARG
    assert L.lp_set_variant(9) == lp.LP_ERR_INVALID_ARG
    assert L.lp_set_tuning(lp.TUNE_TILE_ELEMS, 1000) == lp.LP_ERR_INVALID_ARG
    out = ctypes.c_uint64(0)
    assert L.lp_schedule_steps(4, n, 0, 0, 0, ctypes.byref(out)) == lp.LP_ERR_INVALID_ARG
    assert L.lp_schedule_steps(4, n, 16, 7, 0, ctypes.byref(out)) == lp.LP_ERR_INVALID_ARG
    for code in (0, 1, 2, 3):
        assert lp.status_string(code)


def test_compute_entry_fails_loudly_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    L = lp.lib()
    raw = [np.zeros(80, np.float32) for _ in range(2)]
    ptrs = (ctypes.c_void_p * 2)(*[a.ctypes.data + ((-a.ctypes.data) % 16) for a in raw])
    # valid arguments, no GPU: the library must refuse (LP_ERR_CUDA), never compute on the CPU
    assert L.lp_allreduce(ptrs, 2, 64, 16, ctypes.c_void_p(0)) == lp.LP_ERR_CUDA
    assert L.lp_allreduce(ptrs, 2, 64, 0, ctypes.c_void_p(0)) == lp.LP_ERR_CUDA        # block == 0: library chooses
    assert L.lp_allreduce_op(ptrs, 2, 64, 16, lp.REDUCE_PROD, ctypes.c_void_p(0)) == lp.LP_ERR_CUDA
    assert L.lp_hbm_probe(ptrs, 1, 1, 64, ctypes.c_void_p(0)) == lp.LP_ERR_CUDA
    plan = lp.Plan(ALLREDUCE, 2, 64)
    with pytest.raises(lp.LpError) as ei:
        L_ = ctypes.c_void_p(0)
        rc = L.lp_plan_run(plan.handle, ptrs, None, None, ctypes.c_float(0), ctypes.c_float(0), L_)
        if rc:
            raise lp.LpError(rc, "lp_plan_run")
    assert ei.value.status == lp.LP_ERR_CUDA
    assert "no CUDA device" in lp.status_string(lp.LP_ERR_CUDA)
    # the typed calls, the typed slice lists and the chain: validation first, then the same refusal
    s0 = ctypes.c_void_p(0)
    for dt in (lp.DT_F16, lp.DT_BF16, lp.DT_F64):
        assert L.lp_allreduce_dt(ptrs, 2, 32, 16, dt, lp.REDUCE_SUM, s0) == lp.LP_ERR_CUDA
        assert L.lp_reduce_dt(ptrs, 2, 32, 16, 1, dt, lp.REDUCE_PROD, s0) == lp.LP_ERR_CUDA
        assert L.lp_broadcast_dt(ptrs, 2, 32, 16, 0, dt, s0) == lp.LP_ERR_CUDA
    assert L.lp_allreduce_dt(ptrs, 2, 32, 16, 9, lp.REDUCE_SUM, s0) == lp.LP_ERR_INVALID_ARG
    assert L.lp_allreduce_dt(ptrs, 2, 32, 16, lp.DT_F64, 9, s0) == lp.LP_ERR_INVALID_ARG
    off = (ctypes.c_size_t * 1)(3)
    ln = (ctypes.c_size_t * 1)(8)
    assert L.lp_allreduce_segments_dt(ptrs, 2, 32, off, ln, 1, 16, lp.DT_F16, lp.REDUCE_SUM, s0) == lp.LP_ERR_INVALID_ARG
    off[0] = 4
    assert L.lp_allreduce_segments_dt(ptrs, 2, 32, off, ln, 1, 16, lp.DT_F16, lp.REDUCE_SUM, s0) == lp.LP_ERR_CUDA
    assert L.lp_chain_emulate(ALLREDUCE, ptrs, 2, 64, 16, 0, lp.REDUCE_SUM, 2, 2, 4096, s0) in (lp.LP_ERR_CUDA, lp.LP_ERR_UNSUPPORTED)
    assert lp.lp_dtype_size(lp.DT_F32) == 4 and lp.lp_dtype_size(lp.DT_BF16) == 2 and lp.lp_dtype_size(-1) == 0
    assert not raw[0].any() and not raw[1].any()


def test_plan_validation_and_info_need_no_device():
    # a plan carries its own variant and tuning; creating and querying it is host-only
    with pytest.raises(lp.LpError):
        lp.Plan(9, 4, 1000)                                           # unknown collective
    with pytest.raises(lp.LpError):
        lp.Plan(ALLREDUCE, 0, 1000)
    with pytest.raises(lp.LpError):
        lp.Plan(REDUCE, 4, 1000, root=4)
    with pytest.raises(lp.LpError):
        lp.Plan(ALLREDUCE, 4, 1000, reduce_op=5)
    with pytest.raises(lp.LpError):
        lp.Plan(lp.OP_BSP_SGD, 4, 1000, reduce_op=lp.REDUCE_PROD)     # the SGD steps average: sum only
    with pytest.raises(lp.LpError):
        lp.Plan(ALLREDUCE, 4, 1000, tuning={lp.TUNE_TILE_ELEMS: 1000})
    with pytest.raises(lp.LpError) as ei:
        lp.Plan(ALLREDUCE, 17, 1000, variant=lp.VARIANT_CLUSTER)
    assert ei.value.status == lp.LP_ERR_UNSUPPORTED
    n = 61_000_000
    free = lp.Plan(ALLREDUCE, 6, n, block=65_536)
    conf = lp.Plan(ALLREDUCE, 6, n, block=65_536, tuning={lp.TUNE_GRID_LIMIT: 64})
    a, b = free.info(), conf.info()
    assert a["variant"] == lp.VARIANT_PIPELINE and a["grid"] == 2 * a["sm_count"]
    assert b["variant"] == lp.VARIANT_PIPELINE and b["grid"] == 64 and b["tile_elems"] == 4096
    # the process-wide defaults are untouched by either plan
    assert lp.lp_get_tuning(lp.TUNE_GRID_LIMIT) == 0 and lp.lp_get_variant() == lp.VARIANT_AUTO
    d = lp.Plan(ALLREDUCE, 6, n, variant=lp.VARIANT_DIRECT).info()
    assert d["variant"] == lp.VARIANT_DIRECT and d["block"] == lp.DEFAULT_BLOCK      # block 0 -> LP_DEFAULT_BLOCK


def test_auto_block():
    # block == 0: LP_DEFAULT_BLOCK for the persistent kernels (flat in block), the fitted model's optimum for the
    # copy-engine variant (PAPER.md:81-89 with the B200 constants, profiles/r2_cost_model_fit.md)
    n = 61_000_000
    for v in (lp.VARIANT_AUTO, lp.VARIANT_PIPELINE, lp.VARIANT_DIRECT, lp.VARIANT_CLUSTER):
        assert lp.lp_auto_block(ALLREDUCE, 6, n, v) == lp.DEFAULT_BLOCK
        assert lp.lp_auto_block(ALLREDUCE, 6, 1000, v) == 1000                      # clamped to n
    alpha, beta = lp.lp_fitted_constants(6)
    assert 1e-6 < alpha < 1e-4 and 1e-13 < beta < 1e-11
    a2, b2 = lp.lp_fitted_constants(2)
    assert a2 == pytest.approx(alpha / 5, rel=1e-12) and b2 == beta       # alpha grows with the hops, beta does not
    for op in (BCAST, REDUCE, ALLREDUCE):
        for P in (2, 6, 16):
            alpha, beta = lp.lp_fitted_constants(P)
            b = lp.lp_auto_block(op, P, n, lp.VARIANT_COPY_ENGINE)
            want = lp.lp_optimal_block(op, P, n * 4.0, alpha, beta, 0.0) / 4.0
            assert b % 4 == 0 and 4 <= b <= n and abs(b - want) <= 4, (op, P, b, want)
            # and it does minimise the fitted model over the block sizes a caller might try
            cost = lambda blk: lp.lp_cost_model(lp.ALGO_LP, op, P, n * 4.0, blk * 4.0, alpha, beta, 0.0)  # noqa: E731
            assert all(cost(b) <= cost(x) * (1 + 1e-9) for x in (16_384, 65_536, 1 << 20, 1 << 22, 1 << 24, n))
    assert lp.lp_auto_block(ALLREDUCE, 6, n, lp.VARIANT_COPY_ENGINE) > 100 * 16_384   # far from the paper's 64 KB
    assert lp.lp_auto_block(ALLREDUCE, 1, n, lp.VARIANT_COPY_ENGINE) == n
    assert lp.lp_auto_block(7, 6, n, lp.VARIANT_AUTO) == 0 and lp.lp_auto_block(ALLREDUCE, 0, n, lp.VARIANT_AUTO) == 0
    info = lp.Plan(ALLREDUCE, 6, n, variant=lp.VARIANT_COPY_ENGINE).info()
    assert info["block"] == lp.lp_auto_block(ALLREDUCE, 6, n, lp.VARIANT_COPY_ENGINE)


# ---- cost model of Sec. 3.2 (host only) --------------------------------------------------------------------
def test_cost_model_matches_oracle_table1():
    # the library's Table 1 (own code) against the oracle's, over a grid of p, n, b, alpha, beta, gamma
    from oracle import lpo
    for algo in (lp.ALGO_LP, lp.ALGO_MST, lp.ALGO_BE):
        for op in (BCAST, REDUCE, ALLREDUCE):
            for p in (2, 3, 6, 8, 16):
                for n in (4096.0, 2.44e8, 5.5e8):
                    for b in (4096.0, 65536.0, 1.0e6):
                        for alpha, beta, gamma in ((1e-7, 1e-9, 0.0), (3e-6, 1.5e-13, 2e-14), (0.0, 1e-9, 1e-10)):
                            got = lp.lp_cost_model(algo, op, p, n, b, alpha, beta, gamma)
                            want = lpo.cost(algo, op, p, n, b, alpha, beta, gamma)
                            assert got == pytest.approx(want, rel=1e-12), (algo, op, p, n, b)
    assert lp.lp_cost_model(lp.ALGO_LP, BCAST, 4, 1e6, 0.0, 1e-7, 1e-9) == -1.0      # LP needs a block size
    assert lp.lp_cost_model(7, BCAST, 4, 1e6, 1e4, 1e-7, 1e-9) == -1.0


def test_optimal_block_minimises_the_lp_cost():
    # b* against a brute-force scan of the ORACLE's cost function; and the paper's own numbers: alpha = 1e-7 s,
    # beta = 1e-9 s/byte, AlexNet-sized 244 MB message on 6 GPUs -> tens of KB ("around 64 KB")
    from oracle import lpo
    for op in (BCAST, REDUCE, ALLREDUCE):
        for p, n, alpha, beta, gamma in ((6, 2.44e8, 1e-7, 1e-9, 0.0), (16, 5.52e8, 2.5e-6, 1.4e-13, 1e-14),
                                         (2, 1e6, 1e-6, 1e-10, 1e-10)):
            b_star = lp.lp_optimal_block(op, p, n, alpha, beta, gamma)
            scan = np.geomspace(64.0, n, 4000)
            costs = [lpo.cost(0, op, p, n, b, alpha, beta, gamma) for b in scan]
            best = scan[int(np.argmin(costs))]
            assert abs(np.log(b_star / best)) < 0.01, (op, p, b_star, best)
            assert lpo.cost(0, op, p, n, b_star, alpha, beta, gamma) <= min(costs) * (1 + 1e-9)
    b = lp.lp_optimal_block(BCAST, 6, 2.44e8, 1e-7, 1e-9)
    assert 32e3 < b < 128e3                                   # sqrt(2.44e8 * 1e-7 / (5 * 1e-9)) = 69.9 KB
    assert lp.lp_optimal_block(BCAST, 1, 1e6, 1e-7, 1e-9) == 1e6
    assert lp.lp_optimal_block(BCAST, 4, 1e6, 0.0, 1e-9) == 1e6


def test_auto_variant_resolution():
    # LP_VARIANT_AUTO (the default): register kernel up to ~2 GB of HBM traffic per call (~650 MB for a reduce over
    # >= 4 ranks, never the pipeline for a 2-rank reduce), TMA pipeline above and whenever the grid is confined
    assert lp.lp_get_variant() == lp.VARIANT_AUTO
    small = lp.lp_plan_query(ALLREDUCE, 4, 1 << 20, 65_536)          # 32 MB of traffic
    big = lp.lp_plan_query(ALLREDUCE, 6, 61_000_000, 65_536)         # 2.9 GB
    assert small["variant"] == lp.VARIANT_DIRECT and small["grid"] == small["n_tiles"]
    assert big["variant"] == lp.VARIANT_PIPELINE and big["grid"] == 2 * big["sm_count"]
    assert lp.lp_plan_query(ALLREDUCE, 8, 1 << 24, 65_536)["variant"] == lp.VARIANT_DIRECT     # 1 GB
    assert lp.lp_plan_query(ALLREDUCE, 16, 1 << 24, 65_536)["variant"] == lp.VARIANT_PIPELINE  # 2 GB
    assert lp.lp_plan_query(BCAST, 2, 1 << 27, 65_536)["variant"] == lp.VARIANT_DIRECT         # 1 GB of copy traffic
    assert lp.lp_plan_query(BCAST, 16, 1 << 25, 65_536)["variant"] == lp.VARIANT_PIPELINE      # 2 GB
    assert lp.lp_plan_query(REDUCE, 2, 1 << 27, 65_536)["variant"] == lp.VARIANT_DIRECT        # 2 ranks: always
    assert lp.lp_plan_query(REDUCE, 4, 1 << 24, 65_536)["variant"] == lp.VARIANT_DIRECT        # 320 MB
    assert lp.lp_plan_query(REDUCE, 4, 1 << 25, 65_536)["variant"] == lp.VARIANT_DIRECT        # 640 MB
    assert lp.lp_plan_query(REDUCE, 8, 1 << 25, 65_536)["variant"] == lp.VARIANT_PIPELINE      # 1.1 GB
    assert lp.lp_plan_query(lp.OP_BSP_SGD, 8, 7_000_000, 65_536)["variant"] == lp.VARIANT_DIRECT   # configs[2]: 476 MB
    # the register kernel's tile follows the number of input streams; a broadcast to many ranks is capped in CTAs per SM
    assert lp.lp_plan_query(BCAST, 2, 1 << 24, 65_536)["tile_elems"] == 2048  # one-destination copy: 8 CTAs x 8 KB (profiles/r2_tuning.md 2b)
    assert lp.lp_plan_query(REDUCE, 2, 1 << 24, 65_536)["tile_elems"] == 4096
    assert lp.lp_plan_query(ALLREDUCE, 6, 1 << 24, 65_536)["tile_elems"] == 2048
    assert lp.lp_plan_query(ALLREDUCE, 16, 1 << 22, 65_536)["tile_elems"] == 1024
    assert lp.lp_plan_query(BCAST, 8, 1 << 24, 65_536)["smem_bytes"] > 48 * 1024                # occupancy cap of 3 CTAs
    assert lp.lp_plan_query(BCAST, 3, 1 << 24, 65_536)["smem_bytes"] == 0
    try:
        lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, 32)
        conf = lp.lp_plan_query(ALLREDUCE, 4, 1 << 20, 65_536)
        assert conf["variant"] == lp.VARIANT_PIPELINE and conf["grid"] <= 32
    finally:
        lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, 0)
