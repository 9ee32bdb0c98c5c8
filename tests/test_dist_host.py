"""N > 1 host logic of bench.py on CPU: world_size-2 gloo.  The path does not shard (DESIGN.md "Multi-GPU":
replicas only, no data-path collective), so what N > 1 adds is plumbing: rendezvous, barrier, max-over-ranks
timing, whole-job aggregation, rank-0-only output."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

from tests.conftest import ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r, w, local = bench.dist_setup(world)
    assert (r, w, local) == (rank, world, rank)
    bench.barrier(w)
    slowest = bench.max_over_ranks(10.0 + rank, w)       # rank 1 is the slow one
    total = bench.sum_over_ranks(100.0 * (rank + 1), w)
    bench.barrier(w)
    import torch.distributed as dist
    dist.destroy_process_group()
    q.put((rank, slowest, total))


def test_gloo_world2_max_and_sum_over_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, 11.0, 300.0), (1, 11.0, 300.0)]


class _FakeEndpoint:
    """Stand-in for binding.Chain on the CPU box (no CUDA IPC there): its handle is 64 bytes that name its rank."""
    def __init__(self, rank, P, channels, slots, tile):
        self.rank, self.P, self.connected = rank, P, None
        self.events = []

    def handle(self):
        return bytes([self.rank]) * 64

    def connect(self, handles):
        self.connected = list(handles)

    def disconnect(self):
        self.events.append("disconnect")

    def destroy(self):
        self.events.append("destroy")


def _chain_worker(rank, world, port, q):
    """One rank of the chain with gloo as the link: the per-rank steps csrc/lp_chain.cu takes (lp_chain_plan's roles),
    one message per tile and ring, fp32 numpy adds -- the multi-process path of the chain on the CPU."""
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1611_04255_b200 import binding as lp
    from paper_1611_04255_b200 import chain, inputs
    dist.init_process_group("gloo", rank=rank, world_size=world)
    grp = chain.ChainGroup(endpoint_factory=_FakeEndpoint)
    ok_handles = grp.endpoint.connected == [bytes([r]) * 64 for r in range(world)]
    n, tile = 10_003, 4096
    results = {}
    for op, root in ((lp.OP_ALLREDUCE, 0), (lp.OP_REDUCE, 0), (lp.OP_REDUCE, 1), (lp.OP_BROADCAST, 1)):
        ro = grp.role(op, root)
        x = inputs.uniform([41, 0], rank, n).copy()
        for off in range(0, n, tile):                      # tiles in order, one channel
            sl = slice(off, min(off + tile, n))
            if ro["f_active"]:
                v = x[sl].copy() if ro["f_load"] else None
                if ro["f_recv"]:
                    t = torch.empty(sl.stop - sl.start, dtype=torch.float32)
                    dist.recv(t, src=ro["down"])
                    v = (t.numpy() + v) if ro["f_load"] else t.numpy().copy()     # partial + mine, fp32 RN
                if ro["f_send_up"]:
                    dist.send(torch.from_numpy(v.copy()), dst=ro["up"])
                if ro["f_store"]:
                    x[sl] = v
                if ro["f_send_down"]:
                    dist.send(torch.from_numpy(v.copy()), dst=ro["down"])
            if ro["r_active"]:
                t = torch.empty(sl.stop - sl.start, dtype=torch.float32)
                dist.recv(t, src=ro["up"])
                if ro["r_store"]:
                    x[sl] = t.numpy()
                if ro["r_send_down"]:
                    dist.send(t, dst=ro["down"])
        results[(op, root)] = x.tobytes()
    dist.barrier()
    ep = grp.endpoint
    grp.destroy()      # sync, barrier, unmap the neighbours, barrier, free: never a free before every mapping is closed
    ok_handles = ok_handles and ep.events == ["disconnect", "destroy"]
    dist.destroy_process_group()
    q.put((rank, ok_handles, results))


def test_gloo_world2_chain_handles_and_roles(oracle):
    import numpy as np
    from paper_1611_04255_b200 import binding as lp
    from paper_1611_04255_b200 import inputs
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_chain_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in got), "every rank must see every rank's handle, in rank order"
    n = 10_003
    src = [inputs.uniform([41, 0], r, n) for r in range(2)]
    for (op, root), name in (((lp.OP_ALLREDUCE, 0), "allreduce"), ((lp.OP_REDUCE, 0), "reduce"),
                             ((lp.OP_REDUCE, 1), "reduce"), ((lp.OP_BROADCAST, 1), "broadcast")):
        want = [a.copy() for a in src]
        if name == "allreduce":
            oracle.allreduce(want)
        elif name == "reduce":
            oracle.reduce(want, root=root)
        else:
            oracle.broadcast(want, root=root)
        for r in range(2):
            assert got[r][2][(op, root)] == want[r].tobytes(), (name, root, r)


def test_reference_arm_under_torchrun_prints_once():
    # --impl reference with N = 2: rank 0 alone runs the oracle and prints the line, rank 1 exits 0 silently
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus",
           "2", "--steps", "1", "--warmup", "1", "--config", "1"]
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(ln) for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    # the last stdout line is the headline, and its config has exactly the keys of our arm's
    assert json.loads(out.stdout.strip().splitlines()[-1]) == line
    assert sorted(line["config"]) == ["P", "block", "n", "workload"] and line["config"]["block"] == 65_536


def test_default_workload_is_the_largest_single_gpu_config():
    sys.path.insert(0, ROOT)
    import bench
    old = sys.argv
    sys.argv = ["bench.py"]
    try:
        args = bench.parse_args()
    finally:
        sys.argv = old
    assert args.config == 4
    c = bench.workload(args.config)
    assert (c["P"], c["n"], c["block"]) == (16, 138_000_000, 262_144)
    c = bench.workload(1)
    assert (c["P"], c["n"]) == (6, 61_000_000)
    assert bench.headline_config(4, bench.workload(4), 262_144) == {
        "workload": "BASELINE.json configs[4]: cfg4_P16_vgg16_138M", "P": 16, "n": 138_000_000, "block": 262_144}


def test_headline_line_stays_small():
    """Round 2's single 50 KB line was lost by the driver: the headline must stay a few KB whatever the sections return."""
    sys.path.insert(0, ROOT)
    import bench
    summary = {}
    row = {"lp_us_unchained": 427.1, "lp_frac_8TBs_unchained": 0.8531}
    bench.summarise("configs1", {"allreduce": row}, summary)
    bench.summarise("configs4", {op: row for op in ("allreduce", "reduce", "broadcast")}, summary)
    bench.summarise("configs2", {"lp_bsp_sgd_step": {"us_per_step": 71.5, "frac_8TBs": 0.83}}, summary)
    bench.summarise("sweep", {"summary": {"cells": 84, "lp_min_frac_8TBs": 0.81, "lp_min_frac_8TBs_unchained": 0.81,
                                          "lp_cells_below_0.80_of_8TBs_unchained": ["x"] * 84, "lp_min_vs_mst": 1.0,
                                          "lp_min_vs_be": 1.0}}, summary)
    bench.summarise("sweep_small", {"summary": {"cells": 168, "cells_where_lp_is_not_fastest": 3,
                                                "crossover": {f"allreduce_P{p}": "MST/BE faster up to 64 KB" for p in (2, 4, 8, 16)}}},
                    summary)
    assert len(summary) <= 16
    assert len(bench.compact({"summary": summary})) < 1500
    with pytest.raises(SystemExit):
        bench.workload(3)   # the sweep config is not a single bench workload
