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


def test_reference_arm_under_torchrun_prints_once():
    # --impl reference with N = 2: rank 0 alone runs the oracle and prints the line, rank 1 exits 0 silently
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus",
           "2", "--steps", "1", "--warmup", "1"]
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(ln) for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_default_workload_is_baseline_config1():
    sys.path.insert(0, ROOT)
    import bench
    c = bench.workload(1)
    assert (c["P"], c["n"]) == (6, 61_000_000)
    with pytest.raises(SystemExit):
        bench.workload(3)   # the sweep config is not a single bench workload
