"""The real chain across PROCESSES: every rank is a process of its own with a
real ChainGroup -- lp_chain_create, cudaIpcGetMemHandle, all-gather of the handles over torch.distributed (gloo),
cudaIpcOpenMemHandle of the two neighbours' endpoints -- and the per-rank launches a multi-GPU job makes.  The box has one
GPU, so all ranks live on cuda:0 (CUDA IPC works between processes on one device) and two chain kernels must never have
to wait for one another: only collectives whose data flows one way are run, rank after rank in chain order with a
process barrier between the ranks, and rings that never wrap within a call (tiles per channel <= slots), exactly as
tests/test_gpu_3_chain.py::test_chain_real_entry_points_rank_after_rank does inside one process.  What this adds is the
handle exchange and the peer mappings: pushes and credits really cross a process boundary.  Results byte-equal to the oracle.
"""
import multiprocessing as mp
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

CALLS = [("broadcast", 0), ("reduce", -1), ("broadcast", 1), ("reduce", -1), ("broadcast", -1), ("broadcast", 0)]
N, TILE, CHANNELS, SLOTS = 50_001, 4096, 2, 8          # 13 tiles over 2 channels: 7 <= 8 slots, no ring wraps in a call


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _rank_process(rank, world, port, q):
    try:
        os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK="0", MASTER_ADDR="127.0.0.1",
                          MASTER_PORT=str(port))
        sys.path.insert(0, ROOT)
        import torch
        import torch.distributed as dist
        from paper_1611_04255_b200 import binding as lp
        from paper_1611_04255_b200 import chain, inputs
        torch.cuda.set_device(0)
        dist.init_process_group(backend="gloo", rank=rank, world_size=world)
        grp = chain.ChainGroup(channels=CHANNELS, slots=SLOTS, tile=TILE)     # real endpoints, real IPC handles
        grp.endpoint.set_timeout(1 << 22)                                     # a bug must not hang the GPU lease
        ops = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE}
        x = torch.from_numpy(inputs.uniform([43, world], rank, N)).cuda()
        for op, root in CALLS:
            root = root % world                                               # -1: the chain's last rank
            order = [(root + j) % world for j in range(world)] if op == "broadcast" else list(range(world))
            for r in order:                                                   # rank after rank, nothing runs beside anything
                if r == rank:
                    if op == "broadcast":
                        grp.broadcast(x, root=root, block=TILE)
                    else:
                        grp.reduce(x, root=root, block=TILE)
                    torch.cuda.synchronize()
                dist.barrier()
        err = grp.error()
        out = x.cpu().numpy().tobytes()
        grp.destroy()                                                         # sync, barrier, unmap, barrier, free
        dist.destroy_process_group()
        q.put((rank, err, out, None))
    except Exception as exc:  # noqa: BLE001
        q.put((rank, -1, b"", f"{type(exc).__name__}: {exc}"))


@pytest.mark.parametrize("world", [2, 3])
def test_chain_across_processes_on_one_gpu(oracle, world):
    import numpy as np
    from paper_1611_04255_b200 import inputs
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_process, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        got = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    assert all(e is None for _, _, _, e in got), [e for _, _, _, e in got]
    assert all(p.exitcode == 0 for p in procs)
    host = [inputs.uniform([43, world], r, N).copy() for r in range(world)]
    for op, root in CALLS:
        root = root % world
        if op == "broadcast":
            oracle.broadcast(host, root=root)
        else:
            oracle.reduce(host, root=root)
    for r, err, out, _ in got:
        assert err == 0, (r, "a wait of the chain gave up")
        assert out == host[r].tobytes(), (world, r, int(np.count_nonzero(np.frombuffer(out, np.float32) != host[r])))
