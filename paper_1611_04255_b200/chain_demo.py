"""The LP chain on a machine with >= 2 GPUs (one process per GPU):

    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port 29511 \\
        -m paper_1611_04255_b200.chain_demo [--mb 256] [--iters 20]

Every rank allreduces, reduces and broadcasts a vector through ``ChainGroup`` (csrc/lp_chain.cu: pushes into the
neighbours' rings over NVLink, no NCCL on the data path), checks the bits against what the chain order defines --
``((x0 + x1) + x2) + ...`` computed from an all-gather of the inputs -- runs the fused BSP-SGD step, and rank 0 prints one
JSON line with the device-timed throughput (max over ranks).  This build's box has ONE GPU: there the script runs with
N = 1 only (every collective is then the identity); the chain's device code is covered by ``lp_chain_emulate`` in
tests/test_gpu_3_chain.py.  NOT part of bench.py: north_star's hot path has no inter-GPU collective.
"""
from __future__ import annotations

import argparse
import json
import os


def main():
    import torch
    import torch.distributed as dist
    from . import binding as lp
    from .chain import ChainGroup

    ap = argparse.ArgumentParser()
    ap.add_argument("--mb", type=int, default=256, help="message size per rank in MB (fp32)")
    ap.add_argument("--iters", type=int, default=20)
    ap.add_argument("--channels", type=int, default=0)
    ap.add_argument("--slots", type=int, default=0)
    ap.add_argument("--tile", type=int, default=0)
    args = ap.parse_args()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rank, world = dist.get_rank(), dist.get_world_size()
    grp = ChainGroup(channels=args.channels, slots=args.slots, tile=args.tile)
    n = (args.mb << 20) // 4 + 3
    gen = torch.Generator(device="cuda").manual_seed(1234 + rank)
    x = torch.rand(n, device="cuda", generator=gen) * 2 - 1
    everyone = [torch.empty_like(x) for _ in range(world)]
    dist.all_gather(everyone, x)
    want = everyone[0].clone()
    for r in range(1, world):
        want = want + everyone[r]                       # fp32 RN adds in rank order: the chain's definition (U4)
    checks = {}
    y = x.clone()
    grp.allreduce(y)
    checks["allreduce"] = bool(torch.equal(y, want))
    y = x.clone()
    grp.reduce(y, root=world // 2)
    checks["reduce"] = bool(torch.equal(y, want if rank == world // 2 else x))
    y = x.clone()
    grp.broadcast(y, root=world - 1)
    checks["broadcast"] = bool(torch.equal(y, everyone[world - 1]))
    w = torch.full((n,), 0.5, device="cuda")
    grp.bsp_sgd_step(x, w, lr=0.01)
    inv = torch.ones((), device="cuda") / world            # fl32(1 / P), one RN division (U7)
    checks["bsp_sgd_step"] = bool(torch.equal(w, torch.full((n,), 0.5, device="cuda") - (want * inv) * 0.01))
    times = {}
    for name, fn in (("allreduce", lambda: grp.allreduce(y)), ("broadcast", lambda: grp.broadcast(y, root=0))):
        fn()
        dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.iters):
            fn()
        e1.record()
        torch.cuda.synchronize()
        t = torch.tensor([e0.elapsed_time(e1) / args.iters], device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        times[name] = float(t.item())
    ok = torch.tensor([int(all(checks.values()) and grp.error() == 0)], device="cuda")
    dist.all_reduce(ok, op=dist.ReduceOp.MIN)
    if rank == 0:
        print(json.dumps({"world": world, "msg_MB": n * 4 / 2 ** 20, "bit_exact_on_every_rank": bool(ok.item()),
                          "checks_rank0": checks,
                          "ms": times, "algbw_GBps": {k: n * 4 / v / 1e6 for k, v in times.items()}}), flush=True)
    grp.destroy()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
