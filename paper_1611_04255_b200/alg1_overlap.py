"""Alg. 1 of the paper on one B200: layer-wise non-blocking allreduce overlapped with the backward computation.

    python -m paper_1611_04255_b200.alg1_overlap --out gpurun_out/alg1_overlap [--P 6] [--ratios 0.5,1,2]

PAPER.md:117-138 (Alg. 1) and PAPER.md:182: "GPUs all-reduce or reduce sub-gradients of layer t+1 amidst backward
computations at layer t.  As a result, layer-wise computations partially overlap with communications"; PAPER.md:192
puts the cost of an iteration at max(comm, compt) instead of comm + compt.  This script measures exactly that claim
for the LP allreduce of this library:

  * the message list is an AlexNet-shaped layer list (8 weight tensors, 60,965,224 parameters: BASELINE.json
    configs[1]'s 61 M vector cut at layer boundaries), P virtual ranks, gradients N(0, 1e-3) from seed [1, r];
  * "Backward(i)" is a stand-in: a chain of bf16 matmuls (cuBLAS through torch: compute-bound, real SM / shared-memory
    contention with the collective) or a single-thread spin (`--compute spin`: no contention, the mechanism alone),
    sized so that the whole backward pass takes `ratio` x the time of the layer-wise allreduce alone, 90 % of it in
    the five convolution layers (which hold 4 % of the parameters) as in AlexNet;
  * modes: comm alone, compute alone, serial (Backward(i) then allreduce(i) on one stream: comm + compt) and
    overlapped (Alg. 1: lp_comm_after / lp_allreduce_segments on the comm stream / lp_comm_wait), for several
    LP_TUNE_GRID_LIMIT values (how many persistent CTAs the collective may take from the compute kernels).

Timing: CUDA events on the compute stream around one whole backward pass, median of 5, gradients restored outside the
timed region.  Writes <out>.jsonl and <out>.md.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

from . import binding as lp
from . import inputs

# AlexNet weight tensors (parameter counts incl. biases), forward order; backward visits them in reverse.
LAYERS = [("conv1", 34_944), ("conv2", 307_456), ("conv3", 885_120), ("conv4", 663_936), ("conv5", 442_624),
          ("fc6", 37_752_832), ("fc7", 16_781_312), ("fc8", 4_097_000)]
COMPUTE_SHARE = {"conv1": 0.18, "conv2": 0.18, "conv3": 0.18, "conv4": 0.18, "conv5": 0.18,
                 "fc6": 0.05, "fc7": 0.03, "fc8": 0.02}


def layer_slices():
    off, out = 0, []
    for name, count in LAYERS:
        out.append((name, off, count))
        off += count
    return out, off


def main(argv=None):
    import torch

    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/alg1_overlap")
    ap.add_argument("--P", type=int, default=6)
    ap.add_argument("--block", type=int, default=65_536)
    ap.add_argument("--ratios", default="0.5,1,2")
    ap.add_argument("--limits", default="0,64,32,16")
    ap.add_argument("--compute", default="matmul,spin")
    ap.add_argument("--mode", default="allreduce", choices=["allreduce", "sgd", "broadcast"],
                    help="allreduce: backward pass, layer-wise allreduce of the gradients (default); sgd: backward "
                         "pass, layer-wise fused BSP-SGD step (lp_bsp_sgd_step_segments); broadcast: forward pass, "
                         "layer-wise broadcast of the weights from rank 0 (Alg. 1 lines 2-6)")
    args = ap.parse_args(argv)
    assert torch.cuda.is_available(), "needs a CUDA device"
    dev = torch.device("cuda", 0)
    lp.lib()
    P = args.P
    slices, n = layer_slices()
    pristine = [torch.from_numpy(inputs.normal(1, r, n, 1e-3)).to(dev) for r in range(P)]
    grads = [torch.empty_like(p) for p in pristine]
    ranks = lp.Ranks(grads)
    segs = {name: lp.Segments([(off, cnt)]) for name, off, cnt in slices}
    comm = lp.Comm()
    compute = torch.cuda.Stream()
    back = list(reversed(slices)) if args.mode != "broadcast" else list(slices)  # backward: fc8 ... conv1; forward: conv1 ... fc8
    op = {"allreduce": lp.OP_ALLREDUCE, "sgd": lp.OP_BSP_SGD, "broadcast": lp.OP_BROADCAST}[args.mode]
    min_bytes = lp.lp_min_bytes(op, P, n)
    weights = lp.Ranks([torch.from_numpy(inputs.normal(1, 100, n, 0.05)).to(dev) for _ in range(P)]) if args.mode == "sgd" else None

    def collective(name, stream):
        if args.mode == "allreduce":
            lp.lp_allreduce_segments(ranks, segs[name], args.block, stream=stream)
        elif args.mode == "sgd":
            lp.lp_bsp_sgd_step_segments(ranks, weights, segs[name], args.block, root=0, lr=0.01, stream=stream)
        else:
            lp.lp_broadcast_segments(ranks, segs[name], args.block, root=0, stream=stream)

    a = torch.randn(2048, 2048, device=dev, dtype=torch.bfloat16)
    b = torch.randn(2048, 2048, device=dev, dtype=torch.bfloat16)
    c = torch.empty_like(a)

    def restore():
        for g, p in zip(grads, pristine):
            g.copy_(p)

    def timed(fn, reps=5):
        ms = []
        for it in range(reps + 1):
            restore()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(compute):
                e0.record()
                fn()
                e1.record()
            torch.cuda.synchronize()
            if it:
                ms.append(e0.elapsed_time(e1))
        return float(np.median(ms))

    def comm_only():
        for name, _, _ in back:
            collective(name, compute)

    def unit_ms(kind):
        """Milliseconds of one unit of the compute stand-in (one matmul / 100k spin cycles)."""
        def run():
            for _ in range(50):
                if kind == "matmul":
                    torch.matmul(a, b, out=c)
                else:
                    torch.cuda._sleep(100_000)
        return timed(run, reps=3) / 50

    rows = []
    lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, 0)
    t_comm_full = timed(comm_only)
    for kind in args.compute.split(","):
        u = unit_ms(kind)
        for ratio in [float(x) for x in args.ratios.split(",")]:
            units = {name: max(1, int(round(ratio * t_comm_full * COMPUTE_SHARE[name] / u))) for name, _ in LAYERS}

            def backward(name):
                for _ in range(units[name]):
                    if kind == "matmul":
                        torch.matmul(a, b, out=c)
                    else:
                        torch.cuda._sleep(100_000)

            def compute_only():
                for name, _, _ in back:
                    backward(name)

            def serial():
                for name, _, _ in back:
                    backward(name)
                    collective(name, compute)

            def overlapped():
                if args.mode == "broadcast":            # Alg. 1 lines 1-6: broadcast(w^0); nonblocking_broadcast(w^{i+1}); Forward(i)
                    comm.after(compute)
                    collective(back[0][0], comm.stream)
                    for i, (name, _, _) in enumerate(back):
                        comm.wait(compute)              # layer i's weights have arrived
                        if i + 1 < len(back):
                            collective(back[i + 1][0], comm.stream)
                        backward(name)                  # Forward(i) on the compute stream
                    return
                for name, _, _ in back:
                    backward(name)                      # Backward(i) on the compute stream
                    comm.after(compute)                 # its gradient is ready: nonblocking_allreduce(layer i)
                    collective(name, comm.stream)
                comm.wait(compute)                      # sync_reduce()

            t_comp = timed(compute_only)
            for limit in [int(x) for x in args.limits.split(",")]:
                lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, limit)
                t_comm = timed(comm_only)
                t_ser = timed(serial)
                t_ovl = timed(overlapped)
                row = dict(mode=args.mode, compute=kind, ratio=ratio, grid_limit=limit, P=P, n=n, layers=len(LAYERS),
                           comm_ms=round(t_comm, 4), compute_ms=round(t_comp, 4), serial_ms=round(t_ser, 4),
                           overlapped_ms=round(t_ovl, 4), max_ms=round(max(t_comm, t_comp), 4),
                           sum_ms=round(t_comm + t_comp, 4),
                           hidden_frac=round((t_ser - t_ovl) / min(t_comm, t_comp), 3),
                           comm_GBps=round(min_bytes / t_comm / 1e6, 0))
                rows.append(row)
                print(json.dumps(row), flush=True)
            lp.lp_set_tuning(lp.TUNE_GRID_LIMIT, 0)
    comm.close()
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out + ".jsonl", "w") as f:
        for r in rows:
            f.write(json.dumps(r) + "\n")
    with open(args.out + ".md", "w") as f:
        f.write("# Alg. 1 on one B200: layer-wise LP allreduce overlapped with the backward computation\n\n")
        f.write(f"Command: `python -m paper_1611_04255_b200.alg1_overlap --out {args.out} --P {P} --block {args.block} "
                f"--ratios {args.ratios} --limits {args.limits} --compute {args.compute} --mode {args.mode}`\n\n")
        f.write(f"AlexNet-shaped layer list ({len(LAYERS)} messages, {n:,} fp32 per rank), P={P} virtual ranks; one "
                f"`{ {'allreduce': 'lp_allreduce_segments', 'sgd': 'lp_bsp_sgd_step_segments', 'broadcast': 'lp_broadcast_segments'}[args.mode] }` "
                f"per layer in {'forward' if args.mode == 'broadcast' else 'backward'} order.  PAPER.md:192: the overlapped iteration should cost "
                "max(comm, compt), the serial one comm + compt.  `hidden` = (serial - overlapped) / min(comm, compt): "
                "the fraction of the shorter of the two that the overlap hides.  grid limit 0 = the collective takes "
                "its usual 2 CTAs on every SM.\n\n")
        f.write("| compute | compt/comm | grid limit | comm ms (GB/s) | compt ms | serial ms | overlapped ms | max | sum | hidden |\n")
        f.write("|---|---|---|---|---|---|---|---|---|---|\n")
        for r in rows:
            f.write(f"| {r['compute']} | {r['ratio']} | {r['grid_limit']} | {r['comm_ms']:.3f} ({r['comm_GBps']:.0f}) | "
                    f"{r['compute_ms']:.3f} | {r['serial_ms']:.3f} | {r['overlapped_ms']:.3f} | {r['max_ms']:.3f} | "
                    f"{r['sum_ms']:.3f} | {r['hidden_frac']:.2f} |\n")


if __name__ == "__main__":
    sys.exit(main())
