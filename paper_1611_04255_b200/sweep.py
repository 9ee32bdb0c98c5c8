"""Message-size sweep of BASELINE.json configs[3] (the shape of the paper's Fig. 3 / Fig. 4):
n = 2^10 .. 2^27 fp32 (4 KB .. 512 MB per rank), P in {2, 4, 8, 16} (plus the paper's own 3, 5, 6 by default),
broadcast / reduce / allreduce, LP vs MST (binomial tree) vs BE (recursive halving-doubling) on the same GPU,
uniform[-1,1] inputs from seed [3, r].

    python -m paper_1611_04255_b200.sweep --out gpurun_out/sweep_cfg3 [--min-exp 10] [--max-exp 27] [--P 2,3,4,5,6,8,16]
                                          [--ops broadcast,reduce,allreduce] [--algos lp,mst,be] [--variant auto]
                                          [--tune CHAIN=2,TILE_ELEMS=4096]

Writes <out>.jsonl (one row per cell) and <out>.md (tables).  GB/s is quoted on the ALGORITHM-independent minimum
bytes of the op (broadcast P*n*4, reduce (P+1)*n*4, allreduce 2*P*n*4) so LP, MST and BE rows compare directly;
algbw = n*4 / t.  Timing: CUDA events around one replay of a CUDA graph holding K back-to-back calls (device-side
time per call: the Python / ctypes call overhead of ~10 us is not billed), K chosen for ~2 ms per measurement,
median of 3; working sets rotate through
>= 1 GB (8 x the 126 MB L2) where the arena allows it, and are restored from pristine copies between measurements.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

from . import binding as lp
from . import inputs

OPS = ("broadcast", "reduce", "allreduce")
ALGOS = ("lp", "mst", "be")
OP_ID = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}
L2_BYTES = 126 << 20


def call(algo, op, bufs, block):
    if algo == "lp":
        if op == "allreduce":
            lp.lp_allreduce(bufs, block)
        elif op == "reduce":
            lp.lp_reduce(bufs, block, root=0)
        else:
            lp.lp_broadcast(bufs, block, root=0)
    else:
        f = getattr(lp, f"lp_{algo}_{op}")
        f(bufs) if op == "allreduce" else f(bufs, root=0)


def main(argv=None):
    import torch

    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/sweep_cfg3")
    ap.add_argument("--min-exp", type=int, default=10)
    ap.add_argument("--max-exp", type=int, default=27)
    ap.add_argument("--P", default="2,3,4,5,6,8,16")
    ap.add_argument("--ops", default="broadcast,reduce,allreduce")
    ap.add_argument("--tune", default="", help="comma list of LP_TUNE key=value (names as in binding.TUNE_*), e.g. CHAIN=2")
    ap.add_argument("--tune-grid", default="", help="several named tunings to compare, LP only: 'name:K=V,K=V;name2:K=V' "
                                                     "(an empty list after the colon = library defaults); writes one column per name")
    ap.add_argument("--block", type=int, default=65_536)
    ap.add_argument("--variant", default="auto", choices=["auto", "pipeline", "direct", "cluster"],
                    help="LP realisation timed in the LP column (default: the library default)")
    ap.add_argument("--algos", default="lp,mst,be")
    args = ap.parse_args(argv)
    assert torch.cuda.is_available(), "the sweep needs a CUDA device"
    dev = torch.device("cuda", 0)
    lp.lib()
    lp.lp_set_variant({"auto": lp.VARIANT_AUTO, "pipeline": lp.VARIANT_PIPELINE, "direct": lp.VARIANT_DIRECT,
                       "cluster": lp.VARIANT_CLUSTER}[args.variant])
    for kv in filter(None, args.tune.split(",")):
        k, v = kv.split("=")
        lp.lp_set_tuning(getattr(lp, "TUNE_" + k.strip().upper()), int(v))
    ops = tuple(o for o in OPS if o in args.ops.split(","))
    algos = tuple(a for a in ALGOS if a in args.algos.split(","))
    if args.tune_grid:
        return tune_grid(torch, dev, args, ops)
    peak = 6545.0
    try:
        peak = float(json.load(open(os.path.join(os.path.dirname(__file__), "..", "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        pass
    Ps = [int(x) for x in args.P.split(",")]
    rows = []
    for P in Ps:
        # pristine vectors (seed [3, r]) and the working arena, both P x n_max
        n_max = arena_elems(P, args.max_exp)
        pristine = [torch.from_numpy(inputs.uniform(3, r, 1 << args.max_exp)).to(dev) for r in range(P)]
        work = [torch.empty(n_max, dtype=torch.float32, device=dev) for _ in range(P)]
        for e in range(args.min_exp, args.max_exp + 1):
            n = 1 << e
            n_sets = int(max(1, min(n_max // n, 64, max(2, -(-8 * L2_BYTES // (P * n * 4))))))
            sets = [[w[s * n:(s + 1) * n] for w in work] for s in range(n_sets)]
            for op in ops:
                mb = lp.lp_min_bytes(OP_ID[op], P, n)
                est = max(mb / 3e12, 4e-6)  # seconds per call, rough
                K = int(min(max(2e-3 / est, 3), 20 * n_sets, 400))
                for algo in algos:
                    if algo == "be" and P & (P - 1):
                        continue
                    # K calls captured in one CUDA graph: device-side time per call, no host call overhead
                    rsets = [lp.Ranks(b) for b in sets]
                    call(algo, op, rsets[0], args.block)  # warm-up outside capture (attributes, scratch)
                    torch.cuda.synchronize()
                    graph = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(graph):
                        for i in range(K):
                            call(algo, op, rsets[i % n_sets], args.block)
                    ms = []
                    for rep in range(4):
                        for w, p in zip(work, pristine):   # every set starts from the same seeded vectors
                            for s_ in range(n_sets):
                                w[s_ * n:(s_ + 1) * n].copy_(p[:n])
                        torch.cuda.synchronize()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        graph.replay()
                        e1.record()
                        torch.cuda.synchronize()
                        if rep:  # first repetition is the warm-up
                            ms.append(e0.elapsed_time(e1) / K)
                    del graph
                    t = float(np.median(ms)) * 1e-3
                    row = dict(op=op, algo=algo, P=P, n=n, msg_bytes=n * 4, us=round(t * 1e6, 3),
                               algbw_GBps=round(n * 4 / t / 1e9, 2), hbm_GBps=round(mb / t / 1e9, 1),
                               frac_measured=round(mb / t / 1e9 / peak, 4), frac_8TBs=round(mb / t / 1e9 / 8000, 4),
                               calls=K, sets=n_sets)
                    rows.append(row)
                    print(json.dumps(row), flush=True)
        del pristine, work
        torch.cuda.empty_cache()
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out + ".jsonl", "w") as f:
        for r in rows:
            f.write(json.dumps(r) + "\n")
    write_markdown(rows, args.out + ".md", peak, Ps, args)


def arena_elems(P, max_exp):
    """Elements per rank of the working arena: the largest message, and at least two buffer sets of it or 1 GB over the
    P ranks (8 x the 126 MB L2), whichever is more -- so that no cell is timed on an L2-resident working set."""
    n_max = 1 << max_exp
    need = -(-8 * L2_BYTES // (P * 4))
    return max(2 * n_max if 2 * n_max * P * 4 <= (48 << 30) else n_max, -(-need // n_max) * n_max)


def parse_tuning(text):
    out = {}
    for kv in filter(None, text.split(",")):
        k, v = kv.split("=")
        out[getattr(lp, "TUNE_" + k.strip().upper())] = int(v)
    return out


def tune_grid(torch, dev, args, ops):
    """LP only: the same cells under several named tunings (one column each), same timing method as the sweep."""
    grid = []
    for item in filter(None, args.tune_grid.split(";")):
        name, _, text = item.partition(":")
        grid.append((name.strip(), parse_tuning(text)))
    base = parse_tuning(args.tune)
    Ps = [int(x) for x in args.P.split(",")]
    rows = []
    for P in Ps:
        n_max = arena_elems(P, args.max_exp)
        pristine = [torch.from_numpy(inputs.uniform(3, r, 1 << args.max_exp)).to(dev) for r in range(P)]
        work = [torch.empty(n_max, dtype=torch.float32, device=dev) for _ in range(P)]
        for e in range(args.min_exp, args.max_exp + 1):
            n = 1 << e
            n_sets = int(max(1, min(n_max // n, 64, max(2, -(-8 * L2_BYTES // (P * n * 4))))))
            sets = [lp.Ranks([w[s * n:(s + 1) * n] for w in work]) for s in range(n_sets)]
            for op in ops:
                mb = lp.lp_min_bytes(OP_ID[op], P, n)
                K = int(min(max(2e-3 / max(mb / 3e12, 4e-6), 3), 20 * n_sets, 400))
                row = dict(op=op, P=P, n=n, msg_bytes=n * 4, min_bytes=mb, calls=K, sets=n_sets, us={})
                for name, tuning in grid:
                    for k in range(lp.TUNE_COUNT):
                        lp.lp_set_tuning(k, base.get(k, 0))
                    for k, v in tuning.items():
                        lp.lp_set_tuning(k, v)
                    call("lp", op, sets[0], args.block)
                    torch.cuda.synchronize()
                    graph = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(graph):
                        for i in range(K):
                            call("lp", op, sets[i % n_sets], args.block)
                    ms = []
                    for rep in range(4):
                        for w, p in zip(work, pristine):   # every set starts from the same seeded vectors
                            for s_ in range(n_sets):
                                w[s_ * n:(s_ + 1) * n].copy_(p[:n])
                        torch.cuda.synchronize()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        graph.replay()
                        e1.record()
                        torch.cuda.synchronize()
                        if rep:
                            ms.append(e0.elapsed_time(e1) / K)
                    del graph
                    row["us"][name] = round(float(np.median(ms)) * 1e3, 2)
                rows.append(row)
                print(json.dumps(row), flush=True)
        del pristine, work
        torch.cuda.empty_cache()
    for k in range(lp.TUNE_COUNT):
        lp.lp_set_tuning(k, 0)
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out + ".jsonl", "w") as f:
        for r in rows:
            f.write(json.dumps(r) + "\n")
    with open(args.out + ".md", "w") as f:
        f.write(f"Command: `python -m paper_1611_04255_b200.sweep --out {args.out} --min-exp {args.min_exp} --max-exp {args.max_exp} "
                f"--P {args.P} --ops {args.ops} --variant {args.variant}" + (f" --tune {args.tune}" if args.tune else "")
                + f" --tune-grid '{args.tune_grid}'`\n\n")
        f.write("us per call (CUDA-graph replay of K back-to-back calls / K, median of 3, rotating buffer sets); in brackets the "
                "fraction of 8 TB/s on the op's minimum HBM bytes.\n\n")
        names = [g[0] for g in grid]
        f.write("| op | P | message | " + " | ".join(names) + " |\n|---|---|---|" + "---|" * len(names) + "\n")
        for r in rows:
            best = min(r["us"].values())
            cells = []
            for nme in names:
                u = r["us"][nme]
                txt = f"{u:.2f} ({r['min_bytes'] / u / 1e3 / 8000:.3f})"
                cells.append(f"**{txt}**" if u == best else txt)
            f.write(f"| {r['op']} | {r['P']} | {r['msg_bytes'] >> 20} MB | " + " | ".join(cells) + " |\n")
    return 0


def write_markdown(rows, path, peak, Ps, args):
    def size(b):
        return f"{b >> 20} MB" if b >= 1 << 20 else f"{b >> 10} KB"

    idx = {(r["op"], r["algo"], r["P"], r["n"]): r for r in rows}
    ns = sorted({r["n"] for r in rows})
    with open(path, "w") as f:
        f.write("# Message-size sweep (BASELINE.json configs[3]) — LP vs MST vs BE on one B200\n\n")
        f.write(f"Command: `python -m paper_1611_04255_b200.sweep --out {args.out} --min-exp {args.min_exp} "
                f"--max-exp {args.max_exp} --P {args.P} --block {args.block} --variant {args.variant} --algos {args.algos} "
                f"--ops {args.ops}" + (f" --tune {args.tune}" if args.tune else "") + "`\n\n")
        f.write(f"Cells: GB/s on the op's minimum HBM bytes (fraction of the measured copy peak {peak} GB/s); "
                "LP block 65,536 elements; uniform[-1,1], seed [3, r]. North-star bar: LP >= 80 % of 8 TB/s = 6400 GB/s "
                "for messages >= 64 MB, and LP faster than MST and BE.\n")
        for op in OPS:
            for P in Ps:
                f.write(f"\n## {op}, P = {P}\n\n| message | LP us | LP GB/s (frac) | of 8 TB/s | MST GB/s | BE GB/s | LP/MST | LP/BE |\n"
                        "|---|---|---|---|---|---|---|---|\n")
                for n in ns:
                    a = idx.get((op, "lp", P, n))
                    if not a:
                        continue
                    m, b = idx.get((op, "mst", P, n)), idx.get((op, "be", P, n))
                    nan = float("nan")
                    f.write(f"| {size(n * 4)} | {a['us']:.1f} | {a['hbm_GBps']:.0f} ({a['frac_measured']:.2f}) | "
                            f"{a['frac_8TBs']:.2f} | {(m['hbm_GBps'] if m else nan):.0f} | {(b['hbm_GBps'] if b else nan):.0f} | "
                            f"{(m['us'] / a['us'] if m else nan):.2f}x | {(b['us'] / a['us'] if b else nan):.2f}x |\n")


if __name__ == "__main__":
    sys.exit(main())
