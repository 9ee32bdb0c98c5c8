"""Fit the paper's alpha-beta-gamma model (Eq. 1, Table 1) to B200 measurements and predict the block size.

    python -m paper_1611_04255_b200.cost_fit --out gpurun_out/cost_fit [--P 6] [--n 61000000]

PAPER.md:81-106: a block exchange costs alpha + (beta + gamma) b, an LP allreduce 2(p-1+n/b) alpha + (b(p-1)+n)(2 beta
+ gamma); the paper takes alpha ~ 1e-7 s, beta ~ 1e-9 s/byte for PCI-E and picks b "around 64 KB".  Here the LP
allreduce of configs[1] is timed over a sweep of block sizes in two realisations:

  * copy_engine -- the paper's own design (one cudaMemcpyAsync + one add kernel per hop and block, two streams):
    both terms of the model exist (per-operation submission cost; pipeline fill of p-1 blocks);
  * pipeline    -- the persistent TMA kernel: the running partial never leaves the SM, so there is no fill term
    and the block only matters when it is smaller than a tile.

T(b) = A x1 + W x2 with x1 = p-1+n/b, x2 = b(p-1)+n (bytes) is fitted by least squares (A = 2 alpha, W = 2 beta +
gamma), b* = lp_optimal_block(...) is compared with the measured optimum.  Writes <out>.jsonl and <out>.md.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

from . import binding as lp
from . import inputs


def main(argv=None):
    import torch

    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/cost_fit")
    ap.add_argument("--P", type=int, default=6)
    ap.add_argument("--n", type=int, default=61_000_000)
    ap.add_argument("--min-exp", type=int, default=12)
    ap.add_argument("--max-exp", type=int, default=24)
    args = ap.parse_args(argv)
    assert torch.cuda.is_available(), "needs a CUDA device"
    dev = torch.device("cuda", 0)
    lp.lib()
    P, n = args.P, args.n
    pristine = [torch.from_numpy(inputs.normal(1, r, n, 1e-3)).to(dev) for r in range(P)]
    work = [torch.empty_like(p) for p in pristine]
    ranks = lp.Ranks(work)
    blocks = [1 << e for e in range(args.min_exp, args.max_exp + 1)]
    rows, fits = [], {}
    for variant, vid in (("copy_engine", lp.VARIANT_COPY_ENGINE), ("pipeline", lp.VARIANT_PIPELINE)):
        lp.lp_set_variant(vid)
        ts = []
        for b in blocks:
            ms = []
            for it in range(4):
                for w, p in zip(work, pristine):
                    w.copy_(p)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                lp.lp_allreduce(ranks, b)
                e1.record()
                torch.cuda.synchronize()
                if it:
                    ms.append(e0.elapsed_time(e1))
            t = float(np.median(ms)) * 1e-3
            ts.append(t)
            row = dict(variant=variant, P=P, n=n, block_elems=b, block_bytes=4 * b, nb=-(-n // b), ms=round(t * 1e3, 4))
            rows.append(row)
            print(json.dumps(row), flush=True)
        nbytes = 4.0 * n
        bb = np.array([4.0 * b for b in blocks])
        x1 = (P - 1) + nbytes / bb
        x2 = bb * (P - 1) + nbytes
        # relative least squares (every block size weighs the same)
        X = np.stack([x1, x2], axis=1) / np.array(ts)[:, None]
        sol, *_ = np.linalg.lstsq(X, np.ones(len(ts)), rcond=None)
        A, W = max(float(sol[0]), 0.0), max(float(sol[1]), 0.0)
        pred = A * x1 + W * x2
        b_star = lp.lp_optimal_block(lp.OP_ALLREDUCE, P, nbytes, A / 2, W / 2, 0.0)
        i_best = int(np.argmin(ts))
        fits[variant] = dict(A_us=A * 1e6, W_ps_per_byte=W * 1e12, b_star_bytes=b_star,
                             t_at_b_star_ms=lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, nbytes, b_star, A / 2, W / 2, 0.0) * 1e3,
                             best_block_bytes=float(bb[i_best]), best_ms=ts[i_best] * 1e3,
                             max_rel_err=float(np.max(np.abs(pred - np.array(ts)) / np.array(ts))), pred_ms=(pred * 1e3).tolist())
    lp.lp_set_variant(lp.VARIANT_AUTO)
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out + ".jsonl", "w") as f:
        for r in rows:
            f.write(json.dumps(r) + "\n")
        f.write(json.dumps({"fits": fits}) + "\n")
    with open(args.out + ".md", "w") as f:
        f.write("# The paper's alpha-beta-gamma model (Eq. 1, Table 1) fitted to the LP allreduce on one B200\n\n")
        f.write(f"Command: `python -m paper_1611_04255_b200.cost_fit --out {args.out} --P {P} --n {n} --min-exp {args.min_exp} "
                f"--max-exp {args.max_exp}`\n\n")
        f.write(f"LP allreduce, P={P}, n={n:,} fp32 ({4 * n / 1e6:.0f} MB per rank), single calls timed with CUDA events "
                "(median of 3, inputs restored before each).  Model: T(b) = A (p-1+n/b) + W (b(p-1)+n), A = 2 alpha, "
                "W = 2 beta + gamma, relative least squares over the sweep.\n\n")
        f.write("| block | blocks | copy_engine ms | model ms | pipeline ms | model ms |\n|---|---|---|---|---|---|\n")
        ce = [r for r in rows if r["variant"] == "copy_engine"]
        pi = [r for r in rows if r["variant"] == "pipeline"]
        for i, (a, b) in enumerate(zip(ce, pi)):
            kb = a["block_bytes"] / 1024
            f.write(f"| {kb:.0f} KB | {a['nb']} | {a['ms']:.3f} | {fits['copy_engine']['pred_ms'][i]:.3f} | {b['ms']:.4f} | "
                    f"{fits['pipeline']['pred_ms'][i]:.4f} |\n")
        f.write("\n| realisation | A = 2 alpha | W = 2 beta + gamma | max rel. error of the fit | predicted b* | T(b*) | measured best block | measured best |\n"
                "|---|---|---|---|---|---|---|---|\n")
        for v in ("copy_engine", "pipeline"):
            x = fits[v]
            f.write(f"| {v} | {x['A_us']:.3f} us | {x['W_ps_per_byte']:.4f} ps/B ({1e3 / max(x['W_ps_per_byte'], 1e-9):.0f} GB/s per exchange) | "
                    f"{x['max_rel_err'] * 100:.1f} % | {x['b_star_bytes'] / 1024:.0f} KB | {x['t_at_b_star_ms']:.3f} ms | "
                    f"{x['best_block_bytes'] / 1024:.0f} KB | {x['best_ms']:.3f} ms |\n")


if __name__ == "__main__":
    sys.exit(main())
