"""Fit the paper's alpha-beta-gamma model (Eq. 1, Table 1) to B200 measurements and predict the block size.

    python -m paper_1611_04255_b200.cost_fit --out gpurun_out/cost_fit [--P 2,6,16] [--n 61000000]

PAPER.md:81-106: a block exchange costs alpha + (beta + gamma) b, an LP allreduce 2(p-1+n/b) alpha + (b(p-1)+n)(2 beta
+ gamma); the paper takes alpha ~ 1e-7 s, beta ~ 1e-9 s/byte for PCI-E and picks b "around 64 KB".  Here the LP
allreduce of configs[1] is timed over a sweep of block sizes in two realisations:

  * copy_engine -- the paper's own design (one cudaMemcpyAsync + one add kernel per hop and block, two streams):
    both terms of the model exist (per-operation submission cost; pipeline fill of p-1 blocks);
  * pipeline    -- the persistent TMA kernel: the running partial never leaves the SM, so there is no fill term
    and the block only matters when it is smaller than a tile.

T(b) = A x1 + W x2 with x1 = p-1+n/b, x2 = b(p-1)+n (bytes) is fitted by least squares (A = 2 alpha, W = 2 beta +
gamma), once per rank count p, b* = lp_optimal_block(...) is compared with the measured optimum and with what the
library does for block = 0 (lp_auto_block, the committed constants of lp_fitted_constants), and A(p), W(p) are
tabulated: Eq. 1 assumes they do not depend on p.  Writes <out>.jsonl and <out>.md.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

from . import binding as lp
from . import inputs


def fit_one(torch, dev, P, n, blocks, variants):
    """Times the LP allreduce of (P, n) at every block size in every variant and fits T(b) = A x1 + W x2."""
    pristine = [torch.from_numpy(inputs.normal(1, r, n, 1e-3)).to(dev) for r in range(P)]
    work = [torch.empty_like(p) for p in pristine]
    ranks = lp.Ranks(work)
    rows, fits = [], {}

    def time_block(b):
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
        return float(np.median(ms)) * 1e-3

    for variant, vid in variants:
        lp.lp_set_variant(vid)
        ts = []
        for b in blocks:
            t = time_block(b)
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
        fit = dict(P=P, A_us=A * 1e6, W_ps_per_byte=W * 1e12, b_star_bytes=b_star,
                   t_at_b_star_ms=lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, nbytes, b_star, A / 2, W / 2, 0.0) * 1e3,
                   best_block_bytes=float(bb[i_best]), best_ms=ts[i_best] * 1e3,
                   max_rel_err=float(np.max(np.abs(pred - np.array(ts)) / np.array(ts))), pred_ms=(pred * 1e3).tolist())
        if variant == "copy_engine":
            # what the LIBRARY does with block = 0 (lp_auto_block: the committed constants), and what its committed
            # constants predict for every block of the sweep
            auto_b = int(lp.lp_auto_block(lp.OP_ALLREDUCE, P, n, lp.VARIANT_COPY_ENGINE))
            fit["auto_block_bytes"] = 4.0 * auto_b
            fit["auto_block_ms"] = time_block(0) * 1e3
            al, be = lp.lp_fitted_constants(P)
            lib_pred = np.array([lp.lp_cost_model(lp.ALGO_LP, lp.OP_ALLREDUCE, P, nbytes, x, al, be, 0.0) for x in bb])
            fit["library_constants"] = dict(alpha_us=al * 1e6, beta_ps_per_byte=be * 1e12)
            fit["library_pred_ms"] = (lib_pred * 1e3).tolist()
            fit["library_max_rel_err"] = float(np.max(np.abs(lib_pred - np.array(ts)) / np.array(ts)))
        fits[variant] = fit
    lp.lp_set_variant(lp.VARIANT_AUTO)
    del pristine, work, ranks
    torch.cuda.empty_cache()
    return rows, fits


def main(argv=None):
    import torch

    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/cost_fit")
    ap.add_argument("--P", default="2,6,16", help="comma list of rank counts (Eq. 1 assumes alpha, beta do not depend on p)")
    ap.add_argument("--n", type=int, default=61_000_000)
    ap.add_argument("--min-exp", type=int, default=14)
    ap.add_argument("--max-exp", type=int, default=24)
    args = ap.parse_args(argv)
    assert torch.cuda.is_available(), "needs a CUDA device"
    dev = torch.device("cuda", 0)
    lp.lib()
    n = args.n
    Ps = [int(x) for x in args.P.split(",")]
    blocks = [1 << e for e in range(args.min_exp, args.max_exp + 1)]
    all_rows, all_fits = [], {}
    for P in Ps:
        variants = [("copy_engine", lp.VARIANT_COPY_ENGINE)] + ([("pipeline", lp.VARIANT_PIPELINE)] if P == Ps[len(Ps) // 2] else [])
        rows, fits = fit_one(torch, dev, P, n, blocks, variants)
        all_rows += rows
        all_fits[P] = fits
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out + ".jsonl", "w") as f:
        for r in all_rows:
            f.write(json.dumps(r) + "\n")
        f.write(json.dumps({"fits": {str(k): v for k, v in all_fits.items()}}) + "\n")
    with open(args.out + ".md", "w") as f:
        f.write("# The paper's alpha-beta-gamma model (Eq. 1, Table 1) fitted to the LP allreduce on one B200\n\n")
        f.write(f"Command: `python -m paper_1611_04255_b200.cost_fit --out {args.out} --P {args.P} --n {n} --min-exp {args.min_exp} "
                f"--max-exp {args.max_exp}`\n\n")
        f.write(f"LP allreduce, n={n:,} fp32 ({4 * n / 1e6:.0f} MB per rank), single calls timed with CUDA events "
                "(median of 3, inputs restored before each).  Model (PAPER.md:81-91): T(b) = A (p-1+n/b) + W (b(p-1)+n), "
                "A = 2 alpha, W = 2 beta + gamma, relative least squares over the block sweep, one fit per p.\n")
        for P in Ps:
            fits = all_fits[P]
            ce = [r for r in all_rows if r["variant"] == "copy_engine" and r["P"] == P]
            pi = [r for r in all_rows if r["variant"] == "pipeline" and r["P"] == P]
            f.write(f"\n## p = {P}\n\n| block | blocks | copy_engine ms | own fit ms | library constants ms |"
                    + (" pipeline ms |" if pi else "") + "\n|---|---|---|---|---|" + ("---|" if pi else "") + "\n")
            for i, a in enumerate(ce):
                kb = a["block_bytes"] / 1024
                f.write(f"| {kb:.0f} KB | {a['nb']} | {a['ms']:.3f} | {fits['copy_engine']['pred_ms'][i]:.3f} | "
                        f"{fits['copy_engine']['library_pred_ms'][i]:.3f} |" + (f" {pi[i]['ms']:.4f} |" if pi else "") + "\n")
        f.write("\n## Is the model's assumption (alpha, beta independent of p, PAPER.md:81-89) true on one GPU?\n\n"
                "| p | A = 2 alpha | W = 2 beta + gamma | A / (p-1) | W / (p-1) | A / W | fit error | b* (own fit) | best measured block | "
                "best ms | block = 0 (library) | its ms | library-constant error |\n|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
        for P in Ps:
            x = all_fits[P]["copy_engine"]
            f.write(f"| {P} | {x['A_us']:.2f} us | {x['W_ps_per_byte']:.4f} ps/B | {x['A_us'] / (P - 1):.2f} us | "
                    f"{x['W_ps_per_byte'] / (P - 1):.4f} ps/B | {x['A_us'] * 1e-6 / max(x['W_ps_per_byte'] * 1e-12, 1e-30) / 1e6:.2f} MB | "
                    f"{x['max_rel_err'] * 100:.1f} % | {x['b_star_bytes'] / 2 ** 20:.2f} MB | {x['best_block_bytes'] / 2 ** 20:.2f} MB | "
                    f"{x['best_ms']:.3f} | {x['auto_block_bytes'] / 2 ** 20:.2f} MB | {x['auto_block_ms']:.3f} | "
                    f"{x['library_max_rel_err'] * 100:.1f} % |\n")
        for P in Ps:
            if "pipeline" in all_fits[P]:
                x = all_fits[P]["pipeline"]
                f.write(f"\nPersistent pipeline kernel at p = {P}: A = {x['A_us']:.3f} us, W = {x['W_ps_per_byte']:.4f} ps/B, "
                        f"fit error {x['max_rel_err'] * 100:.1f} % -- the two-term model does not describe it (flat in the block size: "
                        f"{min(r['ms'] for r in all_rows if r['variant'] == 'pipeline'):.4f}-"
                        f"{max(r['ms'] for r in all_rows if r['variant'] == 'pipeline'):.4f} ms over the sweep).\n")


if __name__ == "__main__":
    sys.exit(main())
