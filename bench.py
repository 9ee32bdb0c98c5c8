#!/usr/bin/env python
"""bench.py -- LP allreduce algorithm GB/s and fraction of the HBM roofline on one B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--block B]

A step is one LP allreduce (a1 partition, a2 schedule, a4 reduce stage, a3 broadcast stage = a5) of the
workload -- by default BASELINE.json configs[4], the largest single-GPU configuration: P=16 virtual ranks,
n=138,000,000 fp32 per rank (8.83 GB), N(0,1e-3), seed 4, b=262,144 (--config 1: P=6, n=61,000,000, the
AlexNet-sized vector) -- through the C ABI (lp_allreduce) with the inputs already resident in HBM.  `value` = algbw =
n*4 bytes / t (nccl-tests convention) summed over the N replicas; `roofline.achieved` = minimum HBM bytes
2*P*n*4 / t against the measured copy peak of MEASURED_PEAKS.json.  `e2e` = the same metric through
lp_allreduce_host with pinned HOST buffers (H2D + kernel + D2H inside the timed region).  `cpu_baseline` /
`--impl reference` time the CPU oracle as it stands on the box's host cores, on the FULL vectors of the workload.
The other BASELINE.json configs are measured in the same run and printed FIRST, one compact JSON line per section
(`{"detail": "<section>", ...}`): configs[3] from 64 MB up at P = 2, 3, 4, 5, 6, 8, 16 (`sweep`: LP vs MST vs BE, three
collectives, with the HBM ceiling of the same read : write mix from a plain streaming kernel beside every cell), its
4 KB .. 32 MB half (`sweep_small`: the crossover table of the paper's Fig. 3), configs[1] / configs[4] (all three ops,
variants, block sizes), configs[2] (fused BSP-SGD step, 100 iterations), the pure-stream HBM ceilings, the typed
collectives and the multi-GPU chain's one-GPU emulation.  The LAST line (rank 0) is the headline: a few KB, with a
`summary` of scalars taken from the sections.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1611_04255_b200 import inputs  # noqa: E402

METRIC = "lp_allreduce_algbw"
UNIT = "GB/s (algbw = n*4 bytes per rank / time; roofline on min bytes 2*P*n*4)"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
# roofline.traffic (dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch) cannot be measured
# inside this program (it needs ncu's replays): the line carries the number of the committed `ncu --set full` capture of
# the same command and names it.  config index -> (bytes per launch, source)
TRAFFIC = {
    1: (2_869_328_000, "profiles/r2_ncu_lp_pipeline.md (ncu --set full of `bench.py --config 1`: 0.98 x algorithmic)"),
    4: (17_604_425_000, "profiles/r3_ncu_lp_pipeline_cfg4.md (ncu --set full of this command: read 8.832 GB + write "
                        "8.772 GB = 0.997 x algorithmic)"),
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (4 = the largest, or 1)")
    ap.add_argument("--block", type=int, default=0, help="LP block in elements (0 = the config's)")
    ap.add_argument("--variant", default="auto", choices=["auto", "pipeline", "direct", "cluster", "copy_engine"])
    ap.add_argument("--no-detail", action="store_true", help="skip the secondary measurements")
    ap.add_argument("--detail", default="configs1,configs2,configs4,sweep,sweep_small,ceilings,dtypes,chain",
                    help="comma list of detail sections to run")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args()


def workload(cfg_idx):
    c = inputs.CONFIGS[cfg_idx]
    if "allreduce" not in c["ops"] or not isinstance(c["P"], int):
        raise SystemExit(f"config {cfg_idx} is not a single allreduce workload")
    return c


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ---- clocks ------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: an NVML polling thread (about 1 kHz: the timed
    region of the default run is ~10 ms), or `nvidia-smi -lms 20` when the NVML binding is missing."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.p = self.f = self.thread = None
        self.samples, self.reasons, self.max_mhz, self.stop_flag = [], set(), None, False
        try:
            import threading

            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            masks = {"hw_slowdown": pynvml.nvmlClocksThrottleReasonHwSlowdown,
                     "hw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                     "sw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonSwThermalSlowdown,
                     "sw_power_cap": pynvml.nvmlClocksThrottleReasonSwPowerCap}

            def poll():
                while not self.stop_flag:
                    try:
                        self.samples.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                        for name, m in masks.items():
                            if r & m:
                                self.reasons.add(name)
                    except Exception:  # noqa: BLE001
                        break
                    time.sleep(0.0005)

            self.thread = threading.Thread(target=poll, daemon=True)
            self.thread.start()
            self.how = "nvml thread"
            return
        except Exception:  # noqa: BLE001
            self.thread = None
        self.how = "nvidia-smi -lms 20"
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "how": self.how}
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            if self.samples:
                out.update(sm_mhz=float(np.median(self.samples)), sm_min_mhz=float(min(self.samples)),
                           sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons), samples=len(self.samples))
            return out
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 5]
        os.unlink(self.f.name)
        sm, names = [], ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = set()
        for r in rows:
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
            except ValueError:
                continue
            for name, v in zip(names, r[2:6]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        if sm:
            out["sm_mhz"] = float(np.median(sm))
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


# ---- distributed plumbing (replicas only: no data-path collective) ------------------------------------
def dist_setup(n_gpus):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        import torch
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value, world, device=None):
    """Max of a python float over all ranks (timing rule: the slowest rank counts)."""
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, world, device=None):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ---- the oracle on the host cores (cpu_baseline leg and --impl reference) ------------------------------
def time_oracle(P, n, dist_kind, sigma, seed, passes, warm=2, single_thread_passes=0):
    """Times the oracle's allreduce as it stands on the FULL vectors of the workload (no sample): `passes` timed passes
    of lpo_allreduce_omp (element loop over all host cores) after `warm` untimed ones, and optionally a few passes of
    the canonical single-thread loop lpo_allreduce.  The allreduce is in place (|x| grows ~P per pass): inputs are
    restored outside the timed region before magnitudes could overflow.  Returns (omp seconds list, cores,
    single-thread seconds list)."""
    from oracle import lpo
    src = inputs.rank_vectors(seed, P, n, dist_kind, sigma)
    work = [s.copy() for s in src]
    vmax = max(float(np.abs(h).max()) for h in src)
    safe = max(1, int(np.floor(np.log(1e30 / max(vmax, 1e-30)) / np.log(max(P, 2)))))

    def run(fn_omp, count):
        out, used = [], 0
        for _ in range(count):
            if used >= safe:
                for w, s_ in zip(work, src):
                    np.copyto(w, s_)
                used = 0
            t0 = time.perf_counter()
            lpo.allreduce(work, omp=fn_omp)
            out.append(time.perf_counter() - t0)
            used += 1
        return out

    run(True, warm)  # page faults, thread pool
    omp = run(True, passes)
    single = run(False, single_thread_passes) if single_thread_passes else []
    return omp, lpo.num_threads(), single


def oracle_baseline(c, cfg_idx, passes, single_thread_passes):
    P, n = c["P"], c["n"]
    omp, cores, single = time_oracle(P, n, c["dist"], c.get("sigma", 1.0), cfg_idx, passes,
                                     single_thread_passes=single_thread_passes)
    t = float(np.median(omp))
    out = {"value": n * 4 / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"the full workload: all {n} elements of each of the P={P} vectors ({P * n * 4 / 1e9:.2f} GB), "
                     f"lpo_allreduce_omp, {len(omp)} timed passes after 2 warm-up passes, median {t * 1e3:.1f} ms per pass "
                     f"(min {min(omp) * 1e3:.1f}, mean {sum(omp) / len(omp) * 1e3:.1f})"}
    if single:
        ts = float(np.median(single))
        out["single_thread"] = {"value": n * 4 / ts / 1e9, "unit": UNIT, "cores": 1, "ms_per_pass": ts * 1e3,
                                "passes": len(single), "what": "lpo_allreduce: the canonical plain loop, one host thread"}
    return out, t


def headline_config(cfg_idx, c, block):
    """The `config` object of the headline line: the same keys and values in both arms."""
    return {"workload": f"BASELINE.json configs[{cfg_idx}]: {c['name']}", "P": c["P"], "n": c["n"], "block": block}


def compact(obj):
    return json.dumps(obj, separators=(",", ":"))


def run_reference(args, c, rank, world):
    """--impl reference: the CPU oracle, unmodified, on the host cores, on the whole workload.  Rank 0 only."""
    if rank != 0:
        return
    P, n = c["P"], c["n"]
    block = args.block or c["block"]
    omp, cores, _ = time_oracle(P, n, c["dist"], c.get("sigma", 1.0), args.config, args.steps, warm=max(args.warmup, 1))
    t = float(np.median(omp))
    value = n * 4 / t / 1e9
    sample = (f"the full workload: all {n} elements of each of the P={P} vectors, oracle lpo_allreduce_omp, "
              f"{len(omp)} timed passes after {max(args.warmup, 1)} warm-up passes, median pass "
              f"(mean {sum(omp) / len(omp) * 1e3:.1f} ms, min {min(omp) * 1e3:.1f} ms)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": headline_config(args.config, c, block),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- our arm ------------------------------------------------------------------------------------------------
def timed_steps(torch, step_fn, restore_fn, n_steps, safe_run):
    """Runs n_steps back to back between CUDA events on the current stream; every `safe_run` steps the inputs are
    restored OUTSIDE the event pair (an in-place allreduce multiplies magnitudes by ~P per call).  Returns ms."""
    total_ms, done = 0.0, 0
    while done < n_steps:
        seg = min(safe_run, n_steps - done)
        restore_fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(seg):
            step_fn(done + i)
        e1.record()
        torch.cuda.synchronize()
        total_ms += e0.elapsed_time(e1)
        done += seg
    return total_ms


def run_ours(args, c, rank, world, local):
    import torch

    from paper_1611_04255_b200 import binding as lp

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA library is the product, there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    lp.lib()
    variant = {"pipeline": 0, "direct": 1, "cluster": 2, "copy_engine": 3, "auto": 4}[args.variant]
    lp.lp_set_variant(variant)
    P, n = c["P"], c["n"]
    block = args.block or c["block"]
    sigma = c.get("sigma", 1.0)
    min_bytes = lp.lp_min_bytes(lp.OP_ALLREDUCE, P, n)

    # synthetic inputs, generated on the host, uploaded once
    host = inputs.rank_vectors(args.config, P, n, c["dist"], sigma)
    pristine = [torch.from_numpy(h).to(dev) for h in host]
    n_sets = 3  # rotating buffer sets; one set (P*n*4 bytes) is already >> the 126 MB L2
    free_b, _ = torch.cuda.mem_get_info()
    while n_sets > 1 and n_sets * P * n * 4 > 0.6 * free_b:
        n_sets -= 1
    sets = [[torch.empty_like(p) for p in pristine] for _ in range(n_sets)]

    def restore():
        for s in sets:
            for d, p in zip(s, pristine):
                d.copy_(p)

    def step(i):
        lp.lp_allreduce(sets[i % n_sets], block)

    # growth per call ~P: keep |x| * P^k far below fp32 max
    vmax = max(float(np.abs(h).max()) for h in host)
    safe_uses = max(1, int(np.floor(np.log(1e30 / max(vmax, 1e-30)) / np.log(max(P, 2)))))
    safe_run = safe_uses * n_sets

    barrier(world)
    timed_steps(torch, step, restore, max(args.warmup, 3), safe_run)  # warm-up (>= 3)
    barrier(world)
    torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = lp.lp_launch_count()
    total_ms = timed_steps(torch, step, restore, args.steps, safe_run)
    launches = lp.lp_launch_count() - launches0
    barrier(world)
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    total_ms = max_over_ranks(total_ms, world, dev)
    ms_per_step = total_ms / args.steps
    algbw = world * n * 4 / (ms_per_step * 1e-3) / 1e9
    hbm = min_bytes / (ms_per_step * 1e-3) / 1e9  # per GPU
    peak, peak_src = measured_peak()
    plan = lp.lp_plan_query(lp.OP_ALLREDUCE, P, n, block)
    ran = ["pipeline", "direct", "cluster", "copy_engine"][plan["variant"]]  # what LP_VARIANT_AUTO resolved to

    # e2e: host buffers through lp_allreduce_host, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pinned = [torch.from_numpy(h.copy()).pin_memory() for h in host]
        k_e2e = max(1, min(args.steps, 5))
        lp.lp_allreduce_host(pinned, block)  # warm-up (allocates the staging chunks)
        for p_, h in zip(pinned, host):
            p_.copy_(torch.from_numpy(h))
        barrier(world)
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            lp.lp_allreduce_host(pinned, block)  # synchronous
        t_e2e = (time.perf_counter() - t0) / k_e2e
        t_e2e = max_over_ranks(t_e2e, world, dev)
        e2e = {"value": world * n * 4 / t_e2e / 1e9, "unit": UNIT, "h2d_bytes_per_step": P * n * 4,
               "d2h_bytes_per_step": P * n * 4, "ms_per_step": t_e2e * 1e3, "steps": k_e2e,
               "api": "lp_allreduce_host (pinned host buffers, chunked H2D/kernel/D2H pipeline)"}
        del pinned

    del pristine, sets
    torch.cuda.empty_cache()

    # secondary measurements: one compact JSON line per section, printed as it finishes, BEFORE the headline line
    summary = {}
    if rank == 0 and not args.no_detail:
        want = set(args.detail.split(","))

        def section(name, fn):
            # a secondary measurement that fails must not take the headline line with it
            if name not in want:
                return
            try:
                out = fn()
                summarise(name, out, summary)
            except Exception as exc:  # noqa: BLE001
                out = {"error": f"{type(exc).__name__}: {exc}"}
                summary[f"{name}_error"] = out["error"][:120]
                torch.cuda.synchronize()
            print(compact({"detail": name, **out}), flush=True)

        section("configs1", lambda: cfg1_more(torch, lp, dev, peak))
        section("configs2", lambda: cfg2_steps(torch, lp, dev, peak))
        section("configs4", lambda: cfg4_row(torch, lp, dev, peak))
        section("sweep", lambda: sweep_cfg3(torch, lp, dev, peak))
        section("sweep_small", lambda: sweep_small(torch, lp, dev))
        section("ceilings", lambda: ceilings(torch, lp, dev, peak))
        section("dtypes", lambda: dtype_rows(torch, lp, dev))
        section("chain", lambda: chain_rows(torch, lp, dev))

    cpu = None
    if rank == 0 and not args.no_cpu:
        cpu, _ = oracle_baseline(c, args.config, passes=20 if P * n <= 1 << 29 else 12,
                                 single_thread_passes=3 if P * n <= 1 << 29 else 1)

    if rank != 0:
        return
    traffic, traffic_src = TRAFFIC.get(args.config, (None, "no committed ncu --set full capture of this config"))
    line = {
        "metric": METRIC, "value": algbw, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": headline_config(args.config, c, block),
        "run": {"variant": ran, "grid": plan.get("grid"), "tile_elems": plan.get("tile_elems"),
                "smem_bytes": plan.get("smem_bytes"), "parallelism": f"replicas x{world} (no collective)",
                "l2": f"inputs {P * n * 4 / 1e6:.0f} MB per set >> 126 MB L2, {n_sets} rotating sets"},
        "roofline": {"bound": "hbm", "achieved": hbm, "peak": peak, "unit": "GB/s", "frac": hbm / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "peak_note": "the peak is a 1 read : 1 write torch copy; pure read / write streams reach ~7.4 TB/s "
                                  "here (detail ceilings), so a fraction slightly above 1 is not a ceiling claim",
                     "frac_of_nominal_8TBs": hbm / 8000.0,
                     "kernel": "lp_pipeline_kernel" if ran == "pipeline" else ran,
                     "algorithmic_bytes_per_launch": min_bytes},
        "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "summary": summary,
    }
    print(compact(line), flush=True)


def summarise(name, out, summary):
    """The few scalars of a detail section that the headline line carries (the section's own line has the rest)."""
    if name == "configs1":
        a = out["allreduce"]
        summary["configs1_allreduce_us"] = a["lp_us_unchained"]
        summary["configs1_frac_8TBs_unchained"] = a["lp_frac_8TBs_unchained"]
    elif name == "configs4":
        summary["configs4_frac_8TBs_unchained"] = {op: out[op]["lp_frac_8TBs_unchained"]
                                                   for op in ("allreduce", "reduce", "broadcast")}
    elif name == "configs2":
        summary["configs2_sgd_step_us"] = out["lp_bsp_sgd_step"]["us_per_step"]
        summary["configs2_sgd_step_frac_8TBs"] = out["lp_bsp_sgd_step"]["frac_8TBs"]
    elif name == "sweep":
        sm = out["summary"]
        summary["sweep_ge64MB_cells"] = sm["cells"]
        summary["sweep_min_frac_8TBs"] = sm["lp_min_frac_8TBs"]
        summary["sweep_min_frac_8TBs_unchained"] = sm["lp_min_frac_8TBs_unchained"]
        summary["sweep_cells_below_0.80_unchained"] = len(sm["lp_cells_below_0.80_of_8TBs_unchained"])
        summary["sweep_min_lp_vs_mst"] = sm["lp_min_vs_mst"]
        summary["sweep_min_lp_vs_be"] = sm["lp_min_vs_be"]
    elif name == "sweep_small":
        summary["small_cells"] = out["summary"]["cells"]
        summary["small_cells_where_lp_is_not_fastest"] = out["summary"]["cells_where_lp_is_not_fastest"]
        summary["small_crossover"] = out["summary"]["crossover"]


# ---- detail: the rest of BASELINE.json's configs, driver-measured ---------------------------------------
L2_BYTES = 126 << 20
SWEEP_PS = (2, 3, 4, 5, 6, 8, 16)          # 3, 5, 6: the paper's own Fig. 4 points
SWEEP_EXPS = (24, 25, 26, 27)             # 64, 128, 256, 512 MB per rank: where north_star's 80 % bar applies


def graph_time(torch, fn_of_set, n_sets, restore, traffic_bytes, reps=3, target_ms=2.0, k_max=400):
    """Device time per call: K back-to-back calls captured in one CUDA graph (the host's call overhead is not billed,
    consecutive calls overlap their launches as they do in a training loop), call i on buffer set i mod n_sets,
    inputs restored outside the event pair; median of `reps` replays after one warm-up replay.  Returns (us, K)."""
    est = max(traffic_bytes / 3e12, 4e-6)
    K = int(min(max(target_ms * 1e-3 / est, 3), 20 * n_sets, k_max))
    fn_of_set(0)  # outside capture: function attributes, scratch, claim counters
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for i in range(K):
            fn_of_set(i % n_sets)
    ms = []
    for rep in range(reps + 1):
        restore()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.replay()
        e1.record()
        torch.cuda.synchronize()
        if rep:
            ms.append(e0.elapsed_time(e1) / K)
    del g
    return float(np.median(ms)) * 1e3, K


def lp_call(lp, algo, op, bufs, block):
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


def probe_call(lp, op, bufs):
    """The same read : write mix as `op` over the same buffers, from the plain streaming kernel (lp_hbm_probe)."""
    if op == "allreduce":
        lp.lp_hbm_probe(bufs, bufs)          # P reads, P writes, in place like the collective
    elif op == "reduce":
        lp.lp_hbm_probe(bufs, bufs[:1])      # P reads, 1 write (root 0)
    else:
        lp.lp_hbm_probe(bufs[:1], bufs[1:])  # 1 read, P-1 writes


def cell(lp, torch, op, P, n, block, sets, restore, peak, algos=("lp", "mst", "be")):
    op_id = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}[op]
    mb = lp.lp_min_bytes(op_id, P, n)
    row = {"P": P, "msg_MB": n * 4 / 2 ** 20, "op": op, "min_bytes": mb}
    for algo in algos:
        if algo == "be" and P & (P - 1):
            continue
        us, K = graph_time(torch, lambda s, a=algo: lp_call(lp, a, op, sets[s], block), len(sets), restore, mb)
        row[f"{algo}_us"] = round(us, 2)
        row[f"{algo}_GBps"] = round(mb / us / 1e3, 1)
        row["calls_per_graph"] = K
    # the same LP calls with stream chaining off (LP_TUNE_CHAIN 2): every launch waits for its predecessor to finish
    # before it starts -- what one call costs when the NEXT one depends on it.  Since round 3 this is also what the
    # library's default does between API calls (chaining across calls is opt-in: LP_TUNE_CHAIN 1, lp_chain_optin_us).
    lp.lp_set_tuning(lp.TUNE_CHAIN, 2)
    us, _ = graph_time(torch, lambda s: lp_call(lp, "lp", op, sets[s], block), len(sets), restore, mb)
    row["lp_us_unchained"] = round(us, 2)
    row["lp_GBps_unchained"] = round(mb / us / 1e3, 1)
    lp.lp_set_tuning(lp.TUNE_CHAIN, 1)
    us, _ = graph_time(torch, lambda s: lp_call(lp, "lp", op, sets[s], block), len(sets), restore, mb)
    lp.lp_set_tuning(lp.TUNE_CHAIN, 0)
    row["lp_chain_optin_us"] = round(us, 2)
    us, _ = graph_time(torch, lambda s: probe_call(lp, op, sets[s]), len(sets), restore, mb)
    row["ceiling_GBps"] = round(mb / us / 1e3, 1)      # plain streaming kernel, same mix, same buffers, same method
    g = row["lp_GBps"]
    row["lp_frac_8TBs"] = round(g / 8000.0, 4)
    row["lp_frac_8TBs_unchained"] = round(row["lp_GBps_unchained"] / 8000.0, 4)
    row["lp_frac_measured_copy_peak"] = round(g / peak, 4)
    row["lp_over_ceiling"] = round(g / row["ceiling_GBps"], 4)
    if "mst_us" in row:
        row["lp_vs_mst"] = round(row["mst_us"] / row["lp_us"], 3)
    if "be_us" in row:
        row["lp_vs_be"] = round(row["be_us"] / row["lp_us"], 3)
    row["lp_variant"] = ["pipeline", "direct", "cluster", "copy_engine"][lp.lp_plan_query(op_id, P, n, block)["variant"]]
    return row


def sweep_cfg3(torch, lp, dev, peak, ps=SWEEP_PS, exps=SWEEP_EXPS, block=65_536):
    """BASELINE.json configs[3] at the sizes north_star's bar applies to (>= 64 MB), plus the paper's Fig. 4 rank counts
    3, 5, 6: LP vs MST vs BE, three collectives, uniform[-1,1] from seed [3, r]."""
    n_max = 1 << max(exps)
    host = [inputs.uniform(3, r, n_max) for r in range(max(ps))]
    pristine_all = [torch.from_numpy(h).to(dev) for h in host]
    del host
    rows = []
    for P in ps:
        pristine = pristine_all[:P]
        work = [torch.empty_like(p) for p in pristine]
        for e in exps:
            n = 1 << e
            # rotate through >= 1 GB (8 x L2), and through at least two sets where the arena holds two: consecutive
            # collectives of a training step work on different buffers (the layers of Alg. 1)
            n_sets = int(max(1, min(n_max // n, 64, max(2, -(-8 * L2_BYTES // (P * n * 4))))))
            sets = [lp.Ranks([w[s * n:(s + 1) * n] for w in work]) for s in range(n_sets)]

            def restore(n_sets=n_sets, n=n):
                for w, p in zip(work, pristine):
                    w[:n_sets * n].copy_(p[:n_sets * n])

            for op in ("broadcast", "reduce", "allreduce"):
                row = cell(lp, torch, op, P, n, block, sets, restore, peak)
                row["rotating_sets"] = n_sets
                rows.append(row)
        del work, sets
        torch.cuda.empty_cache()
    del pristine_all
    torch.cuda.empty_cache()
    lp_rows = [r for r in rows]
    summary = {
        "cells": len(rows),
        "lp_min_frac_8TBs": min(r["lp_frac_8TBs"] for r in lp_rows),
        "lp_cells_below_0.80_of_8TBs": [f"{r['op']} P={r['P']} {int(r['msg_MB'])}MB: {r['lp_frac_8TBs']}" for r in lp_rows
                                        if r["lp_frac_8TBs"] < 0.80],
        "lp_min_frac_8TBs_unchained": min(r["lp_frac_8TBs_unchained"] for r in lp_rows),
        "lp_cells_below_0.80_of_8TBs_unchained": [f"{r['op']} P={r['P']} {int(r['msg_MB'])}MB: {r['lp_frac_8TBs_unchained']}"
                                                  for r in lp_rows if r["lp_frac_8TBs_unchained"] < 0.80],
        "lp_min_over_ceiling": min(r["lp_over_ceiling"] for r in lp_rows),
        "lp_min_vs_mst": min(r["lp_vs_mst"] for r in lp_rows if "lp_vs_mst" in r),
        "lp_min_vs_be": min(r["lp_vs_be"] for r in lp_rows if "lp_vs_be" in r),
        "lp_cells_slower_than_mst_or_be": [f"{r['op']} P={r['P']} {int(r['msg_MB'])}MB" for r in lp_rows
                                           if r.get("lp_vs_mst", 9) < 1.0 or r.get("lp_vs_be", 9) < 1.0],
    }
    cols = ["P", "msg_MB", "op", "lp_us", "lp_us_unchained", "lp_chain_optin_us", "mst_us", "be_us", "ceiling_GBps", "lp_frac_8TBs",
            "lp_frac_8TBs_unchained", "lp_over_ceiling", "lp_variant", "rotating_sets"]
    rows = [[r.get(k) for k in cols] for r in rows]
    return {"cols": cols,
            "note": "us per call = CUDA-graph replay of K back-to-back calls / K, median of 3, buffer sets rotating through "
                    ">= 1 GB (8 x L2), inputs restored outside the event pair; GB/s on the op's minimum HBM bytes for every "
                    "algorithm so rows compare; ceiling = lp_hbm_probe (plain streaming kernel, same read:write mix, same "
                    "buffers); block 65,536.  lp_us = library defaults (a call's first launch waits for whatever precedes it on the "
                    "stream; MST / BE tree levels of one call chain); *_unchained = LP_TUNE_CHAIN 2 (every launch waits first); "
                    "lp_chain_optin_us = LP_TUNE_CHAIN 1 (calls on different buffer sets run into each other, rotating_sets > 1)",
            "summary": summary, "rows": rows}


def sweep_small(torch, lp, dev, ps=(2, 4, 8, 16), exps=tuple(range(10, 24)), block=65_536):
    """The 4 KB .. 32 MB half of BASELINE.json configs[3] (Fig. 3; MST's smaller latency term
    should win on short messages): LP (variant auto) vs MST vs BE, three collectives, device time per call from a CUDA
    graph of back-to-back calls on rotating buffer sets.  Messages this short live in the 126 MB L2 -- as they would
    in a training step that has just produced them -- so these cells are launch / latency numbers, not HBM ones."""
    n_max = 2 << max(exps)   # arena per rank: two buffer sets of the longest message
    pristine_all = [torch.from_numpy(inputs.uniform(3, r, n_max)).to(dev) for r in range(max(ps))]
    cols = ["P", "msg_KB", "op", "lp_us", "mst_us", "be_us", "lp_variant"]
    rows, slower = [], []
    crossover = {}
    for P in ps:
        pristine = pristine_all[:P]
        work = [torch.empty_like(p_) for p_ in pristine]
        for e in exps:
            n = 1 << e
            n_sets = int(max(2, min(n_max // n, 16)))
            sets = [lp.Ranks([w[s_ * n:(s_ + 1) * n] for w in work]) for s_ in range(n_sets)]

            def restore(n_sets=n_sets, n=n):
                for w, p_ in zip(work, pristine):
                    w[:n_sets * n].copy_(p_[:n_sets * n])

            for op in ("broadcast", "reduce", "allreduce"):
                op_id = {"broadcast": lp.OP_BROADCAST, "reduce": lp.OP_REDUCE, "allreduce": lp.OP_ALLREDUCE}[op]
                mb = lp.lp_min_bytes(op_id, P, n)
                t = {}
                for algo in ("lp", "mst", "be"):
                    us, _ = graph_time(torch, lambda s_, a=algo: lp_call(lp, a, op, sets[s_], block), n_sets, restore, mb,
                                       reps=2, target_ms=1.0, k_max=200)
                    t[algo] = round(us, 2)
                variant = ["pipeline", "direct", "cluster", "copy_engine"][lp.lp_plan_query(op_id, P, n, block)["variant"]]
                rows.append([P, n * 4 // 1024, op, t["lp"], t["mst"], t["be"], variant])
                best_other = min(t["mst"], t["be"])
                if t["lp"] > 1.03 * best_other:   # 3 %: the timing's own repeatability
                    slower.append(f"{op} P={P} {n * 4 // 1024}KB: lp {t['lp']} us vs {best_other} us")
                    crossover[f"{op}_P{P}"] = n * 4 // 1024
        del work, sets
        torch.cuda.empty_cache()
    return {"cols": cols, "rows": rows,
            "note": "us per call, CUDA-graph replay of K back-to-back calls / K over >= 2 rotating buffer sets (L2-resident), "
                    "median of 2; LP = LP_VARIANT_AUTO with block 65,536; a cell counts as 'LP not fastest' when LP is more "
                    "than 3 % slower than the better of MST and BE",
            "summary": {"cells": len(rows), "cells_where_lp_is_not_fastest": len(slower), "which": slower[:24],
                        "crossover": ("none: LP is the fastest (within 3 %) in every cell from 4 KB to 32 MB" if not slower else
                                      {k: f"MST/BE faster up to {v} KB" for k, v in crossover.items()})}}


def cfg4_row(torch, lp, dev, peak):
    """BASELINE.json configs[4]: P=16, n=138,000,000 (VGG-16-sized), N(0,1e-3) seed 4, b=262,144 -- the largest config."""
    c = inputs.CONFIGS[4]
    P, n, block = c["P"], c["n"], c["block"]
    pristine = [torch.from_numpy(inputs.normal(4, r, n, c["sigma"])).to(dev) for r in range(P)]
    work = [torch.empty_like(p) for p in pristine]
    sets = [lp.Ranks(work)]

    def restore():
        for w, p in zip(work, pristine):
            w.copy_(p)

    out = {"P": P, "n": n, "block": block, "footprint_GB": round(P * n * 4 / 1e9, 2)}
    for op in ("allreduce", "reduce", "broadcast"):
        out[op] = cell(lp, torch, op, P, n, block, sets, restore, peak)
    del pristine, work, sets
    torch.cuda.empty_cache()
    return out


def cfg2_steps(torch, lp, dev, peak):
    """BASELINE.json configs[2]: fused BSP-SGD step, P=8, n=7,000,000, 100 iterations back to back (one CUDA graph of
    100 steps over 3 rotating sets of gradients + weight replicas = 1.3 GB), and the f1 steps beside it."""
    c2 = inputs.CONFIGS[2]
    P, n, block, lr = c2["P"], c2["n"], c2["block"], c2["lr"]
    g_h, w_h = inputs.sgd_inputs(2, P, n, c2["sigma"], c2["w_sigma"])
    n_sets = 3
    g0 = [torch.from_numpy(x).to(dev) for x in g_h]
    w0 = [torch.from_numpy(x).to(dev) for x in w_h]
    gs = [lp.Ranks([x.clone() for x in g0]) for _ in range(n_sets)]
    ws = [lp.Ranks([x.clone() for x in w0]) for _ in range(n_sets)]
    vel = [torch.zeros(n, device=dev) for _ in range(n_sets)]

    def restore():
        for s in range(n_sets):
            for d, p in zip(ws[s], w0):
                d.copy_(p)
            for d, p in zip(gs[s], g0):
                d.copy_(p)
            vel[s].zero_()

    out = {"P": P, "n": n, "block": block, "iterations_per_graph": 100, "rotating_sets": n_sets}

    def add(name, fn, op_id):
        mb = lp.lp_min_bytes(op_id, P, n)
        us, K = graph_time(torch, fn, n_sets, restore, mb, k_max=100, target_ms=1e9)
        out[name] = {"us_per_step": round(us, 2), "hbm_GBps_min_bytes": round(mb / us / 1e3, 1),
                     "frac_8TBs": round(mb / us / 1e3 / 8000, 4), "frac_measured_copy_peak": round(mb / us / 1e3 / peak, 4),
                     "steps_per_graph": K}

    add("lp_bsp_sgd_step", lambda s: lp.lp_bsp_sgd_step(gs[s], ws[s], block, root=0, lr=lr), lp.OP_BSP_SGD)
    add("lp_bsp_sgd_momentum_step", lambda s: lp.lp_bsp_sgd_momentum_step(gs[s], ws[s], vel[s], block, root=0, lr=lr, mu=0.9),
        lp.OP_BSP_SGD_MOM)
    # Alg. 2 (reduce, root update, broadcast: three launches), quoted on the FUSED step's minimum bytes so rows compare
    add("lp_bsp_sgd_alg2_step", lambda s: lp.lp_bsp_sgd_alg2_step(gs[s], ws[s], block, root=0, lr=lr), lp.OP_BSP_SGD)
    add("lp_allreduce_P8_7M", lambda s: lp.lp_allreduce(gs[s], block), lp.OP_ALLREDUCE)
    add("mst_allreduce_P8_7M", lambda s: lp.lp_mst_allreduce(gs[s]), lp.OP_ALLREDUCE)
    add("be_allreduce_P8_7M", lambda s: lp.lp_be_allreduce(gs[s]), lp.OP_ALLREDUCE)
    us, _ = graph_time(torch, lambda s: lp.lp_hbm_probe(list(gs[s]) + [ws[s][0]], list(ws[s])), n_sets, restore,
                       lp.lp_min_bytes(lp.OP_BSP_SGD, P, n), k_max=100, target_ms=1e9)
    out["ceiling_GBps_same_mix"] = round(lp.lp_min_bytes(lp.OP_BSP_SGD, P, n) / us / 1e3, 1)
    out["bar_80pct_of_8TBs_us"] = round(lp.lp_min_bytes(lp.OP_BSP_SGD, P, n) / 6400e9 * 1e6, 2)
    return out


def cfg1_more(torch, lp, dev, peak):
    """BASELINE.json configs[1] (P=6, n=61,000,000, N(0,1e-3) seed 1): the three collectives, every LP variant, the block
    sweep (16K = the paper's 64 KB), MST.  Same graph timing; one working set (1.46 GB >> L2)."""
    c = inputs.CONFIGS[1]
    P, n, block = c["P"], c["n"], c["block"]
    pristine = [torch.from_numpy(h).to(dev) for h in inputs.rank_vectors(1, P, n, c["dist"], c["sigma"])]
    work = [torch.empty_like(p_) for p_ in pristine]
    sets = [lp.Ranks(work)]

    def restore():
        for d, p in zip(work, pristine):
            d.copy_(p)

    out = {}
    for op in ("allreduce", "reduce", "broadcast"):
        out[op] = cell(lp, torch, op, P, n, block, sets, restore, peak, algos=("lp", "mst"))
    mb = lp.lp_min_bytes(lp.OP_ALLREDUCE, P, n)
    cur = lp.lp_get_variant()
    var = {}
    for name, v in (("pipeline", lp.VARIANT_PIPELINE), ("direct", lp.VARIANT_DIRECT), ("cluster", lp.VARIANT_CLUSTER)):
        lp.lp_set_variant(v)
        us, _ = graph_time(torch, lambda s: lp.lp_allreduce(sets[s], block), 1, restore, mb)
        var[name] = {"us": round(us, 2), "hbm_GBps_min_bytes": round(mb / us / 1e3, 1)}
    lp.lp_set_variant(lp.VARIANT_COPY_ENGINE)  # the paper's own design: at the paper's 64 KB block and at block = 0 (fitted optimum)
    for label, b in (("copy_engine_block_auto", 0), ("copy_engine_block_262144", 262_144)):
        lp.lp_allreduce(sets[0], b)  # scratch
        torch.cuda.synchronize()
        restore()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        lp.lp_allreduce(sets[0], b)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        var[label] = {"us": round(ms * 1e3, 1), "hbm_GBps_min_bytes": round(mb / ms / 1e6, 1),
                      "block": int(lp.lp_auto_block(lp.OP_ALLREDUCE, P, n, lp.VARIANT_COPY_ENGINE)) if b == 0 else b}
    lp.lp_set_variant(cur)
    out["allreduce_variants"] = var
    sweep = {}
    for b in (16_384, 65_536, 131_072, 262_144, 524_288, 1_048_576):
        us, _ = graph_time(torch, lambda s, b=b: lp.lp_allreduce(sets[s], b), 1, restore, mb)
        sweep[str(b)] = {"us": round(us, 2), "hbm_GBps_min_bytes": round(mb / us / 1e3, 1)}
    out["allreduce_block_sweep"] = sweep
    del pristine, work, sets
    torch.cuda.empty_cache()
    return out


def ceilings(torch, lp, dev, peak):
    """HBM ceilings of this GPU for pure and mixed streams, 512 MB per stream: lp_hbm_probe (plain kernel) and torch's fill."""
    n = 1 << 27
    bufs = [torch.empty(n, device=dev) for _ in range(6)]
    for b in bufs:
        b.normal_()
    out = {}

    def t(fn, nbytes):
        us, _ = graph_time(torch, lambda s: fn(), 1, lambda: None, nbytes)
        return round(nbytes / us / 1e3, 1)

    out["probe_read_only_4_streams"] = t(lambda: lp.lp_hbm_probe(bufs[:4], []), 4 * n * 4)
    out["probe_write_only_4_streams"] = t(lambda: lp.lp_hbm_probe([], bufs[:4]), 4 * n * 4)
    out["probe_copy_1r_1w"] = t(lambda: lp.lp_hbm_probe(bufs[:1], bufs[1:2]), 2 * n * 4)
    out["probe_1r_5w"] = t(lambda: lp.lp_hbm_probe(bufs[:1], bufs[1:6]), 6 * n * 4)
    out["probe_5r_1w"] = t(lambda: lp.lp_hbm_probe(bufs[:5], bufs[5:6]), 6 * n * 4)
    out["torch_fill_write_only"] = t(lambda: bufs[0].fill_(1.0), n * 4)
    out["measured_peaks_json_hbm_gbs"] = peak
    out["unit"] = "GB/s"
    return out


def dtype_rows(torch, lp, dev, P=6, msg_bytes=256 << 20):
    """SURVEY 8(f)-4 'dtypes': the typed collectives (lp_*_dt, reading U21) on messages of the SAME BYTES per rank in
    every element type -- the path is HBM-bound, so the element type should not change the time.  Same graph timing as
    the sweep; >= 1 GB of rotating buffer sets."""
    types = (("f32", lp.DT_F32, torch.float32), ("f16", lp.DT_F16, torch.float16), ("bf16", lp.DT_BF16, torch.bfloat16),
             ("f64", lp.DT_F64, torch.float64))
    n_sets = max(2, -(-(8 * L2_BYTES) // (P * msg_bytes)))
    out = {"P": P, "msg_MB": msg_bytes / 2 ** 20, "rotating_sets": n_sets,
           "what": "us per call and GB/s on the op's minimum bytes (allreduce 2 P bytes, reduce (P+1) bytes, broadcast P bytes)"}
    raw = [[torch.empty(msg_bytes, dtype=torch.uint8, device=dev) for _ in range(P)] for _ in range(n_sets)]
    for name, dt, tdt in types:
        sets = [[b.view(tdt) for b in s] for s in raw]
        n = sets[0][0].numel()

        def restore():
            for s in sets:
                for r, b in enumerate(s):
                    b.fill_(0.001 * (r + 1))   # repeated in-place sums may reach inf in the 16-bit types: same cost

        row = {"n_elements": n}
        for op, mult in (("allreduce", 2 * P), ("reduce", P + 1), ("broadcast", P)):
            if op == "allreduce":
                fn = lambda s, dt=dt: lp.lp_allreduce_dt(sets[s], 65_536, dtype=dt)
            elif op == "reduce":
                fn = lambda s, dt=dt: lp.lp_reduce_dt(sets[s], 65_536, root=0, dtype=dt)
            else:
                fn = lambda s, dt=dt: lp.lp_broadcast_dt(sets[s], 65_536, root=0, dtype=dt)
            us, _ = graph_time(torch, fn, n_sets, restore, mult * msg_bytes)
            gbs = mult * msg_bytes / us / 1e3
            row[op] = {"us": round(us, 2), "hbm_GBps_min_bytes": round(gbs, 1), "frac_of_8TBs": round(gbs / 8000.0, 4)}
        out[name] = row
    return out


def chain_rows(torch, lp, dev, msg_bytes=64 << 20):
    """the one-rank-per-GPU chain (csrc/lp_chain.cu) as far as ONE GPU can run it -- all P ranks in
    one cooperative launch (lp_chain_emulate), every 'link' being this GPU's own HBM.  So this measures the PROTOCOL
    (push + publish + credit per block), not NVLink: per_link_GBps = message bytes / time is what every emulated link
    direction carried; hbm_GBps counts what the emulation really moves, (6P-4) n 4 bytes for an allreduce (P loads, P stores
    and 2(P-1) ring writes + reads), (3P-2) n 4 for a broadcast.  Eager launches, K back to back between two events."""
    n = msg_bytes // 4
    out = {"msg_MB": msg_bytes / 2 ** 20, "tile_elems": 131_072, "slots": 4, "block": "0 = the cost model's choice",
           "what": "us per call, GB/s per emulated link direction, HBM GB/s of the emulation; NOT an NVLink measurement"}
    for P in (2, 4, 8):
        bufs = [torch.full((n,), 0.001 * (r + 1), device=dev) for r in range(P)]
        row = {"channels": lp.lp_chain_emulate_channels(P)}
        for op, op_id, moved in (("allreduce", lp.OP_ALLREDUCE, 6 * P - 4), ("broadcast", lp.OP_BROADCAST, 3 * P - 2)):
            for _ in range(2):
                lp.lp_chain_emulate(op_id, bufs, block=0)
            torch.cuda.synchronize()
            K = 10
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(K):
                lp.lp_chain_emulate(op_id, bufs, block=0)
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / K
            row[op] = {"us": round(us, 1), "per_link_GBps": round(msg_bytes / us / 1e3, 1),
                       "hbm_GBps": round(moved * msg_bytes / us / 1e3, 1)}
            for r, b in enumerate(bufs):
                b.fill_(0.001 * (r + 1))
        row["error"] = lp.lp_chain_emulate_error(P)
        if P == 2:  # the register realisation of a rank's CTAs beside the default (TMA loads), same protocol
            lp.lp_chain_set_kernel(lp.CHAIN_KERNEL_REGISTER)
            for _ in range(2):
                lp.lp_chain_emulate(lp.OP_ALLREDUCE, bufs, block=0)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(10):
                lp.lp_chain_emulate(lp.OP_ALLREDUCE, bufs, block=0)
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / 10
            row["allreduce_register_kernel"] = {"us": round(us, 1), "per_link_GBps": round(msg_bytes / us / 1e3, 1)}
            lp.lp_chain_set_kernel(lp.CHAIN_KERNEL_DEFAULT)
        out[f"P{P}"] = row
        del bufs
    return out


def main():
    args = parse_args()
    c = workload(args.config)
    if args.impl == "reference":  # no process group: rank 0 alone works, the others exit 0
        run_reference(args, c, int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))
        return
    rank, world, local = dist_setup(args.gpus)
    try:
        run_ours(args, c, rank, world, local)
    finally:
        if world > 1:
            import torch.distributed as dist
            if dist.is_initialized():
                dist.destroy_process_group()


if __name__ == "__main__":
    main()
