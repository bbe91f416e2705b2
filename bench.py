#!/usr/bin/env python
"""Benchmark of the direct-SCF J/K Fock build (the whole hot path) on synthetic input.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A "step" = one te_build_jk over one config (pair lists prebuilt, D resident in HBM).  The default workload is
config 5, the largest one (BASELINE.json north_star: "the largest config's J/K build"); --config 1..4 select the
others.  Metric: unique primitive shell quartets per second (BASELINE.json: "shell-quartet ERIs/s"), with s/iter and
the fraction of the measured FP64 FMA peak alongside.  N > 1 runs N independent replicas (the path does not shard: DESIGN.md section 8),
timed as the max over ranks.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "primitive_shell_quartets_per_s"
UNIT = "quartets/s"
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of a class kernel, taken from a committed
# `ncu --set full` capture of THIS config (profiles/r2_dram_bytes.json: {"<config>": {"(AB|CD)": bytes}}, written from the
# capture named inside that file); a class / config without a capture reports null
DRAM_BYTES_FILE = os.path.join(ROOT, "profiles", "r2_dram_bytes.json")


def ncu_dram_bytes(cfg: int, cls: str):
    try:
        with open(DRAM_BYTES_FILE) as fh:
            return json.load(fh).get(str(cfg), {}).get(cls)
    except (OSError, ValueError):
        return None

CONFIG_NAMES = {1: "cfg1_tiny", 2: "cfg2_small_organic", 3: "cfg3_water16", 4: "cfg4_metal_complex",
                5: "cfg5_large_organic"}


# ------------------------------------------------------------------------------------------- plumbing
def dist_setup(ngpus: int):
    """(rank, world).  Under torchrun, initialise the process group (NCCL with a GPU, gloo without)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if torch.cuda.is_available():
            torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        if not dist.is_initialized():
            dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    return rank, world


def max_over_ranks(x: float, world: int) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda" if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def aggregate(quartets_per_rank: float, seconds_max: float, world: int) -> float:
    """Whole-job throughput of `world` independent replicas: total units / max-over-ranks time."""
    return quartets_per_rank * world / seconds_max


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.stop, self.index = [], threading.Event(), index
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower() == "active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# --------------------------------------------------------------------------------------- reference arm
def oracle_sample(cfg: int):
    """Bounded sample of the workload for the CPU oracle: the first atoms of the config (heavy atoms with
    their H), sized so one O2 build takes seconds.  Returns (problem, description)."""
    from synth import make_config, subset_atoms
    prob = make_config(cfg)
    if cfg == 1:
        return prob, "full config 1 (692,076 unique primitive quartets)"
    if cfg == 3:
        ids = list(range(9))
        return subset_atoms(prob, ids), "first 3 H2O of config 3 (same basis, D sub-block), full O2 build"
    if cfg == 4:
        ids = [0, 1, 2, 49, 50]
        return subset_atoms(prob, ids), "metal + first 2 heavy + their 2 H of config 4, full O2 build"
    nheavy = 12 if cfg == 2 else 120
    k = 3 if cfg == 2 else 5          # config 5: ~1.2e7 live quartets, 5-15 s of oracle work on the box's host threads
    ids = list(range(k)) + [nheavy + i for i in range(k)]
    return subset_atoms(prob, ids), f"first {k} heavy + their {k} H atoms of config {cfg} (same basis, D sub-block), full O2 build"


def run_oracle_steps(cfg: int, steps: int, warmup: int):
    import oracle
    prob, desc = oracle_sample(cfg)
    o = oracle.Oracle(prob)
    o.build_pairs(prob.tau_pair)
    times, live = [], 0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        _, _, st = o.jk_o2(prob.D, prob.tau_jk)
        dt = time.perf_counter() - t0
        live = st["live_quartets"]
        if it >= warmup:
            times.append(dt)
    return live, times, desc, oracle.num_threads()


def main_reference(args, rank, world):
    if rank != 0:
        return
    live, times, desc, cores = run_oracle_steps(args.config, args.steps, min(args.warmup, 1))
    sec = float(np.sum(times))
    val = live * len(times) / sec
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": CONFIG_NAMES[args.config], "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------- roofline ceilings
def main_peaks():
    """FP64 ceilings of this GPU, one JSON line: register-resident DFMA chains (the "alu" roofline denominator), cuBLAS
    float64 matmul 8192^3 (the DMMA / tensor-core FP64 path) and the rate of a DFMA stream fed by one
    lane-private shared-memory load per FMA (the operand pattern of the uniform-ket Hermite -> Cartesian transform)."""
    import torch

    import paper_2406_14920_b200 as te
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --peaks needs a CUDA device")
    torch.cuda.set_device(0)
    n = 8192
    a = torch.randn(n, n, dtype=torch.float64, device="cuda")
    b = torch.randn(n, n, dtype=torch.float64, device="cuda")
    for _ in range(2):
        a @ b
    torch.cuda.synchronize()
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        a @ b
        e1.record()
        torch.cuda.synchronize()
        best = max(best, 2 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
    line = {"fp64_dfma_tflops": te.te_measure_fp64_peak(), "fp64_matmul_8192_tflops": best,
            "fp64_nominal_tflops": 148 * 64 * 2 * 1.965e9 / 1e12,
            "smem_fed_dfma_tflops": {str(w): te.te_measure_smem_dfma_rate(w) for w in (4, 8, 16)}}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------- our arm
def main_ours(args, rank, world):
    import torch

    import paper_2406_14920_b200 as te
    from paper_2406_14920_b200 import flopmodel
    from synth import make_config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path (use --impl reference for the oracle)")
    dev = int(os.environ.get("LOCAL_RANK", "0")) if world > 1 else 0
    torch.cuda.set_device(dev)
    prob = make_config(args.config)
    t0 = time.perf_counter()
    basis = te.Basis.from_problem(prob)
    pairs = basis.shellpair_build(prob.tau_pair)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    n = basis.nbf
    D = torch.tensor(prob.D, device="cuda")
    J = torch.empty_like(D)
    K = torch.empty_like(D)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 256 MB > 126 MB L2

    mixed = args.fp32_below is not None      # te_build_jk_mixed instead of the FP64 build: an extra, not the headline

    def step():
        if mixed:
            pairs.build_jk(D, J, K, threshold=prob.tau_jk, fp32_below=args.fp32_below)
        else:
            pairs.build_jk(D, J, K, threshold=prob.tau_jk)

    for _ in range(max(args.warmup, 0)):
        step()
    torch.cuda.synchronize()
    barrier(world)
    evs = []
    with ClockSampler(dev) as clk:
        torch.cuda.synchronize()
        for _ in range(args.steps):
            flush.fill_(1.0)                                   # evict L2 between timed iterations
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            step()
            e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
    barrier(world)
    sec_local = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    sec = max_over_ranks(sec_local, world)
    q, _ = pairs.stats()
    live = int(q.sum())
    visited, slots = pairs.screening_stats()
    npairs_nonempty = sum(1 for cb in range(10) for ck in range(cb, 10) if pairs.class_count[cb] and pairs.class_count[ck])
    nclasses_nonempty = sum(1 for c in range(10) if pairs.class_count[c])
    # scale, bounds, finish + (Hermite density, Hermite J) per pair class + (schedule, J/K kernel) per class pair
    launches_per_step = 3 + 2 * nclasses_nonempty + 2 * npairs_nonempty

    # end to end through the host entry point: pinned host D in, pinned host J/K out, copies inside the timed region
    Dh = torch.tensor(prob.D).pin_memory()
    Jh = torch.empty_like(Dh).pin_memory()
    Kh = torch.empty_like(Dh).pin_memory()
    pairs.build_jk_host(Dh, prob.tau_jk, Jh, Kh)
    e2e_steps = max(1, min(args.steps, 3))
    barrier(world)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        pairs.build_jk_host(Dh, prob.tau_jk, Jh, Kh)
    e2e_sec = max_over_ranks(time.perf_counter() - t0, world)
    assert float((Jh - J.cpu()).abs().max()) < 1e-9

    if rank != 0:
        return
    # per-class device times (separate profiled pass, CUDA events on the launching stream) -> dominant kernel
    pairs.set_profiling(True)
    step()
    qs, ms = pairs.stats()
    pairs.set_profiling(False)
    peak = te.te_measure_fp64_peak()
    cb, ck = np.unravel_index(int(np.argmax(ms)), ms.shape)
    dom_flops = float(qs[cb, ck]) * flopmodel.class_pair_flops(int(cb), int(ck))
    dom_ach = dom_flops / (float(ms[cb, ck]) * 1e-3) / 1e12
    total_flops = flopmodel.build_flops(qs)
    step_s = sec / args.steps
    per_class = sorted(((float(ms[a, b]), f"({te.CLASS_NAMES[a]}|{te.CLASS_NAMES[b]})", int(qs[a, b]))
                        for a in range(10) for b in range(a, 10) if ms[a, b] > 0), reverse=True)[:8]

    # the oracle, as it stands, on the host cores, on a bounded sample of the same workload
    live_o, t_o, desc, cores = run_oracle_steps(args.config, 1, 0)
    cpu_val = live_o / t_o[0]

    line = {
        "metric": METRIC, "value": aggregate(live * args.steps, sec, world), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * step_s, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if not mixed else "f64/f32 mixed", "data": "synthetic",
        "config": {"workload": CONFIG_NAMES[args.config], "nbf": n, "primitive_pairs_kept": pairs.nkept,
                   "build": "te_build_jk (FP64)" if not mixed else f"te_build_jk_mixed(fp32_below={args.fp32_below}); e2e is the FP64 host path",
                   "live_quartets_per_build": live, "visited_quartets_per_build": int(visited.sum()),
                   "live_over_visited": live / max(int(visited.sum()), 1), "lane_occupancy": live / max(int(slots.sum()), 1),
                   "thresholds": [prob.tau_pair, prob.tau_jk],
                   "l2": "flushed between timed iterations (256 MB fill)", "parallelism": "replicas only"},
        "jk_build_s_per_iter": step_s, "pair_build_s": t_setup,
        "model_flops_per_build": total_flops, "fp64_tflops_algorithmic": total_flops / step_s / 1e12,
        "fp64_frac_of_peak": total_flops / step_s / 1e12 / peak,
        "roofline": {"bound": "alu", "kernel": f"J/K class kernel ({te.CLASS_NAMES[cb]}|{te.CLASS_NAMES[ck]})",
                     "achieved": dom_ach, "peak": peak, "unit": "TFLOP/s", "frac": dom_ach / peak,
                     "traffic": ncu_dram_bytes(args.config, f"({te.CLASS_NAMES[cb]}|{te.CLASS_NAMES[ck]})"),
                     "traffic_source": "profiles/r2_dram_bytes.json (ncu --set full capture of this config) or null",
                     "kernel_ms": float(ms[cb, ck]), "kernel_share_of_step": float(ms[cb, ck]) / float(ms.sum()),
                     "whole_build_frac": total_flops / step_s / 1e12 / peak,
                     "peak_source": "te_measure_fp64_peak: register-resident DFMA chains measured in this run "
                                    "(MEASURED_PEAKS.json has no FP64 entry; nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2)",
                     "top_kernels_ms": per_class},
        "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": aggregate(live * e2e_steps, e2e_sec, world), "unit": UNIT,
                "h2d_bytes_per_step": n * n * 8, "d2h_bytes_per_step": 2 * n * n * 8},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clk.summary(),
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--peaks", action="store_true", help="print the measured FP64 ceilings of this GPU and exit")
    ap.add_argument("--fp32-below", type=float, default=None,
                    help="time te_build_jk_mixed with this density-weighted switch (the paper uses 1e-5) instead of the FP64 build")
    args = ap.parse_args()
    if args.peaks:
        main_peaks()
        return
    if args.impl == "reference":      # rank 0 alone runs the oracle; other ranks exit 0 without work, no rendezvous
        main_reference(args, int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))
        return
    rank, world = dist_setup(args.gpus)
    try:
        main_ours(args, rank, world)
    finally:
        if world > 1:
            import torch.distributed as dist
            if dist.is_initialized():
                dist.destroy_process_group()


if __name__ == "__main__":
    main()
