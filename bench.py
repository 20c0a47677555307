#!/usr/bin/env python
"""bench.py — throughput of the ENCORE hot path (steps a1..a6) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--impl ours|reference] [--all-configs]

A "step" is one encore_compute over one synthetic catalogue (all of a1..a6).  The default workload is c3, the
4PCF configuration BASELINE.json's target is stated on (300 000 lognormal-clustered points, 10 bins in [20,160],
lmax=5); `--all-configs` adds one measured line per config c1..c5 under "per_config".
  value  = primaries/s with the catalogue already resident in HBM (CUDA events over K steps, max over ranks);
  e2e    = the same through encore_compute_host with pinned HOST buffers (H2D of positions+weights and D2H of
           zeta inside the timed region);
  roofline = dominant kernel (the a_lm pair stage), plain FP64 ALU bound, timed live with the library's CUDA events
           on the compute stream; algorithmic flops per DESIGN.md §7;
  cpu_baseline = the oracle as it stands on this box's host cores on a strided subset of primaries.
N > 1: every rank runs an independent catalogue of the same recipe (seed + rank) — separate mocks / D-R splits are
how the paper spends extra nodes — no data-path collective; "scaling": "weak".
`--impl reference` times the CPU oracle (test infrastructure) on the same config and metric.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

SM_COUNT, FP64_LANES_PER_SM = 148, 64
# dram__bytes_read.sum + dram__bytes_write.sum of k_fill + k_harm per step, from the committed `ncu --set full` capture
# profiles/r1_v7_ncu_full.txt (an ALU-bound stage: the traffic is the candidate lists written and read back once)
NCU_PAIR_STAGE_DRAM_BYTES = {"c3": 19.65e9}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


# ---- algorithmic work models ------------------------------------------------
def pair_flops(lmax: int, accepted: int, candidates: int) -> float:
    """per accepted pair 4.5 (lmax+1)^2 + 25 flop, per rejected candidate 12 flop."""
    return accepted * (4.5 * (lmax + 1) ** 2 + 25.0) + max(0, candidates - accepted) * 12.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.stop = [], threading.Event()
        self.index = index
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
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
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def make_catalogue(cfg: W.Config, rank: int):
    if rank:
        cfg = dataclasses.replace(cfg, seed=cfg.seed + 100 * rank)
    return W.make(cfg)


def oracle_sample(cfg: W.Config, pos, w, target_s: float = 15.0):
    """Oracle (as it stands) on primaries 0, stride, 2 stride, ...; returns (primaries/s, description, cores, seconds)."""
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    n = cfg.n
    probe = max(1, n // (8 * cores))              # a first tiny sample to size the real one
    t0 = time.perf_counter()
    oracle.zeta(cfg.order, pos, w, cfg.box, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax, prim_stride=max(1, n // probe))
    dt = time.perf_counter() - t0
    per_prim = dt / max(1, len(range(0, n, max(1, n // probe))))
    want = int(min(n, max(probe, target_s / max(per_prim, 1e-9))))
    stride = max(1, n // want)
    cnt = len(range(0, n, stride))
    t0 = time.perf_counter()
    oracle.zeta(cfg.order, pos, w, cfg.box, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax, prim_stride=stride)
    dt = time.perf_counter() - t0
    return cnt / dt, f"{cnt} of {n} primaries (every {stride}th) against the full catalogue, {dt:.1f} s", cores, dt


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pos, w = make_catalogue(cfg, 0)
    vals = []
    per = max(2.0, 60.0 / max(1, args.steps + args.warmup))
    for it in range(args.warmup + args.steps):
        v, desc, cores, dt = oracle_sample(cfg, pos, w, target_s=per)
        if it >= args.warmup:
            vals.append((v, dt, desc))
    value = statistics.mean(v for v, _, _ in vals)
    line = {
        "impl": "reference", "metric": "primaries_per_s", "value": value, "unit": "primaries/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * statistics.mean(d for _, d, _ in vals),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args),
        "cpu_baseline": {"value": value, "unit": "primaries/s", "cores": cores, "kind": "oracle", "sample": vals[-1][2]},
        "e2e": {"value": value, "unit": "primaries/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def workload_config(cfg, args):
    return {"workload": f"{cfg.name}{' ALLPARITY' if getattr(args, 'allparity', False) else ''}: {cfg.order}PCF, n={cfg.n} {cfg.kind} points, "
                        f"{'periodic L=%g' % cfg.box if cfg.box > 0 else 'open cut-sky shell'}, weights {cfg.weights}, "
                        f"{cfg.nbins} bins in [{cfg.rmin:g},{cfg.rmax:g}], lmax={cfg.lmax}",
            "l2": "256 MiB device memset between steps inside the timed bracket; per-step intermediates (a_lm tiles, "
                  "per-group zeta partials) exceed the 126 MB L2",
            "sharding": "one independent catalogue per rank (seed + 100 rank), no collective"}


def measure_config(E, torch, cfg, rank, steps, warmup, dev, want_e2e=True, allparity=False):
    pos, w = make_catalogue(cfg, rank)
    tp, tw = torch.from_numpy(pos).to(dev), torch.from_numpy(w).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    plan = E.Plan(cfg.order, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax, cfg.box, allparity=allparity)
    E.encore_set_timing(plan.h, True)
    out = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev)
    for _ in range(warmup):
        flush.zero_()
        plan.compute(tp, tw, out=out)
    torch.cuda.synchronize(dev)
    stages = []
    barrier()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        flush.zero_()
        plan.compute(tp, tw, out=out)
        stages.append(E.encore_get_stage_ms(plan.h))   # events of the library's own stream records; syncs that step
    e1.record(stream)
    torch.cuda.synchronize(dev)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = E.encore_get_launch_count(plan.h)
    counts, pairs = E.encore_get_bin_counts(plan.h, cfg.nbins)
    cand = E.encore_get_candidate_pairs(plan.h)
    res = {"ms_total": ms, "stages": {k: statistics.mean(s[k] for s in stages) for k in stages[0]}, "launches": launches,
           "pairs": pairs, "candidates": cand, "flops_contraction": E.encore_contraction_flops(plan.h),
           "nout": plan.n_lambda * plan.n_b, "grid": E.encore_get_grid(plan.h)}
    if want_e2e:
        hp = torch.from_numpy(pos).pin_memory()
        hw = torch.from_numpy(w).pin_memory()
        hz = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64).pin_memory()
        for _ in range(min(warmup, 2)):
            E.encore_compute_host(plan.h, hp, hw, cfg.n, hz)
        barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for _ in range(steps):
            flush.zero_()
            E.encore_compute_host(plan.h, hp, hw, cfg.n, hz)   # synchronises: zeta is on the host when it returns
        torch.cuda.synchronize(dev)
        res["e2e_ms_total"] = 1e3 * (time.perf_counter() - t0)
        res["h2d"] = pos.nbytes + w.nbytes
        res["d2h"] = hz.numel() * 8
    plan.close()
    return res, (pos, w)


_DIST = {"on": False}


def barrier():
    if _DIST["on"]:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(torch, value: float, dev) -> float:
    if not _DIST["on"]:
        return value
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c3", choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--all-configs", action="store_true", help="also measure c1..c5 (2 steps each) into per_config")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--allparity", action="store_true", help="ALLPARITY plan: parity-odd multiplets too (not the headline config)")
    args = ap.parse_args()
    cfg = W.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import paper_2105_08722_b200 as E
    E.lib()                                       # fails loudly if the CUDA library is missing / cannot be built
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
        _DIST["on"] = True
    hbm_gbs, sm_max_mhz, peak_src = peaks()
    steps, warmup = args.steps, max(3, args.warmup)

    with ClockSampler(local) as clocks:
        res, (pos, w) = measure_config(E, torch, cfg, rank, steps, warmup, dev, allparity=args.allparity)
    ms_total = max_over_ranks(torch, res["ms_total"], dev)
    e2e_ms = max_over_ranks(torch, res["e2e_ms_total"], dev)
    ms_per_step = ms_total / steps
    value = world * cfg.n / (ms_per_step * 1e-3)
    st = res["stages"]

    fp64_measured = E.encore_measure_fp64_peak()
    peak_derived = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6
    pf = pair_flops(cfg.lmax, res["pairs"], res["candidates"])
    pair_tflops = pf / (st["pair"] * 1e-3) / 1e12
    ex_flops, ca_flops = res["flops_contraction"]
    grid_bytes = cfg.n * (24 + 4)                        # a1: read x,y,z, write cell id
    sort_bytes = cfg.n * (4 + 4 + 4 + 4 + 4 + 32 + 32)   # a2: cid re-read, scatter idx w+r, rank idx, pos+w gather r+w
    line = {
        "metric": "primaries_per_s", "value": value, "unit": "primaries/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args),
        "pairs_per_s": world * res["pairs"] / (ms_per_step * 1e-3),
        "pairs_per_s_pair_stage": res["pairs"] / (st["pair"] * 1e-3),
        "accepted_pairs": res["pairs"], "candidate_pairs": res["candidates"],
        "contraction_gflops_canonical": cfg.n * ca_flops / (st["contraction"] * 1e-3) / 1e9,
        "contraction_gflops_executed": cfg.n * ex_flops / (st["contraction"] * 1e-3) / 1e9,
        "stage_ms": st,
        "stage_rooflines": {
            "grid_GBps": grid_bytes / (st["grid"] * 1e-3) / 1e9, "sort_GBps": sort_bytes / (st["sort"] * 1e-3) / 1e9,
            "hbm_peak_GBps": hbm_gbs,
            "pair_frac_fp64": pair_tflops * 1e12 / peak_derived,
            "contraction_frac_fp64_executed": cfg.n * ex_flops / (st["contraction"] * 1e-3) / peak_derived,
        },
        "roofline": {"bound": "alu", "kernel": "k_pair (a3+a4)", "achieved": pair_tflops, "peak": peak_derived / 1e12,
                     "unit": "TFLOP/s", "frac": pair_tflops * 1e12 / peak_derived,
                     "traffic": NCU_PAIR_STAGE_DRAM_BYTES.get(cfg.name),
                     "peak_source": f"derived: {SM_COUNT} SM x {FP64_LANES_PER_SM} fp64 FMA lanes x 2 x {sm_max_mhz:g} MHz ({peak_src} clock)",
                     "peak_measured_dfma_chain": fp64_measured / 1e12,
                     "flops_model": "4.5 (lmax+1)^2 + 25 per accepted pair + 12 per rejected candidate (DESIGN.md §7)"},
        "e2e": {"value": world * cfg.n / (e2e_ms / steps * 1e-3), "unit": "primaries/s",
                "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"]},
        "gpu_launches": res["launches"] * steps,
        "clocks": clocks.summary(),
        "grid": {"nc": res["grid"][0], "sub": res["grid"][1]},
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, desc, cores, _ = oracle_sample(cfg, pos, w, target_s=15.0)
        line["cpu_baseline"] = {"value": v, "unit": "primaries/s", "cores": cores, "kind": "oracle", "sample": desc}
    if args.all_configs and world == 1:
        per = {}
        for name in sorted(W.CONFIGS):
            c = W.CONFIGS[name]
            r, _ = measure_config(E, torch, c, 0, 2, 3, dev, want_e2e=False)
            s = r["stages"]
            ex, ca = r["flops_contraction"]
            ms1 = r["ms_total"] / 2
            per[name] = {"order": c.order, "n": c.n, "ms_per_step": ms1, "primaries_per_s": c.n / (ms1 * 1e-3),
                         "pairs_per_s": r["pairs"] / (ms1 * 1e-3), "accepted_pairs": r["pairs"], "stage_ms": s,
                         "pair_frac_fp64": pair_flops(c.lmax, r["pairs"], r["candidates"]) / (s["pair"] * 1e-3) / peak_derived,
                         "contraction_gflops_canonical": c.n * ca / (s["contraction"] * 1e-3) / 1e9,
                         "contraction_frac_fp64_executed": c.n * ex / (s["contraction"] * 1e-3) / peak_derived}
        # the same c3 catalogue with the parity-odd multiplets too (111 instead of 69 multiplets)
        r, _ = measure_config(E, torch, W.CONFIGS["c3"], 0, 2, 3, dev, want_e2e=False, allparity=True)
        ex, ca = r["flops_contraction"]
        per["c3_allparity"] = {"order": 4, "n": W.CONFIGS["c3"].n, "ms_per_step": r["ms_total"] / 2,
                               "primaries_per_s": W.CONFIGS["c3"].n / (r["ms_total"] / 2 * 1e-3), "stage_ms": r["stages"],
                               "n_multiplets": r["nout"] // 120,
                               "contraction_gflops_canonical": W.CONFIGS["c3"].n * ca / (r["stages"]["contraction"] * 1e-3) / 1e9,
                               "contraction_frac_fp64_executed": W.CONFIGS["c3"].n * ex / (r["stages"]["contraction"] * 1e-3) / peak_derived}
        line["per_config"] = per
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
