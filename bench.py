#!/usr/bin/env python
"""bench.py — throughput of the ENCORE hot path (steps a1..a6) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--impl ours|reference] [--no-per-config]

A "step" is one encore_compute over one synthetic catalogue (all of a1..a6).  The default workload is c3, the
4PCF configuration BASELINE.json's target is stated on (300 000 lognormal-clustered points, 10 bins in [20,160],
lmax=5); the default line also carries one measured entry per config c1..c5 under "per_config" (2 steps each).
  value  = primaries/s with the catalogue already resident in HBM (CUDA events over K steps, max over ranks);
  e2e    = the same through encore_compute_host with pinned HOST buffers (H2D of positions+weights and D2H of
           zeta inside the timed region);
  roofline = the kernel that takes the largest share of the step, `roofline_kernels` = one entry per real kernel
           (k_fill, k_harm<..>, k_contract*), each timed live with the library's CUDA events on the compute stream;
           algorithmic flops per DESIGN.md §7; plain FP64 / FP32 ALU bounds;
  cpu_baseline = the oracle as it stands on this box's host cores on a strided subset of primaries, with its own
           split into a_lm-stage and contraction seconds.
N > 1 (torchrun): ONE catalogue sharded over primaries (encore_compute_shard + the NCCL all-gather of
paper_2105_08722_b200.sharded inside the timed region), "scaling": "strong";
the independent-catalogue arm (one mock per rank, no collective) is reported beside it under "replicas".
`--impl reference` times the CPU oracle (test infrastructure) on the same config and metric.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import platform
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

SM_COUNT, FP64_LANES_PER_SM, FP32_LANES_PER_SM = 148, 64, 128
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures of this
# round's kernels (profiles/r2_ncu_full_c3.txt and r2_ncu_full_c5.txt name the commands); None where not captured
NCU_DRAM_BYTES = {"c3": {"k_fill": 1.947e9, "k_harm": 2.958e9, "k_contract": 9.587e9}, "c5": {"k_contract": 9.243e9}}
NCU_PROFILE = {"c3": "profiles/r2_ncu_full_c3.txt", "c5": "profiles/r2_ncu_full_c5.txt"}   # where NCU_DRAM_BYTES comes from


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


# ---- algorithmic work models ------------------------------------------------
def pair_flops(lmax: int, accepted: int, candidates: int) -> float:
    """stage model: per accepted pair 4.5 (lmax+1)^2 + 25 flop, per rejected candidate 12 flop."""
    return accepted * (4.5 * (lmax + 1) ** 2 + 25.0) + max(0, candidates - accepted) * 12.0


def fill_flops(candidates: int) -> float:
    """k_fill's share of the stage model: separation + r^2 + bin of every candidate that reaches the pair test."""
    return 12.0 * candidates


def harm_flops(lmax: int, accepted: int) -> float:
    """k_harm's share: everything of an accepted pair but the 12 flop already charged to k_fill."""
    return accepted * (4.5 * (lmax + 1) ** 2 + 13.0)


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


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return platform.processor() or "unknown"


def oracle_sample(cfg: W.Config, pos, w, target_s: float = 15.0):
    """Oracle (as it stands) on primaries 0, stride, 2 stride, ... against the full catalogue.

    Returns dict(value primaries/s, sample, cores, seconds, pair_stage_seconds, contraction_seconds)."""
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
    o = oracle.zeta(cfg.order, pos, w, cfg.box, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax, prim_stride=stride)
    dt = time.perf_counter() - t0
    return {"value": cnt / dt, "sample": f"{cnt} of {n} primaries (every {stride}th) against the full catalogue, {dt:.1f} s",
            "cores": cores, "seconds": dt, "pair_stage_seconds": o["stage_seconds"][0], "contraction_seconds": o["stage_seconds"][1]}


def cpu_baseline_entry(s):
    return {"value": s["value"], "unit": "primaries/s", "cores": s["cores"], "kind": "oracle", "sample": s["sample"],
            "pair_stage_seconds": s["pair_stage_seconds"], "contraction_seconds": s["contraction_seconds"],
            "nproc": os.cpu_count(), "cpu_model": cpu_model()}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pos, w = make_catalogue(cfg, 0)
    vals = []
    per = max(2.0, 60.0 / max(1, args.steps + args.warmup))
    for it in range(args.warmup + args.steps):
        s = oracle_sample(cfg, pos, w, target_s=per)
        if it >= args.warmup:
            vals.append(s)
    value = statistics.mean(s["value"] for s in vals)
    line = {
        "impl": "reference", "metric": "primaries_per_s", "value": value, "unit": "primaries/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * statistics.mean(s["seconds"] for s in vals),
        "higher_is_better": True, "scaling": "strong" if args.gpus > 1 else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args.gpus),
        "cpu_baseline": dict(cpu_baseline_entry(vals[-1]), value=value),
        "e2e": {"value": value, "unit": "primaries/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def workload_config(cfg, world, allparity=False):
    return {"workload": f"{cfg.name}{' ALLPARITY' if allparity else ''}: {cfg.order}PCF, n={cfg.n} {cfg.kind} points, "
                        f"{'periodic L=%g' % cfg.box if cfg.box > 0 else 'open cut-sky shell'}, weights {cfg.weights}, "
                        f"{cfg.nbins} bins in [{cfg.rmin:g},{cfg.rmax:g}], lmax={cfg.lmax}",
            "l2": "256 MiB device memset between steps inside the timed bracket; per-step intermediates (acceptance-mask rows, "
                  "a_lm tiles) exceed the 126 MB L2",
            "sharding": ("one catalogue, primaries sharded over the ranks (encore_compute_shard), one NCCL all-gather of the "
                         "partial zeta per step" if world > 1 else "single GPU")}


def measure_config(E, torch, cfg, rank, steps, warmup, dev, want_e2e=True, allparity=False, shard=None, fp32_harmonics=False,
                   keep_zeta=False, want_graph=False):
    """shard = (rank, world): time sharded.compute_sharded (one catalogue, all-gather inside); None: the whole catalogue."""
    from paper_2105_08722_b200 import sharded
    pos, w = make_catalogue(cfg, rank if shard is None else 0)
    tp, tw = torch.from_numpy(pos).to(dev), torch.from_numpy(w).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    plan = E.Plan(cfg.order, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax, cfg.box, allparity=allparity, fp32_harmonics=fp32_harmonics)
    E.encore_set_timing(plan.h, True)
    out = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev)

    def one_step():
        flush.zero_()
        if shard is None:
            plan.compute(tp, tw, out=out)
        else:
            sharded.compute_sharded(plan, tp, tw)

    for _ in range(warmup):
        one_step()
    torch.cuda.synchronize(dev)
    kern = []
    barrier()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        one_step()
        kern.append(E.encore_get_kernel_ms(plan.h))   # events of the library's own stream records; syncs that step
    e1.record(stream)
    torch.cuda.synchronize(dev)
    barrier()
    ms = e0.elapsed_time(e1)
    assert E.encore_get_status(plan.h) == E.OK
    launches = E.encore_get_launch_count(plan.h)
    counts, pairs = E.encore_get_bin_counts(plan.h, cfg.nbins)
    cand = E.encore_get_candidate_pairs(plan.h)
    km = {k: statistics.mean(s[k] for s in kern) for k in kern[0]}
    res = {"ms_total": ms, "kernel_ms": km, "launches": launches, "pairs": pairs, "candidates": cand,
           "flops_contraction": E.encore_contraction_flops(plan.h), "nout": plan.n_lambda * plan.n_b,
           "grid": E.encore_get_grid(plan.h), "pair_steps": E.encore_get_pair_steps(plan.h)}
    if keep_zeta and shard is None:
        res["zeta"] = out.cpu().numpy()
    if want_graph and shard is None:
        # encore_compute_enqueue (no read-back, no allocation) captured once into a CUDA graph and replayed: the step without
        # the two host read-backs and the launch latencies of encore_compute (same kernels, same flush between replays)
        E.encore_set_timing(plan.h, False)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            flush.zero_()
            plan.compute_enqueue(tp, tw, out, pos.min(axis=1), pos.max(axis=1))
        g.replay()
        torch.cuda.synchronize(dev)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for _ in range(steps):
            g.replay()
        g1.record(stream)
        torch.cuda.synchronize(dev)
        assert E.encore_get_status(plan.h) == E.OK
        res["graph_replay_ms"] = g0.elapsed_time(g1) / steps
        del g
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


def stage_ms(km):
    return {"grid": km["grid"], "sort": km["sort"], "pair": km["bounds"] + km["k_fill"] + km["k_harm"],
            "contraction": km["k_contract"], "reduce": km["reduce"]}


def kernel_rooflines(cfg, res, fp64_peak, fp32_peak):
    """one entry per real kernel of the step, the one with the largest share of the step first"""
    km = res["kernel_ms"]
    ex, ca = res["flops_contraction"]
    hname = f"k_harm<{cfg.lmax}, 0, {cfg.lmax if cfg.lmax <= 7 else (2 if cfg.lmax == 8 else 3)}, {1 if cfg.box > 0 else 0}, 0>"
    if cfg.lmax > 7:
        hname += f" + k_harm<{cfg.lmax}, {3 if cfg.lmax == 8 else 4}, {cfg.lmax}, {1 if cfg.box > 0 else 0}, 0>"
    cname = {3: f"k_contract3<{cfg.nbins}>", 4: f"k_contract4<{cfg.nbins}>", 5: f"k_contract5<{cfg.nbins}>"}[cfg.order]
    traffic = NCU_DRAM_BYTES.get(cfg.name, {})
    ents = []

    def ent(kernel, ms, flops, peak, bound, unit_peak, **extra):
        ach = flops / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        e = {"kernel": kernel, "bound": bound, "ms": ms, "achieved": ach, "peak": peak / 1e12, "unit": "TFLOP/s",
             "frac": ach * 1e12 / peak, "share_of_step": None, "peak_kind": unit_peak}
        e.update(extra)
        return e
    ents.append(ent(f"k_fill<{1 if cfg.box > 0 else 0}>", km["k_fill"], fill_flops(res["candidates"]), fp32_peak, "alu", "fp32 FMA lanes",
                    model="12 flop per candidate pair that reaches the pair test (fp32 screening, exact fp64 fallback); the kernel is "
                          "bound by instruction issue (integer + fp32 mix), not by the fp32 pipe",
                    traffic=traffic.get("k_fill")))
    ents.append(ent(hname, km["k_harm"], harm_flops(cfg.lmax, res["pairs"]), fp64_peak, "alu", "fp64 FMA lanes",
                    model="4.5 (lmax+1)^2 + 13 flop per accepted pair", traffic=traffic.get("k_harm")))
    ents.append(ent(cname, km["k_contract"], cfg.n * ex, fp64_peak, "alu" if cfg.order > 3 else "hbm", "fp64 FMA lanes",
                    model="executed flops of the factorised kernel (FMA = 2), encore_contraction_flops",
                    canonical_model_tflops=cfg.n * ca / (km["k_contract"] * 1e-3) / 1e12 if km["k_contract"] > 0 else 0.0,
                    traffic=traffic.get("k_contract")))
    tot = sum(km.values())
    for e in ents:
        e["share_of_step"] = e["ms"] / tot if tot > 0 else 0.0
    ents.sort(key=lambda e: -e["ms"])
    return ents


def config_entry(cfg, res, steps, fp64_peak, fp32_peak, fp32_harmonics=False):
    ms1 = res["ms_total"] / steps
    km = res["kernel_ms"]
    st = stage_ms(km)
    ex, ca = res["flops_contraction"]
    pf = pair_flops(cfg.lmax, res["pairs"], res["candidates"])
    if fp32_harmonics:
        # the per-pair arithmetic of k_harm runs on the fp32 lanes here (fp64 only for the 64-pair chunk flushes): its work is
        # set against the fp32 peak; fractions of the fp64 peak would be meaningless for this path and are not reported
        return {"order": cfg.order, "n": cfg.n, "ms_per_step": ms1, "primaries_per_s": cfg.n / (ms1 * 1e-3),
                "pairs_per_s": res["pairs"] / (ms1 * 1e-3), "accepted_pairs": res["pairs"], "candidate_pairs": res["candidates"],
                "pair_steps": res["pair_steps"], "stage_ms": st, "kernel_ms": km,
                "k_harm_frac_fp32": harm_flops(cfg.lmax, res["pairs"]) / (km["k_harm"] * 1e-3) / fp32_peak if km["k_harm"] > 0 else 0.0,
                "contraction_gflops_executed": cfg.n * ex / (st["contraction"] * 1e-3) / 1e9,
                "contraction_frac_fp64_executed": cfg.n * ex / (st["contraction"] * 1e-3) / fp64_peak}
    return {"order": cfg.order, "n": cfg.n, "ms_per_step": ms1, "primaries_per_s": cfg.n / (ms1 * 1e-3),
            "pairs_per_s": res["pairs"] / (ms1 * 1e-3), "accepted_pairs": res["pairs"], "candidate_pairs": res["candidates"],
            "pair_steps": res["pair_steps"], "stage_ms": st, "kernel_ms": km,
            "pair_frac_fp64": pf / (st["pair"] * 1e-3) / fp64_peak,
            "pair_frac_fp64_accepted_only": res["pairs"] * (4.5 * (cfg.lmax + 1) ** 2 + 25.0) / (st["pair"] * 1e-3) / fp64_peak,
            "k_harm_frac_fp64": harm_flops(cfg.lmax, res["pairs"]) / (km["k_harm"] * 1e-3) / fp64_peak if km["k_harm"] > 0 else 0.0,
            "contraction_gflops_canonical": cfg.n * ca / (st["contraction"] * 1e-3) / 1e9,
            "contraction_gflops_executed": cfg.n * ex / (st["contraction"] * 1e-3) / 1e9,
            "contraction_frac_fp64_executed": cfg.n * ex / (st["contraction"] * 1e-3) / fp64_peak}


def measure_next_rows(E, torch, dev, fp64_peak):
    """SURVEY.md §8(f1)-(f3) beside the five configs: 6PCF (literal eq. 44 kernel), edge correction, gridded estimator.
    CUDA events on torch's current stream (the stream the calls are enqueued on), 3 warm-up + 3 timed calls each."""
    import dataclasses
    out = {}
    stream = torch.cuda.current_stream(dev)

    def timed(fn, reps=3):
        for _ in range(3):
            fn()
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize(dev)
        return e0.elapsed_time(e1) / reps

    # (f1) 6PCF on the catalogue of c5 (300 000 lognormal points, 8 bins in [20,160]) at lmax = 2: 327 multiplets x 56 bin
    # quintuples, factorised kernel k_contract6<8>; the literal eq. 44 kernel on a 20 000-point sub-box beside it
    c6 = dataclasses.replace(W.CONFIGS["c5"], order=6, lmax=2, name="c5 catalogue")
    pos, w = W.make(c6)
    tp, tw = torch.from_numpy(pos).to(dev), torch.from_numpy(w).to(dev)
    with E.Plan(6, c6.rmin, c6.rmax, c6.nbins, c6.lmax, c6.box) as plan:
        E.encore_set_timing(plan.h, True)
        z = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
        ms = timed(lambda: plan.compute(tp, tw, out=z))
        km = E.encore_get_kernel_ms(plan.h)
        ex, ca = E.encore_contraction_flops(plan.h)
        out["f1_6pcf"] = {"workload": f"6PCF, n={c6.n} lognormal points (the catalogue of c5), periodic L={c6.box:g}, {c6.nbins} bins in [20,160], "
                                      f"lmax={c6.lmax}: {plan.n_lambda} multiplets x {plan.n_b} bin tuples, {E.encore_num_terms(plan.h)} terms",
                          "ms_per_step": ms, "primaries_per_s": c6.n / (ms * 1e-3), "kernel_ms": km, "kernel": "k_contract6<8> (factorised, contract6.cu)",
                          "contraction_flops_per_primary_executed": ex, "contraction_flops_per_primary_canonical": ca,
                          "contraction_frac_fp64_executed": c6.n * ex / (km["k_contract"] * 1e-3) / fp64_peak}
        sel = (pos[0] < 406.0) & (pos[1] < 406.0) & (pos[2] < 406.0)
        ps, ws = np.ascontiguousarray(pos[:, sel]), np.ascontiguousarray(w[sel])
    with E.Plan(6, c6.rmin, c6.rmax, c6.nbins, c6.lmax, 0.0) as plan:
        tps, tws = torch.from_numpy(ps).to(dev), torch.from_numpy(ws).to(dev)
        E.encore_set_timing(plan.h, True)
        z = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
        res, zs = {}, {}
        for tag, lit in (("factorised", 0), ("literal_eq44", 1)):
            E.encore_set_option(plan.h, "generic_contract", lit)
            timed(lambda: plan.compute(tps, tws, out=z), reps=2)
            res[tag + "_contraction_ms"] = E.encore_get_kernel_ms(plan.h)["k_contract"]
            res[tag + "_flops_per_primary"] = E.encore_contraction_flops(plan.h)[0]
            zs[tag] = z.cpu().numpy().copy()
        # the two kernels share the a_lm tiles and nothing else: their agreement at this depth (hundreds of tiles per CTA)
        # is checked, not just timed
        diff = float(np.abs(zs["factorised"] - zs["literal_eq44"]).max() / np.abs(zs["literal_eq44"]).max())
        assert diff <= 1e-12, f"factorised and literal 6PCF kernels differ by {diff:.3e} of max|zeta|"
        res["max_rel_diff_factorised_vs_literal"] = diff
        out["f1_6pcf"]["sub_box"] = dict(res, n=int(ps.shape[1]), note="open-geometry sub-box of the same catalogue, both contraction kernels")
    # the shapes of the paper's Table 2: ~5e4 uniform points in a periodic box L = 1500, N_r = 10 bins up to
    # r_max = 200, 4PCF at lmax = 5 and 10, 5PCF at lmax = 5.  The paper's seconds (16-core Skylake / best P100 row, a_lm on one
    # CPU core) are context from other hardware, quoted beside this run's time; they are not a target and not a ratio.
    t2 = W.TABLE2
    pos, w = W.make(t2)
    tp, tw = torch.from_numpy(pos).to(dev), torch.from_numpy(w).to(dev)
    rows = {}
    for tag, order, lmax, cpu_s, gpu_s in (("4pcf_lmax5", 4, 5, 4.8, 21.9), ("4pcf_lmax10", 4, 10, 58.8, 38.4), ("5pcf_lmax5", 5, 5, 741.8, 74.3)):
        with E.Plan(order, t2.rmin, t2.rmax, t2.nbins, lmax, t2.box) as plan:
            E.encore_set_timing(plan.h, True)
            z = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
            ms = timed(lambda: plan.compute(tp, tw, out=z))
            km = E.encore_get_kernel_ms(plan.h)
            ex, ca = E.encore_contraction_flops(plan.h)
            rows[tag] = {"outputs": plan.n_lambda * plan.n_b, "ms_per_catalogue": ms, "primaries_per_s": t2.n / (ms * 1e-3), "kernel_ms": km,
                         "contraction_frac_fp64_executed": t2.n * ex / (km["k_contract"] * 1e-3) / fp64_peak,
                         "paper_seconds_16core_cpu": cpu_s, "paper_seconds_best_p100_row": gpu_s}
    out["paper_table2_shapes"] = dict(rows, workload=f"n={t2.n} uniform points, periodic L={t2.box:g}, {t2.nbins} bins in [0,200] (PAPER.md:578)")
    # (f2) edge correction at the shape of c3 / c4: 69 multiplets, 120 bin tuples (120 LU solves of 69 unknowns)
    c3 = W.CONFIGS["c3"]
    with E.Plan(c3.order, c3.rmin, c3.rmax, c3.nbins, c3.lmax, 0.0) as plan:
        g = torch.Generator(device="cpu").manual_seed(42)
        R = torch.randn((plan.n_lambda, plan.n_b), generator=g, dtype=torch.float64) * 0.1
        R[0] = 1.0 + torch.rand(plan.n_b, generator=g, dtype=torch.float64)
        R[1:] *= R[0]
        N = torch.randn((plan.n_lambda, plan.n_b), generator=g, dtype=torch.float64)
        tn, tr = N.to(dev), R.to(dev)
        z = torch.empty_like(tn)
        plan.edge_correct(tn, tr, out=z)          # builds the E G tensor on the host once
        ms = timed(lambda: plan.edge_correct(tn, tr, out=z), reps=10)
        out["f2_edge_correction"] = {"workload": f"eq. 41/42 for {plan.n_lambda} multiplets x {plan.n_b} bin tuples (the shape of c3 / c4)",
                                     "ms_per_call": ms, "kernels": "k_edge_assemble + k_edge_solve (one CTA per bin tuple)"}
    # (f3) gridded estimator: a 64^3 mesh in the box of c3, 4PCF with the bins and lmax of c3
    G = 64
    rng = np.random.default_rng(64)
    delta = torch.from_numpy(rng.standard_normal((G, G, G)) * 0.5).to(dev)
    with E.Plan(c3.order, c3.rmin, c3.rmax, c3.nbins, c3.lmax, c3.box) as plan:
        E.encore_set_timing(plan.h, True)
        z = torch.empty((plan.n_lambda, plan.n_b), dtype=torch.float64, device=dev)
        ms = timed(lambda: plan.compute_grid(delta, out=z))
        out["f3_gridded"] = {"workload": f"4PCF of a {G}^3 mesh, periodic L={c3.box:g}, {c3.nbins} bins in [20,160], lmax={c3.lmax} "
                                         f"({c3.nbins * (c3.lmax + 1) * (c3.lmax + 2) // 2} FFT cross-correlations, then {G ** 3} cells through a5)",
                             "ms_per_step": ms, "cells_per_s": G ** 3 / (ms * 1e-3), "kernel_ms": E.encore_get_kernel_ms(plan.h)}
    return out


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
    ap.add_argument("--no-per-config", action="store_true", help="skip the c1..c5 entries (2 steps each) of per_config")
    ap.add_argument("--all-configs", action="store_true", help="(default now) kept for compatibility")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--allparity", action="store_true", help="ALLPARITY plan: parity-odd multiplets too (not the headline config)")
    ap.add_argument("--fp32-harmonics", action="store_true", help="ENCORE_FP32_HARMONICS plan (a separately reported path, tolerance 1e-5; not the headline)")
    ap.add_argument("--only-next-rows", action="store_true", help="measure and print only `next_rows` (6PCF, edge correction, gridded estimator)")
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
    fp64_peak = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6
    fp32_peak = SM_COUNT * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6
    if args.only_next_rows:
        if rank == 0:
            print(json.dumps({"next_rows": measure_next_rows(E, torch, dev, fp64_peak)}))
        return

    with ClockSampler(local) as clocks:
        res, (pos, w) = measure_config(E, torch, cfg, rank, steps, warmup, dev, allparity=args.allparity,
                                       shard=(rank, world) if world > 1 else None, fp32_harmonics=args.fp32_harmonics)
    ms_total = max_over_ranks(torch, res["ms_total"], dev)
    e2e_ms = max_over_ranks(torch, res["e2e_ms_total"], dev)
    ms_per_step = ms_total / steps
    value = cfg.n / (ms_per_step * 1e-3)          # world > 1: ONE catalogue, sharded (strong scaling)
    km = res["kernel_ms"]
    st = stage_ms(km)

    fp64_measured = E.encore_measure_fp64_peak()
    dmma_measured = E.encore_measure_dmma_peak()
    ents = kernel_rooflines(cfg, res, fp64_peak, fp32_peak)
    top = ents[0]
    pf = pair_flops(cfg.lmax, res["pairs"], res["candidates"])
    ex_flops, ca_flops = res["flops_contraction"]
    grid_bytes = cfg.n * (24 + 4)                        # a1: read x,y,z, write cell id
    sort_bytes = cfg.n * (4 + 4 + 4 + 4 + 4 + 32 + 32)   # a2: cid re-read, scatter idx w+r, rank idx, pos+w gather r+w
    line = {
        "metric": "primaries_per_s", "value": value, "unit": "primaries/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if world > 1 else "weak", "vs_baseline": None,
        "dtype": "f32 harmonics, f64 accumulation / contraction" if args.fp32_harmonics else "f64", "data": "synthetic",
        "config": workload_config(cfg, world, args.allparity),
        "pairs_per_s": res["pairs"] / (ms_per_step * 1e-3) if world == 1 else None,   # (a shard only counts its own pairs)
        "accepted_pairs": res["pairs"], "candidate_pairs": res["candidates"],
        "contraction_gflops_canonical": cfg.n * ca_flops / (st["contraction"] * 1e-3) / 1e9 if world == 1 else None,
        "contraction_gflops_executed": cfg.n * ex_flops / (st["contraction"] * 1e-3) / 1e9 if world == 1 else None,
        "stage_ms": st, "kernel_ms": km,
        "stage_rooflines": {
            "grid_GBps": grid_bytes / (st["grid"] * 1e-3) / 1e9, "sort_GBps": sort_bytes / (st["sort"] * 1e-3) / 1e9,
            "hbm_peak_GBps": hbm_gbs,
            "pair_frac_fp64": pf / (st["pair"] * 1e-3) / fp64_peak,
            "pair_frac_fp64_accepted_only": res["pairs"] * (4.5 * (cfg.lmax + 1) ** 2 + 25.0) / (st["pair"] * 1e-3) / fp64_peak,
            "contraction_frac_fp64_executed": cfg.n * ex_flops / (st["contraction"] * 1e-3) / fp64_peak,
        },
        "roofline": {"bound": top["bound"], "kernel": top["kernel"], "achieved": top["achieved"], "peak": top["peak"],
                     "unit": "TFLOP/s", "frac": top["frac"], "traffic": top.get("traffic"), "traffic_source": NCU_PROFILE.get(cfg.name) if top.get("traffic") is not None else None,
                     "traffic_kind": "from_profile (a constant copied from the named ncu capture of this kernel, not measured by this run)" if top.get("traffic") is not None else None,
                     "ms": top["ms"], "share_of_step": top["share_of_step"], "model": top["model"],
                     "peak_source": f"derived: {SM_COUNT} SM x {FP64_LANES_PER_SM} fp64 (x {FP32_LANES_PER_SM} fp32) FMA lanes x 2 x "
                                    f"{sm_max_mhz:g} MHz ({peak_src} clock); MEASURED_PEAKS.json has no fp64 entry",
                     "peak_measured_dfma_chain": fp64_measured / 1e12,
                     "peak_measured_dmma_m8n8k4": dmma_measured / 1e12},
        "roofline_kernels": ents,
        "e2e": {"value": cfg.n / (e2e_ms / steps * 1e-3), "unit": "primaries/s",
                "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"],
                "note": "encore_compute_host on this rank's GPU (whole catalogue)" if world > 1 else "encore_compute_host"},
        "gpu_launches": res["launches"] * steps,
        "clocks": clocks.summary(),
        "grid": {"nc": res["grid"][0], "sub": res["grid"][1]},
    }
    if world > 1:
        # the independent-catalogue arm: one mock per rank, no data-path collective, weak scaling
        r2, _ = measure_config(E, torch, cfg, rank, max(2, steps // 2), 3, dev, want_e2e=False)
        ms_rep = max_over_ranks(torch, r2["ms_total"], dev) / max(2, steps // 2)
        line["replicas"] = {"value": world * cfg.n / (ms_rep * 1e-3), "unit": "primaries/s", "scaling": "weak", "ms_per_step": ms_rep,
                            "sharding": "one independent catalogue per rank (seed + 100 rank), no collective"}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_entry(oracle_sample(cfg, pos, w, target_s=15.0))
    if world == 1 and not args.no_per_config:
        per, z64, pairs64 = {}, {}, {}
        for name in sorted(W.CONFIGS):
            c = W.CONFIGS[name]
            r, _ = measure_config(E, torch, c, 0, 2, 3, dev, want_e2e=False, want_graph=True, keep_zeta=name in ("c3", "c4"))
            per[name] = config_entry(c, r, 2, fp64_peak, fp32_peak)
            per[name]["graph_replay_ms_per_step"] = r["graph_replay_ms"]   # encore_compute_enqueue replayed from a CUDA graph
            if "zeta" in r:
                z64[name], pairs64[name] = r["zeta"], r["pairs"]
        # the same c3 catalogue with the parity-odd multiplets too (111 instead of 69 multiplets)
        r, _ = measure_config(E, torch, W.CONFIGS["c3"], 0, 2, 3, dev, want_e2e=False, allparity=True)
        per["c3_allparity"] = dict(config_entry(W.CONFIGS["c3"], r, 2, fp64_peak, fp32_peak), n_multiplets=r["nout"] // 120)
        # fp32 harmonics with fp64 accumulation on the c3 and c4 catalogues - a separate path with its own
        # tolerance (1e-5); the difference to this run's fp64 result is reported beside its time
        for name in ("c3", "c4"):
            r32, _ = measure_config(E, torch, W.CONFIGS[name], 0, 2, 3, dev, want_e2e=False, fp32_harmonics=True, keep_zeta=True)
            e32 = config_entry(W.CONFIGS[name], r32, 2, fp64_peak, fp32_peak, fp32_harmonics=True)
            e32["dtype"] = "f32 harmonics, f64 accumulation / contraction"
            e32["max_rel_diff_to_fp64_run"] = float(np.abs(r32["zeta"] - z64[name]).max() / np.abs(z64[name]).max())
            e32["pairs_equal_fp64_run"] = bool(r32["pairs"] == pairs64[name])
            per[name + "_fp32_harmonics"] = e32
        line["per_config"] = per
        line["next_rows"] = measure_next_rows(E, torch, dev, fp64_peak)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
