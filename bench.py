#!/usr/bin/env python
"""bench.py -- throughput of the B200-native CT-AUX walker hot path (contract: see DESIGN.md section 10).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4_6x6_b20] [--sweeps-per-step S]
  python bench.py --impl reference ...     # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole hot path (S1..S5) over one batch of synthetic input:
`ctaux_sweep(S)` for all walkers of the workload, S = rebuild_every sweeps, so that every step holds
the S2 candidate GEMMs, the S3 proposal kernel, the S4 flushes and exactly one S5 rebuild.
The default workload is BASELINE.json configs[3] (6x6 cluster, beta=20, U=6, 8 walkers, delay 64),
the configuration the north_star's performance target is quoted on; all five configs are available
through --config / --all-configs.  Inputs are synthetic (closed-form cluster G0, Philox streams).

Prints ONE JSON line (rank 0).  No file under /root/reference is read.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from ctaux_workloads import CONFIGS, get_config, table_for, walker_seeds  # noqa: E402

METRIC = "accepted vertex updates/sec per B200 (batched walkers)"
UNIT = "updates/s"
# FP64 peak used for the roofline: MEASURED_PEAKS.json holds no FP64 figure, so the rule of the
# profiling guide is applied: measured bf16 dense peak x nominal ratio FP64 : bf16.
NOMINAL_FP64_TFLOPS = 40.0    # NVIDIA B200 datasheet, FP64 (vector = tensor) per GPU
NOMINAL_BF16_TFLOPS = 2250.0
FALLBACK_BF16_TFLOPS = 1590.0
FALLBACK_HBM_GBS = 6650.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the flush kernel from the committed `ncu --set full`
# capture of the SAME launch configuration, keyed (config, walkers per launch, delay): bytes per launch; absent = not
# captured (the field is null then)
FLUSH_TRAFFIC = {("cfg4_6x6_b20", 2, 64): 139.66e6}   # profiles/r2_flush_cand_full.md (third captured launch, k ~ 1700)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            mp = json.load(f)
        return dict(bf16=float(mp["bf16_tflops"]), bf16_sustained=float(mp.get("bf16_tflops_sustained", mp["bf16_tflops"])),
                    hbm=float(mp["hbm_gbs"]), source="measured")
    except Exception:
        return dict(bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0, hbm=FALLBACK_HBM_GBS, source="fallback")


def measure_fp64_peak(dev, n=8192, reps=5):
    """FP64 roofline denominator, measured live on this GPU the way MEASURED_PEAKS.json measures bf16:
    cuBLAS DGEMM (torch.matmul float64) n^3, best of `reps`, CUDA events.  MEASURED_PEAKS.json holds no
    FP64 figure; the figure derived from it by the guide's rule (bf16 x nominal FP64:bf16) is reported
    beside it as `peak_alt`."""
    import torch
    a = torch.randn(n, n, dtype=torch.float64, device=dev)
    b = torch.randn(n, n, dtype=torch.float64, device=dev)
    c = torch.empty_like(a)
    torch.matmul(a, b, out=c)
    torch.cuda.synchronize()
    best = 0.0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
    del a, b, c
    torch.cuda.empty_cache()
    return best


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().split(",")]
                if len(parts) >= 7:
                    self.rows.append(parts)
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in self.rows)
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(float(r[2]) for r in self.rows), "reasons": sorted(reasons),
                "samples": len(self.rows)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# --------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference): the oracle as it stands, never tuned.
ORACLE_WARMUP_SWEEPS = {"cfg1_2x2_b2": 200, "cfg2_2x2_b10": 60, "cfg3_4x4_b10": 40}


def oracle_start_state(cfg, table):
    """A THERMALISED start for the oracle sample, so that the CPU figure is taken at the same <k> and acceptance regime
    as the GPU figure (T1 costs O(k^2) per proposal): the oracle-written configuration of tests/golden when there is one
    (configs 3-5: minutes to hours of CPU to produce), else a warm-up run of the oracle itself (configs 1-2: seconds).
    Returns (site, tau, spin, id, next_id, p, description)."""
    import glob
    from oracle import ctaux_oracle as orc
    files = sorted(glob.glob(os.path.join(ROOT, "tests", "golden", f"thermalised_{cfg['name']}_seed*.txt")))
    if files:
        meta, rows = {}, []
        with open(files[0]) as f:
            for line in f:
                if line.startswith("#"):
                    _, key, val = line.split()
                    meta[key] = val
                elif line.strip():
                    i, s, t, sp = line.split()
                    rows.append((int(i), int(s), float.fromhex(t), int(sp)))
        return ([r[1] for r in rows], [r[2] for r in rows], [r[3] for r in rows], [r[0] for r in rows], int(meta["next_id"]),
                int(meta["p"]), f"oracle-thermalised start {os.path.basename(files[0])} ({meta['sweeps']} oracle sweeps, k = {len(rows)})")
    ns = ORACLE_WARMUP_SWEEPS.get(cfg["name"], 20)
    w = orc.OracleWalker.from_config(cfg, table, 12345, orc.T1)
    w.reset(cfg["init_k"])
    w.sweep(ns)
    c = w.config()
    return (c["site"], c["tau"], c["spin"], c["id"], w.next_id, w.p, f"start thermalised by {ns} oracle sweeps (untimed), k = {w.k}")


# proposals per chain in one bounded oracle sample (about 1-2 s of CPU per chain: T1 costs O(k^2) per proposal)
ORACLE_SAMPLE_PROPOSALS = {"cfg1_2x2_b2": 400000, "cfg2_2x2_b10": 100000, "cfg3_4x4_b10": 10000, "cfg4_6x6_b20": 120,
                           "cfg5_6x6_b40": 30}


class OracleChains:
    """One oracle chain (mode T1) per host thread, all from the common thermalised start, each with its own seed.  The
    start-up (set_state and T1's first from-scratch inverse) is untimed; sample(n) advances every chain by n proposals
    and returns (accepted updates, proposals, seconds)."""

    def __init__(self, cfg, table, n_chains, first_seed=0):
        from concurrent.futures import ThreadPoolExecutor
        from oracle import ctaux_oracle as orc
        self.start = oracle_start_state(cfg, table)
        st = self.start
        self.threads = min(n_chains, os.cpu_count() or 1)
        self.ex = ThreadPoolExecutor(max_workers=self.threads)

        def make(seed):
            w = orc.OracleWalker.from_config(cfg, table, int(seed), orc.T1)
            w.set_state(st[0], st[1], st[2], st[3], st[4], st[5])
            w.propose(1)
            return w

        self.walkers = list(self.ex.map(make, walker_seeds(n_chains, first_seed)))

    def sample(self, n):
        a0 = sum(w.acc_ins + w.acc_rem for w in self.walkers)
        p0 = sum(w.p for w in self.walkers)
        t0 = time.perf_counter()
        list(self.ex.map(lambda w: w.propose(n), self.walkers))
        dt = time.perf_counter() - t0
        return (sum(w.acc_ins + w.acc_rem for w in self.walkers) - a0, sum(w.p for w in self.walkers) - p0, dt)

    def k_mean(self):
        return float(np.mean([w.k for w in self.walkers]))


def cpu_baseline(cfg, table):
    cores = os.cpu_count() or 1
    ch = OracleChains(cfg, table, cores)
    n = 8 * ORACLE_SAMPLE_PROPOSALS.get(cfg["name"], 100)
    acc, props, dt = ch.sample(n)
    return {"value": acc / dt, "unit": UNIT, "cores": ch.threads, "kind": "oracle",
            "proposals_per_s": props / dt, "k_mean": ch.k_mean(),
            "sample": f"oracle T1 (textbook rank-1 updates), {cores} chains (own seeds) x {n} proposals from the "
                      f"{ch.start[6]}, one thread per chain, {dt:.1f} s; T1's once-per-sweep from-scratch inverse is not in the sample"}


def run_reference(args):
    rank, world, local = dist_env()
    if rank != 0:
        return 0
    cfg = get_config(args.config)
    table = table_for(cfg)
    cores = os.cpu_count() or 1
    ch = OracleChains(cfg, table, cores)
    n = ORACLE_SAMPLE_PROPOSALS.get(cfg["name"], 100)
    for _ in range(args.warmup):
        ch.sample(max(1, n // 4))
    acc = props = 0
    dt = 0.0
    for step in range(args.steps):
        a, p, t = ch.sample(n)
        acc += a
        props += p
        dt += t
    value = acc / dt
    threads = ch.threads
    sample = (f"each step = {cores} oracle T1 chains (own seeds) x {n} proposals, continuing from the {ch.start[6]}, one thread "
              f"per chain (bounded sample of {cfg['name']}: {cfg['n_walkers']} walkers x {cfg['sweeps']} sweeps; T1's "
              f"once-per-sweep from-scratch inverse is not in the sample)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "sample": sample, "k_mean": ch.k_mean()},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "proposals_per_s": props / dt, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------------------------
def total_stats(W, n_walkers):
    keys = ("proposals", "acc_ins", "acc_rem", "flops_cand", "flops_cand_alg", "flops_flush", "flops_usinv", "flops_rebuild",
            "flushes", "sum_rank", "blocks", "sum_k", "sweeps", "rebuilds", "guard_ends", "acc_flip")
    tot = {k: 0.0 for k in keys}
    ks = []
    for w in range(n_walkers):
        st = W.get_stats(w)
        for k in keys:
            tot[k] += st[k]
        ks.append(st["k"])
    tot["k_mean"] = float(np.mean(ks))
    return tot


def diff(a, b):
    return {k: a[k] - b[k] for k in a if k != "k_mean"}


DEFAULT_GROUPS = {"cfg3_4x4_b10": 4, "cfg4_6x6_b20": 4, "cfg5_6x6_b40": 2}


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_1901_01047_b200 import WalkerGroups, Walkers
    from paper_1901_01047_b200.replicas import aggregate, rank_seeds

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this package has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = get_config(args.config)
    table = table_for(cfg)
    B = args.walkers or cfg["n_walkers"]
    delay = args.delay or cfg["delay"]
    S = args.sweeps_per_step or cfg["rebuild_every"]
    G = args.groups or DEFAULT_GROUPS.get(cfg["name"], 1)
    if B % G:
        G = 1
    dev = f"cuda:{local}"
    # replicas only: rank r runs its own walkers with disjoint seeds
    seeds = rank_seeds(rank, B)
    fp64_dgemm = measure_fp64_peak(dev) if rank == 0 else 0.0
    from paper_1901_01047_b200 import probe_fp64
    fp64_dmma = probe_fp64(0) if rank == 0 else 0.0
    W = WalkerGroups(G, B, lambda g, nb, stream: Walkers.from_config(
        cfg, table, n_walkers=nb, delay=delay, rebuild_every=S, device=dev, cand_window=args.cand_window, stream=stream,
        rebuild_mode=args.rebuild_mode, flip_moves=args.flips, graph_mode=args.graph))
    W.reset(seeds)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        W.sweep(S)
    barrier()
    # ---- timed region: K steps, all groups concurrently, no per-kernel events
    s0 = total_stats(W, B)
    l0 = W.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record(stream)            # the device is idle here: the region starts now
        for i in range(args.steps):
            W.sweep(S)               # returns when every group has finished the step
        barrier()
        e1.record(stream)
        torch.cuda.synchronize()
    ms_total = e0.elapsed_time(e1)
    s1 = total_stats(W, B)
    l1 = W.launch_count()
    d = diff(s1, s0)
    acc = d["acc_ins"] + d["acc_rem"] + d["acc_flip"]
    # ---- kernel pass: the same step once more, per-class CUDA events on the launching streams; with
    # several groups they run one after the other here, so that each kernel is timed alone
    W.timing_enable(True)
    for g in W.groups:
        g.sweep(S)
    torch.cuda.synchronize()
    s2 = total_stats(W, B)
    tim = W.timing_get()
    W.timing_enable(False)
    dk = diff(s2, s1)
    # the S5 rebuild is latency-bound (pivot search per column), and inside a step all stream groups rebuild AT THE
    # SAME TIME: timed here that way (one ctaux_rebuild per group, concurrently), besides the one-group-at-a-time figure
    torch.cuda.synchronize()
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0.record(stream)
    W.rebuild()
    torch.cuda.synchronize()
    r1.record(stream)
    torch.cuda.synchronize()
    rebuild_concurrent_ms = r0.elapsed_time(r1)
    s3 = total_stats(W, B)
    rebuild_concurrent_flops = s3["flops_rebuild"] - s2["flops_rebuild"]

    # max over ranks of the device time; sum over ranks of the work
    ms_max, (acc_all, props_all) = aggregate(ms_total, [acc, d["proposals"]], device=dev)

    out = None
    if rank == 0:
        peaks = measured_peaks()
        fp64_alt = peaks["bf16_sustained"] * NOMINAL_FP64_TFLOPS / NOMINAL_BF16_TFLOPS
        fp64_peak = fp64_dgemm
        fl = tim["flush_gemm"]
        flush_tf = dk["flops_flush"] / (fl["ms"] * 1e-3) / 1e12 if fl["ms"] > 0 else 0.0
        per_launch_flops = dk["flops_flush"] / max(fl["launches"], 1)
        roofline = {"kernel": "gemm_tma_flush_kernel<2,4,TDescFlush> (S4 rank-r flush: DMMA m8n8k4 on 64x64 tiles, operand tiles "
                              "staged by TMA through a 2-stage mbarrier ring, 4 CTAs/SM, compaction gather into the accumulators)",
                    "bound": "tensor",
                    "achieved": flush_tf, "peak": fp64_peak, "unit": "TFLOP/s", "frac": flush_tf / fp64_peak if fp64_peak else None,
                    "traffic": FLUSH_TRAFFIC.get((cfg["name"], B // G, delay)),
                    "algorithmic_bytes": 2 * (B // G) * 16.0 * (s2["k_mean"] ** 2),   # read + write of N, both spins
                    "peak_source": "cuBLAS DGEMM 8192^3 measured live in this run (FP64 runs at max SM clock: no power cap)",
                    "peak_dmma_issue_rate": fp64_dmma,
                    "peak_alt": fp64_alt,
                    "peak_alt_source": f"{peaks['source']} bf16 sustained {peaks['bf16_sustained']:.1f} TF x nominal FP64:bf16 "
                                       f"{NOMINAL_FP64_TFLOPS:g}:{NOMINAL_BF16_TFLOPS:g}",
                    "frac_alt": flush_tf / fp64_alt,
                    "flops_per_launch": per_launch_flops, "ms_per_launch": fl["ms"] / max(fl["launches"], 1),
                    "launches": fl["launches"], "mean_rank": dk["sum_rank"] / max(dk["flushes"], 1),
                    "walkers_per_launch": B // G,
                    "timed": "kernel pass after the timed region: one more step, groups one after the other"}
        if fl["launches"] == 0:   # fused small-k path: no flush GEMM exists; the walker is one latency-bound kernel
            roofline = {"kernel": "k_walk_fused (whole sweeps in one kernel, N in shared memory; rank-1 updates)",
                        "bound": "alu", "achieved": None, "peak": None, "unit": "TFLOP/s", "frac": None, "traffic": None,
                        "note": "dependent-latency bound chain (one CTA per walker): no roofline applies; see DESIGN.md section 9"}
        steps_ms = {k: v["ms"] for k, v in tim.items()}
        other = {"cand_gemm_tflops": dk["flops_cand"] / (tim["cand_gemm"]["ms"] * 1e-3) / 1e12 if tim["cand_gemm"]["ms"] > 0 else 0.0,
                 "rebuild_tflops": dk["flops_rebuild"] / (tim["rebuild"]["ms"] * 1e-3) / 1e12 if tim["rebuild"]["ms"] > 0 else 0.0,
                 "rebuild_all_groups_concurrent_ms": rebuild_concurrent_ms,
                 "rebuild_all_groups_concurrent_tflops": rebuild_concurrent_flops / (rebuild_concurrent_ms * 1e-3) / 1e12
                 if rebuild_concurrent_ms > 0 else 0.0}
        cand_tf = other["cand_gemm_tflops"]
        cand_alg_tf = dk["flops_cand_alg"] / (tim["cand_gemm"]["ms"] * 1e-3) / 1e12 if tim["cand_gemm"]["ms"] > 0 else 0.0
        roofline_s2 = {"kernel": "gemm_tma_kernel<TDescCandRows/TDescCandCols> (S2 candidate products, the largest share of a "
                                 "large-k step)", "bound": "tensor",
                       "achieved": cand_alg_tf, "peak": fp64_peak, "unit": "TFLOP/s",
                       "frac": cand_alg_tf / fp64_peak if fp64_peak else None,
                       "counting": "SURVEY 8d: 2 m k^2 (rows) + 2 n^2 r_ins (columns of ACCEPTED inserts only), both spins",
                       "achieved_launched": cand_tf, "frac_launched": cand_tf / fp64_peak if fp64_peak else None,
                       "launched_counting": "2 m k^2 + 2 n^2 m: the column product covers every candidate (DESIGN.md section 2)"}
        out = {"metric": METRIC, "value": acc_all / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps,
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": {"workload": cfg["name"], "cluster": f"{cfg['Lx']}x{cfg['Ly']}", "beta": cfg["beta"], "U": cfg["U"],
                          "K": cfg["K"], "walkers_per_gpu": B, "stream_groups": G, "delay": delay, "sweeps_per_step": S,
                          "rebuild_every": S, "rebuild_mode": "lu" if args.rebuild_mode == 0 else "newton-schulz refresh", "graph_mode": args.graph,
                          "moves": "insert/remove/flip" if args.flips else "insert/remove", "l2": "inputs larger than L2" if B * 4 * (s1["k_mean"] ** 2) * 8 > 126e6 else
                          "working set fits L2 (latency-bound chain; no flush between steps)",
                          "parallelism": "replicas only"},
               "proposals_per_s": props_all / (ms_max * 1e-3), "k_mean": s1["k_mean"],
               "mean_k_over_proposals": d["sum_k"] / max(d["proposals"], 1),
               "acceptance": acc / max(d["proposals"], 1),
               "blocks": int(d["blocks"]), "guard_ends": int(d["guard_ends"]),
               "gpu_launches": int(l1 - l0), "roofline": roofline, "roofline_s2": roofline_s2, "kernel_pass_ms_by_class": steps_ms, "gemm": other}
        out["clocks"] = clk.summary()
    return W, cfg, table, out, (rank, world, local)


def run_e2e(W, cfg, B, S, steps, rank):
    """Same metric through the C ABI with HOST buffers: every step uploads the walkers' state from packed host arrays
    (ctaux_set_state: configuration H2D + S1/S5 on the device), runs ctaux_sweep(S) and reads the result back into
    pinned host buffers (ctaux_get_config_all + ctaux_get_stats_all + ctaux_get_N_all, D2H).  The binding's packed forms
    are used (the arrays the C ABI itself takes), so no per-walker Python runs inside the timed region."""
    import torch
    seeds = np.arange(rank * B, rank * B + B, dtype=np.uint64)
    states = W.get_state_packed(with_N=True)      # untimed: also allocates the pinned staging buffers
    acc = 0
    h2d = d2h = 0
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        h2d += sum(int(st["k"].sum()) * (8 + 4 + 8 + 1) + len(st["k"]) * (4 + 8 + 8 + 8) for st in states)
        W.set_state_packed(seeds, states)
        W.sweep(S)
        states = W.get_state_packed(with_N=True)
        for st in states:
            s_ = st["stats"]
            acc += int(s_["acc_ins"].sum() + s_["acc_rem"].sum() + s_["acc_flip"].sum())      # counters restart at set_state
            kk = st["k"].astype(np.int64)
            d2h += int((kk * (8 + 4 + 8 + 1) + 2 * kk * kk * 8).sum()) + len(kk) * 4 + s_.nbytes
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    return {"value": acc / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d / steps), "d2h_bytes_per_step": int(d2h / steps),
            "steps": steps, "ms_per_step": 1e3 * dt / steps,
            "what": "ctaux_set_state(packed host arrays) + ctaux_sweep + ctaux_get_config_all/get_stats_all/get_N_all into pinned host buffers, every step"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4_6x6_b20", choices=[c["name"] for c in CONFIGS])
    ap.add_argument("--walkers", type=int, default=0, help="walkers per GPU (default: the config's)")
    ap.add_argument("--delay", type=int, default=0)
    ap.add_argument("--sweeps-per-step", type=int, default=0)
    ap.add_argument("--groups", type=int, default=0, help="stream groups the walkers are split over (0 = per-config default)")
    ap.add_argument("--rebuild-mode", type=int, default=0, choices=[0, 1],
                    help="periodic rebuild: 0 = from-scratch LU (default, BASELINE.json), 1 = Newton-Schulz refresh (two GEMMs)")
    ap.add_argument("--graph", type=int, default=0, choices=[-1, 0, 1],
                    help="ctaux_params.graph_mode: CUDA graph per poll interval of block steps; 0 = library default (on for max_k <= 512), 1 = every size, -1 = off")
    ap.add_argument("--flips", type=int, default=0, choices=[0, 1],
                    help="1: auxiliary-spin flip as a third move (SURVEY NEXT-1; a different chain than BASELINE.json's)")
    ap.add_argument("--cand-window", type=int, default=0, help="insertion candidates pre-expanded per block")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, replicas only)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    W, cfg, table, out, (rank, world, local) = run_gpu(args)
    B = args.walkers or cfg["n_walkers"]
    S = args.sweeps_per_step or cfg["rebuild_every"]
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(W, cfg, B, S, min(args.steps, 3), rank)
        if world > 1:
            import torch
            import torch.distributed as dist
            t = torch.tensor([e2e["value"]], dtype=torch.float64, device=f"cuda:{local}")
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
            e2e["value"] = float(t.item())
    if rank == 0:
        out["e2e"] = e2e
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(cfg, table)
        print(json.dumps(out))
    W.close()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
