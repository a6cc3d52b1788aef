"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded
inputs and compare element by element.  The oracle and the CUDA package never import each other;
only the tests see both."""
import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from ctaux_workloads import table_for, walker_seeds
from oracle.ctaux_oracle import T0, T1, OracleWalker

EXACT_FIELDS = ("p", "type", "arg", "tau", "spin", "accepted", "u")
# Logged ratios come from different arithmetic (Woodbury block on the device, determinants or
# rank-1 formulas in the oracle).  A ratio is a difference of O(1) terms, so its ABSOLUTE error is
# what the arithmetic bounds; tiny |R| (near-singular A', always rejected by a wide margin) carry a
# large relative error on both sides.  DESIGN.md "tolerances".
R_RTOL = 1e-7
R_ATOL = 1e-10
N_FROB_TOL = 1e-10     # BASELINE.json north_star: relative Frobenius error of N


def run_oracle(cfg, table, seeds, n_sweeps, mode, init_k=None):
    init_k = cfg["init_k"] if init_k is None else init_k

    def one(seed):
        w = OracleWalker.from_config(cfg, table, int(seed), mode)
        w.reset(init_k)
        w.sweep(n_sweeps)
        return w

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        return list(ex.map(one, seeds))


def compare_logs(dev_log, orc_log, what=""):
    assert len(dev_log) == len(orc_log), f"{what}: log length {len(dev_log)} vs {len(orc_log)}"
    for f in EXACT_FIELDS:
        if dev_log[f].tobytes() != orc_log[f].tobytes():
            bad = np.nonzero(dev_log[f] != orc_log[f])[0]
            i = int(bad[0])
            aR = abs(orc_log["R"][i])
            margin = abs(orc_log["u"][i] - aR) / max(aR, 1e-300)
            raise AssertionError(f"{what}: field {f} first differs at entry {i}: dev={dev_log[i]} orc={orc_log[i]} "
                                 f"(oracle margin at that proposal {margin:.3e})")
    both = np.abs(orc_log["R"]) > 0
    err = np.abs(dev_log["R"] - orc_log["R"]) - (R_RTOL * np.abs(orc_log["R"]) + R_ATOL)
    assert err.size == 0 or err.max() < 0, f"{what}: R error beyond tolerance by {err.max():.3e} at entry {err.argmax()}"
    assert np.all(dev_log["R"][~both] == 0.0)


def compare_configs(dev_cfg, orc_cfg, what=""):
    for f in ("id", "site", "tau", "spin"):
        assert dev_cfg[f].tobytes() == orc_cfg[f].tobytes(), f"{what}: configuration field {f} differs"


def frob_rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def compare_N(walkers, w_index, orc, what="", tol=N_FROB_TOL):
    errs = []
    for s in range(2):
        Nd = walkers.get_N(w_index, s)
        No = orc.N(s)
        assert Nd.shape == No.shape, f"{what}: N shape {Nd.shape} vs {No.shape}"
        if No.size:
            e = frob_rel(Nd, No)
            errs.append(e)
            assert e < tol, f"{what}: spin {s} rel Frobenius error {e:.3e}"
    return errs


def full_parity(cfg, n_walkers, n_sweeps, mode, delay=None, rebuild_every=None, init_k=None, seeds=None,
                check_N=True, cand_window=0, max_k=None):
    """reset + n_sweeps on both sides, compare logs, configurations, N, sign, counters."""
    from paper_1901_01047_b200 import Walkers
    table = table_for(cfg)
    seeds = walker_seeds(n_walkers) if seeds is None else np.asarray(seeds, dtype=np.uint64)
    init_k = cfg["init_k"] if init_k is None else init_k
    cap = int(n_sweeps * max(cfg["max_k"], 16) + 64)
    W = Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table,
                delay=cfg["delay"] if delay is None else delay, n_walkers=n_walkers, init_k=init_k,
                max_k=cfg["max_k"] if max_k is None else max_k,
                rebuild_every=cfg["rebuild_every"] if rebuild_every is None else rebuild_every,
                log_capacity=cap, cand_window=cand_window)
    W.reset(seeds)
    W.sweep(n_sweeps)
    orcs = run_oracle(cfg, table, seeds, n_sweeps, mode, init_k)
    worst = 0.0
    for w, o in enumerate(orcs):
        what = f"{cfg['name']} walker {w}"
        compare_logs(W.get_log(w), o.log(), what)
        compare_configs(W.get_config(w), o.config(), what)
        st = W.get_stats(w)
        assert st["k"] == o.k and st["proposals"] == o.p and st["next_id"] == o.next_id, what
        assert st["sign"] == o.sign and st["acc_ins"] == o.acc_ins and st["acc_rem"] == o.acc_rem, what
        assert st["sweeps"] == n_sweeps, what
        if check_N:
            errs = compare_N(W, w, o, what)
            worst = max([worst] + errs)
    return W, orcs, worst
