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
# large relative error on both sides.  The device evaluates R from an N that has drifted for up to
# rebuild_every sweeps and is allowed a relative error of 1e-10 (the bar below); the entries of N
# enter R multiplied by factors up to (e^gamma - 1)^2 * prefactor, so R cannot be held tighter than
# ~100x the N bar.  R is a diagnostic: the BIT-EXACT field is the decision `accepted`.
# DESIGN.md section 5 "tolerances".
R_RTOL = 1e-6
R_ATOL = 1e-8
N_FROB_TOL = 1e-10     # BASELINE.json north_star: relative Frobenius error of N
WORST_R = {"frac": 0.0}   # largest R error seen in this session, in units of the tolerance (printed by conftest.py)


def run_oracle(cfg, table, seeds, n_sweeps, mode, init_k=None, flips=0, pairs=None):
    init_k = cfg["init_k"] if init_k is None else init_k

    def one(seed):
        w = OracleWalker.from_config(cfg, table, int(seed), mode)
        if pairs is not None:
            w.set_pairs(*pairs)
        if flips:
            w.set_flips(True)
        w.reset(init_k)
        w.sweep(n_sweeps)
        return w

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        return list(ex.map(one, seeds))


def compare_logs(dev_log, orc_log, what="", r_rtol=None, r_atol=None):
    r_rtol = R_RTOL if r_rtol is None else r_rtol
    r_atol = R_ATOL if r_atol is None else r_atol
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
    if len(dev_log):
        frac = np.abs(dev_log["R"] - orc_log["R"]) / (r_rtol * np.abs(orc_log["R"]) + r_atol)
        WORST_R["frac"] = max(WORST_R["frac"], float(frac.max()))
    err = np.abs(dev_log["R"] - orc_log["R"]) - (r_rtol * np.abs(orc_log["R"]) + r_atol)
    assert err.size == 0 or err.max() < 0, f"{what}: R error beyond tolerance by {err.max():.3e} at entry {err.argmax()}"
    assert np.all(dev_log["R"][~both] == 0.0)


def compare_configs(dev_cfg, orc_cfg, what=""):
    for f in ("id", "site", "tau", "spin"):
        assert dev_cfg[f].tobytes() == orc_cfg[f].tobytes(), f"{what}: configuration field {f} differs"


def frob_rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def _oracle_N(orc, s):
    """N_sigma = A_sigma^-1 of the oracle's current configuration: the oracle's own plain-C++ inversion below order
    1024; above it the SAME definition through LAPACK (numpy.linalg.inv of the oracle's A: a library primitive as one
    step -- the plain-C++ routine needs 40 s per matrix at k = 3600), cached per (spin, proposal counter)."""
    if orc.k <= 1024:
        return orc.N(s)
    cache = orc.__dict__.setdefault("_N_cache", {})
    key = (s, orc.p, orc.k)
    if key not in cache:
        cache.clear() if len(cache) >= 2 and all(kk[1] != orc.p for kk in cache) else None
        cache[key] = np.linalg.inv(orc.A(s))
    return cache[key]


def compare_N(walkers, w_index, orc, what="", tol=N_FROB_TOL):
    errs = []
    for s in range(2):
        Nd = walkers.get_N(w_index, s)
        No = _oracle_N(orc, s)
        assert Nd.shape == No.shape, f"{what}: N shape {Nd.shape} vs {No.shape}"
        if No.size:
            e = frob_rel(Nd, No)
            errs.append(e)
            assert e < tol, f"{what}: spin {s} rel Frobenius error {e:.3e}"
    return errs


def full_parity(cfg, n_walkers, n_sweeps, mode, delay=None, rebuild_every=None, init_k=None, seeds=None,
                check_N=True, cand_window=0, max_k=None, n_tol=N_FROB_TOL, fused=0, rebuild_mode=0, flips=0, pairs=None,
                r_rtol=None):
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
                log_capacity=cap, cand_window=cand_window, fused_small=fused, rebuild_mode=rebuild_mode, flip_moves=flips,
                pairs=pairs)
    W.reset(seeds)
    W.sweep(n_sweeps)
    orcs = run_oracle(cfg, table, seeds, n_sweeps, mode, init_k, flips=flips, pairs=pairs)
    worst = 0.0
    for w, o in enumerate(orcs):
        what = f"{cfg['name']} walker {w}"
        compare_logs(W.get_log(w), o.log(), what, r_rtol=r_rtol)
        compare_configs(W.get_config(w), o.config(), what)
        st = W.get_stats(w)
        assert st["k"] == o.k and st["proposals"] == o.p and st["next_id"] == o.next_id, what
        assert st["sign"] == o.sign and st["acc_ins"] == o.acc_ins and st["acc_rem"] == o.acc_rem, what
        assert st["sweeps"] == n_sweeps, what
        assert st["acc_flip"] == o.acc_flip, what
        if check_N:
            errs = compare_N(W, w, o, what, tol=n_tol)
            worst = max([worst] + errs)
    return W, orcs, worst


def load_thermalised(name, seed=0):
    """tests/golden/thermalised_<name>_seed<seed>.txt (written by make_thermalised.py from the ORACLE
    only): returns (config dict in list order, next_id, p)."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"thermalised_{name}_seed{seed}.txt")
    meta, rows = {}, []
    with open(path) as f:
        for line in f:
            if line.startswith("#"):
                _, key, val = line.split()
                meta[key] = val
            elif line.strip():
                i, s, t, sp = line.split()
                rows.append((int(i), int(s), float.fromhex(t), int(sp)))
    assert len(rows) == int(meta["k"])
    cfg = dict(id=np.array([r[0] for r in rows], np.uint64), site=np.array([r[1] for r in rows], np.int32),
               tau=np.array([r[2] for r in rows], np.float64), spin=np.array([r[3] for r in rows], np.int8))
    return cfg, int(meta["next_id"]), int(meta["p"])


def parity_from_state(cfg, state, seeds, n_sweeps, mode, n_proposals=None, delay=None, tol=N_FROB_TOL,
                      rebuild_every=0, flips=0, **kw):
    """Both sides start from the SAME given configuration (a thermalised, well-conditioned one), each
    walker with its own seed; no rebuild on the device, so N is the incrementally updated matrix after
    n_sweeps sweeps (or the oracle runs n_proposals single proposals and the device log is compared on
    that prefix).  Logs / configurations bit-exact, N within tol."""
    from paper_1901_01047_b200 import Walkers
    table = table_for(cfg)
    c0, next_id, p0 = state
    nw = len(seeds)
    cap = int(max(n_sweeps, 1) * max(cfg["max_k"], 16) + 64)
    W = Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table,
                delay=cfg["delay"] if delay is None else delay, n_walkers=nw, init_k=0, max_k=cfg["max_k"],
                rebuild_every=rebuild_every, log_capacity=cap, flip_moves=flips, **kw)
    W.set_state(seeds, [c0] * nw, [next_id] * nw, [p0] * nw)

    def one(seed):
        o = OracleWalker.from_config(cfg, table, int(seed), mode)
        if flips:
            o.set_flips(True)
        o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], next_id, p0)
        if n_proposals is None:
            o.sweep(n_sweeps)
        else:
            o.propose(n_proposals)
        return o

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex2:
        orcs_f = [ex2.submit(one, s) for s in seeds]
        W.sweep(n_sweeps)
        orcs = [f.result() for f in orcs_f]
    worst = 0.0
    for w, o in enumerate(orcs):
        what = f"{cfg['name']} thermalised, walker seed {int(seeds[w])}"
        ol = o.log()
        dl = W.get_log(w)
        if n_proposals is not None:
            dl = dl[:len(ol)]
        compare_logs(dl, ol, what)
        if n_proposals is None:
            compare_configs(W.get_config(w), o.config(), what)
            st = W.get_stats(w)
            assert st["k"] == o.k and st["proposals"] == o.p and st["next_id"] == o.next_id, what
            worst = max([worst] + compare_N(W, w, o, what, tol=tol))
    return W, orcs, worst


# ------------------------------------------------------------------ log replay by brute-force determinants
def replay_windows(start_cfg, log, windows):
    """Apply the accepted moves of `log` (entries numbered from the start configuration) to the start configuration and
    return, for every proposal index inside one of the half-open `windows`, the configuration BEFORE that proposal:
    list of (index, site list, tau list, spin list, version), version = number of accepted moves so far (two
    proposals with the same version meet the same configuration)."""
    site, tau, spin = list(start_cfg["site"]), list(start_cfg["tau"]), list(start_cfg["spin"])
    want = sorted(i for lo, hi in windows for i in range(lo, hi))
    out, version, wi = [], 0, 0
    for i, e in enumerate(log):
        if wi < len(want) and want[wi] == i:
            out.append((i, list(site), list(tau), list(spin), version))
            wi += 1
        if wi >= len(want):
            break
        if e["accepted"]:
            if e["type"] == 0:
                site.append(int(e["arg"])); tau.append(float(e["tau"])); spin.append(int(e["spin"]))
            elif e["type"] == 1:
                j = int(e["arg"])
                del site[j], tau[j], spin[j]
            else:
                spin[int(e["arg"])] = -spin[int(e["arg"])]
            version += 1
    return out


def brute_force_verify(cfg, table, start_cfg, log, windows, rtol=1e-7, atol=1e-9, what=""):
    """SURVEY 8d "log-replay verification" (built on P:201 Eq. (27)): every logged ratio R and every decision inside
    the windows is re-derived from scratch -- the configuration before the proposal is rebuilt from the log, the
    matrices A_sigma and A'_sigma are built by the oracle from the two vertex lists, their determinants are taken by
    LAPACK (numpy slogdet), R = prefactor x prod_sigma det A'/det A, decision = (u < |R|).  Nothing of any fast-update
    formula (Woodbury block on the device, rank-1 formulas of the oracle's T1 mode) enters.  Independent per proposal,
    so it runs in parallel over the host cores; by induction a window whose ratios and decisions all check is a piece
    of the brute-force chain.  Returns the largest |R_log - R_bf| / (rtol |R_bf| + atol)."""
    snaps = replay_windows(start_cfg, log, windows)
    K = cfg["K"]
    probe = OracleWalker.from_config(cfg, table, 0, T0)     # only its model data (table, gamma) is used: A_of is const

    def logdets(site, tau, spin):
        if not site:
            return [(0.0, 1.0), (0.0, 1.0)]
        out = []
        for s in range(2):
            sg, la = np.linalg.slogdet(probe.A_of(s, site, tau, spin))
            out.append((la, sg))
        return out

    # the distinct vertex lists whose determinants are needed: the list BEFORE every proposal (shared by all proposals
    # of one version) and the PROPOSED list of every proposal; the proposed list of an accepted proposal IS the list
    # before the next one, so inside a window of n consecutive proposals there are n + 1 distinct lists, not 2 n
    idx_of = {snap[0]: q for q, snap in enumerate(snaps)}
    lists, need = {}, []
    for snap in snaps:
        i, site, tau, spin, version = snap
        e = log[i]
        k = len(site)
        if e["type"] != 0 and k == 0:
            need.append((i, None, None, 0.0))
            continue
        lists.setdefault(("v", version), (site, tau, spin))
        if e["type"] == 0:
            prop = (site + [int(e["arg"])], tau + [float(e["tau"])], spin + [int(e["spin"])])
            pref = K / (k + 1)
        elif e["type"] == 1:
            j = int(e["arg"])
            prop = (site[:j] + site[j + 1:], tau[:j] + tau[j + 1:], spin[:j] + spin[j + 1:])
            pref = k / K
        else:
            j = int(e["arg"])
            prop = (site, tau, spin[:j] + [-spin[j]] + spin[j + 1:])
            pref = 1.0
        if e["accepted"] and (i + 1) in idx_of:
            nxt = snaps[idx_of[i + 1]]
            assert nxt[4] == version + 1 and (nxt[1], nxt[2], nxt[3]) == (list(prop[0]), list(prop[1]), list(prop[2]))
            key = ("v", version + 1)
        else:
            key = ("a", i)
        lists.setdefault(key, prop)
        need.append((i, ("v", version), key, pref))

    keys = list(lists)
    from threadpoolctl import threadpool_limits
    with threadpool_limits(limits=1):      # one LAPACK thread per worker: the vertex lists are the parallel dimension
        with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
            dets = dict(zip(keys, ex.map(lambda kk: logdets(*lists[kk]), keys)))
    res = []
    for i, k0, k1, pref in need:
        if k0 is None:
            res.append((i, 0.0, None))
            continue
        d0, d1 = dets[k0], dets[k1]
        R = pref * d1[0][1] * d1[1][1] * d0[0][1] * d0[1][1] * math.exp(d1[0][0] + d1[1][0] - d0[0][0] - d0[1][0])
        res.append((i, R, None))
    worst = 0.0
    for i, R, _ in res:
        e = log[i]
        err = abs(e["R"] - R) / (rtol * abs(R) + atol)
        worst = max(worst, err)
        assert err < 1.0, f"{what}: proposal {i}: logged R {e['R']!r} vs brute force {R!r} (x{err:.2e} of tolerance)"
        assert int(e["accepted"]) == (1 if e["u"] < abs(R) else 0), f"{what}: proposal {i}: decision differs from brute force"
    return worst
