"""Why the library MEASURES the error of N instead of trusting a rebuild cadence (error_monitor.cuh).

A numpy model of the delayed-block update (the arithmetic of S2-S4 in matrix form, LAPACK-quality kernels, no CUDA)
replays the accepted moves of an oracle chain from the thermalised config-4 state and compares N with the from-scratch
inverse after every block.  The drift is not rounding noise that averages out: every block maps the error N already
carries through (A'^-1 A) . (A A'^-1), so it grows roughly geometrically -- an order of magnitude within a third of a
sweep, 2e-10 after one sweep (measured with this model) -- and it does so for ANY way of obtaining S^-1 (bordering as in the S3 kernel, or a fresh LAPACK solve per
block).  A fixed cadence cannot hold 1e-10 at an acceptable cost; a measured trigger can."""
import numpy as np

from ctaux_workloads import get_config, table_for
from oracle.ctaux_oracle import T1, OracleWalker

from parity_helpers import load_thermalised


def _gmat(T, cfg, si, ta, sj, tb):
    Lx, Ly, beta, M = cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["M"]
    si, sj, ta, tb = np.asarray(si), np.asarray(sj), np.asarray(ta), np.asarray(tb)
    d = ((si[:, None] % Lx - sj[None, :] % Lx) % Lx) + Lx * ((si[:, None] // Lx - sj[None, :] // Lx) % Ly)
    dt = ta[:, None] - tb[None, :]
    sg = np.where(dt < 0, -1.0, 1.0)
    dt = np.where(dt < 0, dt + beta, dt)
    x = dt * (M / beta)
    m = np.minimum(np.floor(x).astype(int), M - 1)
    return -sg * (T[d, m] + (x - m) * (T[d, m + 1] - T[d, m]))


def _replay(cfg, T, c0, log, delay, variant, probe, egp):
    egm = 1.0 / egp
    E = lambda sidx, s: np.where((1 if sidx == 0 else -1) * np.asarray(s) > 0, egm, egp)
    g00 = -T[0, 0]
    site, tau, spin = list(c0["site"]), list(c0["tau"]), list(c0["spin"])
    N = [np.linalg.inv(probe.A_of(s, site, tau, spin)) for s in range(2)]
    errs, i = [], 0
    while i < len(log):
        k0, moves, live, cand = len(site), [], list(range(len(site))), []
        while i < len(log) and len(moves) < delay:
            e = log[i]
            if e["accepted"]:
                if e["type"] == 0:
                    cand.append((int(e["arg"]), float(e["tau"]), int(e["spin"])))
                    live.append(k0 + len(cand) - 1); moves.append((0, k0 + len(cand) - 1))
                else:
                    slot = live[int(e["arg"])]
                    if slot >= k0:
                        break                     # a twice-touched slot ends the block (chain-neutral)
                    del live[int(e["arg"])]; moves.append((1, slot))
            i += 1
        if not moves:
            continue
        m = len(cand)
        es, et, esp = site + [c[0] for c in cand], tau + [c[1] for c in cand], spin + [c[2] for c in cand]
        n = k0 + m
        gx = _gmat(T, cfg, es, et, es[k0:], et[k0:]) if m else np.zeros((n, 0))
        for c in range(m):
            gx[k0 + c, c] = g00
        for s in range(2):
            Ej = E(s, spin)
            Next = np.zeros((n, n)); Next[:k0, :k0] = N[s]
            if m:
                Next[k0:, :k0] = (_gmat(T, cfg, es[k0:], et[k0:], site, tau) * (Ej - 1.0)[None, :]) @ N[s]
                Next[k0:, k0:] = np.eye(m)
            Gx = Next @ gx
            J = [sl for _, sl in moves]
            XJ = np.stack([((np.arange(n) == j) - Next[:, j]) / (Ej[j] - 1.0) if j < k0 else (np.arange(n) == j) - Gx[:, j - k0] for j in J], axis=1)
            dE = np.array([(E(s, esp[sl]) - 1.0) if ty == 0 else (1.0 - E(s, esp[sl])) for ty, sl in moves], dtype=float)
            S = XJ[J, :] + np.diag(1.0 / dE)
            if variant == "border":               # S^-1 grown one accepted move at a time, as in the S3 kernel
                Sinv = np.zeros((0, 0))
                for a in range(len(J)):
                    tv, tpv = Sinv @ S[:a, a], S[a, :a] @ Sinv
                    st = S[a, a] - S[a, :a] @ tv
                    new = np.zeros((a + 1, a + 1))
                    new[:a, :a] = Sinv + np.outer(tv, tpv) / st
                    new[:a, a], new[a, :a], new[a, a] = -tv / st, -tpv / st, 1 / st
                    Sinv = new
                Nn = Next - (XJ @ Sinv) @ Next[J, :]
            else:                                 # a fresh LAPACK solve per block
                Nn = Next - XJ @ np.linalg.solve(S, Next[J, :])
            N[s] = Nn[np.ix_(live, live)]
        site, tau, spin = [es[j] for j in live], [et[j] for j in live], [esp[j] for j in live]
        e_blk = []
        for s in range(2):
            Nd = np.linalg.inv(probe.A_of(s, site, tau, spin))
            e_blk.append(np.linalg.norm(N[s] - Nd) / np.linalg.norm(Nd))
        errs.append(max(e_blk))
    return errs


def test_fast_updates_amplify_the_error_they_carry_whatever_inverts_S():
    cfg = get_config(3)
    T = table_for(cfg)
    c0, nid, p0 = load_thermalised(cfg["name"])
    o = OracleWalker.from_config(cfg, T, 7, T1)
    o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], nid, p0)
    o.propose(650)                                    # a third of a sweep: five to six blocks of rank <= 64
    probe = OracleWalker.from_config(cfg, T, 0, T1)
    out = {}
    for variant in ("border", "solve"):
        out[variant] = _replay(cfg, T, c0, o.log(), cfg["delay"], variant, probe, o.exp_gamma)
    for variant, errs in out.items():
        assert len(errs) >= 5
        assert errs[0] < 2e-12                        # one block from a fresh inverse: rounding level
        assert errs[-1] > 5e-12 and errs[-1] > 8 * errs[0], (variant, errs)       # ... an order of magnitude up five blocks later
    assert 0.1 < out["border"][-1] / out["solve"][-1] < 10.0     # the way S is inverted is not the cause
