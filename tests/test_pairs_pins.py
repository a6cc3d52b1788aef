"""Pins of the oracle's general opposite-spin density-density interaction (Eq. (19)-(25),
PAPER.md:174-194; model parameters U, V of PAPER.md:743-778).  No CUDA path involved."""
import math

import numpy as np
import pytest

from ctaux_workloads import cluster_dispersion, g0_table, get_config, table_for
from oracle.ctaux_oracle import T0, T1, OracleWalker

from test_oracle_pins import _fock_ops, _fock_trace


def extended_hubbard_pairs(Lx, Ly, U, V):
    """On-site U plus V between opposite spins on nearest-neighbour sites: pairs (a up, b down, U_p)."""
    Nc = Lx * Ly
    a, b, u = list(range(Nc)), list(range(Nc)), [U] * Nc
    for i in range(Nc):
        x, y = i % Lx, i // Lx
        nbrs = {((x + 1) % Lx) + Lx * y, ((x - 1) % Lx) + Lx * y, x + Lx * ((y + 1) % Ly), x + Lx * ((y - 1) % Ly)} - {i}
        for j in sorted(nbrs):
            a.append(i); b.append(j); u.append(V)
    return np.array(a, np.int32), np.array(b, np.int32), np.array(u)


def test_gamma_per_pair_eq25_and_identity_pairs_reproduce_the_on_site_model():
    cfg = get_config(1)
    T = table_for(cfg)
    a, b, u = extended_hubbard_pairs(2, 2, 4.0, 1.5)
    w = OracleWalker.from_config(cfg, T, 3, T1)
    w.set_pairs(a, b, u)
    for p in range(a.size):
        ch = 1 + u[p] * cfg["beta"] * a.size / (2 * cfg["K"])         # Eq. (25) with N_corr = number of pairs
        assert abs(math.cosh(math.log(w.pair_exp_gamma(p))) / ch - 1) < 1e-13
    # pairs (i, i, U): N_corr = Nc, one gamma -- the default chain, bit for bit
    ref = OracleWalker.from_config(cfg, T, 3, T1)
    ref.reset(cfg["init_k"]); ref.sweep(5)
    same = OracleWalker.from_config(cfg, T, 3, T1)
    same.set_pairs(np.arange(4), np.arange(4), np.full(4, cfg["U"]))
    same.reset(cfg["init_k"]); same.sweep(5)
    assert ref.log().tobytes() == same.log().tobytes()
    assert np.array_equal(ref.N(0), same.N(0)) and np.array_equal(ref.N(1), same.N(1))


@pytest.mark.parametrize("Lx,Ly,mu", [(2, 2, 0.0), (3, 2, -0.3)])
def test_fock_space_trace_with_pairs(Lx, Ly, mu):
    """Eq. (27) for vertices (p, tau, s) of the extended Hubbard model: det A_up is the single-species Fock-space trace
    with e^{-gamma_p s n} at site a_p, det A_down the one with e^{+gamma_p s n} at site b_p -- different sites, different
    gammas per vertex.  Pins which site and which gamma enter which matrix."""
    beta, K, M = 2.0, 1.0, 256
    T = g0_table(Lx, Ly, beta, mu, M)
    a, b, u = extended_hubbard_pairs(Lx, Ly, 4.0, 1.5)
    rng = np.random.default_rng(7 * Lx + Ly)
    for nv in (1, 2, 3, 4):
        for trial in range(3):
            pairs = rng.integers(0, a.size, nv).astype(np.int32)
            if trial == 0:
                pairs[0] = a.size - 1                                   # an inter-site pair for sure
            taus = rng.choice(np.arange(1, M), nv, replace=False) * beta / M
            spins = rng.choice([-1, 1], nv).astype(np.int8)
            w = OracleWalker(Lx, Ly, beta, 4.0, K, T, 0)
            w.set_pairs(a, b, u)
            w.set_state(pairs, taus, spins)
            for sidx, sigma in enumerate([+1, -1]):
                sites = (a if sidx == 0 else b)[pairs]
                av = [-math.log(w.pair_exp_gamma(int(p))) * sigma * int(s) for p, s in zip(pairs, spins)]
                want = _fock_trace(Lx, Ly, beta, mu, sites, taus, av)
                la, sg = w.logdet(sidx)
                assert abs(sg * math.exp(la) / want - 1) < 1e-10, (nv, trial, sidx)


def test_T1_equals_T0_with_pairs():
    cfg = get_config(0)
    T = table_for(cfg)
    a, b, u = extended_hubbard_pairs(2, 2, 4.0, 2.0)
    logs = []
    for mode in (T0, T1):
        w = OracleWalker.from_config(cfg, T, 5, mode)
        w.set_pairs(a, b, u)
        w.reset(6)
        w.sweep(40)
        logs.append((w.log(), w.config(), w.sign))
    for f in ("p", "type", "arg", "tau", "spin", "accepted", "u"):
        assert logs[0][0][f].tobytes() == logs[1][0][f].tobytes(), f
    assert np.allclose(logs[0][0]["R"], logs[1][0]["R"], rtol=1e-9, atol=1e-300)
    assert logs[0][0]["arg"][logs[0][0]["type"] == 0].max() >= 4          # inter-site pairs were proposed
    assert logs[0][2] == logs[1][2]


def test_mean_order_identity_with_inter_site_interaction_against_exact_diagonalisation():
    """<k> = K - beta <H_int> (from Eq. (22)-(23)) on a two-site cluster with on-site U and inter-site V between opposite
    spins, <H_int> by exact diagonalisation of H0 + H_int in the 16-dimensional Fock space.  Pins the stationary
    distribution for N_corr != Nc: the pair proposal (1/N_corr), the prefactors with Eq. (25)'s N_corr, and the weights."""
    Lx, Ly, beta, K, mu, U, V = 2, 1, 2.0, 1.0, -0.2, 4.0, 2.0
    T = g0_table(Lx, Ly, beta, mu, 128)
    a, b, u = np.array([0, 1, 0, 1], np.int32), np.array([0, 1, 1, 0], np.int32), np.array([U, U, V, V])
    # exact: spin-orbitals 0,1 = up at sites 0,1; 2,3 = down at sites 0,1
    kx, ky, eps = cluster_dispersion(Lx, Ly)
    h = np.array([[np.mean(np.cos(kx * (i - j)) * (eps - mu)) for j in range(2)] for i in range(2)])
    c = _fock_ops(4)
    n = [ci.T @ ci for ci in c]
    H0 = sum(h[i, j] * (c[i].T @ c[j] + c[2 + i].T @ c[2 + j]) for i in range(2) for j in range(2))
    Hint = sum(u[p] * (n[a[p]] @ n[2 + b[p]] - 0.5 * (n[a[p]] + n[2 + b[p]])) for p in range(4))
    ev, Vv = np.linalg.eigh(H0 + Hint)
    wgt = np.exp(-beta * (ev - ev.min()))
    hint_avg = float(np.sum(wgt * np.einsum("ij,jk,ki->i", Vv.T, Hint, Vv)) / wgt.sum())
    want = K - beta * hint_avg
    means = []
    for seed in range(8):
        w = OracleWalker(Lx, Ly, beta, U, K, T, seed, T1)
        w.set_pairs(a, b, u)
        w.reset(4)
        w.propose(120000)
        log = w.log()
        dk = log["accepted"] * np.where(log["type"] == 0, 1, -1)
        kb = 4 + np.concatenate([[0], np.cumsum(dk)[:-1]])
        means.append(kb[5000:].mean())
    means = np.array(means)
    err = means.std(ddof=1) / math.sqrt(len(means))
    assert abs(means.mean() - want) < max(4.5 * err, 0.03), (means.mean(), err, want)
