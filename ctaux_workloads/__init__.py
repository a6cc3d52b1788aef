"""Seeded, synthetic input generators shared by the oracle, the tests and bench.py.

This module holds NONE of the CT-AUX method's arithmetic (no gamma, no A/N matrices,
no Metropolis step, no random-number generator).  It only states the workloads:

* the periodic Lx x Ly Hubbard cluster (site / displacement indexing),
* the closed-form non-interacting cluster propagator G0(r, tau) tabulated on M tau
  intervals (BASELINE.json north_star: G0(k,tau) = -exp(-(eps_k-mu) tau)/(1+exp(-beta (eps_k-mu)))),
* the five BASELINE.json configs as plain dictionaries,
* the walker seeds (walker w uses seed w).

Paper passages: dispersion Eq. (45) with t'=0; `sp-time-intervals`
 for the tau grid; Eq. (20) for what mu means
(the chemical potential of H0 AFTER the U/2 shift, so mu=0 is half filling).

The DCA self-consistency loop that would produce the paper's G0 is out of scope
(SURVEY.md section 8d): these isolated-cluster tables STAND IN for it.
"""
from __future__ import annotations

import math
import numpy as np

__all__ = [
    "cluster_dispersion",
    "g0_exact",
    "g0_table",
    "mu_for_density",
    "CONFIGS",
    "get_config",
    "walker_seeds",
    "atomic_limit_table",
]


def cluster_dispersion(Lx: int, Ly: int, t: float = 1.0):
    """Cluster momenta k = 2*pi*(nx/Lx, ny/Ly) and eps_k = -2t(cos kx + cos ky).

    Eq. (45), t' = 0.  Returns (kx[Nc], ky[Nc], eps[Nc]), index nx + Lx*ny.
    """
    nx = np.arange(Lx)
    ny = np.arange(Ly)
    kx = (2.0 * np.pi * nx / Lx)[None, :].repeat(Ly, 0).reshape(-1)
    ky = (2.0 * np.pi * ny / Ly)[:, None].repeat(Lx, 1).reshape(-1)
    eps = -2.0 * t * (np.cos(kx) + np.cos(ky))
    return kx, ky, eps


def _fermi_weight(xi: np.ndarray, tau: np.ndarray, beta: float) -> np.ndarray:
    """exp(-xi*tau)/(1+exp(-beta*xi)) evaluated without overflow, shape [len(xi), len(tau)]."""
    xi = xi[:, None]
    tau = tau[None, :]
    pos = np.exp(-np.where(xi >= 0, xi, 0.0) * tau) / (1.0 + np.exp(-beta * np.abs(xi)))
    neg = np.exp(np.where(xi < 0, xi, 0.0) * (beta - tau)) / (1.0 + np.exp(-beta * np.abs(xi)))
    return np.where(xi >= 0, pos, neg)


def g0_exact(Lx: int, Ly: int, beta: float, mu: float, tau: np.ndarray, t: float = 1.0) -> np.ndarray:
    """Standard-sign G0(r_d, tau) for tau in [0, beta] (0 means 0+, beta means beta-).

    G0(r,tau) = -(1/Nc) sum_k cos(k.r) exp(-xi_k tau)/(1+exp(-beta xi_k)), xi_k = eps_k - mu.
    Row d = dx + Lx*dy is the displacement (dx, dy).  Shape [Nc, len(tau)], all <= 0 at r=0.
    """
    tau = np.asarray(tau, dtype=np.float64)
    kx, ky, eps = cluster_dispersion(Lx, Ly, t)
    w = _fermi_weight(eps - mu, tau, beta)  # [Nc_k, n_tau]
    Nc = Lx * Ly
    out = np.empty((Nc, tau.size), dtype=np.float64)
    for dy in range(Ly):
        for dx in range(Lx):
            phase = np.cos(kx * dx + ky * dy)  # [Nc_k]
            out[dx + Lx * dy] = -(phase[:, None] * w).sum(axis=0) / Nc
    return out


def g0_table(Lx: int, Ly: int, beta: float, mu: float, M: int = 512, t: float = 1.0) -> np.ndarray:
    """Table T[d][m] = G0(r_d, m*beta/M), m = 0..M (M intervals, M+1 points), C-contiguous f64."""
    tau = np.arange(M + 1, dtype=np.float64) * (beta / M)
    tau[M] = beta
    return np.ascontiguousarray(g0_exact(Lx, Ly, beta, mu, tau, t))


def atomic_limit_table(M: int = 512) -> np.ndarray:
    """Nc=1, xi=0: G0(tau) = -1/2 for every tau (pin P6)."""
    return np.full((1, M + 1), -0.5, dtype=np.float64)


def mu_for_density(Lx: int, Ly: int, beta: float, n: float, t: float = 1.0) -> float:
    """mu solving the NON-interacting cluster density (2/Nc) sum_k f(eps_k - mu) = n (bisection)."""
    _, _, eps = cluster_dispersion(Lx, Ly, t)

    def dens(mu):
        x = beta * (eps - mu)
        return 2.0 * np.mean(0.5 * (1.0 - np.tanh(0.5 * x)))

    lo, hi = -8.0 * t, 8.0 * t
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if dens(mid) < n:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def _cfg(name, Lx, Ly, beta, U, mu, n_walkers, delay, sweeps, warmup_sweeps, init_k, max_k,
         rebuild_every=10, K=1.0, M=512):
    return dict(name=name, Lx=Lx, Ly=Ly, beta=float(beta), U=float(U), K=float(K), mu=float(mu),
                M=M, n_walkers=n_walkers, delay=delay, sweeps=sweeps, warmup_sweeps=warmup_sweeps,
                init_k=init_k, max_k=max_k, rebuild_every=rebuild_every)


# BASELINE.json `configs`, made concrete in SURVEY.md section 8d.  mu values are the frozen
# 6-decimal outputs of mu_for_density.  init_k = round(K + beta U Nc (n/2)(1-n/2)).
# max_k is a capacity: comfortably above the hard bound K + beta U Nc n / 2.
CONFIGS = [
    _cfg("cfg1_2x2_b2", 2, 2, 2.0, 4.0, 0.0, 1, 8, 1000, 200, 9, 64),
    _cfg("cfg2_2x2_b10", 2, 2, 10.0, 4.0, 0.0, 256, 16, 500, 0, 41, 128),
    _cfg("cfg3_4x4_b10", 4, 4, 10.0, 4.0, -0.054654, 64, 32, 200, 0, 159, 384),
    _cfg("cfg4_6x6_b20", 6, 6, 20.0, 6.0, -0.037689, 8, 64, 100, 0, 1070, 2304),
    _cfg("cfg5_6x6_b40", 6, 6, 40.0, 6.0, -0.009099, 2, 128, 50, 0, 2156, 4608),
]


def get_config(i_or_name):
    if isinstance(i_or_name, int):
        return dict(CONFIGS[i_or_name])
    for c in CONFIGS:
        if c["name"] == i_or_name:
            return dict(c)
    raise KeyError(i_or_name)


def walker_seeds(n_walkers: int, first: int = 0) -> np.ndarray:
    """Walker w draws from the counter-based stream keyed by seed first+w (BASELINE.json)."""
    return np.arange(first, first + n_walkers, dtype=np.uint64)


def table_for(cfg: dict) -> np.ndarray:
    return g0_table(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["mu"], cfg["M"])
