"""ORACLE of the bare cluster propagator of the DCA  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/ may import this module; it shares no code with paper_1901_01047_b200/ and never imports it.  Plain numpy,
complex128, written to be read against the paper:

  * Eq. (1)-(4) PAPER.md:55-68   patch functions; "in the standard coarse-graining the patches are defined as the
    Brillouin zones of the superlattice".
  * Eq. (6)  PAPER.md:85   Sigma_DCA(k, iw_n) = sum_K phi_K(k) Sigma_c(K, iw_n)
  * Eq. (7)  PAPER.md:89   Gbar(K, iw_n) = (Nc/V_BZ) int_BZ dk phi_K(k) [G0^-1(k, iw_n) - Sigma_DCA(k, iw_n)]^-1
  * Eq. (8)  PAPER.md:93   G0(k, iw_n) = [i w_n - eps_k + mu]^-1
  * Eq. (9)  PAPER.md:97   cluster exclusion:  G0c(K, iw_n) = [Gbar^-1(K, iw_n) + Sigma_c(K, iw_n)]^-1
  * Eq. (45) PAPER.md:517  eps_k = -2t (cos kx + cos ky)   (t' = 0)

What the walker consumes is G0c(r, tau) on the tau grid of its table (PAPER.md:861 `sp-time-intervals`); the paper does not
say how the Matsubara sum is closed.  Readings:
  G1  Patches of the periodic Lx x Ly square cluster: K = 2 pi (nx/Lx, ny/Ly); patch K = {K + kt : |kt_x| <= pi/Lx,
      |kt_y| <= pi/Ly}.  Quadrature: midpoint rule, n_quad x n_quad points per patch (n_quad = 1 is the patch centre: the
      isolated cluster).  The paper's interlaced patches and Gaussian quadrature are out of scope.
  G2  G0c(r, iw_n) = (1/Nc) sum_K e^{+i K.r} G0c(K, iw_n)   (inverse of the cluster Fourier transform of the accumulator).
  G3  G0c(r, tau) = (1/beta) sum_{n in Z} e^{-i w_n tau} G0c(r, iw_n) with N_w positive frequencies kept, the negative
      ones by G0c(K, -iw_n) = conj G0c(K, iw_n) (real eps_k; Sigma_c(K, -iw_n) = conj Sigma_c(K, iw_n)), and the
      high-frequency tail c1/(iw) + c2/(iw)^2 + c3/(iw)^3 summed analytically: c1 = 1, c2 = <eps - mu>_patch,
      c3 = <(eps - mu)^2>_patch (the first three moments of G0c do not depend on Sigma_c), with
          (1/beta) sum_n e^{-iw tau}/(iw)   = -1/2,   .../(iw)^2 = (2 tau - beta)/4,   .../(iw)^3 = tau (beta - tau)/4
      on 0 < tau < beta.  The truncation error is O(N_w^-3).
  G4  Table: T[d][m] = G0c(r_d, m beta / M), m = 0..M, STANDARD sign; m = 0 is 0+ and m = M is beta- (the tail terms carry
      the jump).  Row d = dx + Lx dy as in the walker's table.
"""
from __future__ import annotations

import math

import numpy as np


def cluster_momenta(Lx, Ly):
    nx, ny = np.meshgrid(np.arange(Lx), np.arange(Ly))
    return (2 * math.pi * nx / Lx).reshape(-1), (2 * math.pi * ny / Ly).reshape(-1)       # index nx + Lx ny


def patch_points(Lx, Ly, n_quad):
    """G1: midpoint offsets kt inside a patch, [n_quad^2] each."""
    ox = ((np.arange(n_quad) + 0.5) / n_quad - 0.5) * (2 * math.pi / Lx)
    oy = ((np.arange(n_quad) + 0.5) / n_quad - 0.5) * (2 * math.pi / Ly)
    gx, gy = np.meshgrid(ox, oy)
    return gx.reshape(-1), gy.reshape(-1)


def coarse_grain(Lx, Ly, t, mu, beta, n_omega, n_quad, sigma_c=None):
    """Eq. (6)-(8): Gbar(K, iw_n) for n = 0..n_omega-1, and the patch moments <eps - mu>, <(eps - mu)^2>."""
    Kx, Ky = cluster_momenta(Lx, Ly)
    ox, oy = patch_points(Lx, Ly, n_quad)
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    Nc = Lx * Ly
    sigma_c = np.zeros((Nc, n_omega), np.complex128) if sigma_c is None else np.asarray(sigma_c, np.complex128)
    Gbar = np.zeros((Nc, n_omega), np.complex128)
    m1, m2 = np.zeros(Nc), np.zeros(Nc)
    for K in range(Nc):
        eps = -2.0 * t * (np.cos(Kx[K] + ox) + np.cos(Ky[K] + oy))                  # Eq. (45) on the patch
        Gbar[K] = (1.0 / (1j * wn[None, :] - eps[:, None] + mu - sigma_c[K][None, :])).mean(axis=0)     # Eq. (7)
        m1[K], m2[K] = (eps - mu).mean(), ((eps - mu) ** 2).mean()
    return Gbar, m1, m2


def cluster_exclusion(Gbar, sigma_c=None):
    """Eq. (9)."""
    sigma_c = 0.0 if sigma_c is None else np.asarray(sigma_c, np.complex128)
    return 1.0 / (1.0 / Gbar + sigma_c)


def g0_table_from_sigma(Lx, Ly, t, mu, beta, n_omega, n_quad, n_tau, sigma_c=None):
    """G2-G4: the table [Nc][n_tau + 1] of G0c(r, tau) (standard sign) the walker consumes."""
    Nc = Lx * Ly
    Gbar, m1, m2 = coarse_grain(Lx, Ly, t, mu, beta, n_omega, n_quad, sigma_c)
    G0K = cluster_exclusion(Gbar, sigma_c)
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    iw = 1j * wn
    rem = G0K - (1.0 / iw[None, :] + m1[:, None] / iw[None, :] ** 2 + m2[:, None] / iw[None, :] ** 3)    # tail removed
    Kx, Ky = cluster_momenta(Lx, Ly)
    tau = np.arange(n_tau + 1) * (beta / n_tau)
    tau[-1] = beta
    out = np.zeros((Nc, n_tau + 1))
    # (1/beta) sum over +-n of e^{-iw tau} f(iw), f(-iw) = conj f(iw)  =  (2/beta) Re sum_{n>=0} e^{-i w_n tau} f(i w_n)
    ph = np.exp(-1j * wn[:, None] * tau[None, :])                                         # [n_omega][n_tau+1]
    for d in range(Nc):
        rx, ry = d % Lx, d // Lx
        fr = (np.exp(1j * (Kx * rx + Ky * ry))[:, None] * rem).sum(axis=0) / Nc         # G2
        c1 = 1.0 if d == 0 else 0.0
        c2 = (np.exp(1j * (Kx * rx + Ky * ry)) * m1).sum().real / Nc
        c3 = (np.exp(1j * (Kx * rx + Ky * ry)) * m2).sum().real / Nc
        # the remainder of a general r is not conjugate-symmetric in n by itself; its K-sum is real-symmetric because the
        # cluster has inversion symmetry (eps_K = eps_-K), which makes fr(-n) = conj fr(n)
        out[d] = (2.0 / beta) * (fr[:, None] * ph).sum(axis=0).real \
                 + c1 * (-0.5) + c2 * (2 * tau - beta) / 4 + c3 * tau * (beta - tau) / 4
    return out
