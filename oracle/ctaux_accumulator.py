"""ORACLE of the single-particle accumulation of CT-AUX  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's CPU-baseline legs may import this module; it shares no code with
paper_1901_01047_b200/ (the CUDA path) and never imports it.  Plain numpy in FP64 / complex128, written to be checked
against the paper by eye:

  * PAPER.md:212  "From a vertex configuration {v}_k and its respective N_sigma-matrices we first compute a function M,
    whose Fourier coefficients are then accumulated."
  * Eq. (28) PAPER.md:214   <G(k, iw_n)> = G0(k, iw_n) - (1/beta) G0(k, iw_n) <M(k, iw_n)> G0(k, iw_n)
  * Eq. (29) PAPER.md:218   Sigma(k, iw_n) = G0^-1(k, iw_n) - <G(k, iw_n)>^-1
  * Eq. (30)-(31) PAPER.md:232-238   non-equispaced FFT: the samples f_i at random times tau_i are convolved with a
    localised, beta-periodic kernel phi onto an equispaced grid of m*N_w points, accumulated there over the whole
    Monte-Carlo run ("delayed"), transformed ONCE at the end and divided by the kernel's Fourier coefficients phi_w;
    "the kernel phi [is approximated] with a low order polynomial at the cost of a controllable interpolation error".

The paper prints neither the definition of M nor the kernel (it cites refs [18], [11], [22]).  Readings:
  R1  M_sigma = (E - 1) N_sigma with the factor on the ROW:  M[j,l] = (E_j - 1) N[j,l],  E_j = e^{-gamma sigma s_j}.
      In the positive convention g = -G0 the Green's function of ONE configuration is
          g_c(x, y) = g(x, y) + sum_jl g(x, j) M[j,l] g(l, y),       x = (site, tau), j / l = vertices,
      i.e. G_c = G0 - G0 M G0 in the standard sign.  Derived from Eq. (27) by bordering A with a row x and a column y;
      pinned by the Fock-space trace with c_x(tau) c+_y(tau') inserted (tests/test_accumulator_pins.py).
  R2  M(r, iw_n) = sum_{j,l : r_j - r_l = r} M[j,l] e^{i w_n (tau_j - tau_l)},  w_n = (2n+1) pi / beta, n = 0..N_w-1
      (positive frequencies; M(r, tau) is real for a real H0, so the negative ones follow by conjugation), and
      M(K, iw_n) = (1/Nc) sum_r e^{-i K.r} M(r, iw_n).  With this normalisation Eq. (28) holds as printed (the 1/beta
      and the 1/Nc are the averages over a rigid shift of all times and all sites).
  R3  Monte-Carlo average with the sign: <M> = sum_c sign_c M_c / sum_c sign_c  (PAPER.md:224 sign problem).
  R4  NFFT grid: L = m * N_w points, spacing beta / L (Eq. (31) as printed; m >= 2 resolves the N_w positive
      frequencies).  A time difference t in (-beta, beta) is folded to [0, beta) with the fermionic sign (M is
      beta-ANTIperiodic); the transform at fermionic frequencies is the FFT of f_l e^{i pi l / L}.
  R5  Kernel: Gaussian window phi(t) = exp(-(t / (s Delta))^2), Delta = beta / L, truncated at |t| <= w Delta (2w grid
      points per sample), with the width of the standard Gaussian NFFT window  s^2 = (2 sigma / (2 sigma - 1)) (w / pi),
      sigma = m / 2 the oversampling against the bandwidth 2 N_w.  phi_w is the Fourier coefficient of the truncated
      window evaluated by its defining sum on the grid refined 64-fold.  Aliasing error ~ 4 exp(-w pi (1 - 1/(2 sigma - 1))).
  R6  "Low order polynomial": the window is tabulated with its derivative at `n_tab` points per grid cell and evaluated by
      cubic Hermite interpolation (error O(n_tab^-4), far below the aliasing error for n_tab = 32).
"""
from __future__ import annotations

import math

import numpy as np


# --------------------------------------------------------------------------------------------- M and G of one configuration
def m_matrix(N: np.ndarray, spins: np.ndarray, sidx: int, exp_gamma: float) -> np.ndarray:
    """R1: M[j,l] = (E_j - 1) N[j,l];  N is the oracle's N_sigma (row-major k x k), E_j = e^{-gamma sigma s_j}."""
    sigma = +1 if sidx == 0 else -1
    E = np.where(sigma * np.asarray(spins) > 0, 1.0 / exp_gamma, exp_gamma)
    return (E - 1.0)[:, None] * N


def g_config(g_xv: np.ndarray, M: np.ndarray, g_vy: np.ndarray, g_xy: float) -> float:
    """R1: g_c(x, y) = g(x, y) + sum_jl g(x, j) M[j,l] g(l, y)   (positive convention g = -G0)."""
    return g_xy + g_xv @ M @ g_vy


# --------------------------------------------------------------------------------------------- T0: direct Fourier sums
def displacement(Lx: int, Ly: int, site_j: np.ndarray, site_l: np.ndarray) -> np.ndarray:
    """index of r_j - r_l on the periodic Lx x Ly cluster (same convention as the walker's table rows)."""
    dx = (site_j[:, None] % Lx - site_l[None, :] % Lx) % Lx
    dy = (site_j[:, None] // Lx - site_l[None, :] // Lx) % Ly
    return dx + Lx * dy


def m_direct(Lx, Ly, beta, site, tau, M, n_omega) -> np.ndarray:
    """R2, brute force: M(r, iw_n) = sum_{jl: r_j - r_l = r} M[j,l] e^{i w_n (tau_j - tau_l)}.  O(k^2 N_w).
    Returns complex128 [Nc][n_omega]."""
    Nc = Lx * Ly
    site = np.asarray(site)
    tau = np.asarray(tau, dtype=np.float64)
    out = np.zeros((Nc, n_omega), np.complex128)
    if site.size == 0:
        return out
    d = displacement(Lx, Ly, site, site)
    dt = tau[:, None] - tau[None, :]
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    for r in range(Nc):
        sel = d == r
        if sel.any():
            out[r] = (M[sel][:, None] * np.exp(1j * dt[sel][:, None] * wn[None, :])).sum(axis=0)
    return out


def m_of_k(Lx, Ly, M_r: np.ndarray) -> np.ndarray:
    """R2: M(K, iw_n) = (1/Nc) sum_r e^{-i K.r} M(r, iw_n); K = 2 pi (nx/Lx, ny/Ly), index nx + Lx ny."""
    Nc = Lx * Ly
    out = np.zeros_like(M_r)
    for ky in range(Ly):
        for kx in range(Lx):
            ph = np.array([np.exp(-2j * math.pi * (kx * (r % Lx) / Lx + ky * (r // Lx) / Ly)) for r in range(Nc)])
            out[kx + Lx * ky] = (ph[:, None] * M_r).sum(axis=0) / Nc
    return out


def greens_function(beta, xi_k: np.ndarray, M_k: np.ndarray):
    """Eq. (28) and (29) for the isolated cluster, G0(K, iw_n) = 1 / (i w_n - xi_K).  Returns (G, Sigma), [Nc][n_omega]."""
    n_omega = M_k.shape[1]
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    G0 = 1.0 / (1j * wn[None, :] - np.asarray(xi_k)[:, None])
    G = G0 - G0 * M_k * G0 / beta
    return G, 1.0 / G0 - 1.0 / G


# --------------------------------------------------------------------------------------------- the method: delayed NFFT
class DelayedNFFT:
    """Eq. (30)-(31) with readings R4-R6.  accumulate() convolves the samples of one configuration onto the grid,
    finalize() does the single FFT and the division by phi_w."""

    def __init__(self, Lx, Ly, beta, n_omega, oversampling=4, window=6, n_tab=32):
        assert oversampling >= 2 and window >= 1
        self.Lx, self.Ly, self.Nc, self.beta = Lx, Ly, Lx * Ly, float(beta)
        self.n_omega, self.m, self.w, self.n_tab = n_omega, oversampling, window, n_tab
        self.L = oversampling * n_omega
        self.delta = self.beta / self.L
        sigma = oversampling / 2.0
        self.s2 = (2.0 * sigma / (2.0 * sigma - 1.0)) * (window / math.pi)          # R5
        # R6: table of phi and phi' at n_tab points per cell over x in [0, w] (x = |t| / Delta)
        x = np.arange(window * n_tab + 1) / n_tab
        self.tab = np.exp(-x * x / self.s2)
        self.dtab = -2.0 * x / self.s2 * self.tab
        self.grid = np.zeros((2, self.Nc, self.L), np.float64)
        self.sign_sum = 0.0
        self.n_meas = 0

    def window_value(self, x: np.ndarray) -> np.ndarray:
        """phi at x = |t| / Delta <= w by cubic Hermite interpolation in the table (R6)."""
        x = np.abs(x)
        u = x * self.n_tab
        i = np.minimum(np.floor(u).astype(np.int64), self.w * self.n_tab - 1)
        f = u - i
        h = 1.0 / self.n_tab
        p0, p1, d0, d1 = self.tab[i], self.tab[i + 1], self.dtab[i] * h, self.dtab[i + 1] * h
        f2, f3 = f * f, f * f * f
        return (2 * f3 - 3 * f2 + 1) * p0 + (f3 - 2 * f2 + f) * d0 + (-2 * f3 + 3 * f2) * p1 + (f3 - f2) * d1

    def window_hat(self) -> np.ndarray:
        """phi_w at the N_w positive fermionic frequencies: the transform of the truncated window, by its defining sum on
        a 64-fold refined grid (R5)."""
        fine = 64
        x = np.arange(-self.w * fine, self.w * fine + 1) / fine
        wn = (2 * np.arange(self.n_omega) + 1) * math.pi / self.beta
        ph = np.exp(-x * x / self.s2)
        ph[0] *= 0.5
        ph[-1] *= 0.5
        return (ph[:, None] * np.cos(wn[None, :] * (x * self.delta)[:, None])).sum(axis=0) / fine

    def accumulate(self, site, tau, M_up, M_dn, sign=1, site_dn=None):
        """Spread sign * M[j,l] at time tau_j - tau_l (folded antiperiodically, R4) and displacement r_j - r_l onto
        the 2w nearest grid points, for both spins.  site_dn: the sites the DOWN matrix is built on when they differ from
        those of the up matrix (general interactions, NEXT-4: vertex p = (a_p up, b_p down))."""
        site = np.asarray(site)
        tau = np.asarray(tau, dtype=np.float64)
        self.sign_sum += sign
        self.n_meas += 1
        k = site.size
        if k == 0:
            return
        d_up = displacement(self.Lx, self.Ly, site, site).reshape(-1)
        d_dn = d_up if site_dn is None else displacement(self.Lx, self.Ly, np.asarray(site_dn), np.asarray(site_dn)).reshape(-1)
        t = (tau[:, None] - tau[None, :]).reshape(-1)
        sg = np.where(t < 0.0, -1.0, 1.0)
        t = np.where(t < 0.0, t + self.beta, t)
        x = t / self.delta
        l0 = np.floor(x).astype(np.int64)
        for sidx, M in enumerate((M_up, M_dn)):
            d = d_up if sidx == 0 else d_dn
            val = sign * sg * np.asarray(M).reshape(-1)
            for o in range(-self.w + 1, self.w + 1):          # grid points l0 - w + 1 ... l0 + w
                l = l0 + o
                wgt = self.window_value(x - l)
                wrap = np.where(l < 0, -1.0, np.where(l >= self.L, -1.0, 1.0))   # beta-antiperiodic grid
                np.add.at(self.grid[sidx], (d, l % self.L), val * wgt * wrap)

    def finalize(self) -> np.ndarray:
        """Eq. (31): ONE FFT of the accumulated grid, divided by phi_w.  Returns sum_c sign_c M_c(r, iw_n) as
        complex128 [2][Nc][n_omega]; the Monte-Carlo average is this divided by sign_sum (R3)."""
        l = np.arange(self.L)
        twist = np.exp(1j * math.pi * l / self.L)                   # fermionic frequencies: w_n = (2n+1) pi / beta
        F = np.fft.ifft(self.grid * twist[None, None, :], axis=2) * self.L   # sum_l f_l e^{+2 pi i n l / L}
        return F[:, :, : self.n_omega] / self.window_hat()[None, None, :]
