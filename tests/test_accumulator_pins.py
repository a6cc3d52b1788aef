"""Pins of the single-particle accumulation oracle (oracle/ctaux_accumulator.py) against what the
paper and the mathematics fix.  None of these tests touches the CUDA path."""
import math

import numpy as np
import pytest

from ctaux_workloads import atomic_limit_table, cluster_dispersion, g0_table, get_config, table_for
from oracle.ctaux_accumulator import DelayedNFFT, g_config, greens_function, m_direct, m_matrix, m_of_k
from oracle.ctaux_oracle import T1, OracleWalker


# ----------------------------------------------------------------------------- Fock-space Green's function of a configuration
def _fock_ops(nsite):
    dim = 1 << nsite
    ops = []
    for i in range(nsite):
        c = np.zeros((dim, dim))
        for st in range(dim):
            if st >> i & 1:
                c[st & ~(1 << i), st] = (-1) ** bin(st & ((1 << i) - 1)).count("1")
        ops.append(c)
    return ops


def _fock_time_ordered(Lx, Ly, beta, mu, events):
    """Tr[T_tau e^{-beta H0} prod O_i(tau_i)] for events (tau, matrix-in-Fock-space), already carrying the fermionic sign
    of the ordering (the caller supplies it); earliest time acts first."""
    Nc = Lx * Ly
    kx, ky, eps = cluster_dispersion(Lx, Ly)
    h = np.zeros((Nc, Nc))
    for i in range(Nc):
        for j in range(Nc):
            dx, dy = i % Lx - j % Lx, i // Lx - j // Lx
            h[i, j] = np.mean(np.cos(kx * dx + ky * dy) * (eps - mu))
    c = _fock_ops(Nc)
    dim = 1 << Nc
    H = sum(h[i, j] * c[i].T @ c[j] for i in range(Nc) for j in range(Nc))
    ev, V = np.linalg.eigh(H)
    prop = lambda t: (V * np.exp(-t * ev)) @ V.T
    op, tprev = np.eye(dim), 0.0
    for t, mat in sorted(events, key=lambda e: e[0]):
        op = mat(c) @ prop(t - tprev) @ op
        tprev = t
    return np.trace(prop(beta - tprev) @ op)


@pytest.mark.parametrize("mu", [0.0, -0.3])
@pytest.mark.parametrize("nv", [1, 2, 3])
def test_M_gives_the_greens_function_of_a_configuration(mu, nv):
    """R1 (Eq. (27)-(28)): with M = (E - 1) N, g_c(x, y) = g(x,y) + sum_jl g(x,j) M[j,l] g(l,y) is
    <T c_x(tau) c+_y(tau') prod e^{a_i n_i}>_0 / <T prod e^{a_i n_i}>_0, evaluated literally in the 16-dimensional Fock
    space of the 2x2 cluster.  A factor on the wrong side of N, a transposed M or a wrong sign fails here."""
    Lx = Ly = 2
    beta, U, K, Mt = 2.0, 4.0, 1.0, 512
    T = g0_table(Lx, Ly, beta, mu, Mt)
    rng = np.random.default_rng(40 + nv)
    for trial in range(4):
        grid = rng.choice(np.arange(1, Mt), nv + 2, replace=False)       # distinct on-grid times: interpolation exact
        taus, (tx, ty) = grid[:nv] * beta / Mt, grid[nv:] * beta / Mt
        sites = rng.integers(0, 4, nv).astype(np.int32)
        spins = rng.choice([-1, 1], nv).astype(np.int8)
        x, y = int(rng.integers(0, 4)), int(rng.integers(0, 4))
        w = OracleWalker(Lx, Ly, beta, U, K, T, 0)
        w.set_state(sites, taus, spins)
        gamma = math.log(w.exp_gamma)
        disp = lambda i, j: ((i % Lx - j % Lx) % Lx) + Lx * ((i // Lx - j // Lx) % Ly)
        for sidx, sigma in enumerate([+1, -1]):
            a = [-gamma * sigma * int(s) for s in spins]
            vert = [(taus[i], (lambda c, i=i: np.eye(16) + (math.exp(a[i]) - 1.0) * c[sites[i]].T @ c[sites[i]])) for i in range(nv)]
            den = _fock_time_ordered(Lx, Ly, beta, mu, vert)
            num = _fock_time_ordered(Lx, Ly, beta, mu, vert + [(tx, lambda c: c[x]), (ty, lambda c: c[y].T)])
            want = (1.0 if tx > ty else -1.0) * num / den          # T-ordering sign of c_x(tx) c+_y(ty)
            M = m_matrix(w.N(sidx), spins, sidx, w.exp_gamma)
            g_xv = np.array([w.g(disp(x, int(sites[j])), tx - taus[j]) for j in range(nv)])
            g_vy = np.array([w.g(disp(int(sites[l]), y), taus[l] - ty) for l in range(nv)])
            got = g_config(g_xv, M, g_vy, w.g(disp(x, y), tx - ty))
            assert abs(got - want) < 1e-11 * max(1.0, abs(want)), (mu, nv, trial, sidx, got, want)


def test_one_vertex_closed_form_of_M_and_window_normalisation():
    """One vertex: N = 1/A, A = E - g00 (E - 1), so M(r=0, iw_n) = (E - 1)/(E - g00 (E - 1)) for EVERY frequency (a delta
    function at tau - tau' = 0) and M(r != 0) = 0.  Pins m_direct, and -- the sample sits exactly on a grid point -- the
    window, its Fourier coefficients phi_w and the fermionic twist of the delayed NFFT."""
    cfg = get_config(0)
    T = table_for(cfg)
    w = OracleWalker.from_config(cfg, T, 0)
    w.set_state([2], [0.7], [1])
    g00 = -T[0, 0]
    n_omega = 64
    nf = DelayedNFFT(cfg["Lx"], cfg["Ly"], cfg["beta"], n_omega, oversampling=8, window=10)
    Ms = []
    for sidx in range(2):
        E = 1.0 / w.exp_gamma if sidx == 0 else w.exp_gamma
        want = (E - 1.0) / (E - g00 * (E - 1.0))
        M = m_matrix(w.N(sidx), [1], sidx, w.exp_gamma)
        assert abs(M[0, 0] / want - 1) < 1e-13
        Mr = m_direct(cfg["Lx"], cfg["Ly"], cfg["beta"], [2], [0.7], M, n_omega)
        assert np.abs(Mr[0] - want).max() < 1e-12 * abs(want) and np.abs(Mr[1:]).max() == 0.0
        Ms.append(M)
    nf.accumulate([2], [0.7], Ms[0], Ms[1], sign=1)
    F = nf.finalize()
    for sidx in range(2):
        assert np.abs(F[sidx, 0] - Ms[sidx][0, 0]).max() < 1e-9 * abs(Ms[sidx][0, 0])
        assert np.abs(F[sidx, 1:]).max() < 1e-12


@pytest.mark.parametrize("ci,m,wnd,tol", [(1, 4, 6, 2e-5), (1, 8, 10, 1e-9), (2, 4, 6, 2e-5), (2, 8, 10, 1e-9)])
def test_delayed_nfft_equals_direct_fourier_sum(ci, m, wnd, tol):
    """Eq. (30)-(31) against the definition: M(r, iw_n) of thermalised configurations (configs 2 and 3, both spins, a
    few configurations accumulated with signs) by the delayed NFFT and by the O(k^2 N_w) direct sum.  The error is the
    aliasing error of the Gaussian window, ~4 exp(-w pi (1 - 1/(2 sigma - 1))): 2e-5 for (m, w) = (4, 6), below 1e-9 for
    (8, 10) -- "a controllable interpolation error"."""
    cfg = get_config(ci)
    T = table_for(cfg)
    n_omega = 128
    nf = DelayedNFFT(cfg["Lx"], cfg["Ly"], cfg["beta"], n_omega, oversampling=m, window=wnd)
    direct = np.zeros((2, cfg["Lx"] * cfg["Ly"], n_omega), np.complex128)
    for seed, sign in ((0, 1), (1, -1), (2, 1)):
        w = OracleWalker.from_config(cfg, T, seed, T1)
        w.reset(cfg["init_k"])
        w.sweep(20 if ci == 1 else 12)
        c = w.config()
        Ms = [m_matrix(w.N(s), c["spin"], s, w.exp_gamma) for s in range(2)]
        nf.accumulate(c["site"], c["tau"], Ms[0], Ms[1], sign=sign)
        for s in range(2):
            direct[s] += sign * m_direct(cfg["Lx"], cfg["Ly"], cfg["beta"], c["site"], c["tau"], Ms[s], n_omega)
    F = nf.finalize()
    assert nf.n_meas == 3 and nf.sign_sum == 1
    scale = np.abs(direct).max()
    assert np.abs(F - direct).max() / scale < tol


def test_atomic_limit_greens_function_from_accumulated_M():
    """Eq. (28) with R2/R3 on the exactly solvable case Nc = 1, xi = 0 (half-filled atom, H = U (n_up - 1/2)(n_dn - 1/2)
    up to constants): G(iw_n) = 1/2 [1/(iw_n - U/2) + 1/(iw_n + U/2)] = -i w_n / (w_n^2 + U^2/4).  The oracle chain
    samples configurations, M is accumulated with the delayed NFFT, and Eq. (28) gives G within the Monte-Carlo error.
    Pins the 1/beta of Eq. (28), the sign of M and the sampling with signs."""
    beta, U, K = 2.0, 4.0, 1.0
    T = atomic_limit_table(64)
    n_omega = 8
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    exact = -1j * wn / (wn ** 2 + U * U / 4)
    runs = []
    for seed in range(8):
        w = OracleWalker(1, 1, beta, U, K, T, seed, T1)
        w.reset(5)
        w.propose(4000)
        nf = DelayedNFFT(1, 1, beta, n_omega, oversampling=8, window=10)
        for meas in range(1500):
            w.propose(12)
            c = w.config()
            if w.k:
                Ms = [m_matrix(w.N(s), c["spin"], s, w.exp_gamma) for s in range(2)]
            else:
                Ms = [np.zeros((0, 0))] * 2
            nf.accumulate(c["site"], c["tau"], Ms[0], Ms[1], sign=w.sign)
        Mk = nf.finalize() / nf.sign_sum
        G, Sigma = greens_function(beta, np.array([0.0]), 0.5 * (Mk[0] + Mk[1]))
        runs.append(G[0])
    runs = np.array(runs)
    mean, err = runs.mean(axis=0), runs.std(axis=0, ddof=1) / math.sqrt(len(runs))
    assert np.all(np.abs(mean - exact) < np.maximum(4.5 * err, 2e-3)), (mean, exact, err)
    # Eq. (29): the atomic self-energy is U^2 / (4 i w_n); checked at the lowest frequency within the propagated error
    sig = 1j * wn - 1.0 / mean
    assert abs(sig[0] - U * U / (4j * wn[0])) < 0.15 * abs(U * U / (4 * wn[0]))


def test_m_of_k_is_the_cluster_fourier_transform():
    """R2: M(K) = (1/Nc) sum_r e^{-iK.r} M(r); a function that is 1 at r = 0 only transforms to 1/Nc at every K, a constant
    to delta_{K,0}; on the 3x2 cluster the phases of x and y are not interchangeable."""
    Lx, Ly = 3, 2
    Mr = np.zeros((6, 1), np.complex128)
    Mr[0] = 1.0
    assert np.allclose(m_of_k(Lx, Ly, Mr), 1.0 / 6)
    assert np.allclose(m_of_k(Lx, Ly, np.ones((6, 1), np.complex128))[:, 0], [1, 0, 0, 0, 0, 0])
    Mr = np.zeros((6, 1), np.complex128)
    Mr[1] = 1.0                                                     # r = (1, 0)
    want = np.array([np.exp(-2j * math.pi * kx / 3) / 6 for ky in range(2) for kx in range(3)])
    assert np.allclose(m_of_k(Lx, Ly, Mr)[:, 0], want)
