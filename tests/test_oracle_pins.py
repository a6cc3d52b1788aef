"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin states which plausible mistake it catches.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest

from ctaux_workloads import (CONFIGS, atomic_limit_table, g0_exact, g0_table, get_config,
                             mu_for_density, table_for)
from oracle.ctaux_oracle import T0, T1, OracleWalker, philox, unif53

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- P1: table
def test_P1_table_closed_form_values():
    """Generator vs the closed-form values of SURVEY 8c.4 P1 (sign, k-grid, phase factors)."""
    cfg = get_config(0)
    T = table_for(cfg)
    M, beta, Lx = cfg["M"], cfg["beta"], cfg["Lx"]
    for line in open(os.path.join(GOLD, "g0_cfg1_closed_form.txt")):
        if line.startswith("#") or not line.strip():
            continue
        dx, dy, tau, g = line.split()
        m = int(round(float(tau) / beta * M))
        assert abs(-T[int(dx) + Lx * int(dy), m] - float(g)) < 2e-14, line
    # textbook special value: g(0; beta/2) = (1 + 1/cosh 4)/4 on the 2x2 cluster at mu = 0
    assert abs(-T[0, M // 2] - 0.25 * (1 + 1 / math.cosh(4.0))) < 1e-15


@pytest.mark.parametrize("ci", range(5))
def test_P1_table_invariants(ci):
    """g(r,0+) + g(r,beta-) = delta_{r,0} (anticommutator); g(0,0+) = 1 - n_sigma."""
    cfg = get_config(ci)
    T = table_for(cfg)
    s = -(T[:, 0] + T[:, -1])
    want = np.zeros(T.shape[0])
    want[0] = 1.0
    assert np.abs(s - want).max() < 1e-13
    # density from mu: n_sigma = 1 - g(0,0+); the frozen mu reproduces the target filling
    target = {0: 1.0, 1: 1.0, 2: 0.9, 3: 0.9, 4: 0.95}[ci]
    assert abs(2 * (1 + T[0, 0]) - target) < 2e-6
    if ci >= 2:
        assert abs(mu_for_density(cfg["Lx"], cfg["Ly"], cfg["beta"], target) - cfg["mu"]) < 1e-6


def test_P1_oracle_interpolation_exact_on_grid_and_second_order_off_grid():
    cfg = get_config(2)
    T = table_for(cfg)
    w = OracleWalker.from_config(cfg, T, 0)
    beta, M = cfg["beta"], cfg["M"]
    rng = np.random.default_rng(1)
    for _ in range(200):
        d = int(rng.integers(0, 16))
        m = int(rng.integers(1, M))
        tau = m * beta / M
        assert abs(w.g(d, tau) - (-T[d, m])) < 1e-14
        # antiperiodicity: g(d, tau - beta) = -g(d, tau)
        assert abs(w.g(d, tau - beta) + (-T[d, m])) < 1e-14
    taus = rng.uniform(0, beta, 300)
    exact = -g0_exact(cfg["Lx"], cfg["Ly"], beta, cfg["mu"], taus)
    for i, tau in enumerate(taus):
        d = i % 16
        # linear interpolation error <= h^2/8 max|g''| ; |g''| <= max xi^2 <= (4+|mu|)^2
        assert abs(w.g(d, tau) - exact[d, i]) < (beta / M) ** 2 / 8 * 17.0


# ----------------------------------------------------------------------------- P2: gamma
def test_P2_gamma_eq25():
    for line in open(os.path.join(GOLD, "exp_gamma.txt")):
        if line.startswith("#"):
            continue
        ci, ch, eg = line.split()
        cfg = get_config(int(ci))
        w = OracleWalker.from_config(cfg, table_for(cfg), 0)
        assert abs(1 + cfg["U"] * cfg["beta"] * cfg["Lx"] * cfg["Ly"] / (2 * cfg["K"]) - float(ch)) < 1e-12
        assert abs(w.exp_gamma / float(eg) - 1) < 1e-14
        assert abs(math.cosh(math.log(w.exp_gamma)) / float(ch) - 1) < 1e-13


# ----------------------------------------------------------------------------- P3: Fock space
def _fock_ops(nsite):
    """Jordan-Wigner c_i (annihilators) on the 2^nsite Fock space."""
    dim = 1 << nsite
    ops = []
    for i in range(nsite):
        c = np.zeros((dim, dim))
        for st in range(dim):
            if st >> i & 1:
                sgn = (-1) ** bin(st & ((1 << i) - 1)).count("1")
                c[st & ~(1 << i), st] = sgn
        ops.append(c)
    return ops


def _fock_trace(Lx, Ly, beta, mu, sites, taus, avals, eps=None):
    """Tr[T_tau e^{-beta H0} prod_i e^{a_i n_{x_i}(tau_i)}] / Tr e^{-beta H0}: Eq. (27) literally.
    `eps`: dispersion on the cluster momenta (default: the isotropic one of Eq. (45))."""
    from ctaux_workloads import cluster_dispersion
    Nc = Lx * Ly
    kx, ky, eps0 = cluster_dispersion(Lx, Ly)
    eps = eps0 if eps is None else eps
    h = np.zeros((Nc, Nc))
    for i in range(Nc):
        for j in range(Nc):
            dx, dy = i % Lx - j % Lx, i // Lx - j // Lx
            h[i, j] = np.mean(np.cos(kx * dx + ky * dy) * (eps - mu))
    c = _fock_ops(Nc)
    dim = 1 << Nc
    H = np.zeros((dim, dim))
    for i in range(Nc):
        for j in range(Nc):
            H += h[i, j] * c[i].T @ c[j]
    ev, V = np.linalg.eigh(H)

    def prop(t):
        return (V * np.exp(-t * ev)) @ V.T

    order = np.argsort(taus)  # earliest time acts first (rightmost)
    op = np.eye(dim)
    tprev = 0.0
    for i in order:
        op = prop(taus[i] - tprev) @ op
        n = c[sites[i]].T @ c[sites[i]]
        op = (np.eye(dim) + (math.exp(avals[i]) - 1.0) * n) @ op
        tprev = taus[i]
    op = prop(beta - tprev) @ op
    return np.trace(op) / np.sum(np.exp(-beta * ev))


@pytest.mark.parametrize("mu", [0.0, -0.3])
@pytest.mark.parametrize("nv", [1, 2, 3, 4])
def test_P3_fock_space_trace_equals_det_A(mu, nv):
    """Pins Q1 (sign of g), Q2 (E = e^{-gamma sigma s}), Q6 (diagonal = g(0,0+)), time ordering,
    antiperiodicity and the column-scaled form of A: a wrong sign, a transposed g or a row-scaled
    A fails here."""
    Lx = Ly = 2
    beta, U, K, M = 2.0, 4.0, 1.0, 512
    T = g0_table(Lx, Ly, beta, mu, M)
    rng = np.random.default_rng(100 + nv)
    for trial in range(6):
        sites = rng.integers(0, 4, nv).astype(np.int32)
        ms = rng.choice(np.arange(1, M), nv, replace=False)  # on-grid distinct times: interpolation exact
        taus = ms * beta / M
        spins = rng.choice([-1, 1], nv).astype(np.int8)
        w = OracleWalker(Lx, Ly, beta, U, K, T, 0)
        w.set_state(sites, taus, spins)
        gamma = math.log(w.exp_gamma)
        for sidx, sigma in enumerate([+1, -1]):
            a = [-gamma * sigma * int(s) for s in spins]
            want = _fock_trace(Lx, Ly, beta, mu, sites, taus, a)
            got = np.linalg.det(w.A(sidx))
            la, sg = w.logdet(sidx)
            assert abs(got / want - 1) < 1e-11
            assert abs(sg * math.exp(la) / want - 1) < 1e-11


@pytest.mark.parametrize("Lx,Ly,ty", [(3, 3, 1.0), (3, 2, 1.0), (2, 3, 1.0), (3, 3, 0.6)])
@pytest.mark.parametrize("mu", [0.0, -0.3])
def test_P3_fock_space_trace_on_3x3_and_3x2_clusters(Lx, Ly, ty, mu):
    """Pins the displacement index d(i,j) = ((xi-xj) mod Lx) + Lx ((yi-yj) mod Ly) beyond the 2x2 cluster, where
    (xi-xj) mod 2 cannot tell a wrap, a wrong row stride or an x<->y mix-up apart (Eq. (27) evaluated literally in
    the 2^Nc-dimensional Fock space, Nc = 9 / 6, against det A of the oracle).  Lx != Ly catches a row stride of Ly
    instead of Lx and swapped moduli; the 3x3 cluster with anisotropic hopping (t_y = 0.6 t_x, table built here from
    the same closed form) catches an x<->y mix-up that the isotropic square cluster hides (g(dx,dy) = g(dy,dx)
    there).  Every parameter set includes pairs whose raw displacement is negative in x, in y and in both (wraps)."""
    from ctaux_workloads import cluster_dispersion
    beta, U, K, M = 2.0, 4.0, 1.0, 256
    Nc = Lx * Ly
    kx, ky, _ = cluster_dispersion(Lx, Ly)
    eps = -2.0 * (np.cos(kx) + ty * np.cos(ky))
    if ty == 1.0:
        T = g0_table(Lx, Ly, beta, mu, M)
    else:   # closed form G0(r,tau) = -(1/Nc) sum_k cos(k.r) e^{-xi tau}/(1+e^{-beta xi}) with the anisotropic xi_k
        tau = np.arange(M + 1) * (beta / M)
        xi = eps - mu
        wgt = np.exp(-xi[:, None] * tau[None, :]) / (1.0 + np.exp(-beta * xi[:, None]))
        T = np.empty((Nc, M + 1))
        for dy in range(Ly):
            for dx in range(Lx):
                T[dx + Lx * dy] = -(np.cos(kx * dx + ky * dy)[:, None] * wgt).sum(axis=0) / Nc
        assert abs(T[1, 7] - T[Lx, 7]) > 1e-3          # g((1,0)) != g((0,1)): the table can tell x from y
    rng = np.random.default_rng(1000 * Lx + 100 * Ly + int(10 * ty))
    wraps = set()
    for nv in (1, 2, 3, 4):
        for trial in range(3):
            sites = rng.integers(0, Nc, nv).astype(np.int32)
            if nv == 2 and trial == 0:
                sites = np.array([0, Nc - 1], np.int32)          # (0,0) and (Lx-1,Ly-1): wraps in x and y both ways
            if nv == 3 and trial == 0:
                sites = np.array([Lx - 1, Lx * (Ly - 1), 1], np.int32)   # x-only and y-only wraps, mixed (dx,dy)
            taus = rng.choice(np.arange(1, M), nv, replace=False) * beta / M
            spins = rng.choice([-1, 1], nv).astype(np.int8)
            for i in sites:
                for j in sites:
                    wraps.add((int(i % Lx < j % Lx), int(i // Lx < j // Lx)))
            w = OracleWalker(Lx, Ly, beta, U, K, T, 0)
            w.set_state(sites, taus, spins)
            gamma = math.log(w.exp_gamma)
            for sidx, sigma in enumerate([+1, -1]):
                a = [-gamma * sigma * int(s) for s in spins]
                want = _fock_trace(Lx, Ly, beta, mu, sites, taus, a, eps=eps)
                la, sg = w.logdet(sidx)
                assert abs(sg * math.exp(la) / want - 1) < 1e-10, (Lx, Ly, ty, mu, nv, trial, sidx)
                assert abs(np.linalg.det(w.A(sidx)) / want - 1) < 1e-10
    assert wraps == {(0, 0), (0, 1), (1, 0), (1, 1)}


# ----------------------------------------------------------------------------- P4: one vertex
@pytest.mark.parametrize("ci", [0, 2])
def test_P4_one_vertex_closed_form(ci):
    """prod_sigma det A = 1 + (U beta Nc / K) g00 (1 - g00); first insertion from empty: R = K * that."""
    cfg = get_config(ci)
    T = table_for(cfg)
    g00 = -T[0, 0]
    want = 1 + cfg["U"] * cfg["beta"] * cfg["Lx"] * cfg["Ly"] / cfg["K"] * g00 * (1 - g00)
    w = OracleWalker.from_config(cfg, T, 3)
    w.set_state([1], [0.3], [1])
    prod = 1.0
    for s in range(2):
        la, sg = w.logdet(s)
        prod *= sg * math.exp(la)
    assert abs(prod / want - 1) < 1e-13
    if ci == 0:
        assert abs(want - 9.0) < 1e-12
    # chain from the empty configuration: first INSERT proposal has R = K/(0+1) * want
    for mode in (T0, T1):
        w = OracleWalker.from_config(cfg, T, 5, mode)
        w.reset(0)
        w.propose(40)
        log = w.log()
        first_ins = log[log["type"] == 0][0]
        k_before = (log["accepted"][: int(first_ins["p"])] * np.where(log["type"][: int(first_ins["p"])] == 0, 1, -1)).sum()
        assert k_before == 0
        assert abs(first_ins["R"] / (cfg["K"] * want) - 1) < 1e-12


# ----------------------------------------------------------------------------- P5: U -> 0
def test_P5_U_zero_poisson():
    """gamma = 0 => A = N = 1, R_ins = K/(k+1), R_rem = k/K, stationary k ~ Poisson(K).
    Pins the 1/2-1/2 move probabilities, both prefactors, the k=0 removal rule, RNG plumbing."""
    K = 1.5
    T = g0_table(2, 2, 2.0, 0.0, 64)
    w = OracleWalker(2, 2, 2.0, 0.0, K, T, 11, T1)
    w.reset(0)
    n = 400000
    w.propose(n)
    log = w.log()
    dk = log["accepted"] * np.where(log["type"] == 0, 1, -1)
    k_before = np.concatenate([[0], np.cumsum(dk)[:-1]])
    ins = log["type"] == 0
    assert np.allclose(log["R"][ins], K / (k_before[ins] + 1), rtol=1e-13)
    assert np.allclose(log["R"][~ins], k_before[~ins] / K, rtol=1e-13)
    assert np.all(log["accepted"][(~ins) & (k_before == 0)] == 0)
    ks = k_before[1000:]
    # mean = variance = K for a Poisson law; chi^2 on the histogram with an autocorrelation allowance
    assert abs(ks.mean() - K) < 0.03
    assert abs(ks.var() - K) < 0.06
    hist = np.bincount(ks, minlength=12)[:8] / ks.size
    pois = np.array([math.exp(-K) * K ** j / math.factorial(j) for j in range(8)])
    assert np.abs(hist - pois).max() < 0.01
    # N is the identity for every spin
    assert np.allclose(w.N(0), np.eye(w.k)) and np.allclose(w.N_incremental(1), np.eye(w.k))
    # about half the proposals are insertions
    assert abs(ins.mean() - 0.5) < 0.005


# ----------------------------------------------------------------------------- P6: <k> identity
def test_P6_atomic_limit_mean_order():
    """<k> = K - beta <H_int> (from Eq. 23).  Nc = 1, xi = 0: <k> = K + (beta U/2)/(1+e^{-beta U/2}).
    Pins the stationary distribution with U != 0 (prefactors together with the determinant weight)."""
    beta, U, K = 2.0, 4.0, 1.0
    want = K + (beta * U / 2) / (1 + math.exp(-beta * U / 2))
    assert abs(want - 4.92806) < 1e-5
    T = atomic_limit_table(64)
    means = []
    for seed in range(8):
        w = OracleWalker(1, 1, beta, U, K, T, seed, T1)
        w.reset(5)
        w.propose(150000)
        log = w.log()
        dk = log["accepted"] * np.where(log["type"] == 0, 1, -1)
        k_before = 5 + np.concatenate([[0], np.cumsum(dk)[:-1]])
        means.append(k_before[5000:].mean())
    means = np.array(means)
    err = means.std(ddof=1) / math.sqrt(len(means))
    assert abs(means.mean() - want) < max(4 * err, 0.02), (means.mean(), err, want)


# ----------------------------------------------------------------------------- P7/P8: invariants
@pytest.mark.parametrize("ci,sweeps", [(0, 60), (1, 6)])
def test_P7_P8_T1_equals_T0_and_inverse_invariant(ci, sweeps):
    """T1 (rank-1 updates) reproduces T0 (brute-force determinants) decision for decision;
    T1's incrementally updated N is the inverse of A rebuilt from the configuration;
    the removal ratio per spin is N_jj."""
    cfg = get_config(ci)
    T = table_for(cfg)
    a = OracleWalker.from_config(cfg, T, 7, T0)
    b = OracleWalker.from_config(cfg, T, 7, T1)
    for w in (a, b):
        w.reset(cfg["init_k"])
        w.sweep(sweeps)
    la, lb = a.log(), b.log()
    assert len(la) == len(lb) and len(la) >= 16 * sweeps
    for f in ("p", "type", "arg", "tau", "spin", "accepted", "u"):
        assert la[f].tobytes() == lb[f].tobytes(), f
    assert np.allclose(la["R"], lb["R"], rtol=1e-9, atol=1e-300)
    ca, cb = a.config(), b.config()
    for f in ca:
        assert ca[f].tobytes() == cb[f].tobytes()
    assert a.sign == b.sign
    k = b.k
    for s in range(2):
        Ninc = b.N_incremental(s)
        A = b.A(s)
        assert np.linalg.norm(Ninc @ A - np.eye(k)) / math.sqrt(k) < 1e-10
        assert np.linalg.norm(Ninc - a.N(s)) / np.linalg.norm(a.N(s)) < 1e-10
        assert np.linalg.norm(a.N(s) - np.linalg.inv(A)) / np.linalg.norm(a.N(s)) < 1e-11


def test_P8_logged_ratios_by_numpy_determinants():
    """Every logged R of a T0 run equals prefactor * prod_sigma det A'/det A with determinants taken
    by numpy on configurations rebuilt from the log (independent LU, independent bookkeeping)."""
    cfg = get_config(0)
    T = table_for(cfg)
    w = OracleWalker.from_config(cfg, T, 21, T0)
    w.reset(cfg["init_k"])
    c0 = w.config()
    w.sweep(12)
    log = w.log()
    site, tau, spin = list(c0["site"]), list(c0["tau"]), list(c0["spin"])
    probe = OracleWalker.from_config(cfg, T, 0, T0)

    def dets(si, ta, sp):
        probe.set_state(si, ta, sp)
        return [np.linalg.det(probe.A(s)) if len(si) else 1.0 for s in range(2)]

    for e in log:
        k = len(site)
        d0 = dets(site, tau, spin)
        if e["type"] == 0:
            s2, t2, p2 = site + [e["arg"]], tau + [e["tau"]], spin + [e["spin"]]
            pref = cfg["K"] / (k + 1)
        else:
            if k == 0:
                assert e["accepted"] == 0 and e["R"] == 0
                continue
            j = e["arg"]
            s2, t2, p2 = site[:j] + site[j + 1:], tau[:j] + tau[j + 1:], spin[:j] + spin[j + 1:]
            pref = k / cfg["K"]
        d1 = dets(s2, t2, p2)
        R = pref * d1[0] * d1[1] / (d0[0] * d0[1])
        assert abs(R / e["R"] - 1) < 1e-9
        assert e["accepted"] == (1 if e["u"] < abs(R) else 0)
        if e["accepted"]:
            site, tau, spin = s2, t2, p2
    fin = w.config()
    assert list(fin["site"]) == site and list(fin["tau"]) == tau and list(fin["spin"]) == spin
    # ids ascend (insert appends, erase is stable: Q15)
    assert np.all(np.diff(fin["id"].astype(np.int64)) > 0)


# ----------------------------------------------------------------------------- P9-P11
def test_P9_reversibility_P10_permutation_P11_spin_symmetry():
    cfg = get_config(2)
    T = table_for(cfg)
    rng = np.random.default_rng(5)
    k = 12
    site = rng.integers(0, 16, k).astype(np.int32)
    tau = rng.uniform(0, cfg["beta"], k)
    spin = rng.choice([-1, 1], k).astype(np.int8)
    w = OracleWalker.from_config(cfg, T, 0)

    def prod_det(si, ta, sp):
        w.set_state(si, ta, sp)
        out = []
        for s in range(2):
            la, sg = w.logdet(s)
            out.append(sg * math.exp(la))
        return out

    d_full = prod_det(site, tau, spin)
    d_less = prod_det(site[:-1], tau[:-1], spin[:-1])
    K = cfg["K"]
    R_ins = K / k * d_full[0] * d_full[1] / (d_less[0] * d_less[1])
    R_rem = k / K * d_less[0] * d_less[1] / (d_full[0] * d_full[1])
    assert abs(R_ins * R_rem - 1) < 1e-12
    # P10: simultaneous row/column permutation leaves det unchanged
    perm = rng.permutation(k)
    d_perm = prod_det(site[perm], tau[perm], spin[perm])
    assert np.allclose(d_perm, d_full, rtol=1e-11)
    # P11: flipping every s swaps A_up <-> A_down
    d_flip = prod_det(site, tau, -spin)
    assert abs(d_flip[0] / d_full[1] - 1) < 1e-12 and abs(d_flip[1] / d_full[0] - 1) < 1e-12
    w.set_state(site, tau, spin)
    Aup, Adn = w.A(0), w.A(1)
    w.set_state(site, tau, -spin)
    assert np.array_equal(w.A(0), Adn) and np.array_equal(w.A(1), Aup)


# ----------------------------------------------------------------------------- P12: Philox
def test_P12_philox_against_curand_host_generator():
    """cuRAND's HOST Philox4_32_10 generator (runs on the CPU) is an independent implementation.
    Its stream is laid out as 65536 subsequences x 4 words, then the next counter value: output
    group g (4 words) is Philox(counter=(c_lo, c_hi, g % 65536, 0), key=seed) with c = g // 65536
    (layout probed once, then used to pin counter words c0, c1, c2 and both key words)."""
    try:
        cr = C.CDLL("libcurand.so.10")
    except OSError:
        try:
            cr = C.CDLL("/usr/local/cuda/lib64/libcurand.so.10")
        except OSError:
            pytest.skip("libcurand not found")
    gen = C.c_void_p()
    assert cr.curandCreateGeneratorHost(C.byref(gen), 161) == 0  # CURAND_RNG_PSEUDO_PHILOX4_32_10
    for seed in (0, 1, 255, 0x0123456789ABCDEF):
        key = [seed & 0xFFFFFFFF, seed >> 32]
        for c in (0, 1, 2, 1000, 2 ** 31 + 5, 2 ** 32 + 3):
            assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
            assert cr.curandSetGeneratorOffset(gen, C.c_ulonglong(c * 65536 * 4)) == 0
            out = np.zeros(4 * 8, np.uint32)
            assert cr.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(out.size)) == 0
            for s in range(8):
                assert out[4 * s: 4 * s + 4].tolist() == philox([c & 0xFFFFFFFF, c >> 32, s, 0], key).tolist()
    cr.curandDestroyGenerator(gen)


def test_P12_philox_against_triton_interpreter():
    """Second independent implementation (covers counter word c3 = 1, which the walker uses):
    triton.language.philox executed by Triton's CPU interpreter."""
    os.environ["TRITON_INTERPRET"] = "1"
    try:
        import torch
        import triton
        import triton.language as tl

        @triton.jit
        def kern(out, seed, c0, c1, c2, c3):
            a, b, c, d = tl.philox(seed, c0, c1, c2, c3)
            tl.store(out + 0, a)
            tl.store(out + 1, b)
            tl.store(out + 2, c)
            tl.store(out + 3, d)

        cases = [(5, [7, 3, 1, 1]), (0, [0, 0, 0, 1]), (255, [12345, 0, 1, 1]), (17, [2 ** 31 - 1, 9, 0, 1])]
        got = []
        for seed, c in cases:
            out = torch.zeros(4, dtype=torch.int32)
            kern[(1,)](out, seed, c[0], c[1], c[2], c[3])
            got.append(out.numpy().view(np.uint32).tolist())
    except Exception as exc:  # interpreter unavailable in this environment
        pytest.skip(f"triton interpreter unavailable: {exc!r}")
    for (seed, c), g in zip(cases, got):
        assert g == philox(c, [seed, 0]).tolist()


def test_unif53_range_and_bits():
    assert unif53(0, 0) == 0.0
    assert unif53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert unif53(1, 0) == 2.0 ** -32
    assert unif53(0, 1 << 11) == 2.0 ** -53


# ----------------------------------------------------------------------------- sweep convention
def test_sweep_length_and_counter_continuity():
    """Q16: a sweep is max(16, k_start) proposals; the counter runs on across sweep() calls."""
    cfg = get_config(1)
    T = table_for(cfg)
    a = OracleWalker.from_config(cfg, T, 3, T1)
    a.reset(cfg["init_k"])
    k0 = a.k
    a.sweep(1)
    assert a.p == max(16, k0)
    k1 = a.k
    a.sweep(1)
    assert a.p == max(16, k0) + max(16, k1)
    b = OracleWalker.from_config(cfg, T, 3, T1)
    b.reset(cfg["init_k"])
    b.sweep(2)
    assert a.log().tobytes() == b.log().tobytes()
    e = OracleWalker.from_config(get_config(0), table_for(get_config(0)), 3, T0)
    e.reset(0)
    e.sweep(1)
    assert e.p == 16


# ----------------------------------------------------------------------------- NEXT-1: auxiliary-spin flips
def test_flip_ratio_equals_ratio_of_fock_space_traces():
    """A flip multiplies the weight by prod_sigma det A'_sigma / det A_sigma (Fig. 5 (c)->(d)).
    The logged ratio of the oracle's first flip proposal, against the ratio of the two Fock-space traces of
    Eq. (27) evaluated literally (independent of every matrix formula in the oracle)."""
    Lx = Ly = 2
    beta, U, K, M, mu = 2.0, 4.0, 1.0, 512, -0.3
    T = g0_table(Lx, Ly, beta, mu, M)
    rng = np.random.default_rng(7)
    checked = 0
    for seed in range(40):
        nv = int(rng.integers(1, 5))
        sites = rng.integers(0, 4, nv).astype(np.int32)
        taus = rng.choice(np.arange(1, M), nv, replace=False) * beta / M
        spins = rng.choice([-1, 1], nv).astype(np.int8)
        for mode in (T0, T1):
            w = OracleWalker(Lx, Ly, beta, U, K, T, seed, mode)
            w.set_flips(True)
            w.set_state(sites, taus, spins)
            w.propose(1)
            e = w.log()[0]
            if e["type"] != 2:
                continue
            j = int(e["arg"])
            gamma = math.log(w.exp_gamma)
            flipped = spins.copy()
            flipped[j] = -flipped[j]
            want = 1.0
            for sigma in (+1, -1):
                num = _fock_trace(Lx, Ly, beta, mu, sites, taus, [-gamma * sigma * int(s) for s in flipped])
                den = _fock_trace(Lx, Ly, beta, mu, sites, taus, [-gamma * sigma * int(s) for s in spins])
                want *= num / den
            assert abs(e["R"] / want - 1) < 1e-9, (seed, mode, e["R"], want)
            assert e["accepted"] == (1 if e["u"] < abs(e["R"]) else 0)
            checked += 1
    assert checked >= 10


@pytest.mark.parametrize("ci,sweeps", [(0, 60), (1, 6)])
def test_flips_T1_equals_T0(ci, sweeps):
    """With flips enabled the rank-1 oracle (column-change formula) reproduces brute force decision for decision."""
    cfg = get_config(ci)
    table = table_for(cfg)
    out = []
    for mode in (T0, T1):
        w = OracleWalker.from_config(cfg, table, 11, mode)
        w.set_flips(True)
        w.reset(cfg["init_k"])
        w.sweep(sweeps)
        out.append((w.log(), w.config(), w.acc_flip, w.sign, w.N(0), w.N(1)))
    a, b = out
    assert a[2] == b[2] > 0 and a[3] == b[3]
    for f in ("p", "type", "arg", "tau", "spin", "accepted", "u"):
        assert a[0][f].tobytes() == b[0][f].tobytes(), f
    assert set(np.unique(a[0]["type"])) == {0, 1, 2}
    assert np.max(np.abs(a[0]["R"] - b[0]["R"]) / np.maximum(np.abs(a[0]["R"]), 1e-300)) < 1e-8
    for f in a[1]:
        assert a[1][f].tobytes() == b[1][f].tobytes()
    # flipping twice is the identity on the weight: R_1 * R_2 = 1 (brute force, T0)
    cfg1 = a[1]
    w = OracleWalker.from_config(cfg, table, 0, T0)
    w.set_state(cfg1["site"], cfg1["tau"], cfg1["spin"])
    l0 = [w.logdet(s) for s in range(2)]
    sp = cfg1["spin"].copy()
    sp[0] = -sp[0]
    w.set_state(cfg1["site"], cfg1["tau"], sp)
    l1 = [w.logdet(s) for s in range(2)]
    r12 = math.exp(sum(x[0] for x in l1) - sum(x[0] for x in l0))
    r21 = math.exp(sum(x[0] for x in l0) - sum(x[0] for x in l1))
    assert abs(r12 * r21 - 1) < 1e-12


def test_flips_keep_the_stationary_distribution():
    """Adding a valid move must not change the stationary law: atomic limit <k> (pin P6) with flips on, and the
    auxiliary spins stay unpolarised on average."""
    beta, U, K = 2.0, 4.0, 1.0
    want = K + (beta * U / 2) / (1 + math.exp(-beta * U / 2))
    T = atomic_limit_table(64)
    means, acc = [], 0
    for seed in range(8):
        w = OracleWalker(1, 1, beta, U, K, T, seed, T1)
        w.set_flips(True)
        w.reset(5)
        w.propose(150000)
        log = w.log()
        dk = log["accepted"] * np.where(log["type"] == 0, 1, np.where(log["type"] == 1, -1, 0))
        k_before = 5 + np.concatenate([[0], np.cumsum(dk)[:-1]])
        means.append(k_before[5000:].mean())
        acc += w.acc_flip
    means = np.array(means)
    err = means.std(ddof=1) / math.sqrt(len(means))
    assert acc > 1000
    assert abs(means.mean() - want) < max(4 * err, 0.02), (means.mean(), err, want)


# ----------------------------------------------------------------------------- T1 at the sizes it referees
@pytest.mark.parametrize("name,seed,nprop", [("cfg4_6x6_b20", 0, 48), ("cfg5_6x6_b40", 1, 16)])
def test_T1_equals_brute_force_at_full_size(name, seed, nprop):
    """The rank-1 oracle (T1) referees the parity tests on configs 4-5 (k ~ 1700-3600, e^gamma = 4322 / 8642), far
    from the k <= 65 where it is compared with T0 proposal by proposal.  Here: from the thermalised configuration of
    tests/golden (written by the oracle), T1 runs `nprop` proposals; every logged ratio and decision is re-derived by
    brute force -- A and A' built from the vertex lists, determinants by LAPACK (Eq. (27); SURVEY 8d log-replay
    protocol) -- and T1's incrementally updated N is compared with LAPACK's inverse of A built from the final list."""
    from parity_helpers import brute_force_verify, load_thermalised
    cfg = get_config(name)
    T = table_for(cfg)
    c0, next_id, p0 = load_thermalised(name, seed)
    o = OracleWalker.from_config(cfg, T, 5, T1)
    o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], next_id, p0)
    o.propose(nprop)
    log = o.log()
    assert log["accepted"].sum() >= nprop // 4 and set(np.unique(log["type"])) == {0, 1}
    worst = brute_force_verify(cfg, T, c0, log, [(0, nprop)], rtol=1e-8, atol=1e-10, what=name)
    assert worst < 1.0
    for s in range(2):
        Ninc, Ndir = o.N_incremental(s), np.linalg.inv(o.A(s))
        assert np.linalg.norm(Ninc - Ndir) / np.linalg.norm(Ndir) < 1e-10
