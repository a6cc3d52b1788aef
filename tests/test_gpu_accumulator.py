"""GPU parity of the single-particle accumulator S6: ctaux_accumulate / ctaux_get_M through the C ABI
against oracle/ctaux_accumulator.py on the same configurations.

Tolerance: both sides evaluate the SAME window table formula and the same transform, so they differ
by (a) the order of the k^2 additions per grid point and (b) the two N matrices, which agree to 1e-10 (relative Frobenius)
-- M is linear in N.  Bar: |M_dev - M_orc| <= 1e-9 max|M_orc| per spin.  Against the DEFINITION (direct Fourier sum) both
carry the aliasing error of the window, ~2e-5 at the default (m, w) = (4, 6), < 1e-9 at (8, 10)."""
import math

import numpy as np
import pytest

from ctaux_workloads import atomic_limit_table, get_config, table_for, walker_seeds
from oracle.ctaux_accumulator import DelayedNFFT, greens_function, m_direct, m_matrix
from oracle.ctaux_oracle import T1, OracleWalker

from parity_helpers import load_thermalised

pytestmark = pytest.mark.gpu

TOL = 1e-9


def _pkg():
    import paper_1901_01047_b200 as pkg
    return pkg


def _rel(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


@pytest.mark.parametrize("ci,nw,sweeps,m,wnd", [(1, 6, 25, 4, 6), (1, 3, 25, 8, 10), (2, 4, 12, 4, 6), (0, 2, 50, 4, 6)])
def test_accumulate_matches_oracle_on_given_configurations(ci, nw, sweeps, m, wnd):
    """Every walker starts from its OWN oracle-thermalised configuration (set_state), one ctaux_accumulate, one
    ctaux_get_M: against the oracle's delayed NFFT (same window parameters) and against the direct Fourier sum."""
    cfg = get_config(ci)
    table = table_for(cfg)
    n_omega = 64
    orcs = []
    for seed in range(nw):
        o = OracleWalker.from_config(cfg, table, 100 + seed, T1)
        o.reset(cfg["init_k"])
        o.sweep(sweeps)
        orcs.append(o)
    W = _pkg().Walkers.from_config(cfg, table, n_walkers=nw, n_omega=n_omega, nfft_oversampling=m, nfft_window=wnd)
    W.set_state(walker_seeds(nw), [o.config() for o in orcs], [o.next_id for o in orcs], [o.p for o in orcs])
    W.accumulate()
    Md, sign_sum, n_meas = W.get_M()
    nf = DelayedNFFT(cfg["Lx"], cfg["Ly"], cfg["beta"], n_omega, oversampling=m, window=wnd)
    direct = np.zeros_like(Md)
    for w, o in enumerate(orcs):
        c = o.config()
        assert W.get_stats(w)["sign"] == o.sign
        Ms = [m_matrix(o.N(s), c["spin"], s, o.exp_gamma) for s in range(2)]
        nf.accumulate(c["site"], c["tau"], Ms[0], Ms[1], sign=o.sign)
        for s in range(2):
            direct[s] += o.sign * m_direct(cfg["Lx"], cfg["Ly"], cfg["beta"], c["site"], c["tau"], Ms[s], n_omega)
    Mo = nf.finalize()
    assert n_meas == nw and sign_sum == sum(o.sign for o in orcs)
    for s in range(2):
        assert _rel(Md[s], Mo[s]) < TOL
        assert _rel(Md[s], direct[s]) < (2e-5 if (m, wnd) == (4, 6) else 2e-9)


def test_accumulation_over_a_chain_with_signs_and_reset():
    """Device chain and oracle chain in lock step (config 2, 8 walkers): 6 x (one sweep, one measurement); the sum of
    sign * M over all measurements, sign_sum and n_meas agree; ctaux_reset_accumulator starts over; a second context
    with the measurements split differently gives the same sums (the accumulation is linear)."""
    cfg = get_config(1)
    table = table_for(cfg)
    nw, n_omega, nmeas = 8, 32, 6
    seeds = walker_seeds(nw, first=30)
    W = _pkg().Walkers.from_config(cfg, table, n_walkers=nw, n_omega=n_omega, rebuild_every=1)
    W.reset(seeds)
    orcs = []
    for s in seeds:
        o = OracleWalker.from_config(cfg, table, int(s), T1)
        o.reset(cfg["init_k"])
        orcs.append(o)
    nf = DelayedNFFT(cfg["Lx"], cfg["Ly"], cfg["beta"], n_omega)
    for it in range(nmeas):
        W.sweep(1)
        W.accumulate()
        for o in orcs:
            o.sweep(1)
            c = o.config()
            nf.accumulate(c["site"], c["tau"], m_matrix(o.N(0), c["spin"], 0, o.exp_gamma),
                          m_matrix(o.N(1), c["spin"], 1, o.exp_gamma), sign=o.sign)
    Md, ss, nm = W.get_M()
    Mo = nf.finalize()
    assert nm == nw * nmeas and ss == nf.sign_sum
    for s in range(2):
        assert _rel(Md[s], Mo[s]) < TOL
    Md2, _, _ = W.get_M()                        # get_M does not reset
    assert np.array_equal(Md, Md2)
    W.reset_accumulator()
    Mz, ss0, nm0 = W.get_M()
    assert nm0 == 0 and ss0 == 0 and np.abs(Mz).max() == 0.0


def test_empty_configuration_and_disabled_accumulator():
    """Degenerate cases: a walker with k = 0 contributes its sign and nothing else; without n_omega the calls are
    refused with CTAUX_ESTATE."""
    pkg = _pkg()
    cfg = get_config(0)
    table = table_for(cfg)
    W = pkg.Walkers.from_config(cfg, table, n_walkers=2, n_omega=16, init_k=0)
    W.reset(walker_seeds(2))
    W.accumulate()
    M, ss, nm = W.get_M()
    assert nm == 2 and ss == 2.0 and np.abs(M).max() == 0.0
    W2 = pkg.Walkers.from_config(cfg, table, n_walkers=1)
    W2.reset([0])
    with pytest.raises(pkg.CtauxError) as ei:
        W2.accumulate()
    assert ei.value.code == -5
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.Walkers.from_config(cfg, table, n_walkers=1, n_omega=16, nfft_window=17)   # 2w > 32 lanes
    assert ei.value.code == -1


@pytest.mark.slow
def test_accumulate_config4_full_size_against_direct_sum():
    """Config 4 at full size (k ~ 1720, 36 displacements, 3 M samples per spin) from the oracle-thermalised start: one
    measurement against the oracle's delayed NFFT and against the direct Fourier sum of the oracle's M."""
    cfg = get_config(3)
    table = table_for(cfg)
    c0, next_id, p0 = load_thermalised(cfg["name"])
    n_omega = 32
    W = _pkg().Walkers(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, delay=cfg["delay"], n_walkers=1,
                       init_k=0, max_k=cfg["max_k"], n_omega=n_omega)
    W.set_state([0], [c0], [next_id], [p0])
    W.accumulate()
    Md, ss, nm = W.get_M()
    o = OracleWalker.from_config(cfg, table, 0, T1)
    o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], next_id, p0)
    Ms = [m_matrix(np.linalg.inv(o.A(s)), c0["spin"], s, o.exp_gamma) for s in range(2)]
    nf = DelayedNFFT(cfg["Lx"], cfg["Ly"], cfg["beta"], n_omega)
    nf.accumulate(c0["site"], c0["tau"], Ms[0], Ms[1], sign=o.sign)
    Mo = nf.finalize()
    assert ss == o.sign and nm == 1
    for s in range(2):
        assert _rel(Md[s], Mo[s]) < TOL
        direct = o.sign * m_direct(cfg["Lx"], cfg["Ly"], cfg["beta"], c0["site"], c0["tau"], Ms[s], n_omega)
        assert _rel(Md[s], direct) < 2e-5


def test_atomic_limit_greens_function_on_the_device():
    """The whole NEXT-2 path on the device, pinned to an exact result (no oracle involved): Nc = 1, xi = 0,
    G(iw_n) = -i w_n / (w_n^2 + U^2/4).  128 device chains, a measurement every sweep, Eq. (28) with <M> = sum / sign_sum."""
    pkg = _pkg()
    beta, U, K = 2.0, 4.0, 1.0
    n_omega, nw = 8, 128
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    exact = -1j * wn / (wn ** 2 + U * U / 4)
    est = []
    for rep in range(4):
        W = pkg.Walkers(1, 1, beta, U, K, atomic_limit_table(64), delay=8, n_walkers=nw, init_k=5, max_k=64,
                        rebuild_every=20, n_omega=n_omega, nfft_oversampling=8, nfft_window=10)
        W.reset(walker_seeds(nw, first=2000 + 1000 * rep))
        W.sweep(100)
        for it in range(150):
            W.sweep(1)
            W.accumulate()
        M, ss, nm = W.get_M()
        assert nm == 150 * nw
        G, Sigma = greens_function(beta, np.array([0.0]), 0.5 * (M[0] + M[1]) / ss)
        est.append(G[0])
        W.close()
    est = np.array(est)
    mean, err = est.mean(axis=0), est.std(axis=0, ddof=1) / 2.0
    assert np.all(np.abs(mean - exact) < np.maximum(4.5 * err, 2e-3)), (mean, exact, err)
