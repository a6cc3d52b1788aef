"""GPU parity with a general opposite-spin density-density interaction (ctaux_params.n_pairs):
extended Hubbard clusters (on-site U plus nearest-neighbour V between opposite spins) and a bilayer
(U in each layer, V between the layers, PAPER.md:752-776 with the layers mapped onto the two rows of an Lx x 2 cluster).
Same bar as everywhere: decisions and configurations bit-exact, N within 1e-10."""
import math

import numpy as np
import pytest

from ctaux_workloads import get_config, table_for, walker_seeds
from oracle.ctaux_accumulator import DelayedNFFT
from oracle.ctaux_oracle import T0, T1, OracleWalker

from parity_helpers import compare_logs, full_parity
from test_pairs_pins import extended_hubbard_pairs

pytestmark = pytest.mark.gpu


def _pkg():
    import paper_1901_01047_b200 as pkg
    return pkg


@pytest.mark.parametrize("fused", [1, -1])
def test_extended_hubbard_2x2_against_brute_force(fused):
    """2x2 cluster, U = 4, V = 1.5: N_corr = 12 pairs.  Config-1 shape (beta = 2) in full lock step with T0, config-2
    shape (beta = 10, <k> ~ 150: needs max_k 320, so the fused path is asked only at beta = 2) on the delayed path."""
    pairs = extended_hubbard_pairs(2, 2, 4.0, 1.5)
    cfg = dict(get_config(0), name="ext_2x2_b2", max_k=96, init_k=12)
    W, orcs, worst = full_parity(cfg, 3, 120, T0, fused=fused, pairs=pairs)
    log = W.get_log(0)
    assert log["arg"][log["type"] == 0].max() >= 4           # inter-site pairs proposed (and the log carries pair indices)
    assert max(o.k for o in orcs) > 12
    if fused < 0:
        cfg2 = dict(get_config(1), name="ext_2x2_b10", max_k=320, init_k=100, delay=32)
        # From this far-from-equilibrium random start (N_corr = 12: cosh gamma = 241) single ratios are differences with a
        # cancellation of ~1e4 (|s_nn| against |s_nn - s_row S^-1 s_col|); with N itself good to 1e-10 a logged R carries up
        # to ~1e-6 relative error -- measured 1.3e-6 against brute force.  Decisions, configurations and N keep their bars.
        full_parity(cfg2, 4, 8, T0, fused=-1, pairs=pairs, r_rtol=1e-5)


def test_extended_hubbard_4x4_delayed_blocks_and_large_k_kernels():
    """4x4 cluster, beta = 5, U = 4, V = 1: N_corr = 80, <k> ~ 200; the delayed-block path with the candidate GEMMs per
    spin sector (the two sectors see different sites), once with the small-k and once with the large-k launch shapes."""
    pairs = extended_hubbard_pairs(4, 4, 4.0, 1.0)
    cfg = dict(get_config(2), name="ext_4x4_b5", beta=5.0, max_k=448, init_k=150)
    # thermalising chains from a random 150-vertex start (cond(A) ~ 1e6): the logged ratios of the two sides agree to a few
    # 1e-7 relative, within a factor of two of parity_helpers' equilibrium tolerance (1e-6), and where a block ends moves
    # them; the bar here is 1e-5 as for the 2x2 thermalising case above, decisions stay bit-exact
    full_parity(cfg, 6, 8, T1, pairs=pairs, r_rtol=1e-5)
    full_parity(dict(cfg, max_k=600), 2, 5, T1, pairs=pairs, delay=128, r_rtol=1e-5)


def test_bilayer_interlayer_interaction_and_flips():
    """Bilayer as a 4 x 2 cluster (row = layer): U = 4 on every site, V = 2 between the two sites of a rung, opposite
    spins, with the auxiliary-spin flip as third move."""
    Lx, Ly = 4, 2
    a = list(range(8)) + [i for i in range(4)] + [4 + i for i in range(4)]
    b = list(range(8)) + [4 + i for i in range(4)] + [i for i in range(4)]
    u = [4.0] * 8 + [2.0] * 8
    pairs = (np.array(a, np.int32), np.array(b, np.int32), np.array(u))
    cfg = dict(get_config(1), name="bilayer_4x2", Lx=Lx, Ly=Ly, beta=3.0, max_k=112, init_k=30)
    for fused in (1, -1):
        full_parity(cfg, 4, 10, T1, fused=fused, pairs=pairs, flips=1)


def test_accumulator_with_pairs_uses_the_sites_of_each_spin_sector():
    """S6 with pairs: the displacement of a sample of M_up is a_j - a_l, of M_down b_j - b_l."""
    from oracle.ctaux_accumulator import m_direct
    pkg = _pkg()
    pa, pb, pu = extended_hubbard_pairs(2, 2, 4.0, 1.5)
    cfg = dict(get_config(0), name="ext_2x2_b2", max_k=96, init_k=12)
    table = table_for(cfg)
    n_omega, nw = 32, 3
    orcs = []
    for seed in range(nw):
        o = OracleWalker.from_config(cfg, table, 70 + seed, T1)
        o.set_pairs(pa, pb, pu)
        o.reset(cfg["init_k"])
        o.sweep(30)
        orcs.append(o)
    W = pkg.Walkers.from_config(cfg, table, n_walkers=nw, n_omega=n_omega, nfft_oversampling=8, nfft_window=10, pairs=(pa, pb, pu))
    W.set_state(walker_seeds(nw), [o.config() for o in orcs], [o.next_id for o in orcs], [o.p for o in orcs])
    W.accumulate()
    Md, ss, nm = W.get_M()
    nf = DelayedNFFT(2, 2, cfg["beta"], n_omega, oversampling=8, window=10)
    direct = np.zeros_like(Md)
    for o in orcs:
        c = o.config()
        Ms = []
        for s in range(2):
            eg = np.array([o.pair_exp_gamma(int(p)) for p in c["site"]])
            E = np.where((1 if s == 0 else -1) * c["spin"] > 0, 1.0 / eg, eg)
            Ms.append((E - 1.0)[:, None] * o.N(s))
        nf.accumulate(pa[c["site"]], c["tau"], Ms[0], Ms[1], sign=o.sign, site_dn=pb[c["site"]])
        direct[0] += o.sign * m_direct(2, 2, cfg["beta"], pa[c["site"]], c["tau"], Ms[0], n_omega)
        direct[1] += o.sign * m_direct(2, 2, cfg["beta"], pb[c["site"]], c["tau"], Ms[1], n_omega)
    Mo = nf.finalize()
    for s in range(2):
        assert np.abs(Md[s] - Mo[s]).max() < 1e-9 * np.abs(Mo[s]).max()
        assert np.abs(Md[s] - direct[s]).max() < 2e-9 * np.abs(direct[s]).max()


def test_pairs_arguments_are_validated():
    pkg = _pkg()
    cfg = get_config(0)
    table = table_for(cfg)
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.Walkers.from_config(cfg, table, pairs=(np.array([0, 4]), np.array([0, 1]), np.array([4.0, 1.0])))   # site 4 of 4
    assert ei.value.code == -1
