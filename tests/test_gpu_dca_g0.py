"""GPU parity of the DCA bare-propagator table: ctaux_g0_table through the C ABI against
oracle/dca_g0.py, element by element, and a walker driven by such a table against the oracle walker on the same table.

Tolerance: both sides evaluate the same sums in a different order (n_quad^2 terms of O(1) per frequency, then N_w terms of
size <= 1/w_n^4 after the tail removal): 1e-12 absolute on table entries of magnitude <= 1."""
import math

import numpy as np
import pytest

from ctaux_workloads import g0_table, get_config, walker_seeds
from oracle.ctaux_oracle import T0
from oracle.dca_g0 import g0_table_from_sigma as orc_table

from parity_helpers import full_parity

pytestmark = pytest.mark.gpu


def _pkg():
    import paper_1901_01047_b200 as pkg
    return pkg


@pytest.mark.parametrize("Lx,Ly,beta,mu,n_omega,n_quad,n_tau,with_sigma",
                         [(2, 2, 2.0, 0.0, 256, 1, 64, False), (2, 2, 2.0, 0.0, 256, 8, 64, True),
                          (4, 4, 10.0, -0.054654, 1024, 6, 512, True), (3, 2, 5.0, -0.3, 300, 5, 37, True),
                          (1, 1, 4.0, 0.1, 128, 16, 16, False), (6, 6, 20.0, -0.037689, 2048, 4, 512, True)])
def test_g0_table_against_oracle(Lx, Ly, beta, mu, n_omega, n_quad, n_tau, with_sigma):
    Nc = Lx * Ly
    sig = None
    if with_sigma:      # a causal-looking, inversion-symmetric test self-energy: static part + 1/(iw) tail, K dependent
        wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
        kx = 2 * math.pi * (np.arange(Nc) % Lx) / Lx
        ky = 2 * math.pi * (np.arange(Nc) // Lx) / Ly
        amp = 1.0 + 0.3 * (np.cos(kx) + np.cos(ky))
        sig = 0.4 * amp[:, None] + (amp[:, None] ** 2) / (1j * wn[None, :] + 0.2)
    dev = _pkg().g0_table_from_sigma(Lx, Ly, 1.0, mu, beta, n_omega, n_quad, n_tau, sigma_c=sig)
    orc = orc_table(Lx, Ly, 1.0, mu, beta, n_omega, n_quad, n_tau, sigma_c=sig)
    assert dev.shape == orc.shape == (Nc, n_tau + 1)
    assert np.abs(dev - orc).max() < 1e-12
    if n_quad == 1 and not with_sigma:      # the isolated cluster: the closed form of ctaux_workloads
        assert np.abs(dev - g0_table(Lx, Ly, beta, mu, n_tau)).max() < 1e-5


def test_walker_on_an_embedded_cluster_table():
    """The walker does not care where its table comes from: configs 1-2 shapes with the coarse-grained (n_quad = 8)
    propagator of the DEVICE generator, device walker against the brute-force oracle walker on that same table."""
    pkg = _pkg()
    cfg = dict(get_config(1), name="cfg2_embedded")
    table = pkg.g0_table_from_sigma(cfg["Lx"], cfg["Ly"], 1.0, cfg["mu"], cfg["beta"], 1024, 8, cfg["M"])
    import parity_helpers
    orig = parity_helpers.table_for
    parity_helpers.table_for = lambda c: table
    try:
        for fused in (1, -1):
            full_parity(cfg, 4, 8, T0, fused=fused)
    finally:
        parity_helpers.table_for = orig


def test_g0_table_refuses_bad_arguments():
    pkg = _pkg()
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.g0_table_from_sigma(2, 2, 1.0, 0.0, 2.0, 0, 4, 64)
    assert ei.value.code == -1
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.g0_table_from_sigma(2, 2, 1.0, 0.0, 2.0, 64, 65, 64)
    assert ei.value.code == -1
