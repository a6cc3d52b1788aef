"""Pins of the DCA bare-propagator oracle (oracle/dca_g0.py).  No CUDA path involved."""
import math

import numpy as np
import pytest

from ctaux_workloads import g0_table, get_config
from oracle.dca_g0 import cluster_exclusion, coarse_grain, g0_table_from_sigma


@pytest.mark.parametrize("Lx,Ly,beta,mu", [(2, 2, 2.0, 0.0), (4, 4, 10.0, -0.054654), (3, 2, 5.0, -0.3)])
def test_patch_centre_quadrature_reproduces_the_isolated_cluster_table(Lx, Ly, beta, mu):
    """n_quad = 1 puts the whole patch weight on its centre K: Gbar(K) = G0(K) (Eq. (8)), the cluster is isolated, and the
    table must be the closed form  G0(r,tau) = -(1/Nc) sum_K cos(K.r) e^{-xi tau}/(1 + e^{-beta xi})  of ctaux_workloads
    (BASELINE.json).  Pins the K -> r phases (3x2: x and y not interchangeable), the Matsubara sum with its analytic tail,
    the one-sided end points 0+ / beta-, and the sign convention of the table."""
    M, n_omega = 64, 4096
    T = g0_table_from_sigma(Lx, Ly, 1.0, mu, beta, n_omega, 1, M)
    want = g0_table(Lx, Ly, beta, mu, M)
    assert np.abs(T - want).max() < 5e-9


def test_cluster_exclusion_removes_a_static_self_energy():
    """Eq. (9): for a static, K-independent Sigma_c = s and the isolated cluster (n_quad = 1), Gbar = [iw - eps + mu - s]^-1
    and G0c = [Gbar^-1 + s]^-1 = [iw - eps + mu]^-1: the table does not depend on s.  A wrong sign in Eq. (9) doubles the shift."""
    Lx = Ly = 2
    beta, mu, M, n_omega = 4.0, -0.2, 32, 2048
    sig = np.full((4, n_omega), 0.7 + 0.0j)
    a = g0_table_from_sigma(Lx, Ly, 1.0, mu, beta, n_omega, 1, M, sigma_c=sig)
    b = g0_table_from_sigma(Lx, Ly, 1.0, mu, beta, n_omega, 1, M)
    assert np.abs(a - b).max() < 1e-12
    # with a real patch integral the static shift does NOT drop out of Gbar, but Eq. (9) still returns a propagator whose
    # inverse differs from Gbar^-1 by exactly Sigma_c
    Gbar, m1, m2 = coarse_grain(Lx, Ly, 1.0, mu, beta, 64, 8, sigma_c=sig[:, :64])
    G0c = cluster_exclusion(Gbar, sig[:, :64])
    assert np.abs(1 / G0c - 1 / Gbar - 0.7).max() < 1e-12


@pytest.mark.parametrize("n_quad", [1, 4, 16])
def test_anticommutator_sum_rule_and_symmetries(n_quad):
    """G0c(r, 0+) + G0c(r, beta-) = -delta_{r,0} for any patch quadrature and any Sigma_c (the 1/(iw) tail carries the
    whole jump); the table is real and inversion symmetric in r."""
    Lx = Ly = 4
    beta, mu, M, n_omega = 5.0, -0.1, 48, 512
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    sig = np.tile((0.3 - 0.5j / (1 + wn))[None, :], (16, 1))           # some causal-looking self-energy
    T = g0_table_from_sigma(Lx, Ly, 1.0, mu, beta, n_omega, n_quad, M, sigma_c=sig)
    s = T[:, 0] + T[:, -1]
    want = np.zeros(16)
    want[0] = -1.0
    assert np.abs(s - want).max() < 1e-12
    for d in range(16):
        rx, ry = d % 4, d // 4
        assert abs(T[d] - T[(-rx) % 4 + 4 * ((-ry) % 4)]).max() < 1e-12
        assert abs(T[d] - T[ry + 4 * rx]).max() < 1e-12               # square cluster, isotropic hopping: x <-> y
    assert np.all(T[0] < 0)                                              # standard sign: G0(r=0, tau) < 0 on (0, beta)


def test_patches_tile_the_brillouin_zone():
    """Eq. (1)-(2): the Nc patches partition the BZ.  With matching meshes the patch average over ALL K of the 2x2 cluster
    (8x8 points per patch) visits exactly the k points of the single patch of the 1x1 cluster (16x16 points), so
    (1/Nc) sum_K Gbar(K, iw_n) is the same local lattice Green's function -- to rounding."""
    beta, mu, n_omega = 3.0, -0.4, 32
    G1, _, _ = coarse_grain(1, 1, 1.0, mu, beta, n_omega, 16)
    G4, _, _ = coarse_grain(2, 2, 1.0, mu, beta, n_omega, 8)
    assert np.abs(G4.mean(axis=0) - G1[0]).max() < 1e-13
    G16, _, _ = coarse_grain(4, 4, 1.0, mu, beta, n_omega, 4)
    assert np.abs(G16.mean(axis=0) - G1[0]).max() < 1e-13
    # high-frequency moments of the local function: G ~ 1/iw + (<eps> - mu)/(iw)^2 with <eps> = 0 on the full zone
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    assert abs(((1j * wn[-1]) ** 2 * (G1[0, -1] - 1 / (1j * wn[-1]))).real - (-mu)) < 0.05


def test_embedding_differs_from_the_isolated_cluster_and_converges_in_n_quad():
    """The coarse-grained propagator is NOT the isolated-cluster one, and the midpoint rule converges."""
    cfg = get_config(2)
    a = g0_table_from_sigma(4, 4, 1.0, cfg["mu"], cfg["beta"], 1024, 1, 64)
    b = g0_table_from_sigma(4, 4, 1.0, cfg["mu"], cfg["beta"], 1024, 8, 64)
    c = g0_table_from_sigma(4, 4, 1.0, cfg["mu"], cfg["beta"], 1024, 16, 64)
    assert np.abs(a - b).max() > 1e-2
    assert np.abs(b - c).max() < 2e-3
