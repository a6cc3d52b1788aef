"""ctaux_g0_table_noalloc (include/ctaux.h): the DCA bare-propagator table for callers that cannot allocate device memory.
Same kernels as ctaux_g0_table, scratch in a static 8 MiB device array inside the library.  Checked against the existing
path (caller workspace) on two calls in a row -- the second smaller and without a self-energy, so that anything it picked
up from what the first call left in the shared array would show -- at the tolerance of tests/test_gpu_dca_g0.py (1e-12
absolute on entries of magnitude <= 1; the two paths run the same arithmetic, so they are expected to agree bit for bit),
then a third call at the first size again.  Collected last on purpose: the suite runs with pytest -x."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _sigma(Lx, Ly, beta, n_omega):
    Nc = Lx * Ly
    wn = (2 * np.arange(n_omega) + 1) * math.pi / beta
    kx = 2 * math.pi * (np.arange(Nc) % Lx) / Lx
    ky = 2 * math.pi * (np.arange(Nc) // Lx) / Ly
    amp = 1.0 + 0.3 * (np.cos(kx) + np.cos(ky))
    return 0.4 * amp[:, None] + (amp[:, None] ** 2) / (1j * wn[None, :] + 0.2)


def test_g0_table_noalloc_matches_the_workspace_path_on_consecutive_calls():
    import paper_1901_01047_b200 as pkg
    big = dict(Lx=4, Ly=4, t=1.0, mu=-0.054654, beta=10.0, n_omega=1024, n_quad=6, n_tau=512)
    small = dict(Lx=3, Ly=2, t=1.0, mu=-0.3, beta=5.0, n_omega=300, n_quad=5, n_tau=37)
    sig_big = _sigma(4, 4, 10.0, 1024)
    ref_big = pkg.g0_table_from_sigma(sigma_c=sig_big, **big)            # existing path: caller workspace
    ref_small = pkg.g0_table_from_sigma(sigma_c=None, **small)
    got_big = pkg.g0_table_from_sigma_noalloc(sigma_c=sig_big, **big)    # call 1
    got_small = pkg.g0_table_from_sigma_noalloc(sigma_c=None, **small)   # call 2, straight after, on the same array
    got_big2 = pkg.g0_table_from_sigma_noalloc(sigma_c=sig_big, **big)   # call 3
    assert got_big.shape == ref_big.shape and got_small.shape == ref_small.shape
    assert np.isfinite(got_big).all() and np.abs(ref_big).max() > 0.1
    assert np.abs(got_big - ref_big).max() < TOL
    assert np.abs(got_small - ref_small).max() < TOL
    assert np.array_equal(got_big2, got_big)      # does not depend on what earlier calls left in the array


def test_g0_table_noalloc_rejects_sizes_beyond_the_static_array():
    import paper_1901_01047_b200 as pkg
    L = pkg.binding.load_library()
    assert L.ctaux_g0_workspace_bytes(6, 6, 2048, 4096) <= pkg.binding.G0_NOALLOC_MAX_BYTES      # the stated example fits
    assert L.ctaux_g0_workspace_bytes(6, 6, 8192, 4096) > pkg.binding.G0_NOALLOC_MAX_BYTES
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.g0_table_from_sigma_noalloc(6, 6, 1.0, 0.0, 20.0, 8192, 2, 4096)
    assert ei.value.code == -2 and "static array holds 8388608" in str(ei.value)
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.g0_table_from_sigma_noalloc(0, 6, 1.0, 0.0, 20.0, 64, 2, 64)
    assert ei.value.code == -1
    # still usable after the refusals
    a = pkg.g0_table_from_sigma_noalloc(2, 2, 1.0, 0.0, 2.0, 256, 1, 64)
    b = pkg.g0_table_from_sigma(2, 2, 1.0, 0.0, 2.0, 256, 1, 64)
    assert np.abs(a - b).max() < TOL
