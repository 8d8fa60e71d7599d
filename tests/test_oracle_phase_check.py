"""Pins for oracle/phase_check.py (rejection sampler vs table) -- CPU only.

Expected values: the Rayleigh phase function 3/8 (1 + mu^2) in closed form, the asymmetry parameter g of the Mie series
(Eq. 12, pinned separately in test_oracle_mie.py against scipy), hand-made tables, and the definition of a quantile table.
"""
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud, mie, phase_check

M_SN = complex(W.M_RE, W.M_IM)
X5 = math.pi * 5e-6 / W.WAVELENGTH


def test_rayleigh_limit_closed_form():
    """x -> 0: I proportional to 1 + mu^2, so p_j = 3/8 [mu + mu^3/3] over the bin; acceptance 2/3 with I_max = I(+-1)."""
    n = 40
    p = phase_check.exact_bin_probabilities(0.01, complex(1.5, 0.0), n)
    e = np.linspace(-1, 1, n + 1)
    F = 0.375 * (e + e ** 3 / 3.0)
    assert np.allclose(p, np.diff(F), rtol=0, atol=2e-6)                 # O(x^2) corrections to Rayleigh
    total, imax = phase_check.intensity_integral_and_max(0.01, complex(1.5, 0.0))
    assert total / (2 * imax) == pytest.approx(2.0 / 3.0, rel=1e-4)
    assert phase_check.acceptance_rate(0.01, complex(1.5, 0.0), imax) == pytest.approx(2.0 / 3.0, rel=1e-4)


@pytest.mark.parametrize("x", [X5, math.pi * 1e-6 / W.WAVELENGTH])
def test_first_moment_of_exact_bins_is_g(x):
    n = 4000
    p = phase_check.exact_bin_probabilities(x, M_SN, n, n_nodes=16)
    centres = -1.0 + (np.arange(n) + 0.5) * 2.0 / n
    g = mie.efficiencies(x, M_SN)[3]
    assert p.sum() == pytest.approx(1.0, abs=1e-12) and np.all(p > 0)
    assert float(np.sum(p * centres)) == pytest.approx(g, abs=2e-6)      # centre rule: error O(bin^2)


def test_table_bin_probabilities_on_hand_made_tables():
    assert np.allclose(phase_check.table_bin_probabilities(np.linspace(-1, 1, 1025), 64), 1.0 / 64)      # isotropic D_K
    assert np.allclose(phase_check.table_bin_probabilities(np.array([-1.0, 0.0, 1.0]), 4), 0.25)
    p = phase_check.table_bin_probabilities(np.array([-1.0, -1.0, 1.0]), 4)                             # point mass at -1
    assert np.allclose(p, [0.5 + 0.125, 0.125, 0.125, 0.125])
    p = phase_check.table_bin_probabilities(np.array([-1.0, 0.5, 0.5, 0.75, 1.0]), 8)                   # mass at an edge
    assert p.sum() == pytest.approx(1.0) and p[6] == pytest.approx(0.25 + 0.25)                         # bin [0.5, 0.75)
    assert p[7] == pytest.approx(0.25) and np.allclose(p[:6], 0.25 / 6)


def test_table_error_of_the_config_cloud_is_small_and_shrinks_with_K():
    """Inside a table cell D_K is uniform in mu while the true density varies: the total variation over 64 bins is tiny and
    falls as K grows -- this number is what the device-side rejection sampler is there to confirm."""
    exact = phase_check.exact_bin_probabilities(X5, M_SN, 64)
    tv = [phase_check.total_variation(phase_check.table_bin_probabilities(cloud.phase_quantile_table(X5, M_SN, K), 64), exact)
          for K in (64, 1024)]
    assert tv[1] < 2e-4 and tv[1] < 0.2 * tv[0]
    assert phase_check.total_variation([1, 1, 2], [1, 1, 2]) == 0.0
    assert phase_check.total_variation([1, 0], [0, 1]) == 1.0
