"""ORACLE (test infrastructure, fp64) -- what the two ways of sampling the scattering angle must produce.

Part of `oracle/`: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it
never imports the CUDA library and shares no code with it.

The paper samples the scattering angle by acceptance-rejection on the exact Mie function (step (4),
PAPER.md:180; Eq. 13-15); the build samples the canonical inverse-CDF table D_K
(SURVEY.md 8(c) step 2).  SURVEY.md 8(f) row f2 asks for the rejection sampler on the device "to report
the table error".  Both samplers draw cos(theta) and histogram it over n_bins equal bins of [-1, 1]; this
file holds the two EXPECTED histograms, as definitions:

* exact_bin_probabilities: p_j = int_bin I(mu) dmu / int_{-1}^{1} I(mu) dmu, I = |S1|^2 + |S2|^2
  (Eq. 13-14), by Gauss-Legendre quadrature inside every bin (I is a polynomial in mu of degree
  2 n_max: 64 nodes per bin integrate it exactly for the size parameters of the configs);
* table_bin_probabilities: D_K puts probability 1/K uniformly on each interval [M_k, M_{k+1}]
  (cos(theta) = M_k + (M_{k+1} - M_k) frac, frac uniform), so p_j = sum_k |[M_k, M_{k+1}] n bin_j| /
  (K (M_{k+1} - M_k)); an interval of zero width is a point mass in the bin that holds M_k;
* acceptance_rate of the rejection sampler with mu uniform on [-1, 1] and bound I_max:
  int I dmu / (2 I_max);
* total_variation between two histograms / probability vectors: the "table error" in one number.
"""
from __future__ import annotations

import numpy as np
from numpy.polynomial import legendre as npleg

from . import mie


def exact_bin_probabilities(x: float, m: complex, n_bins: int, n_nodes: int = 64) -> np.ndarray:
    a, b = mie.coefficients(x, m)
    t, w = npleg.leggauss(n_nodes)
    edges = np.linspace(-1.0, 1.0, n_bins + 1)
    p = np.empty(n_bins)
    for j in range(n_bins):
        lo, hi = edges[j], edges[j + 1]
        mu = 0.5 * (lo + hi) + 0.5 * (hi - lo) * t
        p[j] = 0.5 * (hi - lo) * np.sum(w * mie.intensity(a, b, mu))
    return p / np.sum(p)


def table_bin_probabilities(M: np.ndarray, n_bins: int) -> np.ndarray:
    M = np.asarray(M, dtype=np.float64)
    K = len(M) - 1
    edges = np.linspace(-1.0, 1.0, n_bins + 1)
    p = np.zeros(n_bins)
    for k in range(K):
        lo, hi = M[k], M[k + 1]
        if hi > lo:
            j0 = min(int(np.floor((lo + 1.0) * n_bins / 2.0)), n_bins - 1)
            j1 = min(int(np.floor((hi + 1.0) * n_bins / 2.0)), n_bins - 1)
            for j in range(j0, j1 + 1):
                ov = min(hi, edges[j + 1]) - max(lo, edges[j])
                if ov > 0.0:
                    p[j] += ov / ((hi - lo) * K)
        else:
            p[min(int(np.floor((lo + 1.0) * n_bins / 2.0)), n_bins - 1)] += 1.0 / K
    return p


def intensity_integral_and_max(x: float, m: complex, n_grid: int = 200001):
    """(int_{-1}^{1} I dmu, max I) -- the maximum over a fine uniform grid in theta (both ends included)."""
    a, b = mie.coefficients(x, m)
    t, w = npleg.leggauss(256)
    total = float(np.sum(w * mie.intensity(a, b, t)))
    mu = np.cos(np.linspace(0.0, np.pi, n_grid))
    return total, float(np.max(mie.intensity(a, b, mu)))


def acceptance_rate(x: float, m: complex, i_max: float) -> float:
    total, _ = intensity_integral_and_max(x, m)
    return total / (2.0 * i_max)


def total_variation(p, q) -> float:
    p = np.asarray(p, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    return 0.5 * float(np.sum(np.abs(p / p.sum() - q / q.sum())))
