"""Statistical comparison of two weighted histograms -- test helper (no method arithmetic).

north_star tolerance: |a_k - b_k| <= 5 sqrt(var_a,k + var_b,k) per bin, after scaling both to the same
photon count.  var of a weighted tally = sum of squared weights (hist2).  Reading R23:
the Gaussian rule needs enough counts, so adjacent bins are merged until the merged bin holds an
effective count (sum w)^2 / sum w^2 >= min_eff on BOTH sides; a trailing remainder is merged into
the last group.
"""
from __future__ import annotations

import json
import os
from types import SimpleNamespace

import numpy as np


def load_golden(name: str) -> SimpleNamespace:
    """Stored oracle tallies tests/golden/oracle_hist_<name>.json (written by tests/golden/make_oracle_hists.py, which calls only
    oracle/): an object with .hist, .hist2, .stats, .n_photons like an oracle run of >= 1e8 histories."""
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"oracle_hist_{name}.json")) as f:
        d = json.load(f)
    return SimpleNamespace(hist=np.asarray(d["hist"], dtype=np.float64), hist2=np.asarray(d["hist2"], dtype=np.float64),
                           stats=d["stats"], n_photons=int(d["n_photons"]), run=d["run"], tau_ext=d["tau_ext"],
                           chunk=int(d.get("chunk", 0)), chunk_stats=d.get("chunk_stats", []))


def per_history_variance(o, key: str, min_chunks: int = 8):
    """Batch-means estimate of the variance of ONE history's contribution to the statistic `key`, from the per-chunk statistics a
    stored oracle run carries (equal chunks of o.chunk histories): chunk * var(chunk means).  None when the run has fewer than
    `min_chunks` equal chunks.  With m chunks the estimate is a scaled chi-square of m - 1 degrees of freedom (relative
    standard error sqrt(2 / (m - 1)): 0.53 at 8 chunks, 0.32 at 20)."""
    cs = o.chunk_stats
    if not cs or len(cs) < min_chunks or o.chunk * len(cs) != o.n_photons:
        return None
    means = np.array([float(c[key]) for c in cs], dtype=np.float64) / o.chunk
    return float(means.var(ddof=1) * o.chunk)


def merge_groups(h_a, h2_a, h_b, h2_b, min_eff=25.0):
    """Greedy left-to-right grouping of bins; returns list of (lo, hi) half-open index ranges."""
    n = len(h_a)
    groups, lo = [], 0
    sa = s2a = sb = s2b = 0.0
    for k in range(n):
        sa += h_a[k]; s2a += h2_a[k]; sb += h_b[k]; s2b += h2_b[k]
        ok_a = s2a > 0 and sa * sa / s2a >= min_eff
        ok_b = s2b > 0 and sb * sb / s2b >= min_eff
        if ok_a and ok_b:
            groups.append((lo, k + 1))
            lo = k + 1
            sa = s2a = sb = s2b = 0.0
    if lo < n:
        if groups:
            groups[-1] = (groups[-1][0], n)
        else:
            groups.append((0, n))
    return groups


def compare(h_a, h2_a, n_a, h_b, h2_b, n_b, min_eff=25.0):
    """Returns dict(z=array of normalised deviations per merged group, groups=..., worst=max|z|).

    Both histograms are converted to per-photon rates; z = (a/n_a - b/n_b) / sqrt(var_a/n_a^2 + var_b/n_b^2).
    """
    h_a, h2_a, h_b, h2_b = (np.asarray(x, dtype=np.float64) for x in (h_a, h2_a, h_b, h2_b))
    groups = merge_groups(h_a, h2_a, h_b, h2_b, min_eff)
    z = []
    for lo, hi in groups:
        a, va = h_a[lo:hi].sum(), h2_a[lo:hi].sum()
        b, vb = h_b[lo:hi].sum(), h2_b[lo:hi].sum()
        den = np.sqrt(va / n_a**2 + vb / n_b**2)
        z.append(0.0 if den == 0 else (a / n_a - b / n_b) / den)
    z = np.asarray(z)
    return dict(z=z, groups=groups, worst=float(np.max(np.abs(z))) if z.size else 0.0,
                chi2=float(np.sum(z * z)), ndf=int(z.size))


def compare_to_expectation(h, h2, n, expected_rate, min_eff=25.0):
    """Compare a tallied histogram with an exact expected per-photon rate per bin (no variance on that side)."""
    h, h2, e = (np.asarray(x, dtype=np.float64) for x in (h, h2, expected_rate))
    big = np.full_like(h, 1e100)
    groups = merge_groups(h, h2, big, big, min_eff)          # only the tallied side limits the merge
    z = []
    for lo, hi in groups:
        a, va = h[lo:hi].sum(), h2[lo:hi].sum()
        # variance of a sum of n iid contributions: n (E w^2 - (E w)^2)  ~  sum w^2 - (sum w)^2 / n
        var = max(va - a * a / n, 1e-300)
        z.append((a - n * e[lo:hi].sum()) / np.sqrt(var))
    z = np.asarray(z)
    return dict(z=z, groups=groups, worst=float(np.max(np.abs(z))) if z.size else 0.0,
                chi2=float(np.sum(z * z)), ndf=int(z.size))
