"""ORACLE (test infrastructure, fp64) -- characteristics of the main peak of a PDV spectrum.

Part of `oracle/`: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it
never imports the CUDA library and shares no code with it.

The paper reads three numbers off a simulated spectrum I(x), x = v~/v_fs (section III.B, Eq. 35,
PAPER.md:356-365; compared with the MC spectra in Figs. 13-15):

    position of the main peak      x_peak                     (Eq. 31:  1 + ln(tau0)/beta)
    value at the peak              I(x_peak)                  (Eq. 32:  proportional to beta / (d2bar/dbar))
    relative curvature at the peak I''(x_peak) / I(x_peak)    (Eq. 34:  -beta^2)

The paper does not say how it reads them off a noisy MC histogram; readings R27-R30 fix it:

  R27  the spectrum is the density of detected weight per unit x:  S[k] = hist[k] / (N dx),
       dx = (v_hi - v_lo) / (n_bins v_fs);  bin centre x_k = (v_lo + (k + 1/2) dv) / v_fs.
  R28  the peak bin k* is the arg-max (first one on ties) of the spectrum smoothed by `n_pass` passes
       of a centred moving average of half-width `half` bins (the mean over the bins that exist, at
       the ends of the array), searched over the bins with x_min <= x_k <= x_max -- x_min > 1 keeps
       the free-surface peak of thin clouds out of it.
  R29  an unweighted least-squares parabola a + b u + c u^2, u = x - x_{k*}, through the UNSMOOTHED
       S[k] of the bins |k - k*| <= fit_half (those that exist) gives
           x_peak = x_{k*} - b / (2c),   I_peak = a - b^2 / (4c),   curvature = 2c / I_peak.
  R30  status 0 ok; 1 no bin in the search range or fewer than 3 bins in the fit window;
       2 the parabola has no maximum (c >= 0) -- then x_peak = x_{k*}, I_peak = smoothed S[k*], curvature = 0.

Everything is written out with plain loops / numpy primitives in the order of R27-R29.
"""
from __future__ import annotations

import numpy as np


def moving_average(s: np.ndarray, half: int) -> np.ndarray:
    """One pass of R28's centred moving average: out[k] = mean of s[max(0,k-half) .. min(n-1,k+half)]."""
    s = [float(v) for v in np.asarray(s, dtype=np.float64)]
    n = len(s)
    out = np.empty(n)
    for k in range(n):
        lo, hi = max(0, k - half), min(n - 1, k + half)
        acc = 0.0
        for j in range(lo, hi + 1):                    # in index order: the arg-max of R28 must not depend on a summation trick
            acc += s[j]
        out[k] = acc / (hi - lo + 1)
    return out


def spectrum_peak(hist, n_photons: int, v_lo: float, v_hi: float, v_fs: float, *, half: int = 4, n_pass: int = 2,
                  fit_half: int = 8, x_min: float = 1.02, x_max: float = 1e30) -> dict:
    """R27-R30 for one histogram row.  Returns x_peak, i_peak, curvature, k_peak, status."""
    h = np.asarray(hist, dtype=np.float64)
    n = len(h)
    dv = (v_hi - v_lo) / n
    dx = dv / v_fs
    x = (v_lo + (np.arange(n) + 0.5) * dv) / v_fs                        # R27
    s = h / (float(n_photons) * dx) if n_photons > 0 else np.zeros(n)
    sm = s.copy()
    for _ in range(n_pass):                                              # R28
        sm = moving_average(sm, half)
    k_star, best = -1, -np.inf
    for k in range(n):
        if x_min <= x[k] <= x_max and sm[k] > best:
            k_star, best = k, sm[k]
    if k_star < 0:
        return dict(x_peak=0.0, i_peak=0.0, curvature=0.0, k_peak=-1, status=1, beta_eq35=0.0, tau0_eq35=0.0)
    lo, hi = max(0, k_star - fit_half), min(n - 1, k_star + fit_half)
    if hi - lo + 1 < 3:
        return dict(x_peak=float(x[k_star]), i_peak=float(sm[k_star]), curvature=0.0, k_peak=k_star, status=1, beta_eq35=0.0,
                    tau0_eq35=0.0)
    u = x[lo:hi + 1] - x[k_star]                                         # R29
    design = np.stack([np.ones_like(u), u, u * u], axis=1)
    (a, b, c), *_ = np.linalg.lstsq(design, s[lo:hi + 1], rcond=None)
    if not c < 0.0:
        return dict(x_peak=float(x[k_star]), i_peak=float(sm[k_star]), curvature=0.0, k_peak=k_star, status=2, beta_eq35=0.0,
                    tau0_eq35=0.0)
    i_peak = a - b * b / (4.0 * c)
    x_peak, curv = float(x[k_star] - b / (2.0 * c)), float(2.0 * c / i_peak)
    beta, tau0 = ejecta_from_peak(x_peak, curv)
    return dict(x_peak=x_peak, i_peak=float(i_peak), curvature=curv, k_peak=k_star, status=0, beta_eq35=beta, tau0_eq35=tau0)


def spectrum_peaks(hist, n_photons: int, v_lo: float, v_hi: float, v_fs, **kw) -> list:
    """Rows of a [n_units][n_bins] histogram stack; v_fs a scalar or one value per row."""
    hist = np.atleast_2d(np.asarray(hist, dtype=np.float64))
    v = np.broadcast_to(np.asarray(v_fs, dtype=np.float64), (hist.shape[0],))
    return [spectrum_peak(hist[i], n_photons, v_lo, v_hi, float(v[i]), **kw) for i in range(hist.shape[0])]


def ejecta_from_peak(x_peak: float, curvature: float):
    """Eq. 35 read backwards (section III.C): the relative curvature at the peak gives the velocity
    profile coefficient, beta = sqrt(-I''/I); the peak position then gives the optical thickness, tau0 = exp(beta (x_peak - 1)).
    (For a weight tally, R31, that tau0 is 2 g tau_ext.)  Returns (beta, tau0); (0, 0) if the curvature is not negative."""
    if not curvature < 0.0:
        return 0.0, 0.0
    beta = (-curvature) ** 0.5
    with np.errstate(over="ignore"):                      # a noise spectrum can give any exponent: inf is the honest answer
        return beta, float(np.exp(beta * (x_peak - 1.0)))

