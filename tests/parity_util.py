"""Statistics used by the parity tests."""
from __future__ import annotations

import math

import numpy as np
from scipy import stats


def channel_z(k1, n1, k2, n2, min_pooled=25):
    """Two-sample binomial z per channel with pooled p; channels whose pooled count is < min_pooled are merged
    into one 'rest' bin (G19).  Returns (z array, chi2, ndf)."""
    k1 = np.asarray(k1, np.float64)
    k2 = np.asarray(k2, np.float64)
    small = (k1 + k2) < min_pooled
    if small.any():
        k1 = np.concatenate([k1[~small], [k1[small].sum()]])
        k2 = np.concatenate([k2[~small], [k2[small].sum()]])
    p = (k1 + k2) / (n1 + n2)
    var = p * (1 - p) * (1 / n1 + 1 / n2)
    ok = var > 0
    z = np.zeros_like(p)
    z[ok] = (k1[ok] / n1 - k2[ok] / n2) / np.sqrt(var[ok])
    return z, float((z ** 2).sum()), int(ok.sum())


def assert_time_hist_agrees(k1, n1, k2, n2, label=""):
    """Bin-by-bin 4 sigma for an arrival-time histogram.  Its tail bins hold a handful of photons and the two runs differ in size
    (up to 20 : 1), so the merging rule of G19 is written for what the normal approximation needs: a bin is kept on its own only if
    the SMALLER run expects at least 10 photons in it (pooled count x min(n1, n2) / (n1 + n2) >= 10); the others form one bin."""
    need = int(math.ceil(10.0 * (n1 + n2) / min(n1, n2)))
    return assert_channels_agree(k1, n1, k2, n2, label, min_pooled=max(25, need))


def assert_channels_agree(k1, n1, k2, n2, label="", min_pooled=25):
    z, chi2, ndf = channel_z(k1, n1, k2, n2, min_pooled)
    worst = float(np.abs(z).max()) if z.size else 0.0
    # all |z| <= 4 (BASELINE.json "within 4 sigma binomial"); chi2 sanity: within 5 sigma of ndf
    assert worst <= 4.0, f"{label}: max |z| = {worst:.2f} over {z.size} channels (chi2/ndf = {chi2:.1f}/{ndf})"
    if ndf > 10:
        assert chi2 < ndf + 5 * math.sqrt(2 * ndf), f"{label}: chi2/ndf = {chi2:.1f}/{ndf}"
    return worst, chi2, ndf


def assert_fraction_agrees(k1, n1, k2, n2, abs_tol, label=""):
    """|k1/n1 - k2/n2| <= abs_tol (+ nothing): used for 'total LCE within 0.2% absolute'."""
    d = abs(k1 / n1 - k2 / n2)
    assert d <= abs_tol, f"{label}: {k1 / n1:.5f} vs {k2 / n2:.5f} differ by {d:.5f} > {abs_tol}"
    return d


def assert_binomial_agrees(k1, n1, k2, n2, nsigma=4.0, label=""):
    p = (k1 + k2) / (n1 + n2)
    s = math.sqrt(max(p * (1 - p), 1e-300) * (1 / n1 + 1 / n2))
    d = abs(k1 / n1 - k2 / n2)
    assert d <= nsigma * s + 1e-12, f"{label}: {k1 / n1:.6f} vs {k2 / n2:.6f}: {d / s:.2f} sigma"


def ks_pvalue(a, b):
    """Two-sample Kolmogorov-Smirnov, asymptotic series with effective n = n1 n2 / (n1 + n2)."""
    return float(stats.ks_2samp(a, b, method="asymp").pvalue)


def fates(fate_count, names):
    return {n: int(fate_count[i]) for i, n in enumerate(names)}
