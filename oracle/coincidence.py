"""TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py).

The paper's way of reading the output of two series: the
time-randomised control, simultaneous hits in two series, pseudo-spectra.  Plain numpy and
Python loops; shares nothing with the CUDA path.

Passages: PAPER.md:68 ("control, produced by the same analysis following time-randomisation of
the H1 and L1 data. (Time-randomisation produces data with maximal entropy, keeping histograms
the same.)"); Fig. 6 ("Pseudo-spectra of simultaneous rho > kappa sigma in H1 and
L1 ... by independent counts and by simultaneous counts with frequency pairs within
Delta f = 50 Hz").  The paper gives no formulas; readings T1-T3 of DESIGN.md:

T1  control series: x'[i] = x[perm[i]] for a permutation perm of 0..n-1 that is an INPUT (drawn by
    the seeded generator workloads.permutation; the method itself draws no random numbers).
T2  simultaneous counts: with two count maps M1, M2 of the same geometry [n_tbins][n_fbins] (one
    count per hit; time bin x frequency bin) and w = the half width in frequency bins,
        C1[t][f] = M1[t][f]  if M2[t][f'] > 0 for some |f' - f| <= w, else 0      (C2 likewise):
    the hits of one series that have a partner in the other series in the same time bin with
    a frequency within w bins (Delta f = 50 Hz at 1-Hz bins: w = 50).
T3  pseudo-spectrum: S[f] = sum_t M[t][f], the time marginal of a count map.
"""
from __future__ import annotations

import numpy as np


def time_randomize(x, perm):
    """T1.  perm must be a permutation of range(len(x))."""
    x = np.asarray(x)
    perm = np.asarray(perm)
    if perm.shape != x.shape or not np.array_equal(np.sort(perm), np.arange(len(x))):
        raise ValueError("perm is not a permutation of the sample indices")
    out = np.empty_like(x)
    for i in range(len(x)):
        out[i] = x[perm[i]]
    return out


def coincidence(m1, m2, half_width_bins):
    """T2.  Returns (C1, C2), uint32 arrays of the maps' shape."""
    m1 = np.asarray(m1, np.uint32)
    m2 = np.asarray(m2, np.uint32)
    if m1.shape != m2.shape or m1.ndim != 2 or half_width_bins < 0:
        raise ValueError("maps must be 2-D, of equal shape, and the half width >= 0")
    nt, nf = m1.shape
    c1 = np.zeros_like(m1)
    c2 = np.zeros_like(m2)
    for t in range(nt):
        for f in range(nf):
            lo, hi = max(f - half_width_bins, 0), min(f + half_width_bins, nf - 1)
            if m1[t, f] and m2[t, lo:hi + 1].any():
                c1[t, f] = m1[t, f]
            if m2[t, f] and m1[t, lo:hi + 1].any():
                c2[t, f] = m2[t, f]
    return c1, c2


def pseudo_spectrum(m):
    """T3.  uint64[n_fbins]."""
    m = np.asarray(m, np.uint32)
    out = np.zeros(m.shape[1], np.uint64)
    for t in range(m.shape[0]):
        out += m[t].astype(np.uint64)
    return out
