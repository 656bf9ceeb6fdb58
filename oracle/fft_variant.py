"""Float64 FFT restatement of the correlation (TEST INFRASTRUCTURE).

The paper's own method is FFT-based correlation (forward FFT,
multiply, complex inverse FFT of N = 2^16).  This module states it with numpy.fft in
float64, zero-padded so that no lag wraps (reading C5: valid lags only).  It is used
for pin P4 (direct and FFT correlation agree on tiny inputs) and, once qualified by
P4, as the second reported CPU baseline in bench.py.  It calls oracle.template /
template_norms for the template (the definition C1, C2) and numpy.fft as the library
primitive; it shares nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from . import template, template_norms


def rho_series_fft(x, fs, L, f0, f1):
    """rho(tau) for all valid lags 0..N-L via zero-padded real FFTs (float64)."""
    x = np.asarray(x, dtype=np.float64)
    N = len(x)
    n_lags = N - L + 1
    nfft = 1
    while nfft < N + L:
        nfft *= 2
    hc, hs = template(fs, L, f0, f1)
    nc, ns = template_norms(hc, hs)
    X = np.fft.rfft(x, nfft)
    # correlation: sum_k x[tau+k] h[k]  <->  X * conj(H)
    c = np.fft.irfft(X * np.conj(np.fft.rfft(hc, nfft)), nfft)[:n_lags]
    s = np.fft.irfft(X * np.conj(np.fft.rfft(hs, nfft)), nfft)[:n_lags]
    c = c / nc if nc > 0 else np.zeros(n_lags)
    s = s / ns if ns > 0 else np.zeros(n_lags)
    # sliding squared norm by prefix sums of x^2 (float64)
    cs = np.concatenate(([0.0], np.cumsum(x * x)))
    n2 = cs[L:L + n_lags] - cs[:n_lags]
    rho = np.zeros(n_lags)
    ok = n2 > 0
    rho[ok] = np.sqrt(c[ok] ** 2 + s[ok] ** 2) / np.sqrt(n2[ok])
    return rho


def correlate_fft(x, fs, L, f0, f1):
    """(rho_max, arg_lag) per template with the FFT variant; smallest lag on ties."""
    rho_max = np.empty(len(f0), np.float64)
    arg = np.empty(len(f0), np.int32)
    for j in range(len(f0)):
        r = rho_series_fft(x, fs, L, f0[j], f1[j])
        a = int(np.argmax(r))          # numpy returns the first maximum
        rho_max[j], arg[j] = r[a], a
    return rho_max, arg
