"""Acceptance rules R1-R3 of DESIGN.md ("Acceptance rules"; BASELINE.json north_star:
|d rho| <= 2e-4; argmax exact where the top two values differ by more than 1e-3; map exact
except for templates within 2e-4 of kappa), as helpers for the GPU parity tests.

The expected values come from oracle/ only; the CUDA results are passed in as numpy arrays.
"""
from __future__ import annotations

import numpy as np

import oracle

RHO_TOL = 2e-4       # R1
GAP_STRICT = 1e-3    # R2a
NEAR_MAX = 4e-4      # R2b
KAPPA_BAND = 2e-4    # R3


def check_values_and_argmax(x, fs, L, f0, f1, rho_gpu, arg_gpu, lag_begin=0, lag_end=None,
                            oracle_result=None, f2=None, family="poly"):
    """R1, R2a, R2b for every template.  Returns (rho_oracle, arg_oracle, exempt) where
    exempt[j] is True when template j's argmax is not unique to within GAP_STRICT."""
    f0 = np.asarray(f0, np.float64)
    f1 = np.asarray(f1, np.float64)
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    if oracle_result is None:
        rho_o, arg_o = oracle.correlate(x, fs, L, f0, f1, lag_begin, lag_end, f2=f2, family=family)
    else:
        rho_o, arg_o = oracle_result
    rho_gpu = np.asarray(rho_gpu, np.float64)
    arg_gpu = np.asarray(arg_gpu)
    err = np.abs(rho_gpu - rho_o)
    worst = int(np.argmax(err)) if len(err) else 0
    assert len(err) == 0 or err[worst] <= RHO_TOL, (
        f"R1: |d rho| = {err[worst]:.3e} at template {worst} (f0={f0[worst]}, f1={f1[worst]}): "
        f"gpu {rho_gpu[worst]!r} oracle {rho_o[worst]!r}")
    assert np.all((arg_gpu >= lag_begin) & ((arg_gpu < lag_end) | (lag_end == lag_begin)))
    exempt = np.zeros(len(f0), bool)
    for j in np.nonzero(arg_gpu != arg_o)[0]:
        series = oracle.rho_series(x, fs, L, f0[j], f1[j], lag_begin, lag_end,
                                   f2=0.0 if f2 is None else float(f2[j]), family=family)
        r1 = series[arg_o[j] - lag_begin]
        others = np.delete(series, arg_o[j] - lag_begin)
        r2 = others.max() if len(others) else -np.inf
        # R2a: a mismatch is only allowed when the maximum is not unique to within 1e-3
        assert r1 - r2 <= GAP_STRICT, (
            f"R2a: template {j} argmax gpu {arg_gpu[j]} != oracle {arg_o[j]} with gap {r1 - r2:.3e}")
        # R2b: the lag the GPU reports is a near-maximiser according to the oracle
        at = series[arg_gpu[j] - lag_begin]
        assert at >= r1 - NEAR_MAX, (
            f"R2b: template {j}: oracle rho at the gpu's lag {arg_gpu[j]} is {at!r} < max {r1!r}")
        exempt[j] = True
    return rho_o, arg_o, exempt


def check_map(f0, rho_gpu, arg_gpu, map_gpu, counters_gpu, rho_o, arg_o, exempt, kappa,
              lag_origin, grid):
    """R3: (i) the GPU map is exactly the histogram of the GPU's own outputs; (ii) over the
    unambiguous templates the oracle's and the GPU's maps agree cell by cell; (iii) the L1
    distance of the two full maps is at most twice the number of ambiguous templates."""
    g = grid
    args = (kappa, lag_origin, g["samples_per_tbin"], g["f_lo_hz"], g["df_hz"], g["n_fbins"],
            g["n_tbins"])
    f0 = np.asarray(f0, np.float64)
    # (i): the oracle's map routine applied to the GPU's fp32 outputs (C9: compared in fp32)
    m_self, c_self = oracle.butterfly_map(f0, np.asarray(rho_gpu, np.float32).astype(np.float64),
                                          arg_gpu, *args)
    np.testing.assert_array_equal(np.asarray(map_gpu, np.uint32).reshape(m_self.shape), m_self)
    np.testing.assert_array_equal(np.asarray(counters_gpu, np.uint64), c_self)
    # (ii), (iii)
    k32 = float(np.float32(kappa))
    amb = exempt | (np.abs(rho_o - k32) <= KAPPA_BAND)
    keep = ~amb
    m_o, _ = oracle.butterfly_map(f0[keep], rho_o[keep], arg_o[keep], *args)
    m_g, _ = oracle.butterfly_map(f0[keep], np.asarray(rho_gpu, np.float64)[keep],
                                  np.asarray(arg_gpu)[keep], *args)
    np.testing.assert_array_equal(m_g, m_o)
    m_full, _ = oracle.butterfly_map(f0, rho_o, arg_o, *args)
    l1 = np.abs(m_full.astype(np.int64) - m_self.astype(np.int64)).sum()
    assert l1 <= 2 * int(amb.sum()), f"R3(iii): L1 {l1} > 2 x {int(amb.sum())} ambiguous"
    return int(amb.sum())


SIGMA_RTOL = 1e-3    # R5: relative tolerance on sigma_j


def check_tails(x, fs, L, f0, f1, kappa, sigma_gpu, hit_j, hit_lag, hit_rho, total, lag_begin=0,
                lag_end=None, f2=None, family="poly"):
    """R5: the kappa-sigma tails of the CUDA path against oracle.sigma / the oracle's
    series.  rho_sigma = rho ||x_tau|| / sigma, so north_star's |d rho| <= 2e-4 becomes the
    per-hit tolerance tol = 2e-4 ||x_tau|| / sigma_j + SIGMA_RTOL rho_sigma.  (i) sigma within
    SIGMA_RTOL; (ii) every GPU hit is a hit of the oracle up to tol, with its value within tol;
    (iii) every oracle hit above kappa + tol is in the GPU list; (iv) no duplicates, and the
    total equals the list length when nothing overflowed."""
    f0 = np.asarray(f0, np.float64)
    f1 = np.asarray(f1, np.float64)
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    f2 = np.zeros(len(f0)) if f2 is None else np.asarray(f2, np.float64)
    sig_o = np.array([oracle.sigma(x, fs, L, a, b, c, family=family) for a, b, c in zip(f0, f1, f2)])
    sigma_gpu = np.asarray(sigma_gpu, np.float64)
    ok = sig_o > 0
    assert np.all(sigma_gpu[~ok] == 0.0)
    assert np.abs(sigma_gpu[ok] / sig_o[ok] - 1.0).max(initial=0.0) <= SIGMA_RTOL, \
        f"R5(i): sigma off by {np.abs(sigma_gpu[ok] / sig_o[ok] - 1.0).max():.2e}"
    n2 = oracle.sliding_n2(x, L, lag_begin, lag_end)
    got = {}
    for j, lag, r in zip(np.asarray(hit_j), np.asarray(hit_lag), np.asarray(hit_rho, np.float64)):
        assert (int(j), int(lag)) not in got, "R5(iv): duplicate hit"
        assert lag_begin <= lag < lag_end
        got[(int(j), int(lag))] = r
    assert total >= len(got)
    n_oracle = n_border = 0
    for j in range(len(f0)):
        if not ok[j]:
            continue
        rs = oracle.rho_series(x, fs, L, f0[j], f1[j], lag_begin, lag_end, f2=float(f2[j]),
                               family=family) * np.sqrt(n2) / sig_o[j]
        tol = 2e-4 * np.sqrt(n2) / sig_o[j] + SIGMA_RTOL * rs
        mine = {lag for (jj, lag) in got if jj == j}
        for lag in mine:
            i = lag - lag_begin
            assert rs[i] > kappa - tol[i], f"R5(ii): gpu hit ({j}, {lag}) has oracle rho_sigma {rs[i]}"
            assert abs(got[(j, lag)] - rs[i]) <= tol[i], \
                f"R5(ii): value at ({j}, {lag}): gpu {got[(j, lag)]} oracle {rs[i]} tol {tol[i]}"
        sure = np.nonzero(rs > kappa + tol)[0]
        n_oracle += int((rs > kappa).sum())
        n_border += int(((rs > kappa - tol) & (rs <= kappa + tol)).sum())
        if total == len(got):                       # nothing overflowed: the list is complete
            missing = [lag_begin + int(i) for i in sure if lag_begin + int(i) not in mine]
            assert not missing, f"R5(iii): template {j} misses sure hits at lags {missing[:5]}"
    if total == len(got):
        assert abs(total - n_oracle) <= n_border
    return n_oracle, n_border
