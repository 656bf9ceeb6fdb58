"""Streaming over 16-s chunks with a 1-s overlap (TEST INFRASTRUCTURE).

Reading C11 (BASELINE.json configs[4]: "processed in 16 s chunks with 1 s overlap on
one stream ... butterfly map accumulated over the whole run"; the paper's 16-s
segments): chunk c covers samples [c*H, c*H + chunk) with hop
H = chunk - L; it searches its local lags [0, H) so that no absolute lag is searched
twice; the last chunk takes all the valid lags it has left.  Max / argmax are per
chunk; a template may add one hit per chunk; lag_origin = c*H.
"""
from __future__ import annotations

import numpy as np

from . import butterfly_map, correlate


def chunk_plan(n_samples: int, L: int, chunk: int):
    """List of (start_sample, n_chunk_samples, lag_begin, lag_end) per chunk; lags are
    local to the chunk and the union over chunks of start + [lag_begin, lag_end) is
    exactly the valid lags 0 .. n_samples - L."""
    if chunk <= L:
        raise ValueError("chunk must exceed L")
    total = n_samples - L + 1
    if chunk >= n_samples:                 # a single chunk takes every valid lag
        return [(0, n_samples, 0, total)]
    H = chunk - L
    plan, start = [], 0
    while start < total:
        n = min(chunk, n_samples - start)
        lags_here = n - L + 1
        last = start + H >= total
        lag_end = lags_here if last else min(H, lags_here)
        plan.append((start, n, 0, lag_end))
        start += H
    return plan


def stream(x, fs, L, f0, f1, chunk, kappa, map_grid, n_threads=0):
    """Run the oracle chunk by chunk; returns (map, counters, per_chunk_results)."""
    g = map_grid
    m = np.zeros((g["n_tbins"], g["n_fbins"]), np.uint32)
    counters = np.zeros(2, np.uint64)
    per_chunk = []
    for (start, n, lb, le) in chunk_plan(len(x), L, chunk):
        rho, arg = correlate(x[start:start + n], fs, L, f0, f1, lb, le, n_threads)
        butterfly_map(f0, rho, arg, kappa, start, g["samples_per_tbin"], g["f_lo_hz"],
                      g["df_hz"], g["n_fbins"], g["n_tbins"], m, counters)
        per_chunk.append((start, rho, arg))
    return m, counters, per_chunk
