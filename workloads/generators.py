"""Seeded input generators (numpy, float64, cast once to fp32).

Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe".  All randomness comes from
numpy.random.default_rng(seed).  Nothing here computes a correlation, a template
norm, rho or a map: these are inputs to both the oracle and the CUDA path.
"""
from __future__ import annotations

import math
from typing import Tuple

import numpy as np

from .configs import Config, Injection


def bank_grid(cfg: Config) -> Tuple[np.ndarray, np.ndarray]:
    """The (f0, f1) float64 lists of the config's bank.

    Inclusive uniform grids (numpy.linspace); template j = i_f0 * n_f1 + i_f1
    (SURVEY.md section 8(c) C3).
    """
    f0 = np.linspace(cfg.f0_lo, cfg.f0_hi, cfg.n_f0, dtype=np.float64)
    f1 = np.linspace(cfg.f1_lo, cfg.f1_hi, cfg.n_f1, dtype=np.float64)
    return np.repeat(f0, cfg.n_f1), np.tile(f1, cfg.n_f0)


def _injection_waveform(inj: Injection, fs: float, n_samples: int):
    """Samples [i0, i1) and A*cos(phi) of one injected chirp (float64)."""
    i0 = max(0, int(round(inj.t_start_s * fs)))
    i1 = min(n_samples, int(round(inj.t_stop_s * fs)))
    t = np.arange(i1 - i0, dtype=np.float64) / fs
    if inj.kind == "linear":
        cycles = inj.f_start_hz * t + 0.5 * inj.slope_hzps * t * t
    elif inj.kind == "settle":
        # phi/2pi = integral of f_inf + (f_s - f_inf) exp(-t/tau)
        cycles = inj.f_inf_hz * t + (inj.f_start_hz - inj.f_inf_hz) * inj.tau_c_s * (
            1.0 - np.exp(-t / inj.tau_c_s))
    else:
        raise ValueError(inj.kind)
    return i0, i1, inj.amplitude * np.cos(2.0 * math.pi * cycles)


def _grb_series(rng: np.random.Generator, n: int) -> np.ndarray:
    """Poisson counts, mean 20 per bin, rate modulated at 10 % rms by Gaussian red
    noise with an f^(-5/3) power spectrum; mean-subtracted, variance-normalised."""
    nfreq = n // 2 + 1
    spec = rng.standard_normal(nfreq) + 1j * rng.standard_normal(nfreq)
    f = np.arange(nfreq, dtype=np.float64)
    shape = np.zeros(nfreq)
    shape[1:] = f[1:] ** (-5.0 / 6.0)        # amplitude = sqrt(PSD)
    g = np.fft.irfft(spec * shape, n)
    g = g / g.std()
    rate = np.clip(20.0 * (1.0 + 0.1 * g), 0.0, None)
    counts = rng.poisson(rate).astype(np.float64)
    return (counts - counts.mean()) / counts.std()


def make_data(cfg: Config, n_samples: int | None = None) -> np.ndarray:
    """The config's data series as a C-contiguous fp32 array.

    `n_samples` may shorten the series (prefix of the same random stream is NOT
    guaranteed; a shortened series is its own seeded input)."""
    n = cfg.n_samples if n_samples is None else int(n_samples)
    rng = np.random.default_rng(cfg.seed)
    if cfg.data_kind == "gauss":
        x = rng.standard_normal(n)
    elif cfg.data_kind == "grb":
        x = _grb_series(rng, n)
    else:
        raise ValueError(cfg.data_kind)
    for inj in cfg.injections:
        i0, i1, w = _injection_waveform(inj, cfg.fs_hz, n)
        if i1 > i0:
            x[i0:i1] += w[: i1 - i0]
    return np.ascontiguousarray(x.astype(np.float32))


def default_map_grid(cfg: Config, n_samples: int | None = None):
    """Default butterfly-map grid: 1/16 s x 1 Hz bins,
    f_lo = 0, n_fbins = ceil(f0_hi) + 1, n_tbins = ceil(samples / samples_per_tbin)."""
    n = cfg.n_samples if n_samples is None else int(n_samples)
    spt = cfg.samples_per_tbin
    return dict(samples_per_tbin=spt, f_lo_hz=0.0, df_hz=1.0,
                n_fbins=int(math.ceil(cfg.f0_hi)) + 1,
                n_tbins=(n + spt - 1) // spt)


def _track_nodes(cfg: Config, inj: Injection, halfwidth: int):
    """Grid nodes within +-halfwidth of the (f0, f1) an injection passes through."""
    f0g = np.linspace(cfg.f0_lo, cfg.f0_hi, cfg.n_f0)
    f1g = np.linspace(cfg.f1_lo, cfg.f1_hi, cfg.n_f1)
    out = set()
    ts = np.arange(inj.t_start_s, inj.t_stop_s, 0.5)
    for t in ts:
        dt = t - inj.t_start_s
        if inj.kind == "linear":
            f, fd = inj.f_start_hz + inj.slope_hzps * dt, inj.slope_hzps
        else:
            e = math.exp(-dt / inj.tau_c_s)
            f = inj.f_inf_hz + (inj.f_start_hz - inj.f_inf_hz) * e
            fd = -(inj.f_start_hz - inj.f_inf_hz) / inj.tau_c_s * e
        i0 = int(np.argmin(np.abs(f0g - f)))
        i1 = int(np.argmin(np.abs(f1g - fd)))
        for a in range(max(0, i0 - halfwidth), min(cfg.n_f0, i0 + halfwidth + 1)):
            for b in range(max(0, i1 - halfwidth), min(cfg.n_f1, i1 + halfwidth + 1)):
                out.add(a * cfg.n_f1 + b)
    return out


def sub_bank_indices(cfg: Config, n_random: int, seed: int = 0,
                     halfwidth: int = 1, max_track: int = 512) -> np.ndarray:
    """A sorted, seeded sample of template indices of the config's own grid for
    parity at scale (SURVEY.md section 8(c) "Coverage at scale"): the four grid corners,
    nodes of the last f0 row (f0 = f0_hi; fs/2 at config 4), nodes near each injected
    chirp's track, and a stratified random sample."""
    T = cfg.n_templates
    rng = np.random.default_rng(1000 * cfg.index + seed)
    idx = {0, cfg.n_f1 - 1, T - cfg.n_f1, T - 1}
    last_row = (cfg.n_f0 - 1) * cfg.n_f1
    idx.update(int(last_row + i) for i in rng.integers(0, cfg.n_f1, size=min(8, cfg.n_f1)))
    track = set()
    for inj in cfg.injections:
        track |= _track_nodes(cfg, inj, halfwidth)
    track = sorted(track)
    if len(track) > max_track:
        track = list(rng.choice(track, size=max_track, replace=False))
    idx.update(int(i) for i in track)
    if n_random > 0:
        edges = np.linspace(0, T, n_random + 1).astype(np.int64)
        lo, hi = edges[:-1], np.maximum(edges[1:], edges[:-1] + 1)
        idx.update(int(i) for i in np.minimum(rng.integers(lo, hi), T - 1))
    return np.array(sorted(idx), dtype=np.int64)


def permutation(n: int, seed: int) -> np.ndarray:
    """Seeded uniformly random permutation of range(n) (int32): the input of the time-randomised
    control (reading T1).  Input generation only: both the oracle and the CUDA path
    receive this array."""
    return np.random.default_rng(seed).permutation(n).astype(np.int32)
