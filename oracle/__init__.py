"""Python face of the float64 CPU oracle (oracle/bfly_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It does
not import, and is not imported by, paper_1802_01685_b200.

Argument marshalling only; all arithmetic is in bfly_oracle.c (plus
fft_variant.py, the float64 FFT restatement used for pin P4, and streaming.py, the
chunk plan of reading C11).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, fp, ip = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int32)
        L.bfo_template.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, dp, dp]
        L.bfo_template.restype = None
        L.bfo_template_norms.argtypes = [C.c_int, dp, dp, dp, dp]
        L.bfo_template_norms.restype = None
        L.bfo_rho_at.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_double, C.c_double,
                                 C.c_int64, dp, dp]
        L.bfo_rho_at.restype = C.c_double
        L.bfo_sliding_n2.argtypes = [fp, C.c_int, C.c_int64, C.c_int64, dp]
        L.bfo_sliding_n2.restype = None
        L.bfo_rho_series.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_double, C.c_double,
                                     C.c_int64, C.c_int64, dp, dp, dp]
        L.bfo_rho_series.restype = None
        L.bfo_correlate.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_int64, dp, dp,
                                    C.c_int64, C.c_int64, dp, ip, C.c_int]
        L.bfo_correlate.restype = C.c_int
        L.bfo_map.argtypes = [C.c_int64, dp, dp, ip, C.c_double, C.c_int64, C.c_int32,
                              C.c_double, C.c_double, C.c_int32, C.c_int32,
                              C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)]
        L.bfo_map.restype = None
        L.bfo_template3.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, C.c_double, dp, dp]
        L.bfo_template3.restype = None
        L.bfo_rho_series3.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_double, C.c_double,
                                      C.c_double, C.c_int64, C.c_int64, dp, dp, dp]
        L.bfo_rho_series3.restype = None
        L.bfo_correlate3.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_int64, dp, dp, dp,
                                     C.c_int64, C.c_int64, dp, ip, C.c_int]
        L.bfo_correlate3.restype = C.c_int
        L.bfo_sigma.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_double, C.c_double]
        L.bfo_sigma.restype = C.c_double
        L.bfo_tails.argtypes = [fp, C.c_int64, C.c_double, C.c_int, C.c_int64, dp, dp, C.c_int64,
                                C.c_int64, C.c_double, dp, C.c_int64, ip, ip, dp, C.c_int]
        L.bfo_tails.restype = C.c_int64
        L.bfo_template_settle.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, C.c_double, dp, dp]
        L.bfo_template_settle.restype = None
        L.bfo_template_family.argtypes = [C.c_int, C.c_double, C.c_int, C.c_double, C.c_double,
                                          C.c_double, dp, dp]
        L.bfo_template_family.restype = None
        L.bfo_rho_series_family.argtypes = [C.c_int, fp, C.c_int64, C.c_double, C.c_int, C.c_double,
                                            C.c_double, C.c_double, C.c_int64, C.c_int64, dp, dp, dp]
        L.bfo_rho_series_family.restype = None
        L.bfo_correlate_family.argtypes = [C.c_int, fp, C.c_int64, C.c_double, C.c_int, C.c_int64,
                                           dp, dp, dp, C.c_int64, C.c_int64, dp, ip, C.c_int]
        L.bfo_correlate_family.restype = C.c_int
        L.bfo_sigma_family.argtypes = [C.c_int, fp, C.c_int64, C.c_double, C.c_int, C.c_double,
                                       C.c_double, C.c_double]
        L.bfo_sigma_family.restype = C.c_double
        L.bfo_tails_family.argtypes = [C.c_int, fp, C.c_int64, C.c_double, C.c_int, C.c_int64, dp,
                                       dp, dp, C.c_int64, C.c_int64, C.c_double, dp, C.c_int64, ip,
                                       ip, dp, C.c_int]
        L.bfo_tails_family.restype = C.c_int64
        L.bfo_max_threads.argtypes = []
        L.bfo_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _f32(x):
    x = np.ascontiguousarray(x)
    if x.dtype != np.float32:
        raise TypeError("data must be fp32 (reading C12: fp32 inputs, upcast inside)")
    return x


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def max_threads() -> int:
    return int(lib().bfo_max_threads())


FAMILY = {"poly": 0, "settle": 1}


def _fam(family) -> int:
    """Template family: "poly" = (f0, f1, f2) polynomial phase (readings C1, N1), "settle" =
    (f_inf, D, tc) exponentially settling chirp (reading N2)."""
    return FAMILY[family]


def template(fs, L, f0, f1, f2=0.0, family="poly"):
    """(hc, hs): un-normalised cosine and sine templates, float64[L] each.  family "poly":
    (f0, f1, f2) (f2: reading N1); family "settle": the three arguments are (f_inf, D, tc)."""
    hc = np.empty(L, np.float64)
    hs = np.empty(L, np.float64)
    lib().bfo_template_family(_fam(family), float(fs), int(L), float(f0), float(f1), float(f2),
                              _p(hc, C.c_double), _p(hs, C.c_double))
    return hc, hs


def template_norms(hc, hs):
    hc, hs = _f64(hc), _f64(hs)
    nc, ns = C.c_double(), C.c_double()
    lib().bfo_template_norms(len(hc), _p(hc, C.c_double), _p(hs, C.c_double),
                             C.byref(nc), C.byref(ns))
    return nc.value, ns.value


def rho_at(x, fs, L, f0, f1, tau, components=False):
    """rho of one template at one lag, by the literal definition."""
    x = _f32(x)
    if not (0 <= tau <= len(x) - L):
        raise ValueError("lag outside the valid range")
    cn, sn = C.c_double(), C.c_double()
    r = lib().bfo_rho_at(_p(x, C.c_float), len(x), float(fs), int(L), float(f0), float(f1),
                         int(tau), C.byref(cn), C.byref(sn))
    return (r, cn.value, sn.value) if components else r


def sliding_n2(x, L, lag_begin=0, lag_end=None):
    x = _f32(x)
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    out = np.empty(max(lag_end - lag_begin, 0), np.float64)
    lib().bfo_sliding_n2(_p(x, C.c_float), int(L), int(lag_begin), int(lag_end),
                         _p(out, C.c_double))
    return out


def rho_series(x, fs, L, f0, f1, lag_begin=0, lag_end=None, components=False, f2=0.0,
               family="poly"):
    """rho(tau) of one template over lag_begin <= tau < lag_end (float64)."""
    x = _f32(x)
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    if not (0 <= lag_begin <= lag_end <= len(x) - L + 1):
        raise ValueError("lag range outside the valid lags")
    n = lag_end - lag_begin
    rho = np.empty(n, np.float64)
    if components:
        c = np.empty(n, np.float64)
        s = np.empty(n, np.float64)
        cp, sp = _p(c, C.c_double), _p(s, C.c_double)
    else:
        cp = sp = None
    lib().bfo_rho_series_family(_fam(family), _p(x, C.c_float), len(x), float(fs), int(L),
                                float(f0), float(f1), float(f2), int(lag_begin), int(lag_end),
                                _p(rho, C.c_double), cp, sp)
    return (rho, c, s) if components else rho


def correlate(x, fs, L, f0, f1, lag_begin=0, lag_end=None, n_threads=0, f2=None, family="poly"):
    """(rho_max float64[T], arg_lag int32[T]) over lag_begin <= tau < lag_end.  family "settle":
    (f0, f1, f2) carry (f_inf, D, tc) per template."""
    x = _f32(x)
    f0, f1 = _f64(f0), _f64(f1)
    if f0.shape != f1.shape or f0.ndim != 1:
        raise ValueError("f0 and f1 must be 1-D and of equal length")
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    T = len(f0)
    rho_max = np.empty(T, np.float64)
    arg = np.empty(T, np.int32)
    if f2 is not None:
        f2 = _f64(f2)
        if f2.shape != f0.shape:
            raise ValueError("f2 must have the shape of f0")
    if family == "settle" and f2 is None:
        raise ValueError("the settle family needs tc per template")
    rc = lib().bfo_correlate_family(_fam(family), _p(x, C.c_float), len(x), float(fs), int(L), T,
                                    _p(f0, C.c_double), _p(f1, C.c_double),
                                    _p(f2, C.c_double) if f2 is not None else None, int(lag_begin),
                                    int(lag_end), _p(rho_max, C.c_double), _p(arg, C.c_int32),
                                    int(n_threads))
    if rc < 0:
        raise ValueError("bfo_correlate: bad arguments")
    return rho_max, arg


def butterfly_map(f0, rho_max, arg_lag, kappa, lag_origin, samples_per_tbin, f_lo_hz, df_hz,
                  n_fbins, n_tbins, map_out=None, counters=None):
    """Accumulate hits into a uint32 [n_tbins][n_fbins] map; returns (map, counters).
    kappa is compared as the fp32 value the C ABI would carry (C9)."""
    f0, rho_max = _f64(f0), _f64(rho_max)
    arg_lag = np.ascontiguousarray(arg_lag, dtype=np.int32)
    if map_out is None:
        map_out = np.zeros((n_tbins, n_fbins), np.uint32)
    if counters is None:
        counters = np.zeros(2, np.uint64)
    k32 = float(np.float32(kappa))
    lib().bfo_map(len(f0), _p(f0, C.c_double), _p(rho_max, C.c_double), _p(arg_lag, C.c_int32),
                  k32, int(lag_origin), int(samples_per_tbin), float(f_lo_hz), float(df_hz),
                  int(n_fbins), int(n_tbins), _p(map_out, C.c_uint32), _p(counters, C.c_uint64))
    return map_out, counters


def sigma(x, fs, L, f0, f1, f2=0.0, family="poly"):
    """Reading S1: rms per quadrature of the circular matched-filter output of one template
    over the whole segment."""
    x = _f32(x)
    if len(x) < L:
        raise ValueError("segment shorter than the template")
    return float(lib().bfo_sigma_family(_fam(family), _p(x, C.c_float), len(x), float(fs), int(L),
                                        float(f0), float(f1), float(f2)))


def tails(x, fs, L, f0, f1, kappa, lag_begin=0, lag_end=None, capacity=None, n_threads=0,
          f2=None, family="poly"):
    """Readings S1-S3: (sigma float64[T], hit_template int32[n], hit_lag int32[n],
    hit_rho float64[n], total) with hits = valid lags where sqrt(c^2+s^2)/sigma_j > kappa, in
    ascending (template, lag) order; n = min(total, capacity)."""
    x = _f32(x)
    f0, f1 = _f64(f0), _f64(f1)
    if f2 is not None:
        f2 = _f64(f2)
        if f2.shape != f0.shape:
            raise ValueError("f2 must have the shape of f0")
    elif family == "settle":
        raise ValueError("the settle family needs tc per template")
    p2 = _p(f2, C.c_double) if f2 is not None else None
    fam = _fam(family)
    lag_end = len(x) - L + 1 if lag_end is None else lag_end
    T = len(f0)
    sig = np.empty(T, np.float64)
    if capacity is None:
        # count first, then size the arrays exactly
        total = lib().bfo_tails_family(fam, _p(x, C.c_float), len(x), float(fs), int(L), T,
                                       _p(f0, C.c_double), _p(f1, C.c_double), p2, int(lag_begin),
                                       int(lag_end), float(kappa), _p(sig, C.c_double), 0, None,
                                       None, None, int(n_threads))
        if total < 0:
            raise ValueError("bad arguments")
        capacity = int(total)
    hj = np.empty(max(capacity, 1), np.int32)
    hl = np.empty(max(capacity, 1), np.int32)
    hr = np.empty(max(capacity, 1), np.float64)
    total = lib().bfo_tails_family(fam, _p(x, C.c_float), len(x), float(fs), int(L), T,
                                   _p(f0, C.c_double), _p(f1, C.c_double), p2, int(lag_begin),
                                   int(lag_end), float(kappa), _p(sig, C.c_double), int(capacity),
                                   _p(hj, C.c_int32), _p(hl, C.c_int32), _p(hr, C.c_double),
                                   int(n_threads))
    if total < 0:
        raise ValueError("bad arguments")
    n = int(min(total, capacity))
    return sig, hj[:n], hl[:n], hr[:n], int(total)
