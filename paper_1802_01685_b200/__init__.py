"""Thin Python binding of libbfly (include/bfly.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used here
for device memory and streams only.  The functions carry the C names without the `bfly_`
prefix.  There is no CPU fallback: if the shared library cannot be loaded the import fails,
and every call that returns a negative status raises BflyError.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

__all__ = ["BflyError", "Bank", "make_bank", "make_bank_grid", "correlate", "correlate_form",
           "butterfly_map", "search_host", "launch_count", "lib_path",
           "FORM_DEFAULT", "FORM_FFT", "FORM_DIRECT", "FORM_FFT_TC", "FORM_DENSE_TC", "FORM_FFT_TC5",
           "debug_fft_tc", "debug_fft_tc5", "tails", "hits_map", "time_randomize", "coincidence", "pseudo_spectrum",
           "make_bank_settle", "FAMILY_POLY", "FAMILY_SETTLE", "debug_peak", "PEAK_FFMA", "PEAK_FFMA2", "PEAK_LDS", "PEAK_HMMA", "PEAK_SHFL", "PEAK_L2",
           "PEAK_UMMA"]

FORM_DEFAULT, FORM_FFT, FORM_DIRECT, FORM_FFT_TC, FORM_DENSE_TC, FORM_FFT_TC5 = 0, 1, 2, 3, 4, 5
FAMILY_POLY, FAMILY_SETTLE = 0, 1
PEAK_FFMA, PEAK_FFMA2, PEAK_LDS, PEAK_HMMA, PEAK_SHFL, PEAK_L2, PEAK_UMMA = range(7)


class BflyError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str):
        super().__init__(f"{what}: {detail} (status {status})")
        self.status = status


def _load():
    path = _build.LIB
    if _build.is_stale():
        # Build in-tree when the sources are newer (needs nvcc; works without a GPU).
        path = _build.build()
    lib = C.CDLL(path)
    vp, i32, i64, f64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_double, C.c_float
    lib.bfly_strerror.restype = C.c_char_p
    lib.bfly_strerror.argtypes = [C.c_int]
    lib.bfly_last_error.restype = C.c_char_p
    lib.bfly_last_error.argtypes = []
    lib.bfly_make_bank.argtypes = [f64, i32, i64, vp, vp, C.c_int, C.POINTER(vp)]
    lib.bfly_make_bank3.argtypes = [f64, i32, i64, vp, vp, vp, C.c_int, C.POINTER(vp)]
    lib.bfly_bank_get_f2.argtypes = [vp, i64, i64, vp]
    lib.bfly_make_bank_settle.argtypes = [f64, i32, i64, vp, vp, vp, C.c_int, C.POINTER(vp)]
    lib.bfly_bank_get_settle.argtypes = [vp, i64, i64, vp, vp, vp]
    lib.bfly_bank_family.argtypes = [vp]
    lib.bfly_make_bank_grid.argtypes = [f64, i32, f64, f64, i32, f64, f64, i32, C.c_int,
                                        C.POINTER(vp)]
    lib.bfly_free_bank.argtypes = [vp]
    lib.bfly_free_bank.restype = None
    lib.bfly_bank_size.argtypes = [vp]
    lib.bfly_bank_size.restype = i64
    lib.bfly_bank_get.argtypes = [vp, i64, i64, vp, vp, vp, vp]
    lib.bfly_bank_reserve.argtypes = [vp, i64]
    lib.bfly_correlate.argtypes = [vp, vp, i64, i64, i64, vp, vp, vp]
    lib.bfly_correlate_form.argtypes = [vp, C.c_int, vp, i64, i64, i64, vp, vp, vp]
    lib.bfly_correlate_static.argtypes = [vp, vp, i64, i64, i64, vp, vp, vp]
    lib.bfly_correlate_multi.argtypes = [vp, i32, vp, i64, i64, i64, vp, vp, vp]
    lib.bfly_butterfly_map.argtypes = [vp, vp, vp, f32, i64, i32, f64, f64, i32, i32, vp, vp, vp]
    lib.bfly_tails.argtypes = [vp, vp, i64, i64, i64, f32, vp, i64, vp, vp, vp, vp, vp]
    lib.bfly_hits_map.argtypes = [vp, vp, vp, i64, i64, i32, f64, f64, i32, i32, vp, vp, vp]
    lib.bfly_time_randomize.argtypes = [vp, vp, i64, vp, vp, vp]
    lib.bfly_coincidence.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp]
    lib.bfly_pseudo_spectrum.argtypes = [vp, i32, i32, vp, vp]
    lib.bfly_search_host.argtypes = [vp, vp, i64, i64, f32, i32, f64, f64, i32, i32,
                                     vp, vp, vp, vp, vp]
    lib.bfly_bank_set_timing.argtypes = [vp, C.c_int]
    lib.bfly_bank_core_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.bfly_debug_fft_tc.argtypes = [vp, vp, C.c_int, vp]
    lib.bfly_debug_fft_tc5.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.bfly_debug_peak.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(f64), C.POINTER(f64)]
    lib.bfly_launch_count.argtypes = []
    lib.bfly_launch_count.restype = i64
    for name in ("bfly_make_bank", "bfly_make_bank_grid", "bfly_bank_get", "bfly_bank_reserve",
                 "bfly_bank_set_timing", "bfly_bank_core_ms", "bfly_correlate", "bfly_correlate_form", "bfly_correlate_multi", "bfly_correlate_static", "bfly_butterfly_map",
                 "bfly_search_host", "bfly_debug_fft_tc", "bfly_debug_fft_tc5", "bfly_tails", "bfly_hits_map",
                 "bfly_time_randomize", "bfly_coincidence", "bfly_pseudo_spectrum",
                 "bfly_make_bank3", "bfly_bank_get_f2", "bfly_debug_peak", "bfly_make_bank_settle",
                 "bfly_bank_get_settle", "bfly_bank_family"):
        getattr(lib, name).restype = C.c_int
    return lib, path


_lib, _lib_path = _load()


def lib_path() -> str:
    return _lib_path


def _check(status: int, what: str):
    if status != 0:
        raise BflyError(status, what, (_lib.bfly_last_error() or b"").decode() or
                        _lib.bfly_strerror(status).decode())


def _dev(t: torch.Tensor, dtype, name: str, device=None, numel=None):
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    if device is not None and t.device.index != device:
        raise ValueError(f"{name} is on cuda:{t.device.index}, the bank on cuda:{device}")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"{name} has {t.numel()} elements, needs {numel}")
    return C.c_void_p(t.data_ptr())


def _stream(device: int):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


class Bank:
    """Owner of a bfly_bank handle (device-resident bank parameters and workspace)."""

    def __init__(self, handle, device: int, fs_hz: float, L: int):
        self._h = handle
        self.device = device
        self.fs_hz = float(fs_hz)
        self.L = int(L)

    def __len__(self):
        return int(_lib.bfly_bank_size(self._h))

    def close(self):
        if self._h is not None:
            _lib.bfly_free_bank(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def get(self, first: int = 0, count: int | None = None):
        """(f0, f1, 1/||cos||^2, 1/||sin||^2) of templates [first, first+count) as numpy."""
        count = len(self) - first if count is None else count
        f0 = np.empty(count, np.float64)
        f1 = np.empty(count, np.float64)
        a = np.empty(count, np.float32)
        b = np.empty(count, np.float32)
        _check(_lib.bfly_bank_get(self._h, first, count, f0.ctypes.data, f1.ctypes.data,
                                  a.ctypes.data, b.ctypes.data), "bfly_bank_get")
        return f0, f1, a, b

    def get_f2(self, first: int = 0, count: int | None = None):
        count = len(self) - first if count is None else count
        f2 = np.empty(count, np.float64)
        _check(_lib.bfly_bank_get_f2(self._h, first, count, f2.ctypes.data), "bfly_bank_get_f2")
        return f2

    @property
    def family(self) -> int:
        return int(_lib.bfly_bank_family(self._h))

    def get_settle(self, first: int = 0, count: int | None = None):
        """(f_inf, D, tc) of templates [first, first+count) of a settling-family bank."""
        count = len(self) - first if count is None else count
        a, b, c = (np.empty(count, np.float64) for _ in range(3))
        _check(_lib.bfly_bank_get_settle(self._h, first, count, a.ctypes.data, b.ctypes.data,
                                         c.ctypes.data), "bfly_bank_get_settle")
        return a, b, c

    def set_timing(self, enable: bool):
        _check(_lib.bfly_bank_set_timing(self._h, int(bool(enable))), "bfly_bank_set_timing")

    def core_ms(self) -> float:
        """Device time of the correlation-core kernel of the last correlate call (ms)."""
        ms = C.c_float()
        _check(_lib.bfly_bank_core_ms(self._h, C.byref(ms)), "bfly_bank_core_ms")
        return float(ms.value)

    def reserve(self, max_n_samples: int):
        _check(_lib.bfly_bank_reserve(self._h, int(max_n_samples)), "bfly_bank_reserve")


def make_bank(fs_hz: float, L: int, f0_hz, f1_hzps, device: int = 0, f2_hzps2=None) -> Bank:
    """bfly_make_bank, or bfly_make_bank3 when f2_hzps2 (the second frequency derivative of the
    non-linear family) is given."""
    f0 = np.ascontiguousarray(f0_hz, dtype=np.float64)
    f1 = np.ascontiguousarray(f1_hzps, dtype=np.float64)
    if f0.ndim != 1 or f0.shape != f1.shape:
        raise ValueError("f0 and f1 must be 1-D and of equal length")
    h = C.c_void_p()
    if f2_hzps2 is None:
        _check(_lib.bfly_make_bank(float(fs_hz), int(L), f0.size, f0.ctypes.data, f1.ctypes.data,
                                   int(device), C.byref(h)), "bfly_make_bank")
    else:
        f2 = np.ascontiguousarray(f2_hzps2, dtype=np.float64)
        if f2.shape != f0.shape:
            raise ValueError("f2 must have the shape of f0")
        _check(_lib.bfly_make_bank3(float(fs_hz), int(L), f0.size, f0.ctypes.data, f1.ctypes.data,
                                    f2.ctypes.data, int(device), C.byref(h)), "bfly_make_bank3")
    return Bank(h, int(device), fs_hz, L)


def make_bank_settle(fs_hz: float, L: int, f_inf_hz, delta_hz, tau_c_s, device: int = 0) -> Bank:
    """bfly_make_bank_settle: exponentially settling chirps f(t) = f_inf + D exp(-t/tc)."""
    a = np.ascontiguousarray(f_inf_hz, dtype=np.float64)
    b = np.ascontiguousarray(delta_hz, dtype=np.float64)
    c = np.ascontiguousarray(tau_c_s, dtype=np.float64)
    if a.ndim != 1 or a.shape != b.shape or a.shape != c.shape:
        raise ValueError("f_inf, D and tc must be 1-D and of equal length")
    h = C.c_void_p()
    _check(_lib.bfly_make_bank_settle(float(fs_hz), int(L), a.size, a.ctypes.data, b.ctypes.data,
                                      c.ctypes.data, int(device), C.byref(h)), "bfly_make_bank_settle")
    return Bank(h, int(device), fs_hz, L)


def make_bank_grid(fs_hz, L, f0_lo, f0_hi, n_f0, f1_lo, f1_hi, n_f1, device: int = 0) -> Bank:
    h = C.c_void_p()
    _check(_lib.bfly_make_bank_grid(float(fs_hz), int(L), float(f0_lo), float(f0_hi), int(n_f0),
                                    float(f1_lo), float(f1_hi), int(n_f1), int(device),
                                    C.byref(h)), "bfly_make_bank_grid")
    return Bank(h, int(device), fs_hz, L)


def correlate_form(bank: Bank, form: int, x: torch.Tensor, lag_begin: int = 0,
                   lag_end: int | None = None, rho_max: torch.Tensor | None = None,
                   arg_lag: torch.Tensor | None = None):
    """bfly_correlate_form on torch's current stream; returns (rho_max, arg_lag) tensors."""
    T = len(bank)
    n = x.numel()
    lag_end = n - bank.L + 1 if lag_end is None else lag_end
    dev = torch.device("cuda", bank.device)
    if rho_max is None:
        rho_max = torch.empty(T, dtype=torch.float32, device=dev)
    if arg_lag is None:
        arg_lag = torch.empty(T, dtype=torch.int32, device=dev)
    _check(_lib.bfly_correlate_form(bank._h, int(form), _dev(x, torch.float32, "x", bank.device),
                                    n, int(lag_begin), int(lag_end),
                                    _dev(rho_max, torch.float32, "rho_max", bank.device, T),
                                    _dev(arg_lag, torch.int32, "arg_lag", bank.device, T),
                                    _stream(bank.device)), "bfly_correlate")
    return rho_max, arg_lag


def correlate(bank: Bank, x: torch.Tensor, lag_begin: int = 0, lag_end: int | None = None,
              rho_max: torch.Tensor | None = None, arg_lag: torch.Tensor | None = None):
    return correlate_form(bank, FORM_DEFAULT, x, lag_begin, lag_end, rho_max, arg_lag)


STATIC_MAX_SAMPLES = 65536        # BFLY_STATIC_MAX_SAMPLES (include/bfly.h)


def correlate_static(bank: Bank, x: torch.Tensor, rho_max: torch.Tensor, arg_lag: torch.Tensor,
                     lag_begin: int = 0, lag_end: int | None = None):
    """bfly_correlate_static on torch's current stream: the default form with its scratch in a
    static device array (no allocation inside the library); the caller passes the outputs."""
    T, n = len(bank), x.numel()
    lag_end = n - bank.L + 1 if lag_end is None else lag_end
    _check(_lib.bfly_correlate_static(bank._h, _dev(x, torch.float32, "x", bank.device), n, int(lag_begin),
                                      int(lag_end), _dev(rho_max, torch.float32, "rho_max", bank.device, T),
                                      _dev(arg_lag, torch.int32, "arg_lag", bank.device, T),
                                      _stream(bank.device)), "bfly_correlate_static")
    return rho_max, arg_lag


def correlate_multi(bank: Bank, xs, lag_begin: int = 0, lag_end: int | None = None):
    """bfly_correlate_multi: several segments of equal length (a sequence of CUDA tensors) against
    the same bank in one call; returns (list of rho_max, list of arg_lag), one pair per segment."""
    xs = list(xs)
    if not xs:
        raise ValueError("no segments")
    T, n, S = len(bank), xs[0].numel(), len(xs)
    if any(x.numel() != n for x in xs):
        raise ValueError("the segments must have equal length")
    lag_end = n - bank.L + 1 if lag_end is None else lag_end
    dev = torch.device("cuda", bank.device)
    rho = [torch.empty(T, dtype=torch.float32, device=dev) for _ in range(S)]
    arg = [torch.empty(T, dtype=torch.int32, device=dev) for _ in range(S)]
    PA = C.c_void_p * S
    xp = PA(*[_dev(x, torch.float32, "x", bank.device).value for x in xs])
    rp = PA(*[t.data_ptr() for t in rho])
    ap = PA(*[t.data_ptr() for t in arg])
    _check(_lib.bfly_correlate_multi(bank._h, S, xp, n, int(lag_begin), int(lag_end), rp, ap,
                                     _stream(bank.device)), "bfly_correlate_multi")
    return rho, arg


def butterfly_map(bank: Bank, rho_max: torch.Tensor, arg_lag: torch.Tensor, kappa: float,
                  lag_origin: int, samples_per_tbin: int, f_lo_hz: float, df_hz: float,
                  n_fbins: int, n_tbins: int, map_out: torch.Tensor | None = None,
                  counters: torch.Tensor | None = None):
    """bfly_butterfly_map; map_out (int32 storage of the uint32 counts, [n_tbins, n_fbins]) and
    counters (int64 storage of 2 x uint64) are accumulated into; created zeroed if None."""
    dev = torch.device("cuda", bank.device)
    T = len(bank)
    if map_out is None:
        map_out = torch.zeros((n_tbins, n_fbins), dtype=torch.int32, device=dev)
    if counters is None:
        counters = torch.zeros(2, dtype=torch.int64, device=dev)
    _check(_lib.bfly_butterfly_map(bank._h, _dev(rho_max, torch.float32, "rho_max", bank.device, T),
                                   _dev(arg_lag, torch.int32, "arg_lag", bank.device, T),
                                   float(kappa), int(lag_origin), int(samples_per_tbin),
                                   float(f_lo_hz), float(df_hz), int(n_fbins), int(n_tbins),
                                   _dev(map_out, torch.int32, "map_out", bank.device,
                                        n_fbins * n_tbins),
                                   _dev(counters, torch.int64, "counters", bank.device, 2),
                                   _stream(bank.device)), "bfly_butterfly_map")
    return map_out, counters


def tails(bank: Bank, x: torch.Tensor, kappa: float, capacity: int, lag_begin: int = 0,
          lag_end: int | None = None, n_hits: torch.Tensor | None = None):
    """bfly_tails on torch's current stream.  Returns (sigma fp32[T], hit_template int32[capacity],
    hit_lag int32[capacity], hit_rho fp32[capacity], n_hits int64[1]); the hit arrays are in no
    particular order and valid up to min(n_hits, capacity).  n_hits is incremented (created
    zeroed if None)."""
    T = len(bank)
    n = x.numel()
    lag_end = n - bank.L + 1 if lag_end is None else lag_end
    dev = torch.device("cuda", bank.device)
    sigma = torch.empty(T, dtype=torch.float32, device=dev)
    cap = max(int(capacity), 0)
    hj = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
    hl = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
    hr = torch.empty(max(cap, 1), dtype=torch.float32, device=dev)
    if n_hits is None:
        n_hits = torch.zeros(1, dtype=torch.int64, device=dev)
    _check(_lib.bfly_tails(bank._h, _dev(x, torch.float32, "x", bank.device), n, int(lag_begin),
                           int(lag_end), float(kappa), C.c_void_p(sigma.data_ptr()), cap,
                           C.c_void_p(hj.data_ptr()), C.c_void_p(hl.data_ptr()),
                           C.c_void_p(hr.data_ptr()),
                           _dev(n_hits, torch.int64, "n_hits", bank.device, 1),
                           _stream(bank.device)), "bfly_tails")
    return sigma, hj, hl, hr, n_hits


def hits_map(bank: Bank, hit_template: torch.Tensor, hit_lag: torch.Tensor, n_hits: int,
             lag_origin: int, samples_per_tbin: int, f_lo_hz: float, df_hz: float, n_fbins: int,
             n_tbins: int, map_out: torch.Tensor | None = None,
             counters: torch.Tensor | None = None):
    """bfly_hits_map: one count per hit of a bfly_tails list; accumulates like butterfly_map."""
    dev = torch.device("cuda", bank.device)
    if map_out is None:
        map_out = torch.zeros((n_tbins, n_fbins), dtype=torch.int32, device=dev)
    if counters is None:
        counters = torch.zeros(2, dtype=torch.int64, device=dev)
    _check(_lib.bfly_hits_map(bank._h, _dev(hit_template, torch.int32, "hit_template", bank.device),
                              _dev(hit_lag, torch.int32, "hit_lag", bank.device), int(n_hits),
                              int(lag_origin), int(samples_per_tbin), float(f_lo_hz), float(df_hz),
                              int(n_fbins), int(n_tbins),
                              _dev(map_out, torch.int32, "map_out", bank.device, n_fbins * n_tbins),
                              _dev(counters, torch.int64, "counters", bank.device, 2),
                              _stream(bank.device)), "bfly_hits_map")
    return map_out, counters


def time_randomize(x: torch.Tensor, perm: torch.Tensor):
    """bfly_time_randomize: (x[perm], bad flag int32[1]); perm is an int32 CUDA tensor drawn by the
    caller's seeded generator."""
    n = x.numel()
    dev = x.device.index
    out = torch.empty_like(x)
    bad = torch.zeros(1, dtype=torch.int32, device=x.device)
    with torch.cuda.device(dev):
        _check(_lib.bfly_time_randomize(_dev(x, torch.float32, "x"), _dev(perm, torch.int32, "perm", dev, n),
                                        n, C.c_void_p(out.data_ptr()), C.c_void_p(bad.data_ptr()),
                                        _stream(dev)), "bfly_time_randomize")
    return out, bad


def coincidence(map1: torch.Tensor, map2: torch.Tensor, half_width_bins: int):
    """bfly_coincidence on two [n_tbins, n_fbins] int32-stored count maps; returns (co1, co2)."""
    if map1.shape != map2.shape or map1.dim() != 2:
        raise ValueError("maps must be 2-D and of equal shape")
    dev = map1.device.index
    nt, nf = map1.shape
    c1, c2 = torch.empty_like(map1), torch.empty_like(map2)
    with torch.cuda.device(dev):
        _check(_lib.bfly_coincidence(_dev(map1, torch.int32, "map1"), _dev(map2, torch.int32, "map2", dev),
                                     int(nt), int(nf), int(half_width_bins), C.c_void_p(c1.data_ptr()),
                                     C.c_void_p(c2.data_ptr()), _stream(dev)), "bfly_coincidence")
    return c1, c2


def pseudo_spectrum(map_: torch.Tensor, spectrum: torch.Tensor | None = None):
    """bfly_pseudo_spectrum: adds the time marginal of the map to spectrum (int64 storage of
    uint64 [n_fbins]; created zeroed if None)."""
    dev = map_.device.index
    nt, nf = map_.shape
    if spectrum is None:
        spectrum = torch.zeros(nf, dtype=torch.int64, device=map_.device)
    with torch.cuda.device(dev):
        _check(_lib.bfly_pseudo_spectrum(_dev(map_, torch.int32, "map"), int(nt), int(nf),
                                         _dev(spectrum, torch.int64, "spectrum", dev, nf), _stream(dev)),
               "bfly_pseudo_spectrum")
    return spectrum


def search_host(bank: Bank, x_host, chunk_samples: int, kappa: float, samples_per_tbin: int,
                f_lo_hz: float, df_hz: float, n_fbins: int, n_tbins: int):
    """bfly_search_host: the whole path on a HOST fp32 series (numpy array or pinned CPU
    tensor).  Returns numpy (rho_max, arg_lag) of the last chunk, map [n_tbins, n_fbins]
    uint32 and counters uint64[2]."""
    if isinstance(x_host, torch.Tensor):
        if x_host.is_cuda or x_host.dtype != torch.float32 or not x_host.is_contiguous():
            raise TypeError("x_host must be a contiguous fp32 CPU tensor or numpy array")
        xp, n = x_host.data_ptr(), x_host.numel()
    else:
        x_host = np.ascontiguousarray(x_host)
        if x_host.dtype != np.float32:
            raise TypeError("x_host must be fp32")
        xp, n = x_host.ctypes.data, x_host.size
    T = len(bank)
    rho = np.empty(T, np.float32)
    arg = np.empty(T, np.int32)
    m = np.empty((n_tbins, n_fbins), np.uint32)
    cnt = np.empty(2, np.uint64)
    _check(_lib.bfly_search_host(bank._h, C.c_void_p(xp), n, int(chunk_samples), float(kappa),
                                 int(samples_per_tbin), float(f_lo_hz), float(df_hz),
                                 int(n_fbins), int(n_tbins), rho.ctypes.data, arg.ctypes.data,
                                 m.ctypes.data, cnt.ctypes.data, _stream(bank.device)),
           "bfly_search_host")
    return rho, arg, m, cnt


def debug_fft_tc(y: torch.Tensor, full: bool = False) -> torch.Tensor:
    """bfly_debug_fft_tc: the bare tensor-core transform of FORM_FFT_TC on one complex64[8192]
    device tensor (tests only).  Returns complex64[8192]; entries n >= 4096 are 0 unless full."""
    if y.dtype != torch.complex64 or y.numel() != 8192 or not y.is_cuda or not y.is_contiguous():
        raise TypeError("y must be a contiguous complex64[8192] CUDA tensor")
    z = torch.zeros_like(y)
    _check(_lib.bfly_debug_fft_tc(C.c_void_p(y.data_ptr()), C.c_void_p(z.data_ptr()),
                                  int(bool(full)), _stream(y.device.index)), "bfly_debug_fft_tc")
    return z


def debug_peak(which: int, variant: int = 0, iters: int = 2000, device: int = 0):
    """bfly_debug_peak: one microbenchmark on every SM of `device`.  Returns (value, ms) --
    value is a float (flop/s, bytes/s or shuffles/s) except for PEAK_UMMA, where it is the pair
    (MMA flop per clock and SM, clocks per iteration of the streaming warps)."""
    out = (C.c_double * 2)(0.0, 0.0)
    ms = C.c_double(0.0)
    with torch.cuda.device(device):
        _check(_lib.bfly_debug_peak(int(which), int(variant), int(iters), out, C.byref(ms)),
               "bfly_debug_peak")
    return ((out[0], out[1]) if which == PEAK_UMMA else out[0]), ms.value


def debug_fft_tc5(y: torch.Tensor, reps: int = 1):
    """bfly_debug_fft_tc5: the length-8192 transform on tcgen05 for complex64[2 p, 8192] device
    input (tests only).  Returns (complex64[2 p, 4096], SM clock cycles of the whole loop)."""
    if y.dtype != torch.complex64 or y.dim() != 2 or y.shape[1] != 8192 or y.shape[0] % 2 or not y.is_cuda \
            or not y.is_contiguous():
        raise TypeError("y must be a contiguous complex64[2 p, 8192] CUDA tensor")
    z = torch.zeros((y.shape[0], 4096), dtype=torch.complex64, device=y.device)
    cyc = torch.zeros(1, dtype=torch.int64, device=y.device)
    _check(_lib.bfly_debug_fft_tc5(C.c_void_p(y.data_ptr()), C.c_void_p(z.data_ptr()), y.shape[0] // 2,
                                   int(reps), C.c_void_p(cyc.data_ptr()), _stream(y.device.index)),
           "bfly_debug_fft_tc5")
    return z, cyc


def launch_count() -> int:
    return int(_lib.bfly_launch_count())
