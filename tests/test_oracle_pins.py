"""Pins of the float64 oracle against what the mathematics fixes (CPU only).

The paper prints no worked numeric example (no value of rho, of a lag or of a map
cell anywhere in PAPER.md), so nothing is pinned by printed values.  Each pin below
is a closed form, an invariant, a special case that reduces to numpy.fft, or brute
force on a tiny input (SURVEY.md section 8(c) "Pins", P1-P11).
"""
import math

import numpy as np
import pytest

import oracle
from oracle import fft_variant, streaming


def _noise(n, seed):
    return np.random.default_rng(seed).standard_normal(n).astype(np.float32)


FS, L = 2048.0, 2048
INBAND = [(600.0, -200.0), (333.3, 150.0), (850.0, -390.0), (412.7, 77.7)]


def _gram(fs, L_, f0, f1):
    hc, hs = oracle.template(fs, L_, f0, f1)
    nc, ns = oracle.template_norms(hc, hs)
    return float(np.dot(hc, hs) / (nc * ns))


# ---------------------------------------------------------------- bulk == literal
def test_bulk_paths_equal_the_literal_definition_bit_for_bit():
    x = _noise(1500, 11)
    Lt = 300
    f0 = np.array([100.0, 433.3, 900.0])
    f1 = np.array([250.0, -120.0, 17.0])
    rmax, arg = oracle.correlate(x, FS, Lt, f0, f1)
    for j in range(3):
        series = oracle.rho_series(x, FS, Lt, f0[j], f1[j])
        for tau in (0, 1, 517, 1199, 1200):
            assert series[tau] == oracle.rho_at(x, FS, Lt, f0[j], f1[j], tau)
        a = int(np.argmax(series))
        assert arg[j] == a and rmax[j] == series[a]


def test_template_formula_spot_values():
    # C1 written out by hand for a few k (phase zero at the first sample, t = k/fs)
    hc, hs = oracle.template(1000.0, 8, 100.0, 4000.0)
    assert hc[0] == 1.0 and hs[0] == 0.0
    for k in (1, 3, 7):
        t = k / 1000.0
        ph = 2 * math.pi * (100.0 * t + 0.5 * 4000.0 * t * t)
        assert abs(hc[k] - math.cos(ph)) < 1e-15 and abs(hs[k] - math.sin(ph)) < 1e-15
    # quarter-period check: f0 = fs/4, f1 = 0 -> cos: 1,0,-1,0 ; sin: 0,1,0,-1
    hc, hs = oracle.template(8.0, 4, 2.0, 0.0)
    np.testing.assert_allclose(hc, [1, 0, -1, 0], atol=1e-15)
    np.testing.assert_allclose(hs, [0, 1, 0, -1], atol=1e-15)


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("f0,f1", INBAND + [(1024.0, 3.0), (30.0, -100.0)])
def test_P1_cauchy_schwarz(f0, f1):
    x = _noise(3 * L, 5)
    rho, c, s = oracle.rho_series(x, FS, L, f0, f1, components=True)
    assert np.all(np.abs(c) <= 1 + 1e-12) and np.all(np.abs(s) <= 1 + 1e-12)
    g = abs(_gram(FS, L, f0, f1))
    assert np.all(rho ** 2 <= 1 + g + 1e-12)
    assert np.all(rho >= 0)
    np.testing.assert_allclose(rho, np.sqrt(c * c + s * s), rtol=0, atol=1e-15)


def test_P1_bound_is_attained_by_the_extremal_vector():
    # rho^2 reaches 1 + |g| for x = hc_hat + sign(g) hs_hat: the bound is tight, so a
    # wrong normalisation cannot hide below it.
    f0, f1 = 1024.0, 3.0           # f0 = fs/2: strongly non-orthogonal pair
    hc, hs = oracle.template(FS, L, f0, f1)
    nc, ns = oracle.template_norms(hc, hs)
    g = _gram(FS, L, f0, f1)
    x = (hc / nc + math.copysign(1.0, g) * hs / ns)
    x32 = x.astype(np.float32)
    r = oracle.rho_at(x32, FS, L, f0, f1, 0)
    assert abs(r * r - (1 + abs(g))) < 1e-6      # fp32 cast of x costs ~1e-7


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("f0,f1", INBAND)
@pytest.mark.parametrize("tau0", [0, 777, 2048])
def test_P2_noise_free_injection(f0, f1, tau0):
    N = 2 * L
    hc, hs = oracle.template(FS, L, f0, f1)
    nc, _ = oracle.template_norms(hc, hs)
    x = np.zeros(N)
    x[tau0:tau0 + L] = 3.7 * hc / nc
    x32 = x.astype(np.float32)
    g = _gram(FS, L, f0, f1)
    r, cn, sn = oracle.rho_at(x32, FS, L, f0, f1, tau0, components=True)
    assert abs(cn - 1.0) < 2e-7          # fp32 rounding of the injected samples
    assert abs(r - math.sqrt(1 + g * g)) < 2e-7
    series = oracle.rho_series(x32, FS, L, f0, f1)
    assert int(np.argmax(series)) == tau0
    rmax, arg = oracle.correlate(x32, FS, L, np.array([f0]), np.array([f1]))
    assert arg[0] == tau0 and rmax[0] == series[tau0]


def test_P2_exact_in_float64_representable_case():
    # an injection whose samples are exact in fp32: f0 = fs/4, f1 = 0, hc = 1,0,-1,0,...
    fs, Lt, tau0 = 64.0, 64, 5
    x = np.zeros(160, np.float32)
    hc, hs = oracle.template(fs, Lt, 16.0, 0.0)
    x[tau0:tau0 + Lt] = np.round(hc).astype(np.float32) * 2.0
    r, cn, sn = oracle.rho_at(x, fs, Lt, 16.0, 0.0, tau0, components=True)
    assert abs(cn - 1.0) < 1e-12 and abs(sn) < 1e-12 and abs(r - 1.0) < 1e-12


# ---------------------------------------------------------------- P3
def _orth(c, s, g):
    """Norm of the projection of x_tau/||x_tau|| onto span{hc, hs}, from the oracle's two
    separately normalised components and the pair's Gram coefficient g."""
    return np.sqrt((c * c + s * s - 2 * g * c * s) / (1 - g * g))


@pytest.mark.parametrize("f0,f1", INBAND + [(40.0, -150.0), (1000.0, 300.0)])
def test_P3_time_reversal_maps_ascending_onto_descending(f0, f1):
    # Reversing a template gives the quadrature pair of the mapped template
    # (f0 + f1 (L-1)/fs, -f1) rotated by a constant phase: the two pairs span the same
    # plane, so the projection norm is invariant EXACTLY; rho itself (separate
    # normalisation, reading C2) only up to the pair's non-orthogonality.
    N = 3 * L
    xs = _noise(N, 21).astype(np.float64)
    hc, hs = oracle.template(FS, L, f0, f1)
    xs[1234:1234 + L] += 0.5 * hc
    x = xs.astype(np.float32)
    xr = np.ascontiguousarray(x[::-1])
    f0m, f1m = f0 + f1 * (L - 1) / FS, -f1
    a, ca, sa = oracle.rho_series(x, FS, L, f0, f1, components=True)
    b, cb, sb = oracle.rho_series(xr, FS, L, f0m, f1m, components=True)
    n_lags = N - L + 1
    ga, gb = _gram(FS, L, f0, f1), _gram(FS, L, f0m, f1m)
    np.testing.assert_allclose(_orth(ca, sa, ga), _orth(cb, sb, gb)[::-1], rtol=0, atol=1e-11)
    # rho itself: within (|g| + |nc/ns - 1|) * rho of each side
    def eps(f0_, f1_, g):
        nc, ns = oracle.template_norms(*oracle.template(FS, L, f0_, f1_))
        return abs(g) + abs(nc / ns - 1)
    tol = (eps(f0, f1, ga) + eps(f0m, f1m, gb)) * a.max() + 1e-12
    if (f0, f1) in INBAND:
        assert tol < 6e-4
    np.testing.assert_allclose(a, b[::-1], rtol=0, atol=tol)
    # the peak maps exactly: tau -> N - L - tau
    ta = int(np.argmax(a))
    tb = n_lags - 1 - int(np.argmax(b))
    assert abs(ta - 1234) <= 4           # noise may move a flat peak by a few samples
    assert tb == ta or abs(a[ta] - a[tb]) <= 2 * tol
    ia = int(np.argmax(_orth(ca, sa, ga)))
    ib = n_lags - 1 - int(np.argmax(_orth(cb, sb, gb)))
    assert ia == ib or abs(_orth(ca, sa, ga)[ia] - _orth(ca, sa, ga)[ib]) < 1e-11


def test_P3_wrong_mapping_fails():
    # the pin has teeth: the un-mapped (f0, -f1) pair does NOT satisfy the relation
    N = 3 * L
    x = _noise(N, 22)
    xr = np.ascontiguousarray(x[::-1])
    a = oracle.rho_series(x, FS, L, 600.0, -200.0)
    b = oracle.rho_series(xr, FS, L, 600.0, 200.0)
    assert np.abs(a - b[::-1]).max() > 1e-2


# ---------------------------------------------------------------- P4
def test_P4_direct_equals_fft_tiny():
    rng = np.random.default_rng(3)
    x = rng.standard_normal(64).astype(np.float32)
    for f0, f1 in [(3.0, 5.0), (10.0, -7.5), (1.5, 0.3), (16.0, 2.0)]:
        d = oracle.rho_series(x, 32.0, 16, f0, f1)
        f = fft_variant.rho_series_fft(x, 32.0, 16, f0, f1)
        np.testing.assert_allclose(d, f, rtol=0, atol=1e-11)
        # and against a pure-Python brute force of the definition
        for tau in (0, 7, 48):
            c = s = n2 = 0.0
            hc = [math.cos(2 * math.pi * (f0 * k / 32.0 + 0.5 * f1 * (k / 32.0) ** 2)) for k in range(16)]
            hs = [math.sin(2 * math.pi * (f0 * k / 32.0 + 0.5 * f1 * (k / 32.0) ** 2)) for k in range(16)]
            nc = math.sqrt(sum(v * v for v in hc))
            ns = math.sqrt(sum(v * v for v in hs))
            for k in range(16):
                xv = float(x[tau + k])
                c += xv * hc[k]; s += xv * hs[k]; n2 += xv * xv
            r = math.sqrt((c / nc) ** 2 + (s / ns) ** 2) / math.sqrt(n2)
            assert abs(d[tau] - r) < 1e-13


def test_P4_direct_equals_fft_tiny_config_size():
    x = _noise(4096, 1)
    f0 = np.array([600.0, 246.7, 900.0])
    f1 = np.array([-200.0, 400.0, -400.0])
    rd, ad = oracle.correlate(x, FS, L, f0, f1)
    rf, af = fft_variant.correlate_fft(x, FS, L, f0, f1)
    np.testing.assert_allclose(rd, rf, rtol=0, atol=1e-11)
    np.testing.assert_array_equal(ad, af)


# ---------------------------------------------------------------- P5
@pytest.mark.parametrize("a", [1e-3, 0.5, 8.0, 1024.0])
def test_P5_scale_invariance(a):
    x = _noise(2 * L, 9)
    xa = (x * np.float32(a)).astype(np.float32)     # exact for powers of two
    r0 = oracle.rho_series(x, FS, L, 500.0, 100.0, 0, 200)
    r1 = oracle.rho_series(xa, FS, L, 500.0, 100.0, 0, 200)
    tol = 1e-12 if math.log2(a) == int(math.log2(a)) else 2e-7
    np.testing.assert_allclose(r0, r1, rtol=0, atol=tol)


def test_zero_window_gives_zero_rho():
    x = np.zeros(100, np.float32)
    x[60:] = 1.0
    r = oracle.rho_series(x, 32.0, 20, 3.0, 1.0)
    assert np.all(r[:41] == 0.0) and r[60] > 0


# ---------------------------------------------------------------- P6, P7
def test_P6_dft_special_case():
    fs, Lt = 256.0, 256
    x = _noise(Lt, 4)
    X = np.fft.fft(x.astype(np.float64))
    nx = np.linalg.norm(x.astype(np.float64))
    for f0 in (1, 2, 17, 100, 127):
        r = oracle.rho_at(x, fs, Lt, float(f0), 0.0, 0)
        assert abs(r - math.sqrt(2.0 / Lt) * abs(X[f0]) / nx) < 1e-10
        hc, hs = oracle.template(fs, Lt, float(f0), 0.0)
        nc, ns = oracle.template_norms(hc, hs)
        assert abs(nc - math.sqrt(Lt / 2)) < 1e-10 and abs(ns - math.sqrt(Lt / 2)) < 1e-10
        assert abs(np.dot(hc, hs)) < 1e-10


def test_P7_parseval_sum_over_the_bank():
    fs, Lt = 128.0, 128
    x = _noise(Lt, 6)
    xd = x.astype(np.float64)
    X = np.fft.fft(xd)
    f0 = np.arange(1, Lt // 2, dtype=np.float64)
    r, _ = oracle.correlate(x, fs, Lt, f0, np.zeros_like(f0))
    total = np.sum(r ** 2)
    n2 = np.dot(xd, xd)
    expect = (n2 - X[0].real ** 2 / Lt - X[Lt // 2].real ** 2 / Lt) / n2
    assert abs(total - expect) < 1e-10


# ---------------------------------------------------------------- P8
def test_P8_noise_expectation_is_two_over_L():
    Lt, nwin = 64, 20000
    x = _noise(Lt * nwin + Lt, 8)
    fs = 64.0
    temps = [(5.0, 3.0), (20.0, -10.0), (11.3, 7.1), (31.0, -1.0), (2.0, 25.0), (32.0, 4.0)]
    vals = []
    for f0, f1 in temps:
        r = oracle.rho_series(x, fs, Lt, f0, f1)[::Lt][:nwin]   # independent windows
        vals.append(r ** 2)
    vals = np.array(vals)
    mean = vals.mean()
    # windows are independent; templates are not: use the per-template standard error
    se = vals.std(axis=1).mean() / math.sqrt(nwin)
    assert abs(mean - 2.0 / Lt) < 4 * se
    assert se < 0.02 * (2.0 / Lt)        # the check resolves 2 % of 2/L


# ---------------------------------------------------------------- P9
def test_P9_matched_injection_in_noise():
    A, f0, f1, start = 0.3, 600.0, -200.0, 1000
    hc, _ = oracle.template(FS, L, f0, f1)
    peaks, args = [], []
    for seed in range(16):
        x = np.random.default_rng(100 + seed).standard_normal(4096)
        x[start:start + L] += A * hc
        x = x.astype(np.float32)
        r = oracle.rho_series(x, FS, L, f0, f1)
        peaks.append(r[start])
        args.append(int(np.argmax(r)))
    # signal part A*sqrt(L/2), noise ~ N(0,1) per quadrature, ||x|| ~ sqrt(L(1+A^2/2))
    expect = math.sqrt(A * A * L / 2 + 2) / math.sqrt(L * (1 + A * A / 2))
    assert abs(np.mean(peaks) - expect) < 0.012          # se = 0.0216/4 = 0.0054
    assert abs(expect - A / math.sqrt(2)) < 0.01          # SURVEY: rho ~ A/sqrt(2)
    assert np.all(np.abs(np.array(args) - start) <= 8)


# ---------------------------------------------------------------- P10
def test_P10_map_by_brute_force():
    rng = np.random.default_rng(12)
    T = 500
    f0 = rng.uniform(-20, 950, T)
    rho = rng.uniform(0, 0.3, T)
    arg = rng.integers(0, 5000, T).astype(np.int32)
    kappa = 0.2
    rho[:3] = np.float32(kappa)                 # exactly at threshold: not a hit (strict)
    origin, spt, flo, df, nf, nt = 300, 128, 0.0, 1.0, 901, 32
    m, cnt = oracle.butterfly_map(f0, rho, arg, kappa, origin, spt, flo, df, nf, nt)
    ref = np.zeros((nt, nf), np.uint32)
    hits = dropped = 0
    for j in range(T):
        if rho[j] > float(np.float32(kappa)):
            hits += 1
            tb = (origin + int(arg[j])) // spt
            fb = math.floor((f0[j] - flo) / df)
            if 0 <= tb < nt and 0 <= fb < nf:
                ref[tb, fb] += 1
            else:
                dropped += 1
    np.testing.assert_array_equal(m, ref)
    assert cnt[0] == hits and cnt[1] == dropped and dropped > 0
    assert m.sum() == hits - dropped
    # accumulation: a second call adds on top
    m2, cnt2 = oracle.butterfly_map(f0, rho, arg, kappa, origin, spt, flo, df, nf, nt,
                                    m.copy(), cnt.copy())
    np.testing.assert_array_equal(m2, 2 * ref)
    assert cnt2[0] == 2 * hits


# ---------------------------------------------------------------- P11
def test_P11_chunk_plan_covers_every_valid_lag_once():
    for (N, Lt, chunk) in [(4194304, 4096, 65536), (1000, 50, 200), (1000, 50, 1000),
                           (999, 10, 64), (250, 50, 200), (65536, 4096, 65536)]:
        plan = streaming.chunk_plan(N, Lt, chunk)
        seen = np.zeros(N - Lt + 1, np.int32)
        for (start, n, lb, le) in plan:
            assert 0 <= lb <= le <= n - Lt + 1 and start + n <= N
            seen[start + lb:start + le] += 1
        assert np.all(seen == 1)
    plan = streaming.chunk_plan(4194304, 4096, 65536)
    assert len(plan) == 69 and plan[-1][1] == 16384 and plan[-1][3] == 12289
    assert all(p[3] == 61440 for p in plan[:-1])


def test_P11_chunked_max_equals_one_call():
    N, Lt, chunk = 3000, 100, 400
    x = _noise(N, 31)
    fs = 512.0
    f0 = np.array([30.0, 100.0, 200.0, 77.0])
    f1 = np.array([50.0, -40.0, 10.0, 120.0])
    whole_r, whole_a = oracle.correlate(x, fs, Lt, f0, f1)
    best = np.full(4, -1.0)
    arg = np.zeros(4, np.int64)
    for (start, n, lb, le) in streaming.chunk_plan(N, Lt, chunk):
        r, a = oracle.correlate(x[start:start + n], fs, Lt, f0, f1, lb, le)
        upd = r > best
        best[upd] = r[upd]
        arg[upd] = a[upd] + start
    np.testing.assert_array_equal(best, whole_r)
    np.testing.assert_array_equal(arg, whole_a)


def test_stream_accumulates_one_hit_per_chunk():
    N, Lt, chunk = 2000, 100, 500
    x = _noise(N, 32)
    fs = 512.0
    f0 = np.array([30.0, 100.0])
    f1 = np.array([50.0, -40.0])
    grid = dict(samples_per_tbin=32, f_lo_hz=0.0, df_hz=1.0, n_fbins=201, n_tbins=63)
    m, cnt, per_chunk = streaming.stream(x, fs, Lt, f0, f1, chunk, 0.0, grid)
    # kappa = 0: every template hits once per chunk
    assert cnt[0] == 2 * len(per_chunk) and m.sum() == cnt[0] - cnt[1]
