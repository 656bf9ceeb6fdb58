"""Pins PS1-PS5 of the oracle's kappa-sigma tails (oracle.sigma, oracle.tails; readings S1-S3
of DESIGN.md).  CPU only."""
import numpy as np

import oracle


def _norm_templates(fs, L, f0, f1):
    hc, hs = oracle.template(fs, L, f0, f1)
    nc, ns = oracle.template_norms(hc, hs)
    return hc / nc, hs / ns


def test_ps1_sigma_equals_parseval_prediction():
    # sigma^2 = (1 / (2 N^2)) sum_m |X[m]|^2 (|Hc[m]|^2 + |Hs[m]|^2): Parseval's theorem applied to
    # the circular correlation, with numpy's FFT (the paper's predictor step)
    rng = np.random.default_rng(11)
    fs, L, N = 512.0, 128, 1000                      # N not a power of two, L < N
    x = (rng.standard_normal(N) + 0.3 * np.sin(np.arange(N) * 0.21)).astype(np.float32)
    for f0, f1 in ((40.0, 55.0), (200.0, -120.0), (13.0, 0.0)):
        hc, hs = _norm_templates(fs, L, f0, f1)
        X = np.fft.fft(x.astype(np.float64))
        Hc, Hs = np.fft.fft(hc, N), np.fft.fft(hs, N)
        pred = np.sqrt(np.sum(np.abs(X) ** 2 * (np.abs(Hc) ** 2 + np.abs(Hs) ** 2)) / (2.0 * N * N))
        assert abs(oracle.sigma(x, fs, L, f0, f1) / pred - 1.0) < 1e-12


def test_ps2_sigma_by_brute_force_python_loop():
    rng = np.random.default_rng(12)
    fs, L, N = 64.0, 16, 50
    x = rng.standard_normal(N).astype(np.float32)
    hc, hs = _norm_templates(fs, L, 9.0, 4.0)
    acc = 0.0
    for tau in range(N):
        c = sum(float(x[(tau + k) % N]) * hc[k] for k in range(L))
        s = sum(float(x[(tau + k) % N]) * hs[k] for k in range(L))
        acc += c * c + s * s
    assert abs(oracle.sigma(x, fs, L, 9.0, 4.0) - np.sqrt(acc / (2 * N))) < 1e-13


def test_ps3_white_noise_sigma_is_the_data_rms():
    # unit-norm templates: for white data sum_tau c~^2 = sum_d R_x[d] A_h[d] ~ R_x[0] A_h[0] = ||x||^2
    rng = np.random.default_rng(13)
    fs, L, N = 2048.0, 2048, 16384
    x = (1.7 * rng.standard_normal(N)).astype(np.float32)
    rms = np.sqrt(np.mean(x.astype(np.float64) ** 2))
    for f0, f1 in ((300.0, 100.0), (700.0, -250.0)):
        assert abs(oracle.sigma(x, fs, L, f0, f1) / rms - 1.0) < 0.1


def test_ps4_pure_tone_closed_form():
    # x = cos(w n), template f1 = 0 at the same integer frequency, L = fs, N = 4 L:
    # c~ = sqrt(L/2) cos(w tau), s~ = -sqrt(L/2) sin(w tau)  =>  sigma = sqrt(L)/2 and
    # rho_sigma = sqrt(2) at every lag: every valid lag is a hit below sqrt 2, none above
    fs, L, N, f = 256.0, 256, 1024, 19.0
    x = np.cos(2 * np.pi * f * np.arange(N) / fs).astype(np.float32)
    assert abs(oracle.sigma(x, fs, L, f, 0.0) - np.sqrt(L) / 2) < 1e-5
    sig, hj, hl, hr, total = oracle.tails(x, fs, L, [f], [0.0], 1.41)
    assert total == N - L + 1 and np.array_equal(hl, np.arange(N - L + 1))
    assert np.abs(hr - np.sqrt(2.0)).max() < 1e-5
    assert oracle.tails(x, fs, L, [f], [0.0], 1.42)[4] == 0


def test_ps5_tails_against_the_pinned_series_and_scale_invariance():
    # the hits are exactly the lags where the (already pinned) series rho(tau) ||x_tau|| / sigma
    # exceeds kappa; scaling the data leaves the hits unchanged and scales sigma
    rng = np.random.default_rng(15)
    fs, L, N = 1024.0, 256, 3000
    x = rng.standard_normal(N).astype(np.float32)
    hc, _ = oracle.template(fs, L, 100.0, 60.0)
    x[700:700 + L] += (0.5 * hc).astype(np.float32)
    f0, f1 = np.array([100.0, 150.0, 333.0]), np.array([60.0, -70.0, 5.0])
    kappa = 3.0
    sig, hj, hl, hr, total = oracle.tails(x, fs, L, f0, f1, kappa, 10, 2500)
    assert total == len(hj) > 0
    n2 = oracle.sliding_n2(x, L, 10, 2500)
    want = []
    for j in range(3):
        assert abs(sig[j] - oracle.sigma(x, fs, L, f0[j], f1[j])) == 0.0
        r = oracle.rho_series(x, fs, L, f0[j], f1[j], 10, 2500) * np.sqrt(n2) / sig[j]
        for i in np.nonzero(r > kappa)[0]:
            want.append((j, 10 + int(i), r[i]))
    assert [(a, b) for a, b, _ in want] == list(zip(hj.tolist(), hl.tolist()))
    assert np.abs(np.array([w[2] for w in want]) - hr).max() < 1e-12
    assert 700 in hl[hj == 0]                       # the injected chirp is found at its start
    xs = (x * np.float32(64.0)).astype(np.float32)  # power of two: exact
    sig2, hj2, hl2, hr2, total2 = oracle.tails(xs, fs, L, f0, f1, kappa, 10, 2500)
    assert np.allclose(sig2, 64.0 * sig, rtol=1e-13) and np.array_equal(hl2, hl) and np.array_equal(hj2, hj)
    # capacity smaller than the number of hits: the first `capacity` in (template, lag) order
    _, hj3, hl3, _, total3 = oracle.tails(x, fs, L, f0, f1, kappa, 10, 2500, capacity=5)
    assert total3 == total and np.array_equal(hl3, hl[:5]) and np.array_equal(hj3, hj[:5])
    # an all-zero segment has sigma = 0 and no hits (S3)
    z = np.zeros(N, np.float32)
    sig0, _, _, _, t0 = oracle.tails(z, fs, L, f0, f1, kappa)
    assert t0 == 0 and np.all(sig0 == 0.0)
