"""Pins PN1-PN4 of the oracle's non-linear template family (reading N1 of DESIGN.md: constant
second frequency derivative f2).  CPU only."""
import numpy as np

import oracle


def test_pn1_f2_zero_is_the_linear_chirp_bit_for_bit():
    for f0, f1 in ((600.0, -200.0), (20.0, 1000.0)):
        a = oracle.template(4096.0, 4096, f0, f1)
        b = oracle.template(4096.0, 4096, f0, f1, 0.0)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_pn2_instantaneous_frequency_is_the_quadratic():
    # the frequency read off the template itself -- the phase increment of hc + i hs between
    # neighbouring samples -- equals f0 + f1 t + f2 t^2 / 2 at the mid-points (fixes the factors
    # 1/2 and 1/6 and the sign of every term without retyping the phase formula)
    fs, L = 4096.0, 4096
    for f0, f1, f2 in ((700.0, -250.0, 180.0), (300.0, 90.0, -400.0), (1500.0, -60.0, 25.0)):
        hc, hs = oracle.template(fs, L, f0, f1, f2)
        z = hc + 1j * hs
        dphi = np.angle(z[1:] * np.conj(z[:-1]))              # in (-pi, pi): f < fs/2
        t_mid = (np.arange(L - 1) + 0.5) / fs
        f_inst = dphi * fs / (2 * np.pi)
        want = f0 + f1 * t_mid + 0.5 * f2 * t_mid ** 2
        # the mid-point rule is exact up to the third derivative of the phase: f2 / (24 fs^2)
        assert np.abs(f_inst - want).max() < abs(f2) / (24 * fs * fs) + 1e-7
        assert abs(hc[0] - 1.0) < 1e-15 and abs(hs[0]) < 1e-15   # phase zero at the first sample


def test_pn3_noise_free_injection_of_a_curved_chirp():
    fs, L, N, tau0 = 2048.0, 2048, 6000, 1234
    f0, f1, f2 = 500.0, -150.0, 220.0
    hc, hs = oracle.template(fs, L, f0, f1, f2)
    nc, ns = oracle.template_norms(hc, hs)
    g = float(np.dot(hc / nc, hs / ns))
    x = np.zeros(N)
    x[tau0:tau0 + L] = 2.5 * hc
    x = x.astype(np.float32)
    rho, arg = oracle.correlate(x, fs, L, [f0, f0], [f1, f1], f2=[f2, 0.0])
    assert arg[0] == tau0 and abs(rho[0] - np.sqrt(1 + g * g)) < 1e-6
    assert rho[1] < 0.5                                       # the linear chirp does not match it
    series = oracle.rho_series(x, fs, L, f0, f1, f2=f2)
    assert int(np.argmax(series)) == tau0 and abs(series[tau0] - rho[0]) < 1e-12


def test_pn4_time_reversal_maps_the_family_onto_itself():
    # x'[n] = x[N-1-n]: rho_{(f0, f1, f2)}(x, tau) = rho_{(f(T), -f'(T), f2)}(x', N - L - tau) with
    # T = (L-1)/fs, f(T) = f0 + f1 T + f2 T^2/2, f'(T) = f1 + f2 T (exact up to the quadrature
    # pair's non-orthogonality, as pin P3)
    rng = np.random.default_rng(31)
    fs, L, N = 2048.0, 2048, 5000
    x = rng.standard_normal(N).astype(np.float32)
    xr = np.ascontiguousarray(x[::-1])
    T = (L - 1) / fs
    for f0, f1, f2 in ((400.0, 120.0, -90.0), (800.0, -200.0, 150.0)):
        a = oracle.rho_series(x, fs, L, f0, f1, f2=f2)
        b = oracle.rho_series(xr, fs, L, f0 + f1 * T + 0.5 * f2 * T * T, -(f1 + f2 * T), f2=f2)
        assert np.abs(a - b[::-1]).max() < 5e-5
        wrong = oracle.rho_series(xr, fs, L, f0 + f1 * T + 0.5 * f2 * T * T, -(f1 + f2 * T), f2=-f2)
        assert np.abs(a - wrong[::-1]).max() > 1e-3          # a wrong sign of f2 fails
