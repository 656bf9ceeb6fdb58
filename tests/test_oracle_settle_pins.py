"""Pins PE1-PE5 of the oracle's exponentially settling template family (reading N2 of DESIGN.md:
f(t) = f_inf + D exp(-t/tc)), PD1-PD2 of the phase
reduction modulo one turn (reading C4), and PS6 of the kappa-sigma tails on non-linear banks
(PAPER.md:70, 120).  CPU only."""
import numpy as np

import oracle
from workloads.configs import Config, Injection
from workloads.generators import make_data


# ------------------------------------------------------------------ PD: phase modulo one turn
def test_pd1_quarter_turns_are_exact():
    # (f0 = fs/2, f1 = 0): phase k/2 cycles -> cos = +-1, sin = 0 exactly, so the sine template has
    # norm exactly 0 and contributes nothing (reading C4); (fs/4, 0): the values cycle through
    # (1, 0), (0, 1), (-1, 0), (0, -1) exactly
    for fs, L in ((1024.0, 512), (4096.0, 4096), (2048.0, 2048)):
        hc, hs = oracle.template(fs, L, fs / 2, 0.0)
        assert np.array_equal(hc, np.where(np.arange(L) % 2 == 0, 1.0, -1.0))
        assert np.all(hs == 0.0)
        nc, ns = oracle.template_norms(hc, hs)
        assert ns == 0.0 and abs(nc - np.sqrt(L)) < 1e-12
        hc, hs = oracle.template(fs, L, fs / 4, 0.0)
        k = np.arange(L) % 4
        assert np.array_equal(hc, np.choose(k, [1.0, 0.0, -1.0, 0.0]))
        assert np.array_equal(hs, np.choose(k, [0.0, 1.0, 0.0, -1.0]))
    # and rho of the degenerate template is the cosine component alone
    rng = np.random.default_rng(3)
    x = rng.standard_normal(1500).astype(np.float32)
    r, c, s = oracle.rho_at(x, 1024.0, 512, 512.0, 0.0, 77, components=True)
    assert s == 0.0 and abs(r - abs(c)) < 1e-15


def test_pd2_reduced_phase_agrees_with_extended_precision():
    # the same template with the phase kept in 80-bit extended precision (numpy.longdouble on
    # x86-64) and reduced modulo one turn there: an evaluation that shares no code with the oracle
    ld = np.longdouble
    if np.finfo(ld).eps > 1e-18:
        import pytest
        pytest.skip("no extended precision on this host")
    fs, L = 4096.0, 4096
    t = np.arange(L, dtype=ld) / ld(fs)
    for f0, f1, f2 in ((2048.0, 999.5114802149488, 0.0), (700.0, -250.0, 180.0), (33.3, 0.7, 0.0)):
        cyc = ld(f0) * t + ld(0.5) * ld(f1) * t * t + ld(f2) * t * t * t / ld(6.0)
        frac = cyc - np.floor(cyc)
        two_pi = ld(2) * np.arctan2(ld(0), ld(-1))
        want_c, want_s = np.cos(two_pi * frac), np.sin(two_pi * frac)
        hc, hs = oracle.template(fs, L, f0, f1, f2)
        # float64 rounding of the phase itself: 2500 cycles * 2^-53 * 2 pi ~ 2e-12 rad
        assert np.abs(hc - want_c).max() < 5e-12 and np.abs(hs - want_s).max() < 5e-12


# ------------------------------------------------------------------ PE: the settling family
def test_pe1_slow_settling_limit_is_the_constant_tone():
    # tc -> infinity at fixed D: f(t) -> f_inf + D, i.e. the linear chirp (f0 = f_inf + D, f1 = 0);
    # residual phase D t^2 / (2 tc) = 1.5e-10 cycle at tc = 1e12 s
    fs, L = 4096.0, 4096
    a = oracle.template(fs, L, 1200.0, 300.0, 1e12, family="settle")
    b = oracle.template(fs, L, 1500.0, 0.0)
    assert np.abs(a[0] - b[0]).max() < 2e-9 and np.abs(a[1] - b[1]).max() < 2e-9
    # and D = 0 is the pure tone at f_inf whatever tc
    a = oracle.template(fs, L, 777.0, 0.0, 0.3, family="settle")
    b = oracle.template(fs, L, 777.0, 0.0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_pe2_instantaneous_frequency_settles_exponentially():
    # the frequency read off the template's own phase increments is f_inf + D exp(-t/tc) at the
    # mid-points (fixes the sign of D, the role of tc and the factor D tc in the phase)
    fs, L = 4096.0, 4096
    for f_inf, D, tc in ((1200.0, 300.0, 2.0), (1900.0, 100.0, 4.0), (500.0, -200.0, 0.5)):
        hc, hs = oracle.template(fs, L, f_inf, D, tc, family="settle")
        z = hc + 1j * hs
        f_inst = np.angle(z[1:] * np.conj(z[:-1])) * fs / (2 * np.pi)
        t_mid = (np.arange(L - 1) + 0.5) / fs
        want = f_inf + D * np.exp(-t_mid / tc)
        # mid-point rule: error = f''(t) / (24 fs^2) <= |D| / (24 tc^2 fs^2)
        assert np.abs(f_inst - want).max() < abs(D) / (24 * tc * tc * fs * fs) + 1e-7
        assert hc[0] == 1.0 and hs[0] == 0.0


def test_pe3_noise_free_injection_and_the_other_families_miss_it():
    fs, L, N, tau0 = 2048.0, 2048, 6000, 1500
    f_inf, D, tc = 600.0, 250.0, 0.7            # fast settling: far from any cubic over 1 s
    hc, hs = oracle.template(fs, L, f_inf, D, tc, family="settle")
    nc, ns = oracle.template_norms(hc, hs)
    g = float(np.dot(hc / nc, hs / ns))
    x = np.zeros(N)
    x[tau0:tau0 + L] = 1.5 * hc
    x = x.astype(np.float32)
    rho, arg = oracle.correlate(x, fs, L, [f_inf], [D], f2=[tc], family="settle")
    assert arg[0] == tau0 and abs(rho[0] - np.sqrt(1 + g * g)) < 1e-6
    series = oracle.rho_series(x, fs, L, f_inf, D, f2=tc, family="settle")
    assert int(np.argmax(series)) == tau0 and abs(series[tau0] - rho[0]) < 1e-12
    # the Taylor stand-ins at the template's first sample (reading N1) do not reach it
    f0, f1, f2 = f_inf + D, -D / tc, D / (tc * tc)
    r_lin, _ = oracle.correlate(x, fs, L, [f0], [f1])
    r_cub, _ = oracle.correlate(x, fs, L, [f0], [f1], f2=[f2])
    assert r_lin[0] < 0.5 and r_cub[0] < 0.5


def test_pe4_cubic_reading_agrees_to_the_predicted_residual():
    # settle phase = (f_inf + D) t - D t^2/(2 tc) + D t^3/(6 tc^2) - D t^4/(24 tc^3) + ...: the
    # cubic-phase template with (f0, f1, f2) = (f_inf + D, -D/tc, D/tc^2) differs from it by
    # D t^4 / (24 tc^3) cycles to leading order (alternating series: the next term bounds the error)
    fs, L = 4096.0, 4096
    t = np.arange(L) / fs
    for f_inf, D, tc in ((1200.0, 300.0, 6.0), (1200.0, 300.0, 2.0), (1800.0, 150.0, 3.0)):
        a = oracle.template(fs, L, f_inf, D, tc, family="settle")
        b = oracle.template(fs, L, f_inf + D, -D / tc, D / (tc * tc))
        dphi = np.unwrap(np.angle((b[0] + 1j * b[1]) * np.conj(a[0] + 1j * a[1]))) / (2 * np.pi)
        lead = D * t ** 4 / (24 * tc ** 3)
        nxt = D * t ** 5 / (120 * tc ** 4)
        assert np.all(dphi <= lead + 1e-9) and np.all(dphi >= lead - nxt - 1e-9)
    # 0.058 cycle at tc = 6 s, 1.56 cycles at tc = 2 s after one second (N1)
    assert abs(300.0 / (24 * 6.0 ** 3) - 0.0579) < 1e-4 and abs(300.0 / (24 * 2.0 ** 3) - 1.5625) < 1e-12


def test_pe5_matches_the_generators_settling_injection():
    # workloads.generators states the same chirp independently (numpy, phase from the integral of
    # f_inf + (f_s - f_inf) exp(-t/tau)): a settle template cut from the injected track matches
    # it with rho ~ A / sqrt(2) at the right lag, and beats every linear and cubic stand-in
    fs, L, N = 4096.0, 4096, 40000
    inj = Injection("settle", 0.4, 2.0, 8.0, 1500.0, f_inf_hz=1200.0, tau_c_s=1.5)
    cfg = Config(name="pe5", index=9, seed=99, fs_hz=fs, n_samples=N, L=L, f0_lo=0, f0_hi=1, n_f0=1,
                 f1_lo=0, f1_hi=1, n_f1=1, kappa=0.1, data_kind="gauss", injections=(inj,))
    x = make_data(cfg)
    t_off = 1.25                                   # template starts 1.25 s into the injection
    D0 = inj.f_start_hz - inj.f_inf_hz
    D = D0 * np.exp(-t_off / inj.tau_c_s)
    tau0 = int(round((inj.t_start_s + t_off) * fs))
    rho, arg = oracle.correlate(x, fs, L, [inj.f_inf_hz], [D], f2=[inj.tau_c_s], family="settle",
                                lag_begin=tau0 - 300, lag_end=tau0 + 300)
    assert abs(int(arg[0]) - tau0) <= 1 and abs(rho[0] - 0.4 / np.sqrt(2) / np.sqrt(1 + 0.08)) < 0.03
    f0, f1, f2 = inj.f_inf_hz + D, -D / inj.tau_c_s, D / inj.tau_c_s ** 2
    r_lin, _ = oracle.correlate(x, fs, L, [f0], [f1], lag_begin=tau0 - 300, lag_end=tau0 + 300)
    r_cub, _ = oracle.correlate(x, fs, L, [f0], [f1], f2=[f2], lag_begin=tau0 - 300, lag_end=tau0 + 300)
    assert rho[0] > r_cub[0] + 0.02 and rho[0] > r_lin[0] + 0.1


# ------------------------------------------------------------------ PS6: tails on non-linear banks
def _unit(hc, hs):
    nc, ns = oracle.template_norms(hc, hs)
    return hc / nc, hs / ns


def test_ps6_sigma_and_tails_for_curved_and_settling_templates():
    rng = np.random.default_rng(21)
    fs, L, N = 512.0, 128, 1000
    x = (rng.standard_normal(N) + 0.3 * np.sin(np.arange(N) * 0.21)).astype(np.float32)
    cases = [("poly", 40.0, 55.0, 300.0), ("poly", 200.0, -120.0, -500.0), ("settle", 60.0, 90.0, 0.2)]
    X = np.fft.fft(x.astype(np.float64))
    for fam, a, b, c in cases:
        hc, hs = _unit(*oracle.template(fs, L, a, b, c, family=fam))
        # Parseval with numpy's FFT (PS1 on a non-linear template)
        Hc, Hs = np.fft.fft(hc, N), np.fft.fft(hs, N)
        pred = np.sqrt(np.sum(np.abs(X) ** 2 * (np.abs(Hc) ** 2 + np.abs(Hs) ** 2)) / (2.0 * N * N))
        assert abs(oracle.sigma(x, fs, L, a, b, c, family=fam) / pred - 1.0) < 1e-12
    # brute force with circular indexing (PS2 on a curved template)
    fs, L, N = 64.0, 16, 50
    x = rng.standard_normal(N).astype(np.float32)
    hc, hs = _unit(*oracle.template(fs, L, 9.0, 4.0, 30.0))
    acc = 0.0
    for tau in range(N):
        cc = sum(float(x[(tau + k) % N]) * hc[k] for k in range(L))
        ss = sum(float(x[(tau + k) % N]) * hs[k] for k in range(L))
        acc += cc * cc + ss * ss
    assert abs(oracle.sigma(x, fs, L, 9.0, 4.0, 30.0) - np.sqrt(acc / (2 * N))) < 1e-13
    # f2 = 0 is the linear function bit for bit, hits included
    fs, L, N = 1024.0, 256, 3000
    x = rng.standard_normal(N).astype(np.float32)
    f0, f1 = np.array([100.0, 150.0, 333.0]), np.array([60.0, -70.0, 5.0])
    lin = oracle.tails(x, fs, L, f0, f1, 3.0)
    zer = oracle.tails(x, fs, L, f0, f1, 3.0, f2=np.zeros(3))
    assert all(np.array_equal(p, q) for p, q in zip(lin[:4], zer[:4])) and lin[4] == zer[4]
    # the hits of a curved bank are exactly where the pinned series rho ||x_tau|| / sigma exceeds kappa
    f2 = np.array([400.0, -250.0, 90.0])
    hc, _ = oracle.template(fs, L, f0[0], f1[0], f2[0])
    x[700:700 + L] += (0.5 * hc).astype(np.float32)
    sig, hj, hl, hr, total = oracle.tails(x, fs, L, f0, f1, 3.0, 10, 2500, f2=f2)
    n2 = oracle.sliding_n2(x, L, 10, 2500)
    want = []
    for j in range(3):
        assert sig[j] == oracle.sigma(x, fs, L, f0[j], f1[j], f2[j])
        r = oracle.rho_series(x, fs, L, f0[j], f1[j], 10, 2500, f2=f2[j]) * np.sqrt(n2) / sig[j]
        want += [(j, 10 + int(i)) for i in np.nonzero(r > 3.0)[0]]
    assert want == list(zip(hj.tolist(), hl.tolist())) and total == len(want) > 0
    assert 700 in hl[hj == 0]
