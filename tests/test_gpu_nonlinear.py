"""GPU parity of the non-linear template family (bfly_make_bank3; reading N1)
in every correlation form against the float64 oracle (R1, R2).  Needs a B200."""
import numpy as np
import pytest

import oracle

from parity import check_values_and_argmax

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

FORMS = [pytest.param(3, id="fft_tc"), pytest.param(5, id="fft_tc5"), pytest.param(4, id="dense_tc"),
         pytest.param(1, id="fft"), pytest.param(2, id="direct")]


@pytest.fixture(scope="module")
def bfly():
    import paper_1802_01685_b200 as b
    return b


def _settling(fs, L, f_inf, delta, tc, t0):
    """(f0, f1, f2) of f(t) = f_inf + delta exp(-t / tc) at time t0 (the template's first sample)."""
    e = delta * np.exp(-t0 / tc)
    return f_inf + e, -e / tc, e / (tc * tc)


@pytest.mark.parametrize("form", FORMS)
def test_curved_chirps_match_the_oracle(bfly, form):
    rng = np.random.default_rng(41)
    fs, L, N = 4096.0, 4096, 20000
    x = rng.standard_normal(N)
    # an exponentially settling descending chirp 1500 -> 1200 Hz, tc = 6 s, from sample 3000 on
    # (cubic-phase residual over one template: delta / (24 tc^3) = 0.06 cycle)
    t = np.arange(N - 3000) / fs
    x[3000:] += 0.2 * np.cos(2 * np.pi * (1200.0 * t + 300.0 * 6.0 * (1 - np.exp(-t / 6.0))))
    x = x.astype(np.float32)
    # templates along the track (frequency, slope, curvature at their start) + random curved ones
    starts = np.arange(0.0, 3.0, 0.5)
    tr = np.array([_settling(fs, L, 1200.0, 300.0, 6.0, s) for s in starts])
    f0 = np.concatenate([tr[:, 0], rng.uniform(100, 1900, 31)])
    f1 = np.concatenate([tr[:, 1], rng.uniform(-400, 400, 31)])
    f2 = np.concatenate([tr[:, 2], rng.uniform(-500, 500, 31)])
    bank = bfly.make_bank(fs, L, f0, f1, f2_hzps2=f2)
    np.testing.assert_array_equal(bank.get_f2(), f2)
    xd = torch.from_numpy(x).cuda()
    rho, arg = bfly.correlate_form(bank, form, xd)
    torch.cuda.synchronize()
    rho_n, arg_n = rho.cpu().numpy(), arg.cpu().numpy()
    rho_o, arg_o, _ = check_values_and_argmax(x, fs, L, f0, f1, rho_n, arg_n, f2=f2)
    # the curved templates on the track find the chirp near their start (the peak is broad along
    # the track: a shift of d samples is a mismatch of only slope x d / fs in frequency); the same
    # (f0, f1) without curvature does worse
    for i, s in enumerate(starts[:3]):
        assert arg_n[i] == arg_o[i] and abs(int(arg_n[i]) - (3000 + int(s * fs))) <= 64 and rho_n[i] > 0.11
    lin = bfly.make_bank(fs, L, f0[:3], f1[:3])
    rl, _ = bfly.correlate_form(lin, form, xd)
    assert np.all(rl.cpu().numpy() < rho_n[:3])


def test_f2_zero_bank_equals_the_linear_bank_bit_for_bit(bfly):
    rng = np.random.default_rng(42)
    fs, L, N = 2048.0, 2048, 9000
    x = torch.from_numpy(rng.standard_normal(N).astype(np.float32)).cuda()
    f0, f1 = rng.uniform(100, 900, 50), rng.uniform(-300, 300, 50)
    a = bfly.make_bank(fs, L, f0, f1)
    b = bfly.make_bank(fs, L, f0, f1, f2_hzps2=np.zeros(50))
    for form in (3, 4, 1, 2):
        ra, aa = bfly.correlate_form(a, form, x)
        rb, ab = bfly.correlate_form(b, form, x)
        assert torch.equal(ra, rb) and torch.equal(aa, ab)
    with pytest.raises(bfly.BflyError):
        bfly.make_bank(fs, L, f0, f1, f2_hzps2=np.full(50, np.nan))
