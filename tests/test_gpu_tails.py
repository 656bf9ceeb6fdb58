"""GPU parity of the kappa-sigma tails (bfly_tails, bfly_hits_map; SURVEY 8(f) rank 2,
PAPER.md:70, 120) against the float64 oracle: rule R5 of DESIGN.md.  Needs a B200."""
import numpy as np
import pytest

import oracle
from workloads import bank_grid, default_map_grid, get_config, make_data, sub_bank_indices

from parity import check_tails

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def bfly():
    import paper_1802_01685_b200 as b
    return b


def _tails(bfly, fs, L, f0, f1, x, kappa, capacity, lb=0, le=None, f2=None):
    bank = bfly.make_bank(fs, L, f0, f1, f2_hzps2=f2)
    xd = torch.from_numpy(x).cuda()
    sig, hj, hl, hr, n = bfly.tails(bank, xd, kappa, capacity, lb, le)
    torch.cuda.synchronize()
    total = int(n.item())
    k = min(total, capacity)
    return bank, sig.cpu().numpy(), hj.cpu().numpy()[:k], hl.cpu().numpy()[:k], hr.cpu().numpy()[:k], total, (hj, hl)


def test_tails_small_segment_with_injection(bfly):
    rng = np.random.default_rng(21)
    fs, L, N = 2048.0, 2048, 12000
    x = rng.standard_normal(N)
    f0 = np.concatenate([[600.0], rng.uniform(100, 900, 39)])
    f1 = np.concatenate([[-200.0], rng.uniform(-300, 300, 39)])
    hc, _ = oracle.template(fs, L, 600.0, -200.0)
    x[3000:3000 + L] += 0.25 * hc
    x = x.astype(np.float32)
    kappa = 3.6
    bank, sig, hj, hl, hr, total, dev = _tails(bfly, fs, L, f0, f1, x, kappa, 1 << 16)
    n_oracle, n_border = check_tails(x, fs, L, f0, f1, kappa, sig, hj, hl, hr, total)
    assert n_oracle > 50 and 3000 in hl[hj == 0]
    # the map of the hit list = the histogram of the list (integer, exact)
    grid = dict(samples_per_tbin=128, f_lo_hz=0.0, df_hz=1.0, n_fbins=1001, n_tbins=(N + 127) // 128)
    m, c = bfly.hits_map(bank, dev[0], dev[1], total, 77, **grid)
    want = np.zeros((grid["n_tbins"], grid["n_fbins"]), np.uint32)
    dropped = 0
    for j, lag in zip(hj, hl):
        tb, fb = (77 + int(lag)) // 128, int(np.floor(f0[j]))
        if tb < grid["n_tbins"] and 0 <= fb < grid["n_fbins"]:
            want[tb, fb] += 1
        else:
            dropped += 1
    np.testing.assert_array_equal(m.cpu().numpy().view(np.uint32), want)
    assert c.cpu().numpy().tolist() == [total, dropped]
    # determinism of the SET of hits, and the overflow rule: the count still counts everything
    _, sig2, hj2, hl2, hr2, total2, _ = _tails(bfly, fs, L, f0, f1, x, kappa, 1 << 16)
    assert total2 == total and np.array_equal(sig2, sig)
    assert sorted(zip(hj2.tolist(), hl2.tolist(), hr2.tolist())) == sorted(zip(hj.tolist(), hl.tolist(), hr.tolist()))
    _, _, hj3, hl3, _, total3, _ = _tails(bfly, fs, L, f0, f1, x, kappa, 10)
    assert total3 == total and len(hj3) == 10
    assert set(zip(hj3.tolist(), hl3.tolist())) <= set(zip(hj.tolist(), hl.tolist()))


@pytest.mark.parametrize("index,n_random,kappa", [(4, 24, 4.0), (3, 16, 3.8), (2, 12, 4.2)])
def test_tails_sub_bank_of_config(bfly, index, n_random, kappa):
    cfg = get_config(index)
    n = 65536 if index == 2 else None                # one 16-s segment of the 32-s series
    x = make_data(cfg, n)
    f0a, f1a = bank_grid(cfg)
    idx = sub_bank_indices(cfg, n_random, max_track=8)
    f0, f1 = f0a[idx], f1a[idx]
    bank, sig, hj, hl, hr, total, _ = _tails(bfly, cfg.fs_hz, cfg.L, f0, f1, x, kappa, 1 << 18)
    n_oracle, _ = check_tails(x, cfg.fs_hz, cfg.L, f0, f1, kappa, sig, hj, hl, hr, total)
    assert n_oracle > 0


def test_tails_on_a_cubic_phase_bank(bfly):
    """bfly_tails on a bfly_make_bank3 bank (tc_correlate_kernel<TAILS, CUBIC>): the kappa-sigma
    reduction applies to whatever bank is searched.  R5 against oracle.sigma /
    oracle.rho_series with f2; a curved injection is found at its start by its own template."""
    rng = np.random.default_rng(27)
    fs, L, N = 2048.0, 2048, 12000
    x = rng.standard_normal(N)
    f0 = np.concatenate([[700.0], rng.uniform(100, 900, 29)])
    f1 = np.concatenate([[-250.0], rng.uniform(-300, 300, 29)])
    f2 = np.concatenate([[400.0], rng.uniform(-600, 600, 29)])
    hc, _ = oracle.template(fs, L, f0[0], f1[0], f2[0])
    x[5000:5000 + L] += 0.25 * hc
    x = x.astype(np.float32)
    kappa = 3.6
    for lb, le in ((0, None), (1000, 1000 + 2 * 4096 + 3)):
        _, sig, hj, hl, hr, total, _ = _tails(bfly, fs, L, f0, f1, x, kappa, 1 << 16, lb, le, f2=f2)
        n_oracle, _ = check_tails(x, fs, L, f0, f1, kappa, sig, hj, hl, hr, total, lb,
                                  le, f2=f2)
        assert n_oracle > 30 and 5000 in hl[hj == 0]
    # f2 = 0 for every template: the cubic bank's tails are those of the linear bank, bit for bit
    _, sa, ja, la, ra, ta, _ = _tails(bfly, fs, L, f0, f1, x, kappa, 1 << 16)
    _, sb, jb, lb_, rb, tb, _ = _tails(bfly, fs, L, f0, f1, x, kappa, 1 << 16, f2=np.zeros(30))
    assert ta == tb and np.array_equal(sa, sb)
    assert sorted(zip(ja.tolist(), la.tolist(), ra.tolist())) == sorted(zip(jb.tolist(), lb_.tolist(), rb.tolist()))


def test_tails_cubic_bank_one_paper_scale_segment(bfly):
    """One config-4-sized segment (65536 samples, L = 4096, 15 blocks + the 61441st lag) against a
    cubic-phase sub-bank: R5."""
    cfg = get_config(4)
    x = make_data(cfg)
    rng = np.random.default_rng(28)
    f0a, f1a = bank_grid(cfg)
    idx = sub_bank_indices(cfg, 10, max_track=4)
    f0, f1 = f0a[idx], f1a[idx]
    f2 = rng.uniform(-400, 400, len(idx))
    _, sig, hj, hl, hr, total, _ = _tails(bfly, cfg.fs_hz, cfg.L, f0, f1, x, 4.0, 1 << 18, f2=f2)
    n_oracle, _ = check_tails(x, cfg.fs_hz, cfg.L, f0, f1, 4.0, sig, hj, hl, hr, total, f2=f2)
    assert n_oracle > 0


def test_tails_lag_subrange_scale_and_edges(bfly):
    rng = np.random.default_rng(23)
    fs, L, N = 1024.0, 512, 20000
    x = rng.standard_normal(N).astype(np.float32)
    f0, f1 = rng.uniform(50, 450, 9), rng.uniform(-150, 150, 9)
    for lb, le in ((0, N - L + 1), (1234, 9000), (17, 17 + 4096), (17, 17 + 4097), (17, 17 + 8192 + 4), (500, 501)):
        _, sig, hj, hl, hr, total, _ = _tails(bfly, fs, L, f0, f1, x, 3.5, 1 << 16, lb, le)
        check_tails(x, fs, L, f0, f1, 3.5, sig, hj, hl, hr, total, lb, le)
    xs = (x * np.float32(4096.0)).astype(np.float32)          # rho_sigma is scale invariant
    _, sig_s, hj_s, hl_s, hr_s, total_s, _ = _tails(bfly, fs, L, f0, f1, xs, 3.5, 1 << 16)
    check_tails(xs, fs, L, f0, f1, 3.5, sig_s, hj_s, hl_s, hr_s, total_s)
    z = np.zeros(N, np.float32)                               # S3: sigma = 0, no hits
    _, sig0, hj0, _, _, total0, _ = _tails(bfly, fs, L, f0, f1, z, 3.5, 16)
    assert total0 == 0 and np.all(sig0 == 0.0)
    with pytest.raises(bfly.BflyError):                       # needs L >= BFLY_TC_MIN_L
        _tails(bfly, 512.0, 64, [50.0], [1.0], x, 3.5, 16)
    with pytest.raises(bfly.BflyError):                       # kappa must be > 0
        _tails(bfly, fs, L, f0, f1, x, 0.0, 16)


@pytest.mark.parametrize("fs,L", [(1024.0, 512), (4096.0, 4096)])
def test_tails_hits_on_the_lags_past_the_last_whole_block(bfly, fs, L):
    """n_lags = 4096 + r: the last r lags come from the rows delta >= 8 of the last block's transform
    (L = 512: all r; L = 4096: r = 1) or from direct sums; a chirp injected there makes them hits."""
    rng = np.random.default_rng(int(L))
    f0, f1 = rng.uniform(0.05 * fs, 0.4 * fs, 7), rng.uniform(-0.1 * fs, 0.1 * fs, 7)
    for r in (1, 2, 4):
        lb, n_lags = 23, 4096 + r
        N = lb + n_lags + L - 1 + 5
        x = rng.standard_normal(N)
        hc, _ = oracle.template(fs, L, f0[2], f1[2])
        x[lb + n_lags - 1:lb + n_lags - 1 + L] += 0.6 * hc
        x = x.astype(np.float32)
        _, sig, hj, hl, hr, total, _ = _tails(bfly, fs, L, f0, f1, x, 4.0, 1 << 16, lb, lb + n_lags)
        check_tails(x, fs, L, f0, f1, 4.0, sig, hj, hl, hr, total, lb, lb + n_lags)
        assert np.any((hj == 2) & (hl == lb + n_lags - 1))


def test_tails_full_bank_config4_sampled_against_the_oracle(bfly):
    """bfly_tails over BASELINE.json's paper-scale bank (2^23 templates x 61441 lags, kappa = 5.5:
    ~1.5e5 hits, the launch bench.py times): the hit list of sampled templates -- half of them
    drawn from the templates that have hits, half from those that have none -- against the oracle
    (R5), sigma included; no duplicate (template, lag) in the whole list; a sub-bank run of the same
    templates gives the same sigmas and hits bit for bit (R4)."""
    cfg = get_config(4)
    x = make_data(cfg)
    xd = torch.from_numpy(x).cuda()
    full = bfly.make_bank_grid(cfg.fs_hz, cfg.L, cfg.f0_lo, cfg.f0_hi, cfg.n_f0, cfg.f1_lo, cfg.f1_hi, cfg.n_f1)
    kappa, cap = 5.5, 1 << 22
    sig, hj, hl, hr, n = bfly.tails(full, xd, kappa, cap)
    torch.cuda.synchronize()
    total = int(n.item())
    assert 0 < total < cap
    hj_n, hl_n, hr_n = hj.cpu().numpy()[:total], hl.cpu().numpy()[:total], hr.cpu().numpy()[:total]
    key = hj_n.astype(np.int64) * (1 << 20) + hl_n
    assert len(np.unique(key)) == total                      # no duplicates anywhere
    assert np.all((hl_n >= 0) & (hl_n < cfg.n_lags)) and np.all(hr_n > kappa)
    rng = np.random.default_rng(44)
    with_hits = np.unique(hj_n)
    mask = np.ones(len(full), bool)
    mask[with_hits] = False
    without = np.nonzero(mask)[0]
    idx = np.sort(np.concatenate([rng.choice(with_hits, 60, replace=False), rng.choice(without, 60, replace=False),
                                  [0, len(full) - 1]]))
    idx = np.unique(idx)
    f0a, f1a = bank_grid(cfg)
    pos = {int(j): i for i, j in enumerate(idx)}
    sel = np.isin(hj_n, idx)
    sub_j = np.array([pos[int(j)] for j in hj_n[sel]], np.int32)
    sig_n = sig.cpu().numpy()
    n_or, n_border = check_tails(x, cfg.fs_hz, cfg.L, f0a[idx], f1a[idx], kappa, sig_n[idx], sub_j, hl_n[sel],
                                 hr_n[sel], int(sel.sum()))
    print(f"tails, config 4 full bank: {total} hits; {len(idx)} sampled templates: {int(sel.sum())} gpu hits, "
          f"{n_or} oracle hits, {n_border} within tolerance of kappa")
    sub = bfly.make_bank(cfg.fs_hz, cfg.L, f0a[idx], f1a[idx])
    sig2, hj2, hl2, hr2, n2 = bfly.tails(sub, xd, kappa, 1 << 16)
    torch.cuda.synchronize()
    t2 = int(n2.item())
    assert np.array_equal(sig2.cpu().numpy(), sig_n[idx]) and t2 == int(sel.sum())
    a = sorted(zip(sub_j.tolist(), hl_n[sel].tolist(), hr_n[sel].tolist()))
    b = sorted(zip(hj2.cpu().numpy()[:t2].tolist(), hl2.cpu().numpy()[:t2].tolist(), hr2.cpu().numpy()[:t2].tolist()))
    assert a == b
