"""GPU parity of the control / coincidence / pseudo-spectrum calls (
PAPER.md:68, 124; readings T1-T3) against oracle/coincidence.py: integer and gather work,
bit-exact.  Needs a B200."""
import numpy as np
import pytest

from oracle import coincidence as oc
from workloads import permutation

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def bfly():
    import paper_1802_01685_b200 as b
    return b


@pytest.mark.parametrize("n", [1, 257, 65536, 1_000_003])
def test_time_randomize_is_the_gather(bfly, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n).astype(np.float32)
    p = permutation(n, 7)
    y, bad = bfly.time_randomize(torch.from_numpy(x).cuda(), torch.from_numpy(p).cuda())
    assert int(bad.item()) == 0
    np.testing.assert_array_equal(y.cpu().numpy(), x[p] if n > 5000 else oc.time_randomize(x, p))
    if n > 1:
        p2 = p.copy()
        p2[0] = n                                       # out of range: flagged, written as 0
        y2, bad2 = bfly.time_randomize(torch.from_numpy(x).cuda(), torch.from_numpy(p2).cuda())
        assert int(bad2.item()) == 1 and float(y2[0]) == 0.0


@pytest.mark.parametrize("nt,nf,w", [(1, 1, 0), (5, 33, 2), (40, 2049, 50), (16, 901, 0), (3, 70, 5000),
                                     (300, 129, 7)])
def test_coincidence_and_pseudo_spectrum_match_the_oracle(bfly, nt, nf, w):
    rng = np.random.default_rng(nt * 1000 + nf)
    m1 = ((rng.random((nt, nf)) < 0.03) * rng.integers(1, 5, (nt, nf))).astype(np.uint32)
    m2 = ((rng.random((nt, nf)) < 0.02) * rng.integers(1, 3, (nt, nf))).astype(np.uint32)
    d1 = torch.from_numpy(m1.view(np.int32)).cuda()
    d2 = torch.from_numpy(m2.view(np.int32)).cuda()
    c1, c2 = bfly.coincidence(d1, d2, w)
    o1, o2 = oc.coincidence(m1, m2, w)
    np.testing.assert_array_equal(c1.cpu().numpy().view(np.uint32), o1)
    np.testing.assert_array_equal(c2.cpu().numpy().view(np.uint32), o2)
    s = bfly.pseudo_spectrum(d1)
    s = bfly.pseudo_spectrum(d2, s)                     # accumulates
    want = oc.pseudo_spectrum(m1) + oc.pseudo_spectrum(m2)
    np.testing.assert_array_equal(s.cpu().numpy().view(np.uint64), want)
    big = np.full((3, 2), 4_000_000_000, np.uint32)
    sb = bfly.pseudo_spectrum(torch.from_numpy(big.view(np.int32)).cuda())
    assert sb.cpu().numpy().view(np.uint64).tolist() == [12_000_000_000, 12_000_000_000]


def test_control_and_coincidence_end_to_end(bfly):
    """The paper's reading of two detectors through the CUDA path: two series
    sharing one long ascending chirp (independent noise), their kappa-sigma hit maps, the
    simultaneous counts within 50 Hz, and the time-randomised controls.  Every integer step
    equals the oracle's on the GPU's own maps; the shared chirp shows in the simultaneous
    pseudo-spectrum of the data and not in that of the control."""
    fs, L, N = 4096.0, 4096, 65536
    t = np.arange(N) / fs
    chirp = 0.25 * np.cos(2 * np.pi * (500.0 * t + 0.5 * 40.0 * t * t))     # 500 -> 1140 Hz in 16 s
    rng = np.random.default_rng(99)
    series = [(rng.standard_normal(N) + chirp).astype(np.float32) for _ in range(2)]
    starts = np.arange(0.0, 15.0, 0.25)                                     # 1-s pieces of the track
    f0 = np.concatenate([500.0 + 40.0 * starts, rng.uniform(100, 1900, 40)])
    f1 = np.concatenate([np.full(len(starts), 40.0), rng.uniform(-400, 400, 40)])
    bank = bfly.make_bank(fs, L, f0, f1)
    grid = dict(samples_per_tbin=256, f_lo_hz=0.0, df_hz=1.0, n_fbins=2049, n_tbins=N // 256)
    kappa = 4.5
    maps = {}
    for name, x in zip("hl", series):
        xd = torch.from_numpy(x).cuda()
        for ctrl in (False, True):
            if ctrl:
                xd_use, bad = bfly.time_randomize(xd, torch.from_numpy(permutation(N, 5 + ord(name))).cuda())
                assert int(bad.item()) == 0
            else:
                xd_use = xd
            sig, hj, hl, hr, n = bfly.tails(bank, xd_use, kappa, 1 << 20)
            total = int(n.item())
            assert total < (1 << 20)
            m, c = bfly.hits_map(bank, hj, hl, total, 0, **grid)
            assert int(c[0]) == total
            maps[(name, ctrl)] = m
    co = {}
    for ctrl in (False, True):
        m1, m2 = maps[("h", ctrl)], maps[("l", ctrl)]
        c1, c2 = bfly.coincidence(m1, m2, 50)
        o1, o2 = oc.coincidence(m1.cpu().numpy().view(np.uint32), m2.cpu().numpy().view(np.uint32), 50)
        np.testing.assert_array_equal(c1.cpu().numpy().view(np.uint32), o1)
        np.testing.assert_array_equal(c2.cpu().numpy().view(np.uint32), o2)
        s1 = bfly.pseudo_spectrum(c1).cpu().numpy().view(np.uint64)
        np.testing.assert_array_equal(s1, oc.pseudo_spectrum(o1))
        co[ctrl] = int(s1.sum())
    assert co[False] > 50 and co[False] > 5 * max(co[True], 1)
