"""Pins PC1-PC4 of oracle/coincidence.py (readings T1-T3).  CPU only."""
import numpy as np
import pytest

from oracle import coincidence as oc
from workloads import permutation


def test_pc1_time_randomisation_keeps_the_histogram_and_is_seeded():
    rng = np.random.default_rng(1)
    x = rng.standard_normal(1000).astype(np.float32)
    p = permutation(1000, 42)
    y = oc.time_randomize(x, p)
    assert np.array_equal(np.sort(y), np.sort(x)) and not np.array_equal(y, x)   # same histogram
    assert np.array_equal(p, permutation(1000, 42)) and not np.array_equal(p, permutation(1000, 43))
    assert np.array_equal(oc.time_randomize(x, np.arange(1000)), x)              # identity
    inv = np.argsort(p)
    assert np.array_equal(oc.time_randomize(y, inv), x)                          # x'[i] = x[perm[i]]
    with pytest.raises(ValueError):
        oc.time_randomize(x, np.zeros(1000, np.int64))


def test_pc2_coincidence_against_set_arithmetic_on_hit_lists():
    # build the maps from explicit hit lists and count partners pair by pair
    rng = np.random.default_rng(2)
    nt, nf, w = 7, 40, 3
    h1 = [(int(rng.integers(nt)), int(rng.integers(nf))) for _ in range(60)]
    h2 = [(int(rng.integers(nt)), int(rng.integers(nf))) for _ in range(25)]
    m1 = np.zeros((nt, nf), np.uint32)
    m2 = np.zeros((nt, nf), np.uint32)
    for t, f in h1:
        m1[t, f] += 1
    for t, f in h2:
        m2[t, f] += 1
    c1, c2 = oc.coincidence(m1, m2, w)
    want1 = np.zeros_like(m1)
    for t, f in h1:
        if any(t == t2 and abs(f - f2) <= w for t2, f2 in h2):
            want1[t, f] += 1
    want2 = np.zeros_like(m2)
    for t, f in h2:
        if any(t == t1 and abs(f - f1) <= w for t1, f1 in h1):
            want2[t, f] += 1
    assert np.array_equal(c1, want1) and np.array_equal(c2, want2)


def test_pc3_coincidence_limits_and_symmetry():
    rng = np.random.default_rng(3)
    m1 = (rng.random((5, 30)) < 0.2).astype(np.uint32) * rng.integers(1, 4, (5, 30)).astype(np.uint32)
    m2 = (rng.random((5, 30)) < 0.1).astype(np.uint32)
    c1, c2 = oc.coincidence(m1, m2, 4)
    assert np.all(c1 <= m1) and np.all(c2 <= m2) and np.all((c1 == 0) | (c1 == m1))
    d2, d1 = oc.coincidence(m2, m1, 4)                     # roles swapped
    assert np.array_equal(d1, c1) and np.array_equal(d2, c2)
    a1, a2 = oc.coincidence(m1, m2, 0)                     # zero width: same bin only
    assert np.array_equal(a1, m1 * (m2 > 0)) and np.array_equal(a2, m2 * (m1 > 0))
    b1, _ = oc.coincidence(m1, m2, 1000)                   # infinite width: any partner in the row
    assert np.array_equal(b1, m1 * (m2.sum(axis=1, keepdims=True) > 0))
    z1, z2 = oc.coincidence(m1, np.zeros_like(m2), 4)      # no partner at all
    assert not z1.any() and not z2.any()


def test_pc4_pseudo_spectrum_is_the_time_marginal():
    rng = np.random.default_rng(4)
    m = rng.integers(0, 5, (9, 17)).astype(np.uint32)
    s = oc.pseudo_spectrum(m)
    assert s.dtype == np.uint64 and np.array_equal(s, m.sum(axis=0).astype(np.uint64))
    assert int(s.sum()) == int(m.sum())
    big = np.full((3, 2), 4_000_000_000, np.uint32)        # sums beyond 32 bits
    assert oc.pseudo_spectrum(big).tolist() == [12_000_000_000, 12_000_000_000]
