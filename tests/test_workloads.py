"""The seeded input generators and the golden fixture of the oracle (CPU only)."""
import os

import numpy as np

import oracle
from workloads import (CONFIGS, bank_grid, default_map_grid, get_config, make_data,
                       sub_bank_indices)

HERE = os.path.dirname(os.path.abspath(__file__))


def test_config_sizes_match_the_survey_table():
    want = {1: (256, 2049), 2: (65536, 126977), 3: (1048576, 126001),
            4: (8388608, 61441), 5: (1048576, 4190209)}
    for i, (T, nl) in want.items():
        c = CONFIGS[i]
        assert c.n_templates == T and c.n_lags == nl


def test_bank_grid_ordering_and_endpoints():
    c = get_config(1)
    f0, f1 = bank_grid(c)
    assert f0.dtype == np.float64 and len(f0) == 256
    assert f0[0] == 200.0 and f0[-1] == 900.0 and f1[0] == -400.0 and f1[15] == 400.0
    # j = i_f0 * n_f1 + i_f1
    assert f0[16] == np.linspace(200, 900, 16)[1] and f1[17] == np.linspace(-400, 400, 16)[1]
    # even n_f1 on a symmetric range: f1 = 0 is never a node (the slope cut)
    for c in CONFIGS.values():
        g = np.linspace(c.f1_lo, c.f1_hi, c.n_f1)
        assert not np.any(g == 0.0)


def test_data_is_seeded_fp32_and_unit_variance():
    for i in (1, 2, 3, 4):
        c = get_config(i)
        a, b = make_data(c), make_data(c)
        assert a.dtype == np.float32 and a.flags.c_contiguous and len(a) == c.n_samples
        np.testing.assert_array_equal(a, b)
        assert abs(a.std() - 1.0) < 0.02 and abs(a.mean()) < 0.02


def test_grb_series_has_a_red_spectrum():
    c = get_config(3)
    x = make_data(c).astype(np.float64)
    p = np.abs(np.fft.rfft(x)) ** 2
    lo, hi = p[1:40].mean(), p[20000:60000].mean()
    assert lo > 3 * hi         # Kolmogorov continuum on top of white Poisson noise


def test_sub_bank_is_seeded_and_contains_the_corners():
    c = get_config(4)
    a = sub_bank_indices(c, 64)
    b = sub_bank_indices(c, 64)
    np.testing.assert_array_equal(a, b)
    T = c.n_templates
    for corner in (0, c.n_f1 - 1, T - c.n_f1, T - 1):
        assert corner in a
    assert np.all(np.diff(a) > 0) and a[-1] < T
    assert np.any(a >= (c.n_f0 - 1) * c.n_f1)        # the f0 = fs/2 row


def test_default_map_grid():
    g = default_map_grid(get_config(1))
    assert g == dict(samples_per_tbin=128, f_lo_hz=0.0, df_hz=1.0, n_fbins=901, n_tbins=32)
    g = default_map_grid(get_config(5))
    assert g["n_tbins"] == 16384 and g["n_fbins"] == 2049


def test_oracle_reproduces_its_golden_fixture():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "tiny_oracle.txt"))
            if not l.startswith("#")]
    c = get_config(1)
    x = make_data(c)
    f0, f1 = bank_grid(c)
    rho, arg = oracle.correlate(x, c.fs_hz, c.L, f0, f1)
    assert len(rows) == 256
    for j, r in enumerate(rows):
        assert int(r[0]) == j and float(r[1]) == f0[j] and float(r[2]) == f1[j]
        assert abs(float(r[3]) - rho[j]) < 1e-13 and int(r[4]) == arg[j]
    # the Tiny map is empty at kappa = 0.2 (bank maximum ~0.11)
    assert rho.max() < 0.2
