"""bfly_correlate_static: the default correlation form with its scratch in a file-scope static
device array (no cudaMalloc inside the call), for callers that cannot allocate.  Checked against
the existing path (bfly_correlate) on two calls in a row that share the array, the second one
smaller than the first so that stale contents of the first call lie behind it.  Named to be
collected last (the suite runs with pytest -x).  Needs a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

RHO_TOL = 2e-4          # north_star's tolerance, as in tests/parity.py (the two paths run the same
                        # kernels on the same inputs, so they are expected to agree bit for bit)


@pytest.fixture(scope="module")
def bfly():
    import paper_1802_01685_b200 as b
    return b


def _compare(bfly, bank, x, lag_begin=0, lag_end=None):
    T = len(bank)
    xd = torch.from_numpy(x).cuda()
    rho_s = torch.full((T,), -1.0, dtype=torch.float32, device="cuda")
    arg_s = torch.full((T,), -1, dtype=torch.int32, device="cuda")
    bfly.correlate_static(bank, xd, rho_s, arg_s, lag_begin, lag_end)
    torch.cuda.synchronize()
    rho_r, arg_r = bfly.correlate(bank, xd, lag_begin, lag_end)
    torch.cuda.synchronize()
    d = (rho_s - rho_r).abs().max().item()
    assert d <= RHO_TOL, d
    assert torch.equal(arg_s, arg_r)
    assert torch.equal(rho_s, rho_r)                 # same kernels, same inputs: bit-identical
    return rho_s.cpu().numpy(), arg_s.cpu().numpy()


def test_static_scratch_entry_point_matches_the_existing_path_twice(bfly):
    rng = np.random.default_rng(20)
    fs, L = 4096.0, 4096
    T = 148 + 41                                     # more than one template on some SMs, ragged
    f0 = rng.uniform(30.0, 1900.0, T)
    f1 = rng.uniform(-800.0, 800.0, T)
    bank = bfly.make_bank(fs, L, f0, f1)
    # call 1: the maximum size, one 16-s segment (15 blocks + the 61441st lag), with a chirp in it
    n1 = bfly.STATIC_MAX_SAMPLES
    x1 = rng.standard_normal(n1)
    t = np.arange(L) / fs
    x1[30000:30000 + L] += 0.5 * np.cos(2 * np.pi * (f0[7] * t + 0.5 * f1[7] * t * t))
    rho1, arg1 = _compare(bfly, bank, x1.astype(np.float32))
    assert abs(int(arg1[7]) - 30000) <= 1 and rho1[7] > 0.25
    # call 2, right after it: fewer blocks, a lag sub-range, another scale; the array still holds call 1
    x2 = (rng.standard_normal(20000) * 300.0).astype(np.float32)
    _compare(bfly, bank, x2, 17, 17 + 2 * 4096 + 3)
    # and the first input again: the result does not depend on what the array held before
    rho3, arg3 = _compare(bfly, bank, x1.astype(np.float32))
    assert np.array_equal(rho3, rho1) and np.array_equal(arg3, arg1)


def test_static_scratch_entry_point_rejects_what_does_not_fit(bfly):
    rng = np.random.default_rng(21)
    bank = bfly.make_bank(4096.0, 4096, [100.0, 200.0], [10.0, -10.0])
    rho = torch.empty(2, dtype=torch.float32, device="cuda")
    arg = torch.empty(2, dtype=torch.int32, device="cuda")
    x = torch.from_numpy(rng.standard_normal(bfly.STATIC_MAX_SAMPLES + 1).astype(np.float32)).cuda()
    with pytest.raises(bfly.BflyError) as e:
        bfly.correlate_static(bank, x, rho, arg)
    assert "BFLY_STATIC_MAX_SAMPLES" in str(e.value)
    short = bfly.make_bank(512.0, 64, [50.0], [1.0])          # L < BFLY_TC_MIN_L: not this form
    with pytest.raises(bfly.BflyError):
        bfly.correlate_static(short, x[:4096], rho[:1], arg[:1])
