"""Robustness of the C ABI on a GPU: the bank's workspace handed from stream to
stream, the in-use flag under two host threads, per-device set-up, the caller's current device left
alone.  Results are compared with a plain single-stream call of the same library.  Needs a B200."""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def bfly():
    import paper_1802_01685_b200 as b
    return b


def _inputs(seed, fs=4096.0, L=4096, N=30000, T=200):
    rng = np.random.default_rng(seed)
    f0 = rng.uniform(30.0, 1900.0, T)
    f1 = rng.uniform(-800.0, 800.0, T)
    xs = [rng.standard_normal(N).astype(np.float32) for _ in range(4)]
    return fs, L, f0, f1, xs


def test_two_streams_share_one_bank_without_host_synchronisation(bfly):
    fs, L, f0, f1, xs = _inputs(1)
    bank = bfly.make_bank(fs, L, f0, f1)
    xd = [torch.from_numpy(x).cuda() for x in xs]
    ref = []
    for x in xd:
        r, a = bfly.correlate(bank, x)
        torch.cuda.synchronize()
        ref.append((r.clone(), a.clone()))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    out = []
    for rep in range(5):                                  # alternate streams, no synchronisation in between:
        for i, x in enumerate(xd):                        # the workspace is ordered by the bank's event
            with torch.cuda.stream(s1 if (i + rep) & 1 else s2):
                out.append((i, bfly.correlate(bank, x)))
    torch.cuda.synchronize()
    for i, (r, a) in out:
        assert torch.equal(r, ref[i][0]) and torch.equal(a, ref[i][1])


def test_two_host_threads_on_one_bank_either_succeed_or_are_refused(bfly):
    fs, L, f0, f1, xs = _inputs(2)
    bank = bfly.make_bank(fs, L, f0, f1)
    xd = [torch.from_numpy(x).cuda() for x in xs[:2]]
    ref = [tuple(t.clone() for t in bfly.correlate(bank, x)) for x in xd]
    torch.cuda.synchronize()
    results, errors = [[], []], [[], []]

    def worker(k):
        stream = torch.cuda.Stream()
        with torch.cuda.stream(stream):
            for _ in range(200):
                try:
                    results[k].append(bfly.correlate(bank, xd[k]))
                except bfly.BflyError as e:               # refused, not raced
                    errors[k].append(str(e))
        stream.synchronize()

    th = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    for k in range(2):
        assert results[k], "every call of a thread was refused"
        for r, a in results[k]:
            assert torch.equal(r, ref[k][0]) and torch.equal(a, ref[k][1])
        for msg in errors[k]:
            assert "in use" in msg


def _on_device(bfly, dev, fs, L, f0, f1, x_np):
    bank = bfly.make_bank(fs, L, f0, f1, device=dev)
    x = torch.from_numpy(x_np).to(f"cuda:{dev}")
    with torch.cuda.device(dev):
        r, a = bfly.correlate(bank, x)
        rs, as_ = torch.empty_like(r), torch.empty_like(a)
        bfly.correlate_static(bank, x, rs, as_)           # per-device address of the static scratch
        torch.cuda.synchronize()
    assert torch.equal(r, rs) and torch.equal(a, as_)
    return r.cpu(), a.cpu()


def test_calls_leave_the_current_device_alone(bfly):
    fs, L, f0, f1, xs = _inputs(3, T=60)
    before = torch.cuda.current_device()
    _on_device(bfly, 0, fs, L, f0, f1, xs[0])
    assert torch.cuda.current_device() == before


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs in one process")
def test_banks_on_two_devices_in_one_process(bfly):
    fs, L, f0, f1, xs = _inputs(4, T=60)
    before = torch.cuda.current_device()
    r0 = _on_device(bfly, 0, fs, L, f0, f1, xs[0])
    r1 = _on_device(bfly, 1, fs, L, f0, f1, xs[0])       # function attributes and scratch address are per device
    assert torch.equal(r0[0], r1[0]) and torch.equal(r0[1], r1[1])
    assert torch.cuda.current_device() == before
