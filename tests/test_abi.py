"""The C-ABI library loads and exports every symbol include/bfly.h declares; argument
validation that needs no GPU.  No compute calls (CPU box)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "bfly.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(bfly_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_three_named_calls():
    names = _declared()
    for n in ("bfly_make_bank", "bfly_correlate", "bfly_butterfly_map"):
        assert n in names


def test_library_exports_every_declared_symbol():
    import paper_1802_01685_b200 as bfly
    lib = C.CDLL(bfly.lib_path())
    for name in _declared():
        assert hasattr(lib, name), f"libbfly.so does not export {name}"


def test_strerror_and_launch_count():
    import paper_1802_01685_b200 as bfly
    lib = C.CDLL(bfly.lib_path())
    lib.bfly_strerror.restype = C.c_char_p
    assert lib.bfly_strerror(0) == b"ok"
    assert b"invalid" in lib.bfly_strerror(-1)
    assert bfly.launch_count() >= 0


def test_argument_validation_happens_before_any_device_work():
    import paper_1802_01685_b200 as bfly
    with pytest.raises(bfly.BflyError) as e:
        bfly.make_bank(4096.0, 1, [100.0], [1.0])           # L < 2
    assert e.value.status == -1
    with pytest.raises(bfly.BflyError) as e:
        bfly.make_bank(4096.0, 5000, [100.0], [1.0])        # L beyond the supported maximum
    assert e.value.status == -5
    with pytest.raises(bfly.BflyError) as e:
        bfly.make_bank(4096.0, 4096, [np.nan], [1.0])
    assert e.value.status == -1
    with pytest.raises(bfly.BflyError) as e:
        bfly.make_bank(-1.0, 4096, [100.0], [1.0])
    assert e.value.status == -1
    for tc in (0.0, -1.0, np.inf, np.nan):                   # the settling family: tc finite and > 0
        with pytest.raises(bfly.BflyError) as e:
            bfly.make_bank_settle(4096.0, 4096, [1200.0], [300.0], [tc])
        assert e.value.status == -1


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1802_01685_b200 as bfly
    with pytest.raises(bfly.BflyError) as e:
        bfly.make_bank(4096.0, 4096, [100.0], [1.0])
    assert e.value.status in (-3, -4)


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1802_01685_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|oracle[/.]|bfo_", text), f
