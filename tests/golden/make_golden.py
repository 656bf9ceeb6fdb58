"""Write tests/golden/tiny_oracle.txt: the oracle's per-template results on config 1.

Calls only oracle/ and workloads/ (never the CUDA path).  The paper prints no
numeric example (PAPER.md has no value of rho, lag or map cell), so this file is not
a citation of the paper: it is a regression fixture that freezes the oracle's own
arithmetic, so that any later change to it shows up as a diff that the commit
message has to justify.  Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import bank_grid, get_config, make_data  # noqa: E402


def main():
    cfg = get_config(1)
    x = make_data(cfg)
    f0, f1 = bank_grid(cfg)
    rho, arg = oracle.correlate(x, cfg.fs_hz, cfg.L, f0, f1)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle.txt")
    with open(out, "w") as f:
        f.write("# config 1 (Tiny), seed 1: oracle.correlate over all 2049 lags\n")
        f.write("# written by tests/golden/make_golden.py from oracle/ only\n")
        f.write("# j f0_hz f1_hzps rho_max arg_lag\n")
        for j in range(len(f0)):
            f.write(f"{j} {float(f0[j])!r} {float(f1[j])!r} {float(rho[j])!r} {int(arg[j])}\n")
    print(out)


if __name__ == "__main__":
    main()
