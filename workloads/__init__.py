"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the oracle-side tests and by the CUDA-side tests and
bench: it produces *inputs only* (data series, the (f0, f1) lists of a bank,
template sub-samples for parity at scale).  It holds none of the method's
arithmetic: no correlation, no template norms, no rho, no map.  The chirps
added to the data are part of the input recipe (DESIGN.md
"Input recipe"), not of the search.

The paper's real workloads (LIGO LOSC strain, BeppoSAX light curves;
PAPER.md:64, 68, 124) are not available; these inputs stand in for them.
"""
from .configs import CONFIGS, Config, get_config
from .generators import (bank_grid, make_data, sub_bank_indices,
                         default_map_grid, permutation)

__all__ = ["CONFIGS", "Config", "get_config", "bank_grid", "make_data",
           "sub_bank_indices", "default_map_grid", "permutation"]
