"""The five workload configurations of BASELINE.json, with the exact parameters
SURVEY.md section 8(d) fixes where BASELINE.json gives only rough ones."""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Tuple


@dataclass(frozen=True)
class Injection:
    """One chirp added to the noise as A*cos(phi(t)), t measured from t_start.

    kind "linear":  f(t) = f_start + slope*t
    kind "settle":  f(t) = f_inf + (f_start - f_inf)*exp(-t/tau_c)
    """
    kind: str
    amplitude: float
    t_start_s: float
    t_stop_s: float
    f_start_hz: float
    slope_hzps: float = 0.0      # linear only
    f_inf_hz: float = 0.0        # settle only
    tau_c_s: float = 1.0         # settle only


@dataclass(frozen=True)
class Config:
    name: str
    index: int                   # 1-based, as in BASELINE.json / SURVEY.md
    seed: int
    fs_hz: float
    n_samples: int
    L: int                       # template length in samples ("1 s")
    f0_lo: float
    f0_hi: float
    n_f0: int
    f1_lo: float
    f1_hi: float
    n_f1: int
    kappa: float
    data_kind: str               # "gauss" | "grb"
    injections: Tuple[Injection, ...] = field(default_factory=tuple)
    streaming: bool = False      # config 5: 16-s chunks with 1-s overlap
    chunk_samples: int = 65536

    @property
    def n_templates(self) -> int:
        return self.n_f0 * self.n_f1

    @property
    def n_lags(self) -> int:
        return self.n_samples - self.L + 1

    @property
    def samples_per_tbin(self) -> int:
        # 1/16 s time bins (BASELINE.json configs 2 and 5)
        return int(round(self.fs_hz / 16.0))


CONFIGS = {
    1: Config(
        name="tiny", index=1, seed=1, fs_hz=2048.0, n_samples=4096, L=2048,
        f0_lo=200.0, f0_hi=900.0, n_f0=16, f1_lo=-400.0, f1_hi=400.0, n_f1=16,
        kappa=0.2, data_kind="gauss",
        injections=(Injection("linear", 0.3, 1000 / 2048.0, 3048 / 2048.0,
                              600.0, slope_hzps=-200.0),),
    ),
    2: Config(
        name="ligo_like", index=2, seed=2, fs_hz=4096.0, n_samples=131072, L=4096,
        f0_lo=100.0, f0_hi=2000.0, n_f0=256, f1_lo=-500.0, f1_hi=500.0, n_f1=256,
        kappa=0.1, data_kind="gauss",
        injections=(
            Injection("settle", 0.10, 4.0, 20.0, 2000.0, f_inf_hz=1900.0, tau_c_s=4.0),
            Injection("settle", 0.07, 14.0, 26.0, 1950.0, f_inf_hz=1800.0, tau_c_s=3.0),
            Injection("linear", 0.05, 8.0, 16.0, 300.0, slope_hzps=50.0),
        ),
    ),
    3: Config(
        name="grb_like", index=3, seed=3, fs_hz=2000.0, n_samples=128000, L=2000,
        f0_lo=50.0, f0_hi=1000.0, n_f0=1024, f1_lo=-300.0, f1_hi=300.0, n_f1=1024,
        kappa=0.05, data_kind="grb",
    ),
    4: Config(
        name="paper_scale", index=4, seed=4, fs_hz=4096.0, n_samples=65536, L=4096,
        f0_lo=20.0, f0_hi=2048.0, n_f0=4096, f1_lo=-1000.0, f1_hi=1000.0, n_f1=2048,
        kappa=0.08, data_kind="gauss",
        injections=(Injection("linear", 0.05, 0.0, 13.0, 40.0, slope_hzps=150.0),),
    ),
    5: Config(
        name="streaming", index=5, seed=5, fs_hz=4096.0, n_samples=4194304, L=4096,
        f0_lo=100.0, f0_hi=2048.0, n_f0=1024, f1_lo=-600.0, f1_hi=600.0, n_f1=1024,
        kappa=0.06, data_kind="gauss",
        injections=(Injection("settle", 0.03, 300.0, 360.0, 1500.0,
                              f_inf_hz=1200.0, tau_c_s=12.0),),
        streaming=True, chunk_samples=65536,
    ),
}


def get_config(key) -> Config:
    """Look a config up by 1-based index or by name."""
    if isinstance(key, int):
        return CONFIGS[key]
    for c in CONFIGS.values():
        if c.name == key:
            return c
    raise KeyError(key)
