"""The five run configurations of BASELINE.json:configs[0..4] as plain data.

Shapes follow the paper: 27 antennas / 351 baselines, two polarisations, 256 or
1024 channels, 5-50 ms integrations (Table 1 and its note);
512x512 reference image; 6 sigma / 7 sigma thresholds
(PAPER.md:88); array sizes 1-36 km.  Readings of what
BASELINE.json leaves open (channel centres, Y layout, cell size, ...) are the
ones listed in DESIGN.md ("Readings") and SURVEY.md section 8(c) A2/A13-A15.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Tuple

BASE_SEED = 18020308  # seed = 18020308 + config index


@dataclass(frozen=True)
class Config:
    name: str
    index: int                      # position in BASELINE.json:configs
    layout: str                     # "random" | "Y"
    nant: int
    r_min_m: float
    r_max_m: float
    dec_deg: float
    ha_hours: float                 # hour angle at segment mid-time
    f_start_ghz: float
    chan_width_ghz: float
    nchan: int
    npol: int
    nint: int
    inttime_s: float
    dm_max: float
    ndm: int
    dt_list: Tuple[int, ...]
    npix: int
    threshold: float
    n_transients: int
    amp_range: Tuple[float, float]
    dm_inj_range: Tuple[float, float]
    width_range: Tuple[int, int]    # inclusive
    offset_mode: str                # "fixed" | "central" | "large"
    n_flagged: int = 0
    fixed_transient: Tuple[float, int, int, float, int, int] = field(
        default=(0.0, 0, 0, 0.0, 1, 0))  # amp, l, m, dm, width, t0
    # streaming (config 5)
    n_segments: int = 1
    stride_int: int = 0

    @property
    def nbl(self) -> int:
        return self.nant * (self.nant - 1) // 2

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index


_TINY = Config(
    name="tiny", index=0, layout="random", nant=10, r_min_m=0.0, r_max_m=1000.0,
    dec_deg=30.0, ha_hours=0.0, f_start_ghz=1.0, chan_width_ghz=0.5 / 32, nchan=32,
    npol=2, nint=64, inttime_s=0.010, dm_max=140.0, ndm=8, dt_list=(1,), npix=64,
    threshold=6.0, n_transients=1, amp_range=(2.0, 2.0), dm_inj_range=(50.0, 50.0),
    width_range=(1, 1), offset_mode="fixed",
    fixed_transient=(2.0, 8, -5, 50.0, 1, 20))

_LBAND = Config(
    name="lband", index=1, layout="Y", nant=27, r_min_m=40.0, r_max_m=1000.0,
    dec_deg=20.0, ha_hours=0.0, f_start_ghz=1.0, chan_width_ghz=0.004, nchan=256,
    npol=2, nint=1024, inttime_s=0.005, dm_max=1000.0, ndm=64, dt_list=(1, 2, 4, 8),
    npix=512, threshold=7.0, n_transients=10, amp_range=(0.3, 1.0),
    dm_inj_range=(100.0, 900.0), width_range=(1, 8), offset_mode="central")

_SBAND = Config(
    name="sband", index=2, layout="Y", nant=27, r_min_m=0.04 * 3400.0, r_max_m=3400.0,
    dec_deg=20.0, ha_hours=0.0, f_start_ghz=2.0, chan_width_ghz=0.002, nchan=1024,
    npol=2, nint=2048, inttime_s=0.010, dm_max=3000.0, ndm=200,
    dt_list=(1, 2, 4, 8, 16), npix=1024, threshold=7.0, n_transients=5,
    amp_range=(0.3, 1.0), dm_inj_range=(300.0, 2700.0), width_range=(1, 16),
    offset_mode="central", n_flagged=102)

_HIRES = Config(
    name="hires", index=3, layout="Y", nant=27, r_min_m=0.04 * 36000.0, r_max_m=36000.0,
    dec_deg=20.0, ha_hours=0.0, f_start_ghz=1.0, chan_width_ghz=0.004, nchan=256,
    npol=2, nint=512, inttime_s=0.005, dm_max=600.0, ndm=32, dt_list=(1, 2),
    npix=4096, threshold=7.0, n_transients=3, amp_range=(0.5, 1.0),
    dm_inj_range=(60.0, 540.0), width_range=(1, 2), offset_mode="large")

_STREAM = Config(
    name="stream", index=4, layout="Y", nant=27, r_min_m=40.0, r_max_m=1000.0,
    dec_deg=20.0, ha_hours=-1.0, f_start_ghz=1.0, chan_width_ghz=0.004, nchan=256,
    npol=2, nint=1024, inttime_s=0.005, dm_max=1000.0, ndm=64, dt_list=(1, 2, 4, 8),
    npix=512, threshold=7.0, n_transients=2, amp_range=(0.3, 1.0),
    dm_inj_range=(100.0, 900.0), width_range=(1, 8), offset_mode="central",
    n_segments=32, stride_int=400)

# The paper's GOAL workload ("1 ms ... 1.4 GB/s"; Table 1 row "L"): the config-5 array,
# band and trial grid sampled at 1 ms.  Segment stride 2.0 s as in config 5 (2000 integrations), overlap = the
# DM 1000 sweep at 1 ms = 3118 integrations, 8 consecutive segments.  New data per segment:
# 2000 x 351 x 256 x 2 x 8 B = 2.875 GB per 2.0 s = 1.44 GB/s.
_STREAM1MS = Config(
    name="stream1ms", index=5, layout="Y", nant=27, r_min_m=40.0, r_max_m=1000.0,
    dec_deg=20.0, ha_hours=-1.0, f_start_ghz=1.0, chan_width_ghz=0.004, nchan=256,
    npol=2, nint=5118, inttime_s=0.001, dm_max=1000.0, ndm=64, dt_list=(1, 2, 4, 8),
    npix=512, threshold=7.0, n_transients=2, amp_range=(0.3, 1.0),
    dm_inj_range=(100.0, 900.0), width_range=(1, 8), offset_mode="central",
    n_segments=8, stride_int=2000)

CONFIGS = {c.name: c for c in (_TINY, _LBAND, _SBAND, _HIRES, _STREAM, _STREAM1MS)}


def get_config(name: str) -> Config:
    return CONFIGS[name]
