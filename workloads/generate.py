"""Seeded synthetic observation generator (geometry, noise, mock transients).

Everything here is INPUT construction.  The recipe:

* antenna positions: ``random`` = seeded uniform disc (config 1); ``Y`` = three
  arms at azimuth 0/120/240 deg (from North through East), 9 antennas per arm,
  radii ``geomspace(r_min, r_max, 9)`` (BASELINE.json:configs[1..4]).
* uvw from ENU by the textbook rotation at the VLA latitude, one uvw per
  segment at its mid-time hour angle.
* channel centres f_k = f_start + (k + 1/2) * width.
* noise: complex64, N(0,1) per real/imag part per polarisation, one counter
  based Philox stream PER ABSOLUTE INTEGRATION so any row range of any segment
  can be regenerated independently (streaming segments overlap bit-for-bit).
* mock transients: a point source of amplitude A at pixel offset
  (l, m) whose arrival time in each channel follows the cold-plasma law
  (footnote 1) relative to the top channel.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence, Tuple

import numpy as np

from .configs import Config

C_M_S = 299792458.0
VLA_LAT_DEG = 34.0784
# dispersion constant of the SIGNAL model, s GHz^2 cm^3 / pc (PAPER.md:45 prints 4.15 ms)
K_DM_S = 4.148808e-3


@dataclass(frozen=True)
class Transient:
    amp: float
    l_pix: int
    m_pix: int
    dm: float
    width: int
    t0: int          # absolute native integration of arrival at the top channel


def antenna_enu(cfg: Config) -> np.ndarray:
    """[nant][3] East, North, Up in metres."""
    if cfg.layout == "random":
        rng = np.random.Generator(np.random.Philox(key=np.array([cfg.seed, 1], dtype=np.uint64)))
        r = cfg.r_max_m * np.sqrt(rng.random(cfg.nant))
        az = 2.0 * np.pi * rng.random(cfg.nant)
    elif cfg.layout == "Y":
        per_arm = cfg.nant // 3
        radii = np.geomspace(cfg.r_min_m, cfg.r_max_m, per_arm)
        r = np.tile(radii, 3)
        az = np.repeat(np.deg2rad([0.0, 120.0, 240.0]), per_arm)
    else:
        raise ValueError(cfg.layout)
    enu = np.zeros((cfg.nant, 3))
    enu[:, 0] = r * np.sin(az)
    enu[:, 1] = r * np.cos(az)
    return enu


def baseline_uvw_m(cfg: Config, ha_hours: float | None = None) -> np.ndarray:
    """[nbl][3] (u, v, w) in metres for baselines (i<j), value = ant j - ant i."""
    enu = antenna_enu(cfg)
    lat = np.deg2rad(VLA_LAT_DEG)
    dec = np.deg2rad(cfg.dec_deg)
    ha = np.deg2rad(15.0 * (cfg.ha_hours if ha_hours is None else ha_hours))
    e, n, up = enu[:, 0], enu[:, 1], enu[:, 2]
    x = -n * np.sin(lat) + up * np.cos(lat)
    y = e
    z = n * np.cos(lat) + up * np.sin(lat)
    u = x * np.sin(ha) + y * np.cos(ha)
    v = -x * np.sin(dec) * np.cos(ha) + y * np.sin(dec) * np.sin(ha) + z * np.cos(dec)
    w = x * np.cos(dec) * np.cos(ha) - y * np.cos(dec) * np.sin(ha) + z * np.sin(dec)
    ant = np.stack([u, v, w], axis=1)
    i, j = np.triu_indices(cfg.nant, k=1)
    return np.ascontiguousarray(ant[j] - ant[i])


def channel_freqs_hz(cfg: Config) -> np.ndarray:
    k = np.arange(cfg.nchan, dtype=np.float64)
    return (cfg.f_start_ghz + (k + 0.5) * cfg.chan_width_ghz) * 1e9


def dm_list(cfg: Config) -> np.ndarray:
    return np.linspace(0.0, cfg.dm_max, cfg.ndm)


def default_cell_rad(cfg: Config, uvw_m: np.ndarray | None = None) -> float:
    """cell = 1 / (3 * max|uv|_lambda) (BASELINE.json:configs[0]; applied to all configs)."""
    uvw = baseline_uvw_m(cfg) if uvw_m is None else uvw_m
    f = channel_freqs_hz(cfg)
    ul = uvw[:, 0:1] * f[None, :] / C_M_S
    vl = uvw[:, 1:2] * f[None, :] / C_M_S
    return float(1.0 / (3.0 * np.hypot(ul, vl).max()))


def chan_weights(cfg: Config) -> np.ndarray:
    """float32 [nchan] of 0/1; config 3 flags 102 seeded channels."""
    w = np.ones(cfg.nchan, dtype=np.float32)
    if cfg.n_flagged:
        rng = np.random.Generator(np.random.Philox(key=np.array([cfg.seed, 2], dtype=np.uint64)))
        w[rng.choice(cfg.nchan, size=cfg.n_flagged, replace=False)] = 0.0
    return w


def _sweep_integrations(cfg: Config, dm: float) -> np.ndarray:
    """Arrival delay of the mock signal per channel, in whole integrations."""
    f = channel_freqs_hz(cfg) / 1e9
    tau = K_DM_S * dm * (1.0 / (f * f) - 1.0 / (f.max() * f.max()))
    return np.floor(tau / cfg.inttime_s + 0.5).astype(np.int64)


def transients(cfg: Config) -> List[Transient]:
    """The seeded mock transients of a config (absolute arrival times)."""
    if cfg.offset_mode == "fixed":
        a, l, m, dm, w, t0 = cfg.fixed_transient
        return [Transient(float(a), int(l), int(m), float(dm), int(w), int(t0))]
    rng = np.random.Generator(np.random.Philox(key=np.array([cfg.seed, 3], dtype=np.uint64)))
    n_abs = cfg.nint if cfg.n_segments == 1 else cfg.stride_int * cfg.n_segments
    out = []
    for _ in range(cfg.n_transients):
        amp = float(rng.uniform(*cfg.amp_range))
        dm = float(rng.uniform(*cfg.dm_inj_range))
        width = int(rng.integers(cfg.width_range[0], cfg.width_range[1] + 1))
        if cfg.offset_mode == "central":
            lim = cfg.npix // 3
            l, m = (int(v) for v in rng.integers(-lim, lim + 1, size=2))
        else:  # "large": |l|, |m| in [N/4, N/2.5]
            lo, hi = cfg.npix // 4, int(cfg.npix / 2.5)
            l, m = (int(s * v) for s, v in zip(rng.choice([-1, 1], size=2),
                                               rng.integers(lo, hi + 1, size=2)))
        sweep = int(_sweep_integrations(cfg, dm).max())
        t_hi = max(1, n_abs - sweep - width) if cfg.n_segments == 1 else n_abs - width
        t0 = int(rng.integers(0, t_hi))
        out.append(Transient(amp, l, m, dm, width, t0))
    return out


def noise_rows(cfg: Config, t_abs: Sequence[int], out: np.ndarray | None = None) -> np.ndarray:
    """complex64 [len(t_abs)][nbl][nchan][npol]; row t depends on (seed, t) only."""
    if out is None:
        out = np.empty((len(t_abs), cfg.nbl, cfg.nchan, cfg.npol), dtype=np.complex64)
    flat = out.view(np.float32).reshape(len(t_abs), -1)
    for k, t in enumerate(t_abs):
        rng = np.random.Generator(
            np.random.Philox(key=np.array([cfg.seed, (1 << 32) + int(t)], dtype=np.uint64)))
        rng.standard_normal(out=flat[k], dtype=np.float32)
    return out


def make_segment(cfg: Config, segment: int = 0, *, noise: bool = True,
                 inject: bool = True, uvw_m: np.ndarray | None = None,
                 cell_rad: float | None = None,
                 sources: Sequence[Transient] | None = None,
                 rows: Tuple[int, int] | None = None, out: np.ndarray | None = None,
                 persistent: Sequence[Tuple[float, int, int]] = ()) -> np.ndarray:
    """Visibilities of one segment: complex64 [nint][nbl][nchan][npol].

    Segment ``s`` of a streaming config covers absolute integrations
    [s*stride, s*stride + nint).  ``sources`` overrides the seeded transients.
    ``rows = (lo, hi)`` returns only the segment-relative integrations [lo, hi)
    (the same values ``make_segment(...)[lo:hi]`` would hold); ``out`` receives them in place.
    ``persistent`` = (amplitude, l_pix, m_pix) of constant point sources present in every
    integration (what the mean-visibility subtraction of PAPER.md:84-86 removes).
    """
    lo, hi = (0, cfg.nint) if rows is None else rows
    t_first = segment * cfg.stride_int
    t_abs = np.arange(t_first + lo, t_first + hi)
    shape = (hi - lo, cfg.nbl, cfg.nchan, cfg.npol)
    vis = np.empty(shape, dtype=np.complex64) if out is None else out
    assert vis.shape == shape and vis.dtype == np.complex64
    if noise:
        noise_rows(cfg, t_abs, out=vis)
    else:
        vis[...] = 0
    if not inject:
        return vis
    uvw = baseline_uvw_m(cfg, segment_ha_hours(cfg, segment)) if uvw_m is None else uvw_m
    cell = default_cell_rad(cfg, uvw) if cell_rad is None else cell_rad
    f = channel_freqs_hz(cfg)
    ul = uvw[:, 0:1] * f[None, :] / C_M_S          # [nbl][nchan]
    vl = uvw[:, 1:2] * f[None, :] / C_M_S
    for (amp, l_pix, m_pix) in persistent:
        sig = (amp * np.exp(-2j * np.pi * (ul * l_pix + vl * m_pix) * cell)).astype(np.complex64)
        vis += sig[None, :, :, None]
    for src in (transients(cfg) if sources is None else sources):
        phase = np.exp(-2j * np.pi * (ul * src.l_pix + vl * src.m_pix) * cell)
        sig = (src.amp * phase).astype(np.complex64)
        sweep = _sweep_integrations(cfg, src.dm)
        for q in range(src.width):
            t_ch = src.t0 + q + sweep - t_first           # per channel, segment-relative
            for t in np.unique(t_ch):
                if lo <= t < hi:
                    ch = np.nonzero(t_ch == t)[0]
                    vis[t - lo][:, ch, :] += sig[:, ch, None]
    return vis


def segment_ha_hours(cfg: Config, segment: int) -> float:
    """Hour angle at a segment's mid-time; config 5 advances -1 h -> +1 h over its segments."""
    if cfg.n_segments == 1:
        return cfg.ha_hours
    return cfg.ha_hours + 2.0 * segment / (cfg.n_segments - 1)
