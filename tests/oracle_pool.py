"""Test helper: the float64 oracle evaluated on many (dm, dt, j) images of one segment, in parallel on the
host cores (fork pool; the segment is inherited, not pickled).  Imports oracle/ and workloads/ only.

For every key it returns  (peak, y, x, sigma, snr, peak2, y2, x2):  O.image_stats of the oracle image plus the
second-largest pixel and its position, which the GPU tests need for reading A20 (the peak pixel is unique only up
to ties within float32 rounding: when the two largest float64 pixels agree to a few float32 ulps either position
is correct, otherwise the position must be the oracle's)."""
from __future__ import annotations

import multiprocessing as mp
import os
from typing import Dict, Iterable, Optional, Sequence, Tuple

import numpy as np

import oracle as O

Key = Tuple[int, int, int]
_STATE: dict = {}


def _stats8(img: np.ndarray):
    peak, y, x, sigma, snr = O.image_stats(img)
    flat = img.reshape(-1)
    k = y * img.shape[1] + x
    saved = flat[k]
    flat[k] = -np.inf
    k2 = int(np.argmax(flat))
    peak2 = float(flat[k2])
    flat[k] = saved
    y2, x2 = divmod(k2, img.shape[1])
    return (peak, y, x, sigma, snr, peak2, y2, x2)


def _work(keys: Sequence[Key]):
    st = _STATE
    out = []
    for (d, k, j) in keys:
        s = O.dedisperse_resample(st["vis"], st["delays"][d], int(st["dts"][k]), j)
        img = O.image_from_grid(O.grid_visibilities(s, st["iu"], st["iv"], st["keep"], st["npix"]), st["n_w"])
        out.append(((d, k, j), _stats8(img)))
    return out


def host_cores(limit: int = 64) -> int:
    return max(1, min(len(os.sched_getaffinity(0)), limit))


def oracle_stats(vis: np.ndarray, freqs_hz, uvw_m, inttime_s: float, npix: int, cell_rad: float, dm_list,
                 dt_list: Sequence[int], keys: Iterable[Key], chan_weights: Optional[np.ndarray] = None,
                 max_procs: int = 64) -> Dict[Key, tuple]:
    """{key: (peak, y, x, sigma, snr, peak2, y2, x2)} for the given keys, oracle steps O1-O6 per image."""
    keys = list(keys)
    delays = O.delay_table(freqs_hz, dm_list, inttime_s)
    iu, iv, keep = O.cell_table(uvw_m, freqs_hz, npix, cell_rad, chan_weights)
    _STATE.clear()
    _STATE.update(vis=vis, delays=delays, dts=list(dt_list), iu=iu, iv=iv, keep=keep, npix=npix, n_w=int(keep.sum()))
    n = max(1, min(host_cores(max_procs), len(keys)))
    os.environ.setdefault("OMP_NUM_THREADS", "1")
    if n == 1:
        res = [_work(keys)]
    else:
        # small interleaved chunks: the cost per image varies with dt, so static halves would straggle
        chunks = [keys[i::n * 8] for i in range(n * 8)]
        with mp.get_context("fork").Pool(n) as pool:
            res = pool.map(_work, [c for c in chunks if c], chunksize=1)
    _STATE.clear()
    return {k: v for part in res for (k, v) in part}


def all_keys(delays: np.ndarray, nint: int, dt_list: Sequence[int], span: int = 0):
    """Every (dm_idx, dt_idx, j) of the search loop (readings A6, A16)."""
    out = []
    for d in range(delays.shape[0]):
        md = int(delays[d].max())
        for k, dt in enumerate(dt_list):
            out.extend((d, k, j) for j in range(O.n_images(nint, md, int(dt), span)))
    return out


def candidates_from_stats(stats: Dict[Key, tuple], npix: int, threshold: float):
    """The oracle's candidate list (O7) from per-image statistics."""
    out = []
    for (d, k, j), st in stats.items():
        peak, y, x, sigma, snr = st[:5]
        if sigma > 0.0 and snr >= threshold:
            out.append(O.Candidate(d, k, j, x if x < npix // 2 else x - npix, y if y < npix // 2 else y - npix,
                                   peak, sigma, snr))
    return out


def peak_pixel_ok(gpu_l: int, gpu_m: int, st: tuple, npix: int, rel: float = 4e-7) -> bool:
    """Reading A20: the GPU's peak pixel is the oracle's, or the oracle's runner-up when the two largest
    float64 pixels agree within a few float32 ulps (rel = 4e-7 ~ 3 ulp)."""
    peak, y, x, _, _, peak2, y2, x2 = st
    gx, gy = gpu_l % npix, gpu_m % npix
    if (gx, gy) == (x, y):
        return True
    return (gx, gy) == (x2, y2) and abs(peak - peak2) <= rel * abs(peak)
