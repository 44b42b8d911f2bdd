"""Plain float64 CPU oracle of the realfast search loop.  TEST INFRASTRUCTURE.

Slow, unblocked, unfused: each function is the definition written out, in the
order the paper gives it (PAPER.md = /root/reference/PAPER.md; readings A1-A20
are DESIGN.md "Readings", taken from SURVEY.md section 8(c)).

    O0  mean-visibility subtraction (prep)
    O1  delay table            PAPER.md:45 (footnote 1: tau = 4.15 ms DM / nu^2)
    O2  uv cell table          PAPER.md:72, 84 (FFT imaging, no gridding kernel)
    O3  dedisperse + resample  PAPER.md:63, 104 (loops over DM and sampling time), 118
    O4  gridding
    O5  2-D FFT Stokes-I image PAPER.md:88, 118
    O6  peak and robust sigma  PAPER.md:86-88 ("thresholding each image")
    O7  threshold              PAPER.md:88 ("S/N greater than a threshold")
    O8  candidate cut-out: image + phased, dedispersed spectrum
    O9  mock-transient injection
    O10 periodicity search: Fourier transform in time, image each frequency   PAPER.md:100 (footnote 4), 104

Pins (tests/test_oracle_tables.py, test_oracle_imaging.py, test_oracle_prep.py, test_oracle_cutout.py,
test_oracle_inject.py, test_oracle_periodic.py): every function below is pinned to something
other than itself -- closed forms, exact rational arithmetic, a direct DFT,
Parseval, the analytic noise variance, an injected source, brute force.  The
one free choice the paper does not fix is the sigma ESTIMATOR (reading A9:
1.4826 x MAD over all pixels): "parity unpinned" by the paper for that choice;
it is pinned only statistically (MAD-sigma ~ rms ~ analytic value on noise).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
legs may import this module.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Iterable, List, Optional, Sequence, Tuple

import numpy as np

K_DM = 4.148808e-3      # s GHz^2 cm^3/pc; reading A1 (paper prints 4.15 ms)
C_LIGHT = 299792458.0   # m/s
MAD_TO_SIGMA = 1.4826   # reading A9


@dataclass(frozen=True)
class Candidate:
    dm_idx: int
    dt_idx: int
    t_idx: int      # index j in the dt-resampled series
    l_pix: int      # signed x offset in [-npix/2, npix/2)
    m_pix: int      # signed y offset
    peak: float
    sigma: float
    snr: float

    @property
    def key(self) -> Tuple[int, int, int]:
        return (self.dm_idx, self.dt_idx, self.t_idx)


# --------------------------------------------------------------------------- O0
def mean_subtract(vis: np.ndarray) -> np.ndarray:
    """complex128 [nint][nbl][nchan][npol]: vis minus its mean over the integrations of the segment,
    separately for every (baseline, channel, polarisation).

    "subtracting the mean visibility in time on timescales less [than] the VLA fringe rate";
    the segment IS that timescale ("the largest size for which mean visibility subtraction is accurate",
    PAPER.md:108).  Reading A21: one plain arithmetic mean over all nint integrations of the
    segment; flagged channels are simply never gridded afterwards (A17), no weights enter the mean."""
    v = np.asarray(vis).astype(np.complex128)
    return v - v.mean(axis=0, keepdims=True)


# --------------------------------------------------------------------------- O1
def delay_table(freqs_hz: np.ndarray, dm_list: np.ndarray, inttime_s: float) -> np.ndarray:
    """int32 [ndm][nchan]: dispersion delay in whole integrations relative to the
    highest channel (readings A1, A3, A4: round half up)."""
    f = np.asarray(freqs_hz, dtype=np.float64) / 1e9
    fmax = f.max()
    dm = np.asarray(dm_list, dtype=np.float64)[:, None]
    # elementwise IEEE float64, evaluated left to right exactly as written (A4)
    x = K_DM * dm * (1.0 / (f * f) - 1.0 / (fmax * fmax))[None, :] / inttime_s
    return np.floor(x + 0.5).astype(np.int32)


# --------------------------------------------------------------------------- O2
def cell_table(uvw_m: np.ndarray, freqs_hz: np.ndarray, npix: int, cell_rad: float,
               chan_weights: Optional[np.ndarray] = None):
    """(iu, iv, keep): int32 [nbl][nchan] signed cell indices and the kept mask.

    u_lambda = u_m f / c; cell size du = 1/(npix*cell); nearest cell, round half
    up; kept iff inside [-npix/2, npix/2) on both axes and channel weight != 0
    (readings A8, A17).  w is ignored (A8)."""
    uvw = np.asarray(uvw_m, dtype=np.float64)
    f = np.asarray(freqs_hz, dtype=np.float64)
    du = 1.0 / (npix * cell_rad)
    half = npix // 2
    ul = uvw[:, 0:1] * f[None, :] / C_LIGHT          # [nbl][nchan], (u*f)/c in this order
    vl = uvw[:, 1:2] * f[None, :] / C_LIGHT
    iu = np.floor(ul / du + 0.5).astype(np.int32)
    iv = np.floor(vl / du + 0.5).astype(np.int32)
    keep = (iu >= -half) & (iu < half) & (iv >= -half) & (iv < half)
    if chan_weights is not None:
        keep &= (np.asarray(chan_weights) != 0)[None, :]
    return iu, iv, keep


# --------------------------------------------------------------------------- O3
def n_images(nint: int, max_delay: int, dt: int, span: int = 0) -> int:
    """Number of output indices j of one (dm, dt): all j with (j+1)*dt <= n_search.

    n_search = nint - max_ch delay[dm] for a single segment (reading A16) or
    min(that, span) when a streaming search span is set (config 5)."""
    n_search = nint - max_delay
    if span > 0:
        n_search = min(n_search, span)
    return max(0, n_search // dt)


def dedisperse_resample(vis: np.ndarray, delay_dm: np.ndarray, dt: int, j: int) -> np.ndarray:
    """complex128 [nbl][nchan]: Stokes-I visibility of resampled integration j.

    s[bl][ch] = mean over q < dt and over pol of vis[j*dt + q + delay[ch]][bl][ch][pol]
    (readings A5 native-resolution delays, A6 decimating boxcar, A7 Stokes I = pol mean)."""
    nint, nbl, nchan, npol = vis.shape
    s = np.zeros((nbl, nchan), dtype=np.complex128)
    for c in range(nchan):
        for q in range(dt):
            t = j * dt + q + int(delay_dm[c])
            s[:, c] += vis[t, :, c, :].astype(np.complex128).sum(axis=1)
    return s / (dt * npol)


# --------------------------------------------------------------------------- O4
def grid_visibilities(s: np.ndarray, iu: np.ndarray, iv: np.ndarray, keep: np.ndarray,
                      npix: int) -> np.ndarray:
    """complex128 [npix][npix] grid G[iv mod N][iu mod N] += s and its Hermitian
    conjugate at the mirrored cell (reading A8; no fftshift in storage, A12)."""
    g = np.zeros((npix, npix), dtype=np.complex128)
    a = iu[keep].astype(np.int64)
    e = iv[keep].astype(np.int64)
    val = s[keep]
    np.add.at(g, (e % npix, a % npix), val)                 # unbuffered scatter-add
    np.add.at(g, ((-e) % npix, (-a) % npix), np.conj(val))
    return g


# --------------------------------------------------------------------------- O5
def image_from_grid(g: np.ndarray, n_w: int) -> np.ndarray:
    """float64 [npix][npix]: Re(ifft2(G)) * N^2 / (2 N_w); a unit point source at
    the phase centre gives 1.0 (reading A8).  numpy ifft2 has the +i sign."""
    n = g.shape[0]
    return np.real(np.fft.ifft2(g)) * (n * n) / (2.0 * n_w)


def image_direct_dft(s: np.ndarray, iu: np.ndarray, iv: np.ndarray, keep: np.ndarray,
                     npix: int) -> np.ndarray:
    """The same image as the direct sum (1/N_w) sum_kept Re(s e^{+2 pi i (iu x + iv y)/N});
    O(N^2 N_vis): tiny grids only.  Used to pin O4+O5."""
    n_w = int(keep.sum())
    y, x = np.mgrid[0:npix, 0:npix]
    img = np.zeros((npix, npix), dtype=np.float64)
    nbl, nchan = s.shape
    for b in range(nbl):
        for c in range(nchan):
            if keep[b, c]:
                ph = 2.0 * np.pi * (int(iu[b, c]) * x + int(iv[b, c]) * y) / npix
                img += s[b, c].real * np.cos(ph) - s[b, c].imag * np.sin(ph)
    return img / n_w


# --------------------------------------------------------------------------- O6
def image_stats(img: np.ndarray):
    """(peak, y, x, sigma, snr): maximum pixel (first in row-major order on ties),
    sigma = 1.4826 * median(|img - median(img)|) over all pixels, snr = peak/sigma
    (0 when sigma == 0) -- readings A9, A10."""
    flat = img.reshape(-1)
    k = int(np.argmax(flat))
    peak = float(flat[k])
    y, x = divmod(k, img.shape[1])
    med = float(np.median(flat))
    sigma = MAD_TO_SIGMA * float(np.median(np.abs(flat - med)))
    snr = peak / sigma if sigma > 0.0 else 0.0
    return peak, y, x, sigma, snr


# --------------------------------------------------------------------------- O8
def candidate_spectrum(vis: np.ndarray, delay_dm: np.ndarray, iu: np.ndarray, iv: np.ndarray,
                       keep: np.ndarray, npix: int, dt: int, j: int, l_pix: int, m_pix: int,
                       half_window: int) -> np.ndarray:
    """float64 [2*half_window + 1][nchan]: the dedispersed dynamic spectrum of the array phased towards
    the candidate pixel -- the "spectrum" half of a candidate visualisation ("candidate
    visualizations", 124-131 "image and spectrum").

    Reading A22: row r is output integration jj = j - half_window + r of the candidate's
    (DM, dt) series; spec[r][ch] = (1/n_ch) sum over the kept baselines of channel ch of
    Re( s[bl][ch] e^{+2 pi i (iu x + iv y)/N} ) with s = dedisperse_resample(vis, delay, dt, jj) (O3),
    (x, y) = (l_pix mod N, m_pix mod N), n_ch = kept baselines of that channel (0 for a channel without
    any: flagged).  The phase uses the GRIDDED cell of each sample, so that the image pixel is exactly the
    weighted channel sum:  image(dm, dt, jj)[y][x] = sum_ch n_ch spec[r][ch] / N_w   (pinned).
    Rows whose integrations fall outside the segment are zero."""
    nint, nbl, nchan, npol = vis.shape
    x, y = l_pix % npix, m_pix % npix
    out = np.zeros((2 * half_window + 1, nchan), dtype=np.float64)
    n_ch = keep.sum(axis=0)
    phase = np.exp(2j * np.pi * ((iu.astype(np.int64) * x + iv.astype(np.int64) * y) % npix) / npix)
    for r in range(2 * half_window + 1):
        jj = j - half_window + r
        if jj < 0 or (jj + 1) * dt + int(np.max(delay_dm)) > nint:
            continue
        s = dedisperse_resample(vis, delay_dm, dt, jj)
        for c in range(nchan):
            if n_ch[c] > 0:
                out[r, c] = np.real(s[keep[:, c], c] * phase[keep[:, c], c]).sum() / n_ch[c]
    return out


# --------------------------------------------------------------------------- O9
def inject_transient(vis: np.ndarray, freqs_hz, uvw_m, inttime_s: float, cell_rad: float, amp: float,
                     l_pix: float, m_pix: float, dm: float, width: int, t0: int) -> np.ndarray:
    """complex128 copy of vis with a mock transient added ("randomly insert mock transient sources into
    data ... inserted after calibration").

    Reading A18: a point source of amplitude `amp` at pixel offset (l, m), i.e. direction cosines
    (l*cell, m*cell), has visibility amp * e^{-2 pi i (u_lambda l + v_lambda m) cell} (sign convention A12);
    it is added to every polarisation product at native integrations t0 + q + delay[ch], q < width, where
    delay[ch] is the O1 delay of DM `dm` (arrival at the top channel at t0); samples that fall outside
    the segment are dropped."""
    out = np.asarray(vis).astype(np.complex128)
    nint = out.shape[0]
    f = np.asarray(freqs_hz, dtype=np.float64)
    uvw = np.asarray(uvw_m, dtype=np.float64)
    delay = delay_table(f, np.array([dm], dtype=np.float64), inttime_s)[0]
    ul = uvw[:, 0:1] * f[None, :] / C_LIGHT
    vl = uvw[:, 1:2] * f[None, :] / C_LIGHT
    sig = amp * np.exp(-2j * np.pi * (ul * l_pix + vl * m_pix) * cell_rad)       # [nbl][nchan]
    for c in range(f.size):
        for q in range(width):
            t = t0 + q + int(delay[c])
            if 0 <= t < nint:
                out[t, :, c, :] += sig[:, c, None]
    return out


# --------------------------------------------------------------------------- O10
LN2 = 0.6931471805599453


def periodicity_nt(nint: int, max_delay: int, max_nt: int = 4096) -> int:
    """Length of the time transform of one DM trial: the largest power of two <= nint - max_delay
    (0 when that is below 64), at most max_nt = 4096 integrations (reading A23: the search transforms
    the first 4096 dedispersed integrations of longer segments)."""
    n = nint - max_delay
    if n < 64:
        return 0
    return min(1 << (int(n).bit_length() - 1), max_nt)


def periodicity_spectrum(vis: np.ndarray, delay_dm: np.ndarray, nt: int) -> np.ndarray:
    """complex128 [nt][nbl][nchan]: S[k] = (1/nt) sum_t s[t] e^{-2 pi i k t / nt} of the dedispersed
    Stokes-I series s[t][bl][ch] = mean_pol vis[t + delay[ch]][bl][ch][pol], t < nt ("reading a time
    segment, transforming it to frequencies with a Fourier transform", PAPER.md:100 footnote 4)."""
    nint, nbl, nchan, npol = vis.shape
    s = np.empty((nt, nbl, nchan), dtype=np.complex128)
    for c in range(nchan):
        d = int(delay_dm[c])
        s[:, :, c] = vis[d:d + nt, :, c, :].astype(np.complex128).mean(axis=2)
    return np.fft.fft(s, axis=0) / nt


def periodicity_image(spec_k: np.ndarray, iu: np.ndarray, iv: np.ndarray, keep: np.ndarray, npix: int) -> np.ndarray:
    """complex128 [npix][npix]: I_k[y][x] = (1/N_w) sum_kept S[k][bl][ch] e^{+2 pi i (iu x + iv y)/N}
    ("imaging each frequency", footnote 4).  S[k] is not the visibility of a real sky, so there is no
    Hermitian completion: the image is complex and its POWER |I_k|^2 is searched (reading A23)."""
    g = np.zeros((npix, npix), dtype=np.complex128)
    np.add.at(g, (iv[keep].astype(np.int64) % npix, iu[keep].astype(np.int64) % npix), spec_k[keep])
    return np.fft.ifft2(g) * (npix * npix) / int(keep.sum())


def periodicity_stats(power: np.ndarray):
    """(peak_amp, y, x, sigma, snr) of one power image: peak_amp = sqrt(max P) (first maximum in
    row-major order), sigma = sqrt(median(P) / ln 2) -- the rms amplitude of a complex Gaussian field
    whose power has that median (P is exponentially distributed on noise) --, snr = peak_amp / sigma
    (reading A23; the estimator is this build's choice: parity unpinned by the paper)."""
    flat = power.reshape(-1)
    k = int(np.argmax(flat))
    y, x = divmod(k, power.shape[1])
    med = float(np.median(flat))
    sigma = float(np.sqrt(med / LN2))
    amp = float(np.sqrt(flat[k]))
    return amp, y, x, sigma, (amp / sigma if sigma > 0.0 else 0.0)


def periodicity_search(vis: np.ndarray, freqs_hz, uvw_m, inttime_s: float, npix: int, cell_rad: float,
                       dm_list, threshold: float, chan_weights: Optional[np.ndarray] = None,
                       keys: Optional[Iterable[Tuple[int, int]]] = None, return_all_stats: bool = False):
    """Periodicity search of one segment: for every DM trial and every positive
    fluctuation frequency k = 1 .. nt/2 image S[k] and threshold the power image.  Candidates carry
    dt_idx = -1 and t_idx = k; order (dm, k)."""
    nint = vis.shape[0]
    delays = delay_table(freqs_hz, dm_list, inttime_s)
    iu, iv, keep = cell_table(uvw_m, freqs_hz, npix, cell_rad, chan_weights)
    want = None if keys is None else set(keys)
    cands: List[Candidate] = []
    stats = {}
    for d in range(len(dm_list)):
        nt = periodicity_nt(nint, int(delays[d].max()))
        ks = [k for k in range(1, nt // 2 + 1) if want is None or (d, k) in want]
        if not ks or not keep.any():
            continue
        spec = periodicity_spectrum(vis, delays[d], nt)
        for k in ks:
            img = periodicity_image(spec[k], iu, iv, keep, npix)
            amp, y, x, sigma, snr = periodicity_stats(img.real ** 2 + img.imag ** 2)
            if return_all_stats:
                stats[(d, k)] = (amp, y, x, sigma, snr)
            if sigma > 0.0 and snr >= threshold:
                cands.append(Candidate(d, -1, k, x if x < npix // 2 else x - npix, y if y < npix // 2 else y - npix,
                                       amp, sigma, snr))
    return (cands, stats) if return_all_stats else cands


# --------------------------------------------------------------------------- O3-O7
def search_image(vis, delays, iu, iv, keep, npix, dm_idx, dt, j) -> np.ndarray:
    """Image of one (dm, dt, j): O3 -> O4 -> O5."""
    s = dedisperse_resample(vis, delays[dm_idx], dt, j)
    g = grid_visibilities(s, iu, iv, keep, npix)
    return image_from_grid(g, int(keep.sum()))


def search(vis: np.ndarray, freqs_hz, uvw_m, inttime_s: float, npix: int, cell_rad: float,
           dm_list, dt_list: Sequence[int], threshold: float,
           chan_weights: Optional[np.ndarray] = None, span: int = 0,
           keys: Optional[Iterable[Tuple[int, int, int]]] = None,
           return_all_stats: bool = False):
    """The whole loop of Fig. 2 for one segment.

    Returns the list of Candidate with snr >= threshold (order: dm, dt, j).  An image with sigma = 0
    (all-zero image) has snr := 0 and yields no candidate whatever the threshold (SURVEY.md 8(b):
    "All-zero image (sigma = 0) => snr := 0, no candidate"; reading A24).  With
    ``keys`` only those (dm_idx, dt_idx, j) are evaluated (sampled parity at full
    sizes).  With ``return_all_stats`` also returns {key: (peak,y,x,sigma,snr)}.
    """
    nint = vis.shape[0]
    delays = delay_table(freqs_hz, dm_list, inttime_s)
    iu, iv, keep = cell_table(uvw_m, freqs_hz, npix, cell_rad, chan_weights)
    n_w = int(keep.sum())
    cands: List[Candidate] = []
    stats = {}
    if keys is None:
        keys = []
        for d in range(len(dm_list)):
            md = int(delays[d].max())
            for k, dt in enumerate(dt_list):
                keys.extend((d, k, j) for j in range(n_images(nint, md, dt, span)))
    for (d, k, j) in keys:
        dt = int(dt_list[k])
        s = dedisperse_resample(vis, delays[d], dt, j)
        g = grid_visibilities(s, iu, iv, keep, npix)
        img = image_from_grid(g, n_w) if n_w > 0 else np.zeros((npix, npix))
        peak, y, x, sigma, snr = image_stats(img)
        if return_all_stats:
            stats[(d, k, j)] = (peak, y, x, sigma, snr)
        if sigma > 0.0 and snr >= threshold:      # sigma = 0 (all-zero image): snr := 0, never a candidate (A24)
            l = x if x < npix // 2 else x - npix
            m = y if y < npix // 2 else y - npix
            cands.append(Candidate(d, k, j, l, m, peak, sigma, snr))
    if return_all_stats:
        return cands, stats
    return cands
