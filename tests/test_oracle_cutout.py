"""Pins of the cut-out oracle O8 (phased, dedispersed spectrum at a candidate pixel; PAPER.md:88, 124-131;
SURVEY.md 8f-2): the channel-sum identity with the imaging oracle, the dispersion sweep of an injected
source seen at a wrong DM, and a pure-Python brute force."""
import cmath
import math

import numpy as np

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401


def _setup(cfg, dms):
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    return f, uvw, cell, iu, iv, keep, O.delay_table(f, np.asarray(dms, dtype=float), cfg.inttime_s)


def test_weighted_channel_sum_is_the_image_pixel():
    """image(dm, dt, jj)[y][x] = sum_ch n_ch spec[r][ch] / N_w for every row of the window, any pixel,
    on noisy data: pins O8 to O3-O5 (ifft2 route) through a different route (per-channel direct sum)."""
    cfg = W.get_config("tiny")
    f, uvw, cell, iu, iv, keep, delays = _setup(cfg, W.dm_list(cfg))
    w = np.ones(cfg.nchan); w[[3, 17]] = 0
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell, w)
    vis = W.make_segment(cfg)
    n_w, n_ch = keep.sum(), keep.sum(axis=0)
    for (d, dt, j, l, m) in [(2, 1, 21, 8, -5), (5, 2, 7, -20, 13), (0, 4, 3, 0, 0)]:
        spec = O.candidate_spectrum(vis, delays[d], iu, iv, keep, cfg.npix, dt, j, l, m, 2)
        assert spec.shape == (5, cfg.nchan) and (spec[:, [3, 17]] == 0).all()
        for r in range(5):
            img = O.search_image(vis, delays, iu, iv, keep, cfg.npix, d, dt, j - 2 + r)
            assert abs((spec[r] * n_ch).sum() / n_w - img[m % cfg.npix, l % cfg.npix]) < 1e-12


def test_sweep_of_an_injected_source():
    """Noise-free width-1 source at DM 50, t0 = 20, pixel (8, -5).  At the matched trial every channel
    lights up in the row of t0 with the closed-form amplitude A * (gridding decorrelation of that channel);
    at DM 0 the same power runs along the dispersion sweep row = t0 + delay_inj[ch]."""
    cfg = W.get_config("tiny")
    dms = [0.0, 50.0]
    f, uvw, cell, iu, iv, keep, delays = _setup(cfg, dms)
    vis = W.make_segment(cfg, noise=False)
    hw = 12
    spec = O.candidate_spectrum(vis, delays[1], iu, iv, keep, cfg.npix, 1, 20, 8, -5, hw)
    du = 1.0 / (cfg.npix * cell)
    ul = uvw[:, 0:1] * f[None, :] / O.C_LIGHT
    vl = uvw[:, 1:2] * f[None, :] / O.C_LIGHT
    decor = np.cos(2 * np.pi * ((iu * du - ul) * 8 + (iv * du - vl) * (-5)) * cell).mean(axis=0)   # per channel
    assert np.abs(spec[hw] - 2.0 * decor).max() < 1e-6
    rest = np.delete(spec, hw, axis=0)
    assert np.abs(rest).max() < 1e-6
    sweep = O.candidate_spectrum(vis, delays[0], iu, iv, keep, cfg.npix, 1, 20, 8, -5, hw)
    for c in range(cfg.nchan):
        r = hw + int(delays[1][c])
        if r < 2 * hw + 1:
            assert abs(sweep[r, c] - 2.0 * decor[c]) < 1e-6
            assert np.abs(np.delete(sweep[:, c], r)).max() < 1e-6


def test_brute_force_tiny():
    rng = np.random.default_rng(2)
    nint, nbl, nchan, npol, n = 12, 3, 4, 2, 8
    vis = (rng.normal(size=(nint, nbl, nchan, npol)) + 1j * rng.normal(size=(nint, nbl, nchan, npol))).astype(np.complex64)
    iu = rng.integers(-4, 4, size=(nbl, nchan)).astype(np.int32)
    iv = rng.integers(-4, 4, size=(nbl, nchan)).astype(np.int32)
    keep = rng.random((nbl, nchan)) > 0.25
    keep[:, 1] = False
    delay = np.array([3, 2, 1, 0], dtype=np.int32)
    dt, j, l, m, hw = 2, 2, -3, 2, 3
    spec = O.candidate_spectrum(vis, delay, iu, iv, keep, n, dt, j, l, m, hw)
    for r in range(2 * hw + 1):
        jj = j - hw + r
        for c in range(nchan):
            acc, cnt = 0.0, 0
            ok = jj >= 0 and (jj + 1) * dt + 3 <= nint
            for b in range(nbl):
                if ok and keep[b, c]:
                    s = sum(complex(vis[jj * dt + q + delay[c], b, c, p]) for q in range(dt) for p in range(npol)) / (dt * npol)
                    acc += (s * cmath.exp(2j * math.pi * (int(iu[b, c]) * (l % n) + int(iv[b, c]) * (m % n)) / n)).real
                    cnt += 1
            assert abs(spec[r, c] - (acc / cnt if cnt else 0.0)) < 1e-12
