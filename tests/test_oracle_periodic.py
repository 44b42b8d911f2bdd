"""Pins of the periodicity oracle O10 (PAPER.md:100 footnote 4, 104): the inverse time
transform of the frequency images is the transient-search image, a pulse train lands on its harmonics with
the closed-form amplitude, the noise level has its analytic value, and a pure-Python brute force."""
import cmath
import math

import numpy as np

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401


def _geo(cfg, npix=None):
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    iu, iv, keep = O.cell_table(uvw, f, npix or cfg.npix, cell)
    return f, uvw, cell, iu, iv, keep


def test_transform_length():
    assert O.periodicity_nt(1024, 0) == 1024 and O.periodicity_nt(1024, 624) == 256
    assert O.periodicity_nt(64, 0) == 64 and O.periodicity_nt(64, 1) == 0 and O.periodicity_nt(200, 9) == 128


def test_inverse_time_transform_is_the_transient_image():
    """Re( sum_k I_k e^{+2 pi i k t / nt} ) = image(dm, dt = 1, t) of O3-O5 for every t < nt: ties the time
    transform, its 1/nt scale, the un-mirrored gridding and the 1/N_w scale to the pinned imaging oracle."""
    cfg = W.get_config("tiny")
    f, uvw, cell, iu, iv, keep = _geo(cfg)
    import dataclasses
    vis = W.make_segment(dataclasses.replace(cfg, nint=70))
    dms = np.array([0.0, 20.0])
    delays = O.delay_table(f, dms, cfg.inttime_s)
    nt = O.periodicity_nt(70, int(delays[1].max()))
    assert nt == 64
    spec = O.periodicity_spectrum(vis, delays[1], nt)
    imgs = np.stack([O.periodicity_image(spec[k], iu, iv, keep, cfg.npix) for k in range(nt)])
    for t in (0, 21, 63):
        back = np.tensordot(np.exp(2j * np.pi * np.arange(nt) * t / nt), imgs, axes=1)
        ref = O.search_image(vis, delays, iu, iv, keep, cfg.npix, 1, 1, t)
        assert np.abs(back.real - ref).max() < 1e-12 * max(1.0, np.abs(ref).max())


def test_pulse_train_lands_on_its_harmonics():
    cfg = W.get_config("tiny")
    f, uvw, cell, iu, iv, keep = _geo(cfg)
    zero = np.zeros((cfg.nint, cfg.nbl, cfg.nchan, cfg.npol), dtype=np.complex64)
    vis = zero.astype(np.complex128)
    for t0 in range(3, cfg.nint, 8):                          # period 8 integrations, width 1, DM 0
        vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.6, 8, -5, 0.0, 1, t0)
    cands, stats = O.periodicity_search(vis, f, uvw, cfg.inttime_s, cfg.npix, cell,
                                        np.array([0.0]), 5.0, return_all_stats=True)
    du = 1.0 / (cfg.npix * cell)
    ul, vl = uvw[:, 0:1] * f[None, :] / O.C_LIGHT, uvw[:, 1:2] * f[None, :] / O.C_LIGHT
    # |mean e^{i delta}|, delta = phase error of snapping each sample to its cell (the power image keeps the
    # imaginary part that the real transient image drops)
    decor = abs(np.exp(2j * np.pi * ((iu * du - ul) * 8 + (iv * du - vl) * (-5)) * cell)[keep].mean())
    assert sorted(stats) == [(0, k) for k in range(1, 33)]
    for k in (8, 16, 24, 32):                                 # harmonics of nt / period = 64 / 8
        amp, y, x, sigma, snr = stats[(0, k)]
        assert (y, x) == (cfg.npix - 5, 8) and abs(amp - 1.6 / 8 * decor) < 1e-12
    assert max(stats[(0, k)][0] for k in range(1, 33) if k % 8) < 1e-12
    assert {c.t_idx for c in cands} >= {8, 16, 24, 32} and all(c.dt_idx == -1 for c in cands)


def test_noise_level_and_statistics():
    power = np.array([[1.0, 9.0, 4.0], [9.0, 2.0, 3.0]])
    amp, y, x, sigma, snr = O.periodicity_stats(power)
    assert (amp, y, x) == (3.0, 0, 1) and abs(sigma - math.sqrt(3.5 / math.log(2.0))) < 1e-15
    assert O.periodicity_stats(np.zeros((4, 4)))[4] == 0.0
    # noise: E|I_k|^2 = 2 / (npol nt N_w) for unit-variance parts; the median estimator agrees to a few per cent
    cfg = W.get_config("tiny")
    f, uvw, cell, iu, iv, keep = _geo(cfg)
    vis = W.make_segment(cfg, inject=False)
    _, stats = O.periodicity_search(vis, f, uvw, cfg.inttime_s, cfg.npix, cell, np.array([0.0]), 1e9, return_all_stats=True)
    est = np.mean([s[3] ** 2 for s in stats.values()])
    assert abs(est / (2.0 / (cfg.npol * 64 * keep.sum())) - 1.0) < 0.05


def test_brute_force_tiny():
    rng = np.random.default_rng(9)
    nint, nbl, nchan, npol, n = 70, 3, 3, 2, 8
    vis = (rng.normal(size=(nint, nbl, nchan, npol)) + 1j * rng.normal(size=(nint, nbl, nchan, npol))).astype(np.complex64)
    iu = rng.integers(-4, 4, size=(nbl, nchan)).astype(np.int32)
    iv = rng.integers(-4, 4, size=(nbl, nchan)).astype(np.int32)
    keep = np.ones((nbl, nchan), dtype=bool); keep[1, 2] = False
    delay = np.array([5, 2, 0], dtype=np.int32)
    nt = O.periodicity_nt(nint, 5)
    spec = O.periodicity_spectrum(vis, delay, nt)
    k = 5
    img = O.periodicity_image(spec[k], iu, iv, keep, n)
    for (y, x) in [(0, 0), (3, 6), (7, 1)]:
        acc = 0j
        for b in range(nbl):
            for c in range(nchan):
                if keep[b, c]:
                    sk = sum(sum(complex(vis[t + delay[c], b, c, p]) for p in range(npol)) / npol
                             * cmath.exp(-2j * math.pi * k * t / nt) for t in range(nt)) / nt
                    acc += sk * cmath.exp(2j * math.pi * (int(iu[b, c]) * x + int(iv[b, c]) * y) / n)
        assert abs(img[y, x] - acc / keep.sum()) < 1e-12
