"""Pins of the prep oracle O0 (mean-visibility subtraction).
-m "not gpu": closed forms, invariants, brute force, and the imaging identity it exists for."""
import numpy as np

import oracle as O
import workloads as W


def test_closed_form_constant_plus_impulse():
    """vis[t] = c + a*delta(t, t0)  ->  out[t] = a*(delta(t, t0) - 1/n): hand-computed numbers."""
    n = 8
    vis = np.full((n, 1, 1, 1), 3.0 - 2.0j, dtype=np.complex64)
    vis[5] += 4.0 + 8.0j
    out = O.mean_subtract(vis)
    expect = np.full(n, -(4.0 + 8.0j) / 8)           # -0.5 - 1.0j
    expect[5] = (4.0 + 8.0j) * 7 / 8                 # 3.5 + 7.0j
    assert out.dtype == np.complex128 and out.shape == vis.shape
    assert np.allclose(out[:, 0, 0, 0], expect, rtol=0, atol=1e-15)


def test_zero_mean_idempotent_and_per_element():
    rng = np.random.default_rng(5)
    vis = (rng.normal(size=(16, 3, 4, 2)) + 1j * rng.normal(size=(16, 3, 4, 2))).astype(np.complex64)
    out = O.mean_subtract(vis)
    assert np.abs(out.mean(axis=0)).max() < 1e-15
    assert np.abs(O.mean_subtract(out) - out).max() < 1e-15
    # every (bl, ch, pol) uses its own mean: changing one element's offset changes only that element
    vis2 = vis.copy()
    vis2[:, 1, 2, 0] += 10.0
    assert np.abs(O.mean_subtract(vis2) - out).max() < 1e-5
    # brute force, pure Python
    for b in range(3):
        for c in range(4):
            for p in range(2):
                m = sum(complex(vis[t, b, c, p]) for t in range(16)) / 16
                for t in range(16):
                    assert abs(out[t, b, c, p] - (complex(vis[t, b, c, p]) - m)) < 1e-14


def test_constant_source_vanishes_and_transient_survives():
    """What the step is for ("This removes constant sources"): the image of a persistent
    source is 1.0 x amplitude before and identically zero after; by linearity the image of a width-1
    transient keeps (1 - 1/nint) of its peak at its own time at the matched DM (DM 0 here)."""
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    delays = O.delay_table(f, np.array([0.0]), cfg.inttime_s)
    const = W.make_segment(cfg, noise=False, sources=[], persistent=[(3.0, -7, 4)])
    img = O.search_image(const, delays, iu, iv, keep, cfg.npix, 0, 1, 11)
    peak, y, x, _, _ = O.image_stats(img)
    assert (y, x) == (4, cfg.npix - 7) and 0.9 * 3.0 < peak <= 3.0      # gridding decorrelation only
    gone = O.search_image(O.mean_subtract(const), delays, iu, iv, keep, cfg.npix, 0, 1, 11)
    assert np.abs(gone).max() < 1e-6 * peak                            # float32 rounding of the input phases
    src = [W.generate.Transient(2.0, 8, -5, 0.0, 1, 20)]
    both = W.make_segment(cfg, noise=False, sources=src, persistent=[(3.0, -7, 4)])
    only = W.make_segment(cfg, noise=False, sources=src)
    a = O.search_image(O.mean_subtract(both), delays, iu, iv, keep, cfg.npix, 0, 1, 20)
    b = O.search_image(only, delays, iu, iv, keep, cfg.npix, 0, 1, 20)
    assert np.abs(a - (1.0 - 1.0 / cfg.nint) * b).max() < 1e-6 * np.abs(b).max()
    off = O.search_image(O.mean_subtract(both), delays, iu, iv, keep, cfg.npix, 0, 1, 40)
    assert np.abs(off + b / cfg.nint).max() < 1e-6 * np.abs(b).max()   # the -a/n pedestal at every other time
