"""Pins of the injection oracle O9 (mock transients): energy and placement
counted by hand, the closed-form image response, recovery by the search oracle, and agreement with the
independently written signal model of the input generator."""
import numpy as np

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401


def _geo(cfg):
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    return f, uvw, W.default_cell_rad(cfg, uvw)


def test_energy_placement_and_drop_outside():
    cfg = W.get_config("tiny")
    f, uvw, cell = _geo(cfg)
    zero = np.zeros((cfg.nint, cfg.nbl, cfg.nchan, cfg.npol), dtype=np.complex64)
    out = O.inject_transient(zero, f, uvw, cfg.inttime_s, cell, 2.0, 8, -5, 50.0, 3, 20)
    # unit-modulus phases: every (bl, ch, pol) carries |A|^2 in exactly `width` integrations
    assert abs((np.abs(out) ** 2).sum() - 4.0 * cfg.nbl * cfg.nchan * cfg.npol * 3) < 1e-9
    delay = O.delay_table(f, np.array([50.0]), cfg.inttime_s)[0]
    assert delay[0] == 11 and delay[-1] == 0                 # the config-1 DM-50 sweep
    for c in (0, 13, 31):
        on = np.nonzero(np.abs(out[:, 0, c, 0]) > 0)[0]
        assert list(on) == [20 + delay[c] + q for q in range(3)]
    assert np.allclose(out[20, :, 31, 0], out[20, :, 31, 1])  # both polarisation products
    # top channel phase: A e^{-2 pi i (u l + v m) cell}, checked against a hand-expanded cos/sin
    b = 7
    arg = 2 * np.pi * (uvw[b, 0] * f[31] / O.C_LIGHT * 8 + uvw[b, 1] * f[31] / O.C_LIGHT * (-5)) * cell
    assert abs(out[20, b, 31, 0] - 2.0 * (np.cos(arg) - 1j * np.sin(arg))) < 1e-12
    # a source starting 2 integrations before the end: low channels fall off the segment and are dropped
    late = O.inject_transient(zero, f, uvw, cfg.inttime_s, cell, 1.0, 0, 0, 50.0, 1, cfg.nint - 2)
    kept = (np.abs(late[:, 0, :, 0]) > 0).sum()
    assert kept == int((delay <= 1).sum()) and kept < cfg.nchan


def test_image_response_closed_form_and_recovery():
    """at the matched DM and width the image peaks at (m mod N, l mod N) with amplitude
    (A/N_w) sum cos(2 pi ((iu du - u) l + (iv du - v) m) cell); the search oracle recovers it."""
    cfg = W.get_config("tiny")
    f, uvw, cell = _geo(cfg)
    zero = np.zeros((cfg.nint, cfg.nbl, cfg.nchan, cfg.npol), dtype=np.complex64)
    dms = W.dm_list(cfg)
    vis = O.inject_transient(zero, f, uvw, cfg.inttime_s, cell, 1.5, -12, 9, float(dms[3]), 2, 16)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    img = O.search_image(vis, delays, iu, iv, keep, cfg.npix, 3, 2, 8)
    peak, y, x, _, _ = O.image_stats(img)
    du = 1.0 / (cfg.npix * cell)
    ul, vl = uvw[:, 0:1] * f[None, :] / O.C_LIGHT, uvw[:, 1:2] * f[None, :] / O.C_LIGHT
    expect = 1.5 * np.cos(2 * np.pi * ((iu * du - ul) * (-12) + (iv * du - vl) * 9) * cell)[keep].mean()
    assert (y, x) == (9, cfg.npix - 12) and abs(peak - expect) < 1e-9
    noisy = O.inject_transient(W.make_segment(cfg, inject=False), f, uvw, cfg.inttime_s, cell, 1.5, -12, 9,
                               float(dms[3]), 2, 16)
    cands = O.search(noisy, f, uvw, cfg.inttime_s, cfg.npix, cell, dms, (1, 2), cfg.threshold)
    best = max(cands, key=lambda c: c.snr)
    # the S/N of the image statistic is limited by the source's own sidelobes, so the width-1
    # and width-2 images of the burst score alike: the best one is at its DM, pixel and native time
    assert (best.dm_idx, best.l_pix, best.m_pix) == (3, -12, 9)
    assert best.t_idx * (1, 2)[best.dt_idx] in (16, 17)
    matched = [c for c in cands if c.key == (3, 1, 8)]
    assert matched and (matched[0].l_pix, matched[0].m_pix) == (-12, 9)


def test_agrees_with_the_generator_signal_model():
    """workloads.make_segment was written separately (float32 signal); same source, same samples."""
    cfg = W.get_config("tiny")
    f, uvw, cell = _geo(cfg)
    src = W.generate.Transient(0.7, 21, -30, 90.0, 4, 5)
    gen = W.make_segment(cfg, noise=False, sources=[src])
    zero = np.zeros_like(gen)
    ref = O.inject_transient(zero, f, uvw, cfg.inttime_s, cell, 0.7, 21, -30, 90.0, 4, 5)
    assert np.abs(gen - ref).max() < 2e-7
