"""GPU parity of the candidate cut-out: rf_cand_spectrum against oracle O8, element by
element, including rows that fall outside the segment, flagged channels and the fused mean subtraction."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu


def _plan(cfg, nint, dms, dts, weights=None):
    import paper_1802_03084_b200 as R
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    plan = R.Plan(f, uvw, cfg.npol, nint, cfg.inttime_s, cfg.npix, cell, dms, dts, cfg.threshold)
    if weights is not None:
        plan.set_chan_weights(weights)
    return plan, f, uvw, cell


def _check(got, ref):
    assert got.shape == ref.shape and got.dtype == np.float32
    assert np.abs(got - ref).max() <= 1e-5 * np.abs(ref).max()
    assert ((ref == 0) <= (got == 0)).all()              # rows / channels that must be exactly zero


def test_spectrum_tiny_all_cases():
    import torch
    cfg = W.get_config("tiny")
    dms, dts = W.dm_list(cfg), (1, 2, 3)
    w = np.ones(cfg.nchan, dtype=np.float32); w[[3, 17]] = 0
    plan, f, uvw, cell = _plan(cfg, cfg.nint, dms, dts, w)
    vis = W.make_segment(cfg, persistent=[(3.0, -7, 4)])
    d = torch.from_numpy(vis).cuda()
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell, w)
    cases = [(2, 0, 21, 8, -5, 12), (3, 1, 9, -20, 13, 6), (0, 0, 2, 0, 0, 5), (7, 2, 9, 31, -32, 4), (5, 0, 40, 8, -5, 10)]
    for (dm, k, j, l, m, hw) in cases:              # windows reach before t = 0 and past the valid range
        ref = O.candidate_spectrum(vis, delays[dm], iu, iv, keep, cfg.npix, dts[k], j, l, m, hw)
        _check(plan.cand_spectrum(d, dm, k, j, l, m, hw), ref)
    # with the fused mean subtraction the constant source disappears from the spectrum
    plan.set_meansub(True)
    sub = O.mean_subtract(vis)
    ref = O.candidate_spectrum(sub, delays[2], iu, iv, keep, cfg.npix, 1, 21, -7, 4, 8)
    got = plan.cand_spectrum(d, 2, 0, 21, -7, 4, 8)
    assert np.abs(got - ref).max() <= 2e-5 * max(np.abs(ref).max(), 1.0)
    raw = O.candidate_spectrum(vis, delays[2], iu, iv, keep, cfg.npix, 1, 21, -7, 4, 8)
    assert raw.mean() > 2.5 and abs(got.mean()) < 0.1
    plan.destroy()


def test_spectrum_lband_at_a_candidate():
    """Full-size L-band segment: search, take the strongest candidate, cut out its spectrum; the weighted
    channel sum of the centre row reproduces the candidate's peak (the image pixel), and the whole window
    matches the oracle."""
    import torch
    cfg = W.get_config("lband")
    dms = W.dm_list(cfg)
    plan, f, uvw, cell = _plan(cfg, cfg.nint, dms, cfg.dt_list)
    vis = W.make_segment(cfg)
    d = torch.from_numpy(vis).cuda()
    gpu, n = plan.search(d, capacity=1 << 17)
    best = max(gpu, key=lambda c: c["snr"])
    dm, k, j, l, m = (int(best[x]) for x in ("dm_idx", "dt_idx", "t_idx", "l_pix", "m_pix"))
    hw = 8
    got = plan.cand_spectrum(d, dm, k, j, l, m, hw)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    ref = O.candidate_spectrum(vis, delays[dm], iu, iv, keep, cfg.npix, cfg.dt_list[k], j, l, m, hw)
    _check(got, ref)
    n_ch = keep.sum(axis=0)
    pixel = float((got[hw].astype(np.float64) * n_ch).sum() / keep.sum())
    assert abs(pixel - float(best["peak"])) <= 1e-4 * float(best["peak"])
    plan.destroy()
