"""GPU parity of the prep stage: mean-visibility subtraction in place
(rf_prep_meansub) and fused into the search (rf_plan_set_meansub), against oracle O0 + the search oracle."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu

PIX_TOL, SNR_TOL, NEAR_THR = 1e-4, 1e-3, 2e-3


def _plan(cfg, nint, dms, dts, thr, npix=None):
    import paper_1802_03084_b200 as R
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    return R.Plan(f, uvw, cfg.npol, nint, cfg.inttime_s, npix or cfg.npix, cell, dms, dts, thr), f, uvw, cell


def test_meansub_in_place_matches_oracle():
    """Element by element on a ragged shape (nint not a multiple of the kernel's time slices)."""
    import torch
    cfg = W.get_config("tiny")
    nint = 61
    vis = W.make_segment(cfg, persistent=[(3.0, -7, 4)])[:nint].copy()
    vis[:, 3, 5, 1] += 1000.0 + 500.0j                       # a large offset on one element only
    plan, *_ = _plan(cfg, nint, W.dm_list(cfg), cfg.dt_list, cfg.threshold)
    d = torch.from_numpy(vis).cuda()
    plan.prep_meansub(d)
    torch.cuda.synchronize()
    ref = O.mean_subtract(vis)
    got = d.cpu().numpy()
    # float32 storage: the only error is the rounding of (x - mean) and of the mean itself
    scale = np.maximum(np.abs(vis), 1.0)
    assert (np.abs(got - ref) <= 2.5e-7 * scale).all()
    assert np.abs(got.astype(np.complex128).mean(axis=0)).max() < 1e-4
    plan.destroy()


def _compare(gpu, ref_cands, thr):
    g = {(int(c["dm_idx"]), int(c["dt_idx"]), int(c["t_idx"])): c for c in gpu}
    o = {c.key: c for c in ref_cands}
    for key in set(g) ^ set(o):
        snr = o[key].snr if key in o else float(g[key]["snr"])
        assert abs(snr - thr) <= NEAR_THR * thr, (key, snr)
    for key in set(g) & set(o):
        assert abs(float(g[key]["snr"]) - o[key].snr) <= SNR_TOL * o[key].snr, key
        assert (int(g[key]["l_pix"]), int(g[key]["m_pix"])) == (o[key].l_pix, o[key].m_pix), key
    return len(set(g) & set(o))


def test_search_with_meansub_tiny_full_parity():
    """Config 1 with a bright persistent source: without prep it dominates every image; with prep the
    candidate list equals the oracle's on mean_subtract(vis) (exact statistics path, npix 64)."""
    import torch
    cfg = W.get_config("tiny")
    vis = W.make_segment(cfg, persistent=[(5.0, -7, 4)])
    plan, f, uvw, cell = _plan(cfg, cfg.nint, W.dm_list(cfg), cfg.dt_list, cfg.threshold)
    d = torch.from_numpy(vis).cuda()
    raw, _ = plan.search(d)
    assert len(raw) > 300 and (np.abs(raw["l_pix"] + 7) <= 0).mean() > 0.9      # the constant source everywhere
    plan.set_meansub(True)
    gpu, n = plan.search(d)
    assert np.array_equal(d.cpu().numpy(), vis)                                # the input is not modified
    ref = O.search(O.mean_subtract(vis), f, uvw, cfg.inttime_s, cfg.npix, cell, W.dm_list(cfg), cfg.dt_list,
                   cfg.threshold)
    assert _compare(gpu, ref, cfg.threshold) >= 20
    best = max(gpu, key=lambda c: c["snr"])
    assert (int(best["l_pix"]), int(best["m_pix"])) == (8, -5)                 # the transient, not the constant
    # pixel parity of one image through the debug hook
    delays = O.delay_table(f, W.dm_list(cfg), cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    refimg = O.search_image(O.mean_subtract(vis), delays, iu, iv, keep, cfg.npix, 2, 1, 21)
    img, st = plan.debug_image(d, 2, 0, 21)
    assert np.abs(img - refimg).max() <= PIX_TOL * np.sqrt((refimg ** 2).mean())
    plan.destroy()


def test_search_with_meansub_lband_tree_and_generic():
    """npix 512, widths on the boxcar tree (1, 2, 4) and off it (3): fused subtraction in both readers,
    against the oracle on sampled images and on the candidate keys of those images."""
    import torch
    cfg = W.get_config("lband")
    nint, dts = 160, (1, 2, 3, 4)
    dms = W.dm_list(cfg)[:12:4]
    src = [W.generate.Transient(0.3, 40, -77, float(dms[1]), 2, 50)]
    vis = W.make_segment(cfg, sources=src, persistent=[(1.0, 100, 30), (0.5, -20, -60)])[:nint].copy()
    plan, f, uvw, cell = _plan(cfg, nint, dms, dts, 6.5)
    plan.set_meansub(True)
    d = torch.from_numpy(vis).cuda()
    gpu, n = plan.search(d, capacity=1 << 14)
    g = {(int(c["dm_idx"]), int(c["dt_idx"]), int(c["t_idx"])): c for c in gpu}
    sub = O.mean_subtract(vis)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    hits = 0
    for (dm, k, j) in [(1, 0, 50), (1, 1, 25), (1, 2, 16), (1, 3, 12), (0, 0, 3), (2, 2, 20), (2, 1, 7)]:
        ref = O.search_image(sub, delays, iu, iv, keep, cfg.npix, dm, dts[k], j)
        peak, y, x, sigma, snr = O.image_stats(ref)
        img, st = plan.debug_image(d, dm, k, j)
        assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean()), (dm, k, j)
        assert abs(float(st["snr"]) - snr) <= SNR_TOL * snr, (dm, k, j)
        if abs(snr - 6.5) > NEAR_THR * 6.5:
            assert ((dm, k, j) in g) == (snr >= 6.5), (dm, k, j, snr)
        hits += (dm, k, j) in g
    assert hits >= 2
    plan.destroy()
