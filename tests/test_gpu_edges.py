"""GPU parity on the edges of the hot path: image sizes and polarisation counts the five configs do not
use, degenerate plans (nothing kept, a DM that sweeps past the segment), unsorted trial lists, candidate
overflow, ragged time ranges.  Everything is compared with the float64 oracle on the same bytes."""
import numpy as np
import pytest

import oracle as O
import oracle_pool as OP
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu

PIX_TOL, SNR_TOL, NEAR_THR = 1e-4, 1e-3, 2e-3


def _rand_vis(shape, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(shape, dtype=np.float32) + 1j * rng.standard_normal(shape, dtype=np.float32)).astype(np.complex64)


def _compare_all(plan, dvis, vis, f, uvw, cell, npix, dms, dts, thr, inttime, weights=None, min_match=1):
    """Whole candidate list against the oracle's statistics of EVERY image of the loop: membership away from the
    threshold (A11), S/N, peak pixel up to float32-rounding ties (A20), device-counted images."""
    gpu, n = plan.search(dvis, capacity=1 << 15)
    assert n == len(gpu)
    delays = O.delay_table(f, dms, inttime)
    keys = OP.all_keys(delays, vis.shape[0], dts)
    stats = OP.oracle_stats(vis, f, uvw, inttime, npix, cell, dms, dts, keys, chan_weights=weights)
    assert plan.num_images() == len(stats)
    ctr = plan.get_counters()
    assert ctr["images"] == len(stats) or ctr["n_kept"] == 0          # counted on the device
    g = {(int(c["dm_idx"]), int(c["dt_idx"]), int(c["t_idx"])): c for c in gpu}
    assert len(g) == len(gpu)
    o = {c.key: c for c in OP.candidates_from_stats(stats, npix, thr)}
    for key in set(g) ^ set(o):
        assert abs(stats[key][4] - thr) <= NEAR_THR * max(thr, 1e-30), (key, stats[key][4])
    for key in set(g) & set(o):
        assert abs(float(g[key]["snr"]) - o[key].snr) <= SNR_TOL * o[key].snr, key
        assert abs(float(g[key]["peak"]) - o[key].peak) <= 1e-4 * abs(o[key].peak) + 1e-7, key
        assert OP.peak_pixel_ok(int(g[key]["l_pix"]), int(g[key]["m_pix"]), stats[key], npix), (key, stats[key])
    assert len(set(g) & set(o)) >= min_match
    assert ctr["stats_overflow"] == 0
    return g


@pytest.mark.parametrize("npix,npol,dts", [(256, 2, (1, 2, 4, 8)), (128, 1, (1, 2, 5)), (256, 4, (1, 3)), (64, 4, (2, 4))])
def test_small_sizes_every_image(npix, npol, dts):
    """Whole candidate lists at threshold 0 (every image is emitted): npix 256 runs the boxcar tree with two
    rows per warp, 128 / 64 the exact-statistics kernel; npol 1 and 4; widths on and off the tree."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * (1.0 if npix <= 128 else 0.8)
    nint = 43                                               # ragged: not a multiple of any width or block
    dms = np.array([0.0, 60.0, 25.0])                       # unsorted trials
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, npol), 100 + npix + npol)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 5, -9, 60.0, 2, 12).astype(np.complex64)
    plan = R.Plan(f, uvw, npol, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    g = _compare_all(plan, torch.from_numpy(vis).cuda(), vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s,
                     min_match=20)
    assert len(g) == plan.num_images()
    # pixel parity of one image per width through the debug hook
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    d = torch.from_numpy(vis).cuda()
    for k, dt in enumerate(dts):
        ref = O.search_image(vis, delays, iu, iv, keep, npix, 1, dt, 12 // dt)
        img, _ = plan.debug_image(d, 1, k, 12 // dt)
        assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean()), (npix, dt)
    plan.destroy()


def test_offtree_widths_per_image_fallback():
    """Widths off the tree whose boxcar-sum arrays do not fit the workspace budget take the per-image path
    (B7).  rf_plan_set_tuning(RF_TUNE_AUX_WIDTHS, 0) forces that decision on a small plan; the
    candidate list must be the oracle's either way, and identical keys to the plan that uses the sum arrays."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    npix, npol, nint, dts = 256, 2, 43, (1, 3, 6)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * 0.8
    dms = np.array([0.0, 25.0, 60.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, npol), 777)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 5, -9, 60.0, 3, 12).astype(np.complex64)
    d = torch.from_numpy(vis).cuda()
    plan_aux = R.Plan(f, uvw, npol, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    g_aux = _compare_all(plan_aux, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=20)
    plan_aux.destroy()
    plan = R.Plan(f, uvw, npol, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    plan.set_tuning(R.binding.RF_TUNE_AUX_WIDTHS, 0)
    g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=20)
    plan.destroy()
    assert set(g) == set(g_aux) and len(g) == len(g_aux)
    for key in g:
        assert abs(float(g[key]["snr"]) - float(g_aux[key]["snr"])) <= SNR_TOL * float(g[key]["snr"]), key


def test_degenerate_plans():
    """Nothing kept (all channels flagged): zero candidates, zero image, no crash.  A DM whose sweep is
    longer than the segment contributes no images.  Unsorted channel order gives the same tables as the oracle."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    vis = W.make_segment(cfg)
    d = torch.from_numpy(vis).cuda()
    dms = np.array([0.0, 50.0, 400.0])                      # DM 400: max delay 89 > 64 integrations
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, dms, (1,), cfg.threshold)
    assert plan.num_t(2, 0) == 0 and plan.num_t(0, 0) == 64 and plan.num_t(1, 0) == 64 - 11
    gpu, n = plan.search(d)
    assert n > 0 and (gpu["dm_idx"] < 2).all()
    plan.set_chan_weights(np.zeros(cfg.nchan, dtype=np.float32))
    gpu, n = plan.search(d)
    assert n == 0 and plan.get_counters()["n_kept"] == 0
    img, st = plan.debug_image(d, 0, 0, 5)
    assert not img.any() and float(st["snr"]) == 0.0
    plan.destroy()
    # channels given in reverse order: tables and candidates follow the caller's order
    perm = np.arange(cfg.nchan)[::-1].copy()
    plan = R.Plan(f[perm], uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, W.dm_list(cfg), (1,), cfg.threshold)
    delay, cells, keep = plan.get_tables()
    assert np.array_equal(delay, O.delay_table(f[perm], W.dm_list(cfg), cfg.inttime_s))
    vis_p = np.ascontiguousarray(vis[:, :, perm, :])
    a, _ = plan.search(torch.from_numpy(vis_p).cuda())
    ref = O.search(vis, f, uvw, cfg.inttime_s, cfg.npix, cell, W.dm_list(cfg), (1,), cfg.threshold)
    ka = {(int(c["dm_idx"]), int(c["t_idx"])) for c in a}
    kr = {(c.dm_idx, c.t_idx) for c in ref if abs(c.snr - cfg.threshold) > NEAR_THR * cfg.threshold}
    assert kr <= ka and len(ka) - len(kr) <= 2
    plan.destroy()


def test_candidate_overflow_keeps_counting():
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, W.dm_list(cfg), (1,), 0.0)
    d = torch.from_numpy(W.make_segment(cfg)).cuda()
    rec, n = plan.search(d, capacity=10)
    assert n == plan.num_images() == 388 and len(rec) == 10           # count runs past capacity, items are capped
    keys = {(int(c["dm_idx"]), int(c["t_idx"])) for c in rec}
    assert len(keys) == 10 and all(float(c["sigma"]) > 0 for c in rec)
    plan.destroy()


def test_npix_2048_tree_path():
    """npix 2048 is used by none of the five configs: the boxcar tree with 256-thread row-pass CTAs and 32-bit
    histograms (two 128-thread transform groups per CTA), every image at threshold 0 plus one image pixel by pixel."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    npix, nint, dts = 2048, 14, (1, 2, 4)
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * 0.8
    dms = np.array([0.0, 30.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 2048)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 300, -700, 30.0, 2, 4).astype(np.complex64)
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    d = torch.from_numpy(vis).cuda()
    g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=10)
    assert len(g) == plan.num_images()
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    ref = O.search_image(vis, delays, iu, iv, keep, npix, 1, 2, 2)
    img, _ = plan.debug_image(d, 1, 1, 2)
    assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean())
    plan.destroy()


def _tiny_setup(npix, oversample=0.8):
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * (1.0 if npix <= 128 else oversample)
    return cfg, f, uvw, cell


@pytest.mark.parametrize("npix,dts,nint", [(256, (2, 8), 43), (512, (8, 2), 37), (256, (1, 1, 2), 30), (256, (2, 4, 2), 30),
                                           (256, (4, 8), 11), (512, (1, 2, 4, 8), 9), (1024, (1, 2, 4, 8, 16), 45)])
def test_tree_plans_without_dt1_duplicates_short_and_ragged(npix, dts, nint):
    """Shapes of the loop the five configs never use (PAPER.md:104 loops over sampling time): a boxcar-tree plan
    whose dt_list lacks 1 (the dt = 1 level exists only as an intermediate), widths listed twice (the second copy
    takes another path and must give the same images), segments shorter than two blocks (nint < 2 TB), and a
    ragged nint at npix 1024 with a width off the tree.  Every image at threshold 0 against the oracle."""
    import torch
    import paper_1802_03084_b200 as R
    cfg, f, uvw, cell = _tiny_setup(npix)
    dms = np.array([0.0, 25.0, 60.0]) if nint > 20 else np.array([0.0, 8.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 31 * npix + nint)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 5, -9, float(dms[-1]), 2, 3).astype(np.complex64)
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    g = _compare_all(plan, torch.from_numpy(vis).cuda(), vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=4)
    assert len(g) == plan.num_images()
    for a in range(len(dts)):               # duplicate widths: identical statistics through different kernels
        for b in range(a + 1, len(dts)):
            if dts[a] == dts[b]:
                for (d, k, j), c in g.items():
                    if k == a:
                        c2 = g[(d, b, j)]
                        assert abs(float(c["snr"]) - float(c2["snr"])) <= SNR_TOL * float(c["snr"])
                        assert (c["l_pix"], c["m_pix"]) == (c2["l_pix"], c2["m_pix"])
    plan.destroy()


def test_capacity_zero_and_repeated_searches_on_one_plan():
    """capacity = 0 (count only; items may be NULL) and two rf_search calls on ONE plan with different data:
    the second result must not depend on the first (self-cleaning histograms, grown workspaces, device counters)."""
    import torch
    import paper_1802_03084_b200 as R
    npix, nint, dts = 512, 40, (1, 2, 4, 8, 3)
    cfg, f, uvw, cell = _tiny_setup(npix)
    dms = np.array([0.0, 30.0, 60.0])
    thr = 4.5
    va = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 901)
    va = O.inject_transient(va, f, uvw, cfg.inttime_s, cell, 1.5, 40, 17, 30.0, 4, 8).astype(np.complex64)
    vb = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 902)
    vb = O.inject_transient(vb, f, uvw, cfg.inttime_s, cell, 1.0, -90, 3, 60.0, 1, 20).astype(np.complex64)
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, thr)
    da, db = torch.from_numpy(va).cuda(), torch.from_numpy(vb).cuda()
    # capacity 0: no item is written, the count is the number of candidates
    count = torch.zeros(1, dtype=torch.int32, device="cuda")
    plan.search_raw(da.data_ptr(), torch.cuda.current_stream().cuda_stream, 0, 0, count.data_ptr())
    torch.cuda.synchronize()
    n0 = int(count.item())
    ga = _compare_all(plan, da, va, f, uvw, cell, npix, dms, dts, thr, cfg.inttime_s, min_match=3)
    assert n0 == len(ga) > 0
    gb = _compare_all(plan, db, vb, f, uvw, cell, npix, dms, dts, thr, cfg.inttime_s, min_match=1)
    ga2 = _compare_all(plan, da, va, f, uvw, cell, npix, dms, dts, thr, cfg.inttime_s, min_match=3)
    assert set(ga2) == set(ga) and set(gb) != set(ga)
    for k in ga:                                      # bit-identical records on the repeat
        assert ga[k].tobytes() == ga2[k].tobytes()
    plan.destroy()


def test_npix_2048_width_8_rides_the_phase_sums():
    """npix >= 2048 caps the boxcar tree at TB = 4 (one 32-bit histogram per image in the row pass), so a width
    of 8 in dt_list is searched on its phase-decimated sums (B7) instead of failing at search time."""
    import torch
    import paper_1802_03084_b200 as R
    npix, nint, dts = 2048, 20, (1, 2, 4, 8)
    cfg, f, uvw, cell = _tiny_setup(npix)
    dms = np.array([0.0, 30.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 2049)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 300, -700, 30.0, 8, 4).astype(np.complex64)
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    d = torch.from_numpy(vis).cuda()
    g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=10)
    assert len(g) == plan.num_images() and any(k[1] == 3 for k in g)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    ref = O.search_image(vis, delays, iu, iv, keep, npix, 1, 8, 0)
    img, _ = plan.debug_image(d, 1, 3, 0)
    assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean())
    plan.destroy()


@pytest.mark.parametrize("dts", [(1, 2), (1, 2, 4)])
def test_npix_2048_column_pass_forms_agree(dts):
    """npix >= 2048 with TB = 2 (row-pair hand-off) runs the column pass as a pruned DFT over the occupied cells of each uv
    column (k_tree_coldft); RF_TUNE_COL_DFT = 0 keeps the column FFTs, and so does TB = 4 whatever the knob says.  Every
    setting against the oracle on every image, and against each other record by record; several blocks per CTA and a
    ragged tail."""
    import torch
    import paper_1802_03084_b200 as R
    npix, nint = 2048, 23
    cfg, f, uvw, cell = _tiny_setup(npix)
    dms = np.array([0.0, 45.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 2050 + len(dts))
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, -411, 640, 45.0, 2, 6).astype(np.complex64)
    d = torch.from_numpy(vis).cuda()
    lists = {}
    for form in (4, 0, 1):
        plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
        plan.set_tuning(R.binding.RF_TUNE_COL_DFT, form)
        g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=10)
        assert len(g) == plan.num_images()
        lists[form] = g
        if form == 4:
            delays = O.delay_table(f, dms, cfg.inttime_s)
            iu, iv, keep = O.cell_table(uvw, f, npix, cell)
            ref = O.search_image(vis, delays, iu, iv, keep, npix, 1, dts[-1], 1)
            img, _ = plan.debug_image(d, 1, len(dts) - 1, 1)
            assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean())
        plan.destroy()
    for form in (0, 1):
        assert set(lists[form]) == set(lists[4])
        for key, c in lists[4].items():
            o = lists[form][key]
            assert abs(float(c["snr"]) - float(o["snr"])) <= 2e-4 * float(o["snr"]), (form, key)
    plan2 = R.Plan(f, uvw, 2, nint, cfg.inttime_s, 2048, cell, dms, (1,), 6.0)
    with pytest.raises(R.RealfastError):
        plan2.set_tuning(R.binding.RF_TUNE_COL_DFT, 65)
    plan2.destroy()


@pytest.mark.parametrize("cell_mult,u_scale,dts", [(70, 1e-3, (1, 2, 4)), (70, 1e-3, (1, 2)), (40, 0.03, (1, 2))])
def test_npix_2048_dense_columns(cell_mult, u_scale, dts):
    """Nearly north-south baselines and a wide field: the samples fall into a few uv columns that hold hundreds of cells
    (column 0, with its Hermitian mirror, more than a thousand).  First case (TB = 4): column FFTs on these columns;
    second (TB = 2): the pruned column DFT runs on a column of > 1000 cells; third: on ~18 columns of 100-200 cells, many
    per row class.
    Every image against the oracle."""
    import torch
    import paper_1802_03084_b200 as R
    npix, nint = 2048, 11
    cfg, f, uvw, cell = _tiny_setup(npix)
    cell *= cell_mult
    uvw = uvw.copy()
    uvw[:, 0] *= u_scale
    dms = np.array([0.0, 45.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 2060)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 5, 640, 45.0, 2, 3).astype(np.complex64)
    d = torch.from_numpy(vis).cuda()
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=10)
    assert len(g) == plan.num_images()
    delays = O.delay_table(f, dms, cfg.inttime_s)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    assert keep.sum() > 1000 and np.abs(iu[keep]).max() <= (1 if u_scale < 0.01 else 40)
    ref = O.search_image(vis, delays, iu, iv, keep, npix, 0, 1, 2)
    img, _ = plan.debug_image(d, 0, 0, 2)
    assert np.abs(img - ref).max() <= PIX_TOL * np.sqrt((ref ** 2).mean())
    plan.destroy()


@pytest.mark.parametrize("array", ["tiny", "lband"])
def test_npix_4096_north_south_array(array):
    """All baselines north-south at npix 4096: every sample lands in uv column 0, which with its Hermitian mirror then
    holds ~1,800 cells for the 45-baseline array (the pruned column DFT runs on it: the largest list the kernel sees
    in any test) and ~3,000 for the 351-baseline one (three value buffers would need > 100 KB, so the plan keeps the
    column FFTs for that geometry).  Every image against the oracle."""
    import torch
    import paper_1802_03084_b200 as R
    npix, nint, dts = 4096, 9, (1, 2)
    cfg = W.get_config("tiny")
    f = W.channel_freqs_hz(cfg)
    uvw = W.baseline_uvw_m(W.get_config(array)).copy()
    uvw[:, 0] *= 1e-5
    cell = 1900.0 / (np.abs(uvw[:, 1]).max() * f.max() / 299792458.0 * npix)       # |iv| <= 1900 < npix / 2
    dms = np.array([0.0, 45.0])
    vis = _rand_vis((nint, uvw.shape[0], f.size, 2), 4097)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.0, 3, -1500, 45.0, 1, 2).astype(np.complex64)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    rows = set((iv[keep] % npix).tolist()) | set((-iv[keep] % npix).tolist())
    assert np.abs(iu[keep]).max() == 0 and (1500 < len(rows) < 1950 if array == "tiny" else len(rows) > 2200)
    d = torch.from_numpy(vis).cuda()
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    g = _compare_all(plan, d, vis, f, uvw, cell, npix, dms, dts, 0.0, cfg.inttime_s, min_match=8)
    assert len(g) == plan.num_images()
    plan.destroy()


def test_wrong_device_or_knob_is_an_error():
    import torch
    import paper_1802_03084_b200 as R
    cfg, f, uvw, cell = _tiny_setup(64)
    plan = R.Plan(f, uvw, 2, 16, cfg.inttime_s, 64, cell, np.array([0.0]), (1,), 6.0)
    with pytest.raises(R.RealfastError):
        plan.set_tuning(99, 1)
    with pytest.raises(R.RealfastError):
        plan.set_tuning(R.binding.RF_TUNE_DM_GROUP, 0)
    plan.set_tuning(R.binding.RF_TUNE_DM_GROUP, 3)
    plan.destroy()


@pytest.mark.parametrize("npix,radius", [(512, 130), (1024, 180)])
def test_robust_sigma_when_rms_far_exceeds_mad(npix, radius):
    """The case the robust sigma exists for (thresholding an image that holds a bright source): the
    histogram of the row pass spans +-3.5 sigma_rms (B1), so its resolution in units of sigma_MAD degrades by
    sigma_rms / sigma_MAD.  That ratio is bounded by the dirty beam: a single sample gives 1 (a fringe), the VLA-like
    coverages of the configs 1.1-2.4, and the most concentrated beam a gridded snapshot can have -- a completely FILLED
    aperture of `radius` cells, one sample per cell, built here on a lattice -- about 11 at 512^2 and 12 at 1024^2.  Even there
    the S/N must stay within 1e-3 of the oracle and no image may report a histogram overflow."""
    import torch
    import paper_1802_03084_b200 as R
    cell, f = 1.0e-4, np.array([1.4e9])
    du = 1.0 / (npix * cell)
    pts = [(a, b) for a in range(0, radius + 1) for b in range(-radius, radius + 1)
           if a * a + b * b <= radius * radius and (a > 0 or b > 0)]
    nbl = len(pts)
    uvw = np.zeros((nbl, 3))
    uvw[:, 0] = [(a + 0.1) * du * O.C_LIGHT / f[0] for a, _ in pts]
    uvw[:, 1] = [(b - 0.2) * du * O.C_LIGHT / f[0] for _, b in pts]
    nint, dms, dts, inttime = 6, np.array([0.0]), (1, 2), 0.005
    rng = np.random.default_rng(npix)
    vis = (0.01 * (rng.standard_normal((nint, nbl, 1, 2)) + 1j * rng.standard_normal((nint, nbl, 1, 2)))).astype(np.complex64)
    vis = O.inject_transient(vis, f, uvw, inttime, cell, 1.0, 40, -25, 0.0, 2, 2).astype(np.complex64)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    assert keep.all() and len(set(zip(iu.ravel().tolist(), iv.ravel().tolist()))) == nbl      # one sample per cell
    delays = O.delay_table(f, dms, inttime)
    img = O.search_image(vis, delays, iu, iv, keep, npix, 0, 1, 2)
    ratio = np.sqrt((img ** 2).mean()) / O.image_stats(img)[3]
    assert ratio > 10.0, ratio
    plan = R.Plan(f, uvw, 2, nint, inttime, npix, cell, dms, dts, 0.0)
    g = _compare_all(plan, torch.from_numpy(vis).cuda(), vis, f, uvw, cell, npix, dms, dts, 0.0, inttime, min_match=8)
    assert (int(g[(0, 0, 2)]["l_pix"]), int(g[(0, 0, 2)]["m_pix"])) == (40, -25)
    plan.destroy()
