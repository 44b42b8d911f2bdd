"""GPU parity of the periodicity search (PAPER.md:100 footnote 4): rf_search_periodic and
rf_debug_periodic_image against oracle O10 on the same bytes -- power images pixel by pixel, statistics of
every (dm, k) at threshold 0, the candidate list of an injected pulse train, tree blocks of 2, 4 and 8,
ragged transform lengths, flagged channels and the fused mean subtraction."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu

PIX_TOL, SNR_TOL, NEAR_THR = 1e-4, 1e-3, 2e-3


def _rand_vis(shape, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(shape, dtype=np.float32) + 1j * rng.standard_normal(shape, dtype=np.float32)).astype(np.complex64)


def _pulse_train(vis, f, uvw, inttime, cell, amp, l, m, dm, period, t_first):
    out = vis.astype(np.complex128)
    for t0 in range(t_first, vis.shape[0], period):
        out = O.inject_transient(out, f, uvw, inttime, cell, amp, l, m, dm, 1, t0)
    return out.astype(np.complex64)


def _compare(plan, d, vis, f, uvw, cell, npix, dms, thr, inttime, weights=None):
    gpu, n = plan.search_periodic(d, capacity=1 << 15)
    assert n == len(gpu)
    ref, stats = O.periodicity_search(vis, f, uvw, inttime, npix, cell, dms, thr, chan_weights=weights,
                                      return_all_stats=True)
    assert all(int(c["dt_idx"]) == -1 for c in gpu)
    g = {(int(c["dm_idx"]), int(c["t_idx"])): c for c in gpu}
    o = {(c.dm_idx, c.t_idx): c for c in ref}
    assert len(g) == len(gpu)                              # no key twice
    for key in set(g) ^ set(o):
        assert abs(stats[key][4] - thr) <= NEAR_THR * thr, (key, stats[key][4])
    for key in set(g) & set(o):
        assert abs(float(g[key]["snr"]) - o[key].snr) <= SNR_TOL * o[key].snr, key
        assert abs(float(g[key]["peak"]) - o[key].peak) <= 1e-4 * o[key].peak, key
        assert (int(g[key]["l_pix"]), int(g[key]["m_pix"])) == (o[key].l_pix, o[key].m_pix), key
    assert plan.get_counters()["stats_overflow"] == 0
    return g, o, stats


@pytest.mark.parametrize("dts,npol,nint", [((1, 2, 4, 8), 2, 150), ((1, 2), 1, 64), ((4, 3), 4, 100)])
def test_every_frequency_image(dts, npol, nint):
    """Threshold 0: every (dm, k) is emitted and compared; transform lengths differ between the DM trials
    (150 - maxdelay -> 128 and 64; a trial whose sweep leaves fewer than 64 integrations is skipped)."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    npix = 256
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * 0.8
    dms = np.array([0.0, 140.0, 60.0, 600.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, npol), 7 + nint)
    vis = _pulse_train(vis, f, uvw, cfg.inttime_s, cell, 0.5, 20, -31, 60.0, 8, 3)
    plan = R.Plan(f, uvw, npol, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    nts = [O.periodicity_nt(nint, int(delays[i].max())) for i in range(len(dms))]
    assert [plan.periodic_nt(i) for i in range(len(dms))] == nts
    d = torch.from_numpy(vis).cuda()
    g, o, stats = _compare(plan, d, vis, f, uvw, cell, npix, dms, 0.0, cfg.inttime_s)
    assert len(g) == sum(nt // 2 for nt in nts) == len(stats) and len(g) >= 32
    # pixel parity through the debug hook: first, last and a middle bin of a trial
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    for dm_idx in (0, 2):
        nt = nts[dm_idx]
        if nt == 0:
            continue
        spec = O.periodicity_spectrum(vis, delays[dm_idx], nt)
        for k in (1, nt // 8, nt // 2 - 1, nt // 2):
            img = O.periodicity_image(spec[k], iu, iv, keep, npix)
            ref = img.real ** 2 + img.imag ** 2
            got, st = plan.debug_periodic_image(d, dm_idx, k)
            # amplitude |I_k| within 1e-4 of the rms amplitude (the pixel tolerance of the transient images)
            assert np.abs(np.sqrt(got) - np.sqrt(ref)).max() <= PIX_TOL * np.sqrt(ref.mean()), (dm_idx, k)
            amp, y, x, sigma, snr = stats[(dm_idx, k)]
            assert abs(float(st["snr"]) - snr) <= SNR_TOL * snr and int(st["t_idx"]) == k
    plan.destroy()


def test_pulse_train_is_found_on_its_harmonics():
    """A dispersed pulse train of period 8 integrations: at threshold 7 the candidates are exactly the
    oracle's, at the harmonics of nt / 8, at the injected pixel and the matching DM trial."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    npix, nint, thr = 512, 300, 7.0
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * 0.8
    dms = np.array([0.0, 40.0, 80.0, 120.0])
    w = np.ones(cfg.nchan, dtype=np.float32); w[[5, 6, 20]] = 0
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 99)
    vis = _pulse_train(vis, f, uvw, cfg.inttime_s, cell, 0.35, -100, 57, 80.0, 8, 2)
    vis += np.complex64(3.0)                                # a constant source at the phase centre
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, (1, 2, 4, 8), thr)
    plan.set_chan_weights(w)
    plan.set_meansub(True)
    d = torch.from_numpy(vis).cuda()
    g, o, stats = _compare(plan, d, O.mean_subtract(vis), f, uvw, cell, npix, dms, thr, cfg.inttime_s, weights=w)
    nt = plan.periodic_nt(2)
    assert nt == 256
    hits = [key for key in g if key[0] == 2]
    assert set(hits) >= {(2, nt // 8), (2, 2 * nt // 8), (2, 3 * nt // 8)}
    for key in hits:
        assert key[1] % (nt // 8) == 0
        # nearest-cell gridding at a large offset may move the peak by one pixel (the oracle agrees: _compare)
        assert abs(int(g[key]["l_pix"]) + 100) <= 1 and abs(int(g[key]["m_pix"]) - 57) <= 1
    plan.destroy()


def test_needs_the_tree_kernels():
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, W.default_cell_rad(cfg, uvw),
                  W.dm_list(cfg), (1,), 6.0)
    d = torch.from_numpy(W.make_segment(cfg)).cuda()
    with pytest.raises(R.RealfastError):
        plan.search_periodic(d)
    plan.destroy()


def test_lband_full_size_sampled():
    """BASELINE.json configs[1] at full size (351 baselines x 256 channels, 1024 integrations, 512^2, 64 DM trials):
    the whole rf_search_periodic, then sampled (dm, k) images against the oracle -- power image amplitude pixel by
    pixel, S/N, peak pixel, presence in the candidate list; transform lengths 1024, 512 and 256 all occur."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("lband")
    f, uvw, dms = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg), W.dm_list(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, dms, cfg.dt_list, cfg.threshold)
    d_true = 20                                                      # a pulse train at trial 20's DM, period 16
    train = [W.generate.Transient(0.06, -40, 25, float(dms[d_true]), 1, t0) for t0 in range(5, 700, 16)]
    vis = W.make_segment(cfg, sources=train)                         # the seeded generator: both sides read these bytes
    d = torch.from_numpy(vis).cuda()
    gpu, n = plan.search_periodic(d, capacity=1 << 16)
    assert n == len(gpu) and plan.get_counters()["stats_overflow"] == 0
    g = {(int(c["dm_idx"]), int(c["t_idx"])): c for c in gpu}
    delays = O.delay_table(f, dms, cfg.inttime_s)
    nts = [O.periodicity_nt(cfg.nint, int(delays[i].max())) for i in range(len(dms))]
    assert [plan.periodic_nt(i) for i in range(len(dms))] == nts and {1024, 512, 256} <= set(nts)
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
    rng = np.random.default_rng(5)
    found_harmonic = False
    for dm_idx in (0, d_true, 63):
        nt = nts[dm_idx]
        spec = O.periodicity_spectrum(vis, delays[dm_idx], nt)
        ks = sorted({1, nt // 2, nt // 16, 2 * (nt // 16)} | set(int(x) for x in rng.integers(1, nt // 2 + 1, 3)))
        for k in ks:
            img = O.periodicity_image(spec[k], iu, iv, keep, cfg.npix)
            ref = img.real ** 2 + img.imag ** 2
            amp, y, x, sigma, snr = O.periodicity_stats(ref)
            got, st = plan.debug_periodic_image(d, dm_idx, k)
            assert np.abs(np.sqrt(got) - np.sqrt(ref)).max() <= PIX_TOL * np.sqrt(ref.mean()), (dm_idx, k)
            assert abs(float(st["snr"]) - snr) <= SNR_TOL * snr, (dm_idx, k)
            lm = (x if x < cfg.npix // 2 else x - cfg.npix, y if y < cfg.npix // 2 else y - cfg.npix)
            if snr > cfg.threshold * (1 + NEAR_THR):
                assert (dm_idx, k) in g and (int(g[(dm_idx, k)]["l_pix"]), int(g[(dm_idx, k)]["m_pix"])) == lm
                found_harmonic |= dm_idx == d_true and lm == (-40, 25)
            elif snr < cfg.threshold * (1 - NEAR_THR):
                assert (dm_idx, k) not in g
    assert found_harmonic                                            # the pulse train is seen at its DM and pixel
    plan.destroy()


def test_periodic_npix_2048_tb4():
    """The power variant of the row pass at npix 2048 with TB = 4 (512 threads, TB/2 32-bit histograms of 4096
    bins): its shared memory must fit the 227 KB opt-in limit (sized per power image, not per tree node)."""
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    npix, nint, dts = 2048, 70, (1, 2, 4)
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * 0.8
    dms = np.array([0.0, 20.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), 2050)
    vis = _pulse_train(vis, f, uvw, cfg.inttime_s, cell, 0.5, 200, -310, 20.0, 8, 3)
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, 0.0)
    d = torch.from_numpy(vis).cuda()
    gpu, n = plan.search_periodic(d, capacity=1 << 10)
    assert n == len(gpu) == 64 == plan.get_counters()["images"]      # 2 trials x NT/2 = 32 frequency images
    keys = [(0, 1), (1, 8), (1, 32), (0, 17)]
    ref, stats = O.periodicity_search(vis, f, uvw, cfg.inttime_s, npix, cell, dms, 0.0, keys=keys, return_all_stats=True)
    g = {(int(c["dm_idx"]), int(c["t_idx"])): c for c in gpu}
    for key in keys:
        amp, y, x, sigma, snr = stats[key]
        assert abs(float(g[key]["snr"]) - snr) <= SNR_TOL * snr, key
        assert (int(g[key]["l_pix"]) % npix, int(g[key]["m_pix"]) % npix) == (x, y), key
    plan.destroy()
