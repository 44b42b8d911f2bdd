"""rf_search_host (host buffers, copies inside the call; the `e2e` leg of bench.py): the chunked upload with the
search running behind it returns exactly the candidates of rf_search on the resident segment, and those match the
oracle; covers ragged segment lengths (last chunk partial), pageable and pinned input, the plain-upload fallbacks
(mean subtraction, plans without the boxcar tree) and candidate overflow."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu


def _rand_vis(shape, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(shape, dtype=np.float32) + 1j * rng.standard_normal(shape, dtype=np.float32)).astype(np.complex64)


def _keyed(c):
    return {(int(x["dm_idx"]), int(x["dt_idx"]), int(x["t_idx"])): (int(x["l_pix"]), int(x["m_pix"]), float(x["peak"]), float(x["snr"])) for x in c}


@pytest.mark.parametrize("nint,npix,dts,meansub", [(150, 256, (1, 2, 4, 8), False), (64, 256, (1, 2, 3), False),
                                                   (333, 512, (1, 2, 4, 8), False), (150, 256, (1, 2, 4, 8), True),
                                                   (64, 64, (1, 2), False)])
def test_host_search_equals_device_search(nint, npix, dts, meansub):
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    cell = W.default_cell_rad(cfg, uvw) * 64 / npix * (1.0 if npix <= 128 else 0.8)
    dms = np.array([0.0, 100.0, 40.0, 140.0])
    vis = _rand_vis((nint, cfg.nbl, cfg.nchan, 2), nint + npix)
    vis = O.inject_transient(vis, f, uvw, cfg.inttime_s, cell, 1.2, 11, -7, 40.0, 2, 20).astype(np.complex64)
    thr = 4.0
    plan = R.Plan(f, uvw, 2, nint, cfg.inttime_s, npix, cell, dms, dts, thr)
    plan.set_meansub(meansub)
    dev, n_dev = plan.search(torch.from_numpy(vis).cuda(), capacity=1 << 14)
    assert n_dev == len(dev) and n_dev > 0
    for host_in in (vis, torch.from_numpy(vis).pin_memory()):          # pageable numpy, pinned torch
        for _ in range(2):                                             # staging buffers are reused
            got, n = plan.search_host(host_in, capacity=1 << 14)
            assert n == n_dev
            assert _keyed(got) == _keyed(dev)                          # same kernels: identical records
    # and the records are right: against the oracle on the same bytes
    ref = O.search(O.mean_subtract(vis) if meansub else vis, f, uvw, cfg.inttime_s, npix, cell, dms, dts, thr)
    o = {c.key: c for c in ref}
    g = _keyed(dev)
    common = set(o) & set(g)
    assert len(common) >= 1
    for k in set(o) ^ set(g):                                          # only keys AT the threshold may differ (A11)
        snr = o[k].snr if k in o else g[k][3]
        assert abs(snr - thr) <= 2e-3 * thr, (k, snr)
    for k in common:
        assert abs(g[k][3] - o[k].snr) <= 1e-3 * o[k].snr
    # overflow: the count keeps counting, only `capacity` records come back
    got, n = plan.search_host(vis, capacity=3)
    assert n == n_dev and len(got) == 3 and set(_keyed(got)) <= set(g)
    plan.destroy()
