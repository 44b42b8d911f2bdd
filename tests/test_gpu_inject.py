"""GPU parity of the device-side mock injection: rf_inject against oracle O9,
element by element, and the injected source found by rf_search where it was put."""
import numpy as np
import pytest

import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu


def test_inject_matches_oracle_and_is_recovered():
    import torch
    import paper_1802_03084_b200 as R
    cfg = W.get_config("tiny")
    f, uvw, dms = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg), W.dm_list(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, dms, (1, 2), cfg.threshold)
    base = W.make_segment(cfg, inject=False)
    d = torch.from_numpy(base).cuda()
    sources = [(1.5, -12.0, 9.0, float(dms[3]), 2, 16), (0.8, 3.25, -20.5, 133.0, 3, cfg.nint - 4),
               (2.0, 0.0, 0.0, 0.0, 1, -1)]           # sub-pixel offsets; one runs off the end; one starts before 0
    ref = base.astype(np.complex128)
    for (a, l, m, dm, w, t0) in sources:
        plan.inject(d, a, l, m, dm, w, t0)
        ref = O.inject_transient(ref, f, uvw, cfg.inttime_s, cell, a, l, m, dm, w, t0)
    torch.cuda.synchronize()
    got = d.cpu().numpy()
    assert np.abs(got - ref).max() <= 2.5e-7 * np.abs(ref).max()      # one float32 rounding per touched sample
    untouched = np.abs(ref - base) == 0
    assert np.array_equal(got[untouched], base[untouched])
    gpu, n = plan.search(d)
    best = max(gpu, key=lambda c: c["snr"])
    assert (int(best["dm_idx"]), int(best["l_pix"]), int(best["m_pix"])) == (3, -12, 9)
    assert int(best["t_idx"]) * (1, 2)[int(best["dt_idx"])] in (16, 17)
    plan.destroy()
