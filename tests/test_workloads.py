"""Seeded input generator (workloads/): properties the streaming bench and the parity tests rely on.
The generator holds none of the search arithmetic; these tests pin its bookkeeping only."""
import numpy as np

import workloads as W


def test_row_ranges_equal_slices_of_the_full_segment():
    cfg = W.get_config("tiny")
    full = W.make_segment(cfg)
    for lo, hi in [(0, 7), (10, 40), (50, 64)]:
        assert np.array_equal(W.make_segment(cfg, rows=(lo, hi)), full[lo:hi])
    out = np.empty((5,) + full.shape[1:], dtype=np.complex64)
    assert W.make_segment(cfg, rows=(20, 25), out=out) is out
    assert np.array_equal(out, full[20:25])          # the injected source arrives around t = 20


def test_streaming_noise_overlaps_bit_for_bit():
    """Config 5: segment s covers absolute integrations [s*stride, s*stride + nint); the noise of an
    absolute integration does not depend on the segment it is generated for."""
    cfg = W.get_config("stream")
    overlap = cfg.nint - cfg.stride_int
    a = W.make_segment(cfg, 3, inject=False, rows=(cfg.stride_int, cfg.stride_int + 2))
    b = W.make_segment(cfg, 4, inject=False, rows=(0, 2))
    assert overlap == 624 and np.array_equal(a, b)
    assert a.dtype == np.complex64 and a.shape == (2, cfg.nbl, cfg.nchan, cfg.npol)


def test_goal_workload_1ms_matches_the_paper_rate():
    """PAPER.md:94 / Table 1 row "L": 1 ms sampling of the L-band array is 1.4 GB/s; the
    stream1ms config keeps config 5's 2.0 s stride and overlaps by its own DM 1000 sweep."""
    import oracle as O
    cfg = W.get_config("stream1ms")
    rate = cfg.nbl * cfg.nchan * cfg.npol * 8 / cfg.inttime_s
    assert abs(rate / 1.4e9 - 1.0) < 0.03
    delays = O.delay_table(W.channel_freqs_hz(cfg), W.dm_list(cfg), cfg.inttime_s)
    assert int(delays.max()) == cfg.nint - cfg.stride_int == 3118
    assert cfg.stride_int * cfg.inttime_s == W.get_config("stream").stride_int * W.get_config("stream").inttime_s == 2.0
    n_img = sum(O.n_images(cfg.nint, int(delays[d].max()), dt, cfg.stride_int) for d in range(cfg.ndm) for dt in cfg.dt_list)
    assert n_img == 64 * (2000 + 1000 + 500 + 250)
