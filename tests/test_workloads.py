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
