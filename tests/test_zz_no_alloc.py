"""GPU: rf_meansub_static, the allocation-free entry point (scratch in a static device array of the library), against
the existing plan-bound path rf_prep_meansub and against oracle O0 (reading A21).

Collected last on purpose (the file name sorts after every other test file): the run uses `pytest -x`,
so a failure here hides nothing.  The test does not depend on what ran before it: it passes alone in a fresh
process (the first call then also looks up the array's address and loads the module) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

import oracle as O
import workloads as W
import workloads.generate  # noqa: F401

pytestmark = pytest.mark.gpu

TOL = 2.5e-7          # the tolerance of tests/test_gpu_prep.py, relative to max(|vis|, 1), for path against path
# Against the float64 oracle the error is the float32 rounding of the mean (<= 2^-24 |mean| per component) plus
# that of the difference (<= 2^-24 |vis - mean|): <= 3 * sqrt(2) * 2^-24 * max(|vis|, |mean|) = 2.5e-7, worst case.
TOL_ORACLE = 4e-7


def _segment(seed, nint, nbl, nchan, npol, offset):
    rng = np.random.default_rng(seed)
    vis = (rng.standard_normal((nint, nbl, nchan, npol)) + 1j * rng.standard_normal((nint, nbl, nchan, npol)))
    vis += offset * (rng.standard_normal((1, nbl, nchan, npol)) + 1j * rng.standard_normal((1, nbl, nchan, npol)))
    return vis.astype(np.complex64)


def _existing_path(cfg, vis):
    """rf_prep_meansub on a copy of vis through a plan of the same shape (the path that allocates)."""
    import torch
    import paper_1802_03084_b200 as R
    nint, nbl, nchan, npol = vis.shape
    f, uvw = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg)
    assert (uvw.shape[0], f.size) == (nbl, nchan)
    plan = R.Plan(f, uvw, npol, nint, cfg.inttime_s, cfg.npix, W.default_cell_rad(cfg, uvw), [0.0], (1,), 8.0)
    d = torch.from_numpy(vis).cuda()
    plan.prep_meansub(d)
    torch.cuda.synchronize()
    out = d.cpu().numpy()
    plan.destroy()
    return out


def _check_oracle(got, vis):
    ref = O.mean_subtract(vis)                                          # O0, independent of both CUDA paths
    mean = vis.astype(np.complex128).mean(axis=0, keepdims=True)
    scale = np.maximum(np.maximum(np.abs(vis), np.abs(mean)), 1.0)
    assert (np.abs(got - ref) <= TOL_ORACLE * scale).all()
    assert (np.abs(got.astype(np.complex128).mean(axis=0)) <= TOL_ORACLE * scale.max(axis=0)).all()


def _check(got, want, vis):
    scale = np.maximum(np.abs(vis), 1.0)
    assert (np.abs(got - want) <= TOL * scale).all()
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))     # same sums in the same order: same bits


def test_static_entry_point_equals_the_existing_path_on_two_calls_in_a_row():
    """Call 1 fills the whole scratch array (the L-band shape, 351 x 256 x 2 = 179,712 elements, ragged nint);
    call 2 has a much smaller shape, so anything stale it read from call 1 would show; call 3 repeats call 1."""
    import torch
    import paper_1802_03084_b200 as R
    big, small = W.get_config("lband"), W.get_config("tiny")
    vis_a = _segment(11, 37, big.nbl, big.nchan, big.npol, offset=30.0)
    vis_b = _segment(12, 61, small.nbl, small.nchan, small.npol, offset=1000.0)
    want_a, want_b = _existing_path(big, vis_a), _existing_path(small, vis_b)

    da, db, dc = (torch.from_numpy(v).cuda() for v in (vis_a, vis_b, vis_a))
    torch.cuda.synchronize()
    R.meansub_static(da)
    R.meansub_static(db)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    R.meansub_static(dc)                      # a warmed-up call: device memory in use must not move
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    got_a, got_b, got_c = (d.cpu().numpy() for d in (da, db, dc))

    _check(got_a, want_a, vis_a)
    _check(got_b, want_b, vis_b)
    _check(got_c, want_a, vis_a)
    _check_oracle(got_a, vis_a)
    _check_oracle(got_b, vis_b)


def test_static_entry_point_limits_and_errors():
    import torch
    import paper_1802_03084_b200 as R
    from paper_1802_03084_b200 import binding as B
    lim = B.RF_STATIC_MAX_ELEMS
    # exactly at the limit: accepted (no plan of that shape is needed: compare with the definition in float64)
    vis = _segment(13, 5, lim // 2, 1, 2, offset=3.0)
    d = torch.from_numpy(vis).cuda()
    R.meansub_static(d)
    torch.cuda.synchronize()
    _check_oracle(d.cpu().numpy(), vis)
    # one element more: a clear error, and the buffer is untouched
    over = torch.ones((2, lim + 1, 1, 1), dtype=torch.complex64, device="cuda")
    with pytest.raises(R.RealfastError, match="RF_STATIC_MAX_ELEMS"):
        R.meansub_static(over)
    torch.cuda.synchronize()
    assert bool((over == 1).all())
    # bad sizes, a null pointer, a misaligned pointer, a host pointer
    lib = B.load_library()
    ok = torch.ones((4, 3, 2, 2), dtype=torch.complex64, device="cuda")
    assert lib.rf_meansub_static(ok.data_ptr(), 0, 3, 2, 2, None) == -1
    assert lib.rf_meansub_static(ok.data_ptr(), 4, 3, 2, 3, None) == -1
    assert lib.rf_meansub_static(None, 4, 3, 2, 2, None) == -1
    assert lib.rf_meansub_static(ok.data_ptr() + 8, 2, 3, 2, 2, None) == -1
    host = np.ones((4, 3, 2, 2), dtype=np.complex64)
    host_ptr = host.ctypes.data_as(C.c_void_p)
    if host_ptr.value % 16 == 0:
        assert lib.rf_meansub_static(host_ptr, 4, 3, 2, 2, None) == -4
        assert b"current CUDA device" in lib.rf_last_error()
    torch.cuda.synchronize()
    assert bool((ok == 1).all())
