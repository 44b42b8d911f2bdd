"""ctypes binding with the same names as include/realfast.h: argument marshalling only.

Every step of the search runs in the CUDA kernels of librealfast_b200.so; torch is used
here for device memory and streams.  If the library is missing, loading fails loudly --
there is no fallback path.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB: Optional[C.CDLL] = None

RF_OK = 0
EXPORTS = [
    "rf_plan_create", "rf_search", "rf_plan_destroy", "rf_plan_set_chan_weights", "rf_plan_set_uvw",
    "rf_plan_set_search_span", "rf_plan_get_tables", "rf_plan_num_images", "rf_plan_num_t",
    "rf_debug_image", "rf_plan_get_counters", "rf_plan_set_batch", "rf_last_error",
    "rf_search_host", "rf_plan_set_profiling", "rf_plan_get_kernel_times", "rf_plan_set_mode",
    "rf_plan_set_meansub", "rf_prep_meansub", "rf_cand_spectrum", "rf_inject",
    "rf_search_periodic", "rf_plan_periodic_nt", "rf_debug_periodic_image", "rf_plan_set_tuning",
    "rf_plan_fft_work", "rf_meansub_static",
]
RF_STATIC_MAX_ELEMS = 196608     # include/realfast.h
RF_TUNE_AUX_WIDTHS, RF_TUNE_DM_GROUP, RF_TUNE_FEED_BATCH, RF_TUNE_TREE_MAXPIX = 1, 2, 3, 4
RF_TUNE_GATHER_ORDER, RF_TUNE_COL_DFT = 5, 6

# numpy view of rf_cand (32 bytes)
CAND_DTYPE = np.dtype([("dm_idx", "<i4"), ("dt_idx", "<i4"), ("t_idx", "<i4"), ("l_pix", "<i4"),
                       ("m_pix", "<i4"), ("peak", "<f4"), ("sigma", "<f4"), ("snr", "<f4")])
assert CAND_DTYPE.itemsize == 32


class RealfastError(RuntimeError):
    pass


class _CandOut(C.Structure):
    _fields_ = [("items", C.c_void_p), ("capacity", C.c_int32), ("count", C.c_void_p)]


class _Counters(C.Structure):
    _fields_ = [("images", C.c_int64), ("vis_gridded", C.c_int64), ("n_kept", C.c_int32),
                ("n_dropped", C.c_int32), ("stats_overflow", C.c_int32), ("kernel_launches", C.c_int32)]


def lib_path() -> str:
    return os.path.join(_HERE, "librealfast_b200.so")


def load_library() -> C.CDLL:
    """dlopen the in-tree library and declare the prototypes; raises if it is not built."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise RealfastError(f"{path} is not built: run `python -m paper_1802_03084_b200.build` "
                            "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(path)
    dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_void_p
    lib.rf_plan_create.argtypes = [C.POINTER(vp), dp, C.c_int, dp, C.c_int, C.c_int, C.c_int, C.c_double,
                                   C.c_int, C.c_double, dp, C.c_int, ip, C.c_int, C.c_float]
    lib.rf_search.argtypes = [vp, vp, vp, C.POINTER(_CandOut)]
    lib.rf_plan_destroy.argtypes = [vp]
    lib.rf_plan_set_chan_weights.argtypes = [vp, C.POINTER(C.c_float)]
    lib.rf_plan_set_uvw.argtypes = [vp, dp, C.c_double]
    lib.rf_plan_set_search_span.argtypes = [vp, C.c_int]
    lib.rf_plan_set_batch.argtypes = [vp, C.c_int]
    lib.rf_plan_set_tuning.argtypes = [vp, C.c_int, C.c_int]
    lib.rf_plan_get_tables.argtypes = [vp, ip, ip, C.POINTER(C.c_uint8)]
    lib.rf_plan_num_images.argtypes = [vp]
    lib.rf_plan_num_images.restype = C.c_int64
    lib.rf_plan_num_t.argtypes = [vp, C.c_int, C.c_int]
    lib.rf_plan_fft_work.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.rf_debug_image.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp, vp]
    lib.rf_plan_get_counters.argtypes = [vp, C.POINTER(_Counters)]
    lib.rf_last_error.restype = C.c_char_p
    lib.rf_search_host.argtypes = [vp, vp, vp, C.c_int32, ip]
    lib.rf_plan_set_profiling.argtypes = [vp, C.c_int]
    lib.rf_plan_set_mode.argtypes = [vp, C.c_int]
    lib.rf_plan_get_kernel_times.argtypes = [vp, C.POINTER(C.c_float), ip]
    lib.rf_plan_set_meansub.argtypes = [vp, C.c_int]
    lib.rf_prep_meansub.argtypes = [vp, vp, vp]
    lib.rf_meansub_static.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp]
    lib.rf_inject.argtypes = [vp, vp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, vp]
    lib.rf_cand_spectrum.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp]
    lib.rf_search_periodic.argtypes = [vp, vp, vp, C.POINTER(_CandOut)]
    lib.rf_plan_periodic_nt.argtypes = [vp, C.c_int]
    lib.rf_debug_periodic_image.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp, vp]
    for name in EXPORTS:
        if name not in ("rf_plan_num_images", "rf_last_error"):
            getattr(lib, name).restype = C.c_int
    _LIB = lib
    return lib


def _check(rc: int) -> None:
    if rc != RF_OK:
        raise RealfastError(f"realfast error {rc}: {load_library().rf_last_error().decode()}")


def meansub_static(vis, stream=None) -> None:
    """rf_meansub_static: rf_prep_meansub without a plan and without any allocation (scratch in a static device
    array of the library; nbl*nchan*npol <= RF_STATIC_MAX_ELEMS; overlapping calls race).  vis: torch complex64
    CUDA tensor [nint][nbl][nchan][npol], modified in place."""
    import torch
    assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous() and vis.dim() == 4
    nint, nbl, nchan, npol = (int(n) for n in vis.shape)
    st = torch.cuda.current_stream(vis.device) if stream is None else stream
    with torch.cuda.device(vis.device):
        _check(load_library().rf_meansub_static(vis.data_ptr(), nint, nbl, nchan, npol, st.cuda_stream))


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Plan:
    """rf_plan wrapper.  Methods mirror the C entry points one to one."""

    def __init__(self, freqs_hz, uvw_m, npol: int, nint: int, inttime_s: float, npix: int,
                 cell_rad: float, dm_list, dt_list: Sequence[int], threshold: float):
        self._lib = load_library()
        self._h = C.c_void_p()
        f = np.ascontiguousarray(freqs_hz, dtype=np.float64)
        u = np.ascontiguousarray(uvw_m, dtype=np.float64)
        d = np.ascontiguousarray(dm_list, dtype=np.float64)
        t = np.ascontiguousarray(dt_list, dtype=np.int32)
        if u.ndim != 2 or u.shape[1] != 3:
            raise ValueError("uvw_m must be [nbl][3]")
        self.nchan, self.nbl, self.npol, self.nint = f.size, u.shape[0], npol, nint
        self.npix, self.ndm, self.ndt = npix, d.size, t.size
        _check(self._lib.rf_plan_create(C.byref(self._h), _dptr(f), f.size, _dptr(u), u.shape[0], npol, nint,
                                        inttime_s, npix, cell_rad, _dptr(d), d.size,
                                        t.ctypes.data_as(C.POINTER(C.c_int32)), t.size, threshold))

    # -- lifetime
    def destroy(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.rf_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- rf_plan_set_*
    def set_chan_weights(self, w) -> None:
        w = np.ascontiguousarray(w, dtype=np.float32)
        assert w.size == self.nchan
        _check(self._lib.rf_plan_set_chan_weights(self._h, w.ctypes.data_as(C.POINTER(C.c_float))))

    def set_uvw(self, uvw_m, cell_rad: float = 0.0) -> None:
        u = np.ascontiguousarray(uvw_m, dtype=np.float64)
        assert u.shape == (self.nbl, 3)
        _check(self._lib.rf_plan_set_uvw(self._h, _dptr(u), cell_rad))

    def set_search_span(self, n: int) -> None:
        _check(self._lib.rf_plan_set_search_span(self._h, n))

    def set_batch(self, n: int) -> None:
        _check(self._lib.rf_plan_set_batch(self._h, n))

    def set_tuning(self, knob: int, value: int) -> None:
        """rf_plan_set_tuning: knobs RF_TUNE_* (no effect on results)."""
        _check(self._lib.rf_plan_set_tuning(self._h, knob, value))

    # -- queries
    def get_tables(self):
        delay = np.empty((self.ndm, self.nchan), dtype=np.int32)
        cell = np.empty((self.nbl, self.nchan, 2), dtype=np.int32)
        keep = np.empty((self.nbl, self.nchan), dtype=np.uint8)
        _check(self._lib.rf_plan_get_tables(self._h, delay.ctypes.data_as(C.POINTER(C.c_int32)),
                                            cell.ctypes.data_as(C.POINTER(C.c_int32)),
                                            keep.ctypes.data_as(C.POINTER(C.c_uint8))))
        return delay, cell, keep

    def num_images(self) -> int:
        return int(self._lib.rf_plan_num_images(self._h))

    def num_t(self, dm_idx: int, dt_idx: int) -> int:
        return int(self._lib.rf_plan_num_t(self._h, dm_idx, dt_idx))

    def fft_work(self):
        """rf_plan_fft_work: (column transforms, row pair transforms) of npix points per rf_search."""
        a, b = C.c_int64(0), C.c_int64(0)
        _check(self._lib.rf_plan_fft_work(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def get_counters(self) -> dict:
        c = _Counters()
        _check(self._lib.rf_plan_get_counters(self._h, C.byref(c)))
        return {k: getattr(c, k) for k, _ in _Counters._fields_}

    # -- rf_search / rf_debug_image: device pointers and a stream, nothing else
    def search_raw(self, vis_ptr: int, stream: int, items_ptr: int, capacity: int, count_ptr: int) -> None:
        out = _CandOut(items_ptr, capacity, count_ptr)
        _check(self._lib.rf_search(self._h, vis_ptr, stream, C.byref(out)))

    def search(self, vis, capacity: int = 1 << 16, stream=None, sync: bool = True):
        """vis: torch complex64 CUDA tensor [nint][nbl][nchan][npol].  Returns (cands, count) where
        cands is a numpy structured array (CAND_DTYPE) of min(count, capacity) records."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape) == (self.nint, self.nbl, self.nchan, self.npol), tuple(vis.shape)
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        items = torch.empty(max(1, capacity) * 32, dtype=torch.uint8, device=vis.device)
        count = torch.zeros(1, dtype=torch.int32, device=vis.device)
        self.search_raw(vis.data_ptr(), st.cuda_stream, items.data_ptr(), capacity, count.data_ptr())
        if not sync:
            return items, count
        st.synchronize()
        n = int(count.item())
        rec = items[: min(n, capacity) * 32].cpu().numpy().view(CAND_DTYPE).copy()
        return rec, n

    def search_host(self, vis_host, cand_host=None, capacity: int = 1 << 16):
        """rf_search_host: vis_host is a host array/tensor (numpy complex64 or pinned torch tensor);
        the host->device copy, the search and the candidate read-back all happen inside the call."""
        if hasattr(vis_host, "data_ptr"):
            ptr, nbytes = vis_host.data_ptr(), vis_host.numel() * vis_host.element_size()
        else:
            assert vis_host.flags["C_CONTIGUOUS"] and vis_host.dtype == np.complex64
            ptr, nbytes = vis_host.ctypes.data, vis_host.nbytes
        assert nbytes == self.nint * self.nbl * self.nchan * self.npol * 8
        if cand_host is None:
            cand_host = np.empty(capacity, dtype=CAND_DTYPE)
        count = C.c_int32(0)
        _check(self._lib.rf_search_host(self._h, ptr, cand_host.ctypes.data, capacity, C.byref(count)))
        return cand_host[: min(count.value, capacity)], count.value

    def set_profiling(self, enable: bool) -> None:
        _check(self._lib.rf_plan_set_profiling(self._h, int(enable)))

    def get_kernel_times(self):
        """(ms[4], launches[4]) of the last search: 0 = grid+column FFT, 1 = row FFT+statistics, 2 = prep."""
        ms = (C.c_float * 4)()
        n = (C.c_int32 * 4)()
        _check(self._lib.rf_plan_get_kernel_times(self._h, ms, n))
        return [float(v) for v in ms], [int(v) for v in n]

    def set_mode(self, use_tree: bool) -> None:
        """rf_plan_set_mode: image-domain boxcar tree (default) or per-image resampling at the read."""
        _check(self._lib.rf_plan_set_mode(self._h, int(use_tree)))

    def set_meansub(self, enable: bool) -> None:
        """rf_plan_set_meansub: search vis - mean_t(vis) without modifying vis."""
        _check(self._lib.rf_plan_set_meansub(self._h, int(enable)))

    def prep_meansub(self, vis, stream=None) -> None:
        """rf_prep_meansub: subtract the time mean in place in a torch complex64 CUDA tensor."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape) == (self.nint, self.nbl, self.nchan, self.npol), tuple(vis.shape)
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        _check(self._lib.rf_prep_meansub(self._h, vis.data_ptr(), st.cuda_stream))

    def inject(self, vis, amp: float, l_pix: float, m_pix: float, dm: float, width: int, t0: int, stream=None) -> None:
        """rf_inject: add a mock transient in place to a torch complex64 CUDA segment."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape) == (self.nint, self.nbl, self.nchan, self.npol), tuple(vis.shape)
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        _check(self._lib.rf_inject(self._h, vis.data_ptr(), amp, l_pix, m_pix, dm, width, t0, st.cuda_stream))

    def cand_spectrum(self, vis, dm_idx: int, dt_idx: int, t_idx: int, l_pix: int, m_pix: int,
                      half_window: int, stream=None):
        """rf_cand_spectrum: float32 numpy [2*half_window + 1][nchan] (phased, dedispersed spectrum)."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        spec = torch.empty((2 * half_window + 1, self.nchan), dtype=torch.float32, device=vis.device)
        _check(self._lib.rf_cand_spectrum(self._h, vis.data_ptr(), dm_idx, dt_idx, t_idx, l_pix, m_pix,
                                          half_window, spec.data_ptr(), st.cuda_stream))
        st.synchronize()
        return spec.cpu().numpy()

    def debug_image(self, vis, dm_idx: int, dt_idx: int, t_idx: int, stream=None):
        """Returns (image float32 [npix][npix] numpy, stats record) of one (dm, dt, t)."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        img = torch.empty((self.npix, self.npix), dtype=torch.float32, device=vis.device)
        stats = torch.zeros(32, dtype=torch.uint8, device=vis.device)
        _check(self._lib.rf_debug_image(self._h, vis.data_ptr(), dm_idx, dt_idx, t_idx, img.data_ptr(),
                                        stats.data_ptr(), st.cuda_stream))
        st.synchronize()
        return img.cpu().numpy(), stats.cpu().numpy().view(CAND_DTYPE)[0].copy()

    def periodic_nt(self, dm_idx: int) -> int:
        """rf_plan_periodic_nt: length of the time transform of one DM trial (0 = trial skipped)."""
        return int(self._lib.rf_plan_periodic_nt(self._h, dm_idx))

    def search_periodic_raw(self, vis_ptr: int, stream: int, items_ptr: int, capacity: int, count_ptr: int) -> None:
        out = _CandOut(items_ptr, capacity, count_ptr)
        _check(self._lib.rf_search_periodic(self._h, vis_ptr, stream, C.byref(out)))

    def search_periodic(self, vis, capacity: int = 1 << 16, stream=None):
        """rf_search_periodic: candidates (dt_idx = -1, t_idx = fluctuation-frequency bin k) and their count."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape) == (self.nint, self.nbl, self.nchan, self.npol), tuple(vis.shape)
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        items = torch.empty(max(1, capacity) * 32, dtype=torch.uint8, device=vis.device)
        count = torch.zeros(1, dtype=torch.int32, device=vis.device)
        out = _CandOut(items.data_ptr(), capacity, count.data_ptr())
        _check(self._lib.rf_search_periodic(self._h, vis.data_ptr(), st.cuda_stream, C.byref(out)))
        st.synchronize()
        n = int(count.item())
        return items[: min(n, capacity) * 32].cpu().numpy().view(CAND_DTYPE).copy(), n

    def debug_periodic_image(self, vis, dm_idx: int, k: int, stream=None):
        """Returns (power image float32 [npix][npix] numpy, stats record) of one (dm, k)."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        st = torch.cuda.current_stream(vis.device) if stream is None else stream
        img = torch.empty((self.npix, self.npix), dtype=torch.float32, device=vis.device)
        stats = torch.zeros(32, dtype=torch.uint8, device=vis.device)
        _check(self._lib.rf_debug_periodic_image(self._h, vis.data_ptr(), dm_idx, k, img.data_ptr(),
                                                 stats.data_ptr(), st.cuda_stream))
        st.synchronize()
        return img.cpu().numpy(), stats.cpu().numpy().view(CAND_DTYPE)[0].copy()
