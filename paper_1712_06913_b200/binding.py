"""Thin ctypes binding of libmuser.so (include/muser.h): same names, argument marshalling only.

Every step of the imaging path runs inside the CUDA library.  PyTorch is used for device memory and streams:
tensors are passed as `data_ptr()`, the stream as `torch.cuda.current_stream().cuda_stream`.  If the library is
missing or no CUDA device is present the calls raise -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmuser.so")

MUSER_OK, MUSER_EINVAL, MUSER_ECUDA, MUSER_ENOMEM, MUSER_ESTATE, MUSER_EUNSUPPORTED = range(6)
MUSER_KERNEL_PSWF, MUSER_KERNEL_GAUSS = 0, 1
MUSER_STRATEGY_AUTO, MUSER_STRATEGY_TILED, MUSER_STRATEGY_OWNER, MUSER_STRATEGY_WPLANE = 0, 2, 3, 4
MUSER_TUNE_ITEM_SIZE, MUSER_TUNE_BIN_ITERS, MUSER_TUNE_COLS_TMA, MUSER_TUNE_FFT_SUBBATCH = 0, 1, 2, 3
MUSER_WEIGHT_NATURAL, MUSER_WEIGHT_UNIFORM = 0, 1
MUSER_POLS_SUM, MUSER_POLS_SPLIT = 0, 1
STAGES = ("bin", "grid", "pack", "fft", "correct")

_c = ctypes
_vp, _i, _d, _ll = _c.c_void_p, _c.c_int, _c.c_double, _c.c_longlong

# name -> (restype, argtypes): the complete export list of include/muser.h
SIGNATURES = {
    "muser_imager_create": (_vp, [_i, _i, _d, _i, _i]),
    "muser_imager_destroy": (_i, [_vp]),
    "muser_set_kernel": (_i, [_vp, _i, _d]),
    "muser_set_batch": (_i, [_vp, _i]),
    "muser_set_wplanes": (_i, [_vp, _i, _vp, _vp, _vp]),
    "muser_set_strategy": (_i, [_vp, _i]),
    "muser_set_tuning": (_i, [_vp, _i, _i]),
    "muser_set_grid_correction": (_i, [_vp, _i]),
    "muser_set_weighting": (_i, [_vp, _i]),
    "muser_set_phase_offset": (_i, [_vp, _d, _d]),
    "muser_set_psf2x": (_i, [_vp, _i]),
    "muser_psf2x": (_i, [_vp, _vp, _vp]),
    "muser_get_counts": (_i, [_vp, _vp, _vp]),
    "muser_get_weighted_grid": (_i, [_vp, _vp, _vp, _vp]),
    "muser_set_peak_search": (_i, [_vp, _i]),
    "muser_get_peak": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "muser_histogram": (_i, [_vp, _vp, _i, _c.c_float, _c.c_float, _vp, _vp]),
    "muser_histogram_static": (_i, [_vp, _ll, _i, _i, _vp, _vp, _vp, _i]),
    "muser_reset": (_i, [_vp, _vp]),
    "muser_grid": (_i, [_vp, _vp, _vp, _vp, _vp, _ll, _vp]),
    "muser_grid_batched": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _ll, _vp]),
    "muser_grid_rows": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _ll, _i, _i, _i, _i, _vp]),
    "muser_dirty": (_i, [_vp, _vp, _vp]),
    "muser_psf": (_i, [_vp, _vp, _vp]),
    "muser_dirty_psf": (_i, [_vp, _vp, _vp, _vp]),
    "muser_frame_host": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _ll, _vp, _vp, _vp]),
    "muser_frame_host_async": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _ll, _vp, _vp, _vp]),
    "muser_get_grid": (_i, [_vp, _vp, _vp, _vp]),
    "muser_get_table": (_i, [_vp, _i, _vp, _vp]),
    "muser_get_stats": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "muser_last_error": (_c.c_char_p, [_vp]),
    "muser_set_profiling": (_i, [_vp, _i]),
    "muser_get_profile": (_i, [_vp, _vp, _vp]),
    "muser_get_launch_count": (_ll, [_vp]),
    "muser_host_table": (_i, [_i, _i, _i, _d, _vp]),
    "muser_host_wtable": (_i, [_i, _i, _d, _d, _vp]),
    "muser_host_corrector": (_i, [_vp, _i, _i, _i, _vp]),
    "muser_version": (_c.c_char_p, []),
    "muser_microbench": (_i, [_i, _vp]),
}

_lib = None


class MuserError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"muser error {code}: {msg}")
        self.code = code


def lib():
    """Load libmuser.so (built by `python -m paper_1712_06913_b200.build`); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1712_06913_b200.build` "
                               "(the imaging path has no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _ptr(t):
    """Device/host address of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return t.data_ptr()
    assert t.flags["C_CONTIGUOUS"]
    return t.ctypes.data


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return int(stream)


class Imager:
    """One muser_imager handle.  Methods mirror the C ABI one to one (muser_<name>)."""

    def __init__(self, nx, ny, cell_arcsec, support, oversample):
        L = lib()
        self._h = L.muser_imager_create(nx, ny, float(cell_arcsec), support, oversample)
        if not self._h:
            raise MuserError(-1, L.muser_last_error(None).decode())
        self.nx, self.ny, self.support, self.oversample = nx, ny, support, oversample
        self.ngrids, self.nplanes = 1, 0

    def _ck(self, rc):
        if rc != MUSER_OK:
            raise MuserError(rc, lib().muser_last_error(self._h).decode())

    def destroy(self):
        if self._h:
            lib().muser_imager_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- setup
    def set_kernel(self, kind, param=0.0):
        self._ck(lib().muser_set_kernel(self._h, kind, float(param)))
        self.nplanes = 0

    def set_batch(self, ngrids):
        self._ck(lib().muser_set_batch(self._h, ngrids))
        self.ngrids = ngrids

    def set_wplanes(self, w_centres, supports, tables=None):
        """w_centres: float64 array, supports: int array, tables: list of complex64 numpy arrays or None."""
        import numpy as np
        P = len(w_centres)
        wc = np.ascontiguousarray(w_centres, np.float64)
        sp = np.ascontiguousarray(supports, np.int32)
        tp = None
        keep = []
        if tables is not None:
            keep = [np.ascontiguousarray(t, np.complex64) for t in tables]
            tp = (ctypes.c_void_p * P)(*[t.ctypes.data for t in keep])
        self._ck(lib().muser_set_wplanes(self._h, P, wc.ctypes.data if P else None, sp.ctypes.data if P else None,
                                         ctypes.cast(tp, ctypes.c_void_p) if tp is not None else None))
        self.nplanes = P

    def set_strategy(self, strategy):
        self._ck(lib().muser_set_strategy(self._h, strategy))

    def set_tuning(self, key, value):
        self._ck(lib().muser_set_tuning(self._h, key, int(value)))

    def set_grid_correction(self, enabled):
        self._ck(lib().muser_set_grid_correction(self._h, 1 if enabled else 0))

    def set_weighting(self, mode):
        self._ck(lib().muser_set_weighting(self._h, mode))

    def set_phase_offset(self, dl, dm):
        self._ck(lib().muser_set_phase_offset(self._h, float(dl), float(dm)))

    def set_psf2x(self, enabled):
        self._ck(lib().muser_set_psf2x(self._h, 1 if enabled else 0))

    def psf2x(self, beam2x_out, stream=None):
        self._ck(lib().muser_psf2x(self._h, _ptr(beam2x_out), _stream(stream)))

    def set_peak_search(self, enabled):
        self._ck(lib().muser_set_peak_search(self._h, 1 if enabled else 0))

    def get_peak(self):
        """Per grid: (peak value, x, y, minimum) of the last dirty image."""
        n = self.ngrids
        v, m = (ctypes.c_float * n)(), (ctypes.c_float * n)()
        x, y = (ctypes.c_int * n)(), (ctypes.c_int * n)()
        self._ck(lib().muser_get_peak(self._h, v, x, y, m))
        return [(v[i], x[i], y[i], m[i]) for i in range(n)]

    def histogram(self, image, nbins, lo, hi, hist_out, stream=None):
        self._ck(lib().muser_histogram(self._h, _ptr(image), nbins, lo, hi, _ptr(hist_out), _stream(stream)))

    # ---- path
    def reset(self, stream=None):
        self._ck(lib().muser_reset(self._h, _stream(stream)))

    def grid(self, uvw_m, freq_hz, vis, weight, stream=None):
        self._ck(lib().muser_grid(self._h, _ptr(uvw_m), _ptr(freq_hz), _ptr(vis), _ptr(weight),
                                  int(vis.shape[0]), _stream(stream)))

    def grid_batched(self, uvw_m, freq_hz, vis, weight, grid_id, stream=None):
        self._ck(lib().muser_grid_batched(self._h, _ptr(uvw_m), _ptr(freq_hz), _ptr(vis), _ptr(weight),
                                          _ptr(grid_id), int(vis.shape[0]), _stream(stream)))

    def grid_rows(self, uvw_m, freq_hz, vis, weight, grid_id=None, pol_mode=MUSER_POLS_SUM, stream=None):
        """uvw_m [ntime][nrow][3], freq_hz [nchan], vis / weight [ntime][npol][nchan][nrow] (device tensors)."""
        ntime, npol, nchan, nrow = (int(x) for x in vis.shape[:4])
        self._ck(lib().muser_grid_rows(self._h, _ptr(uvw_m), _ptr(freq_hz), _ptr(vis), _ptr(weight), _ptr(grid_id),
                                       nrow, nchan, npol, ntime, pol_mode, _stream(stream)))

    def dirty(self, image_out, stream=None):
        self._ck(lib().muser_dirty(self._h, _ptr(image_out), _stream(stream)))

    def psf(self, beam_out, stream=None):
        self._ck(lib().muser_psf(self._h, _ptr(beam_out), _stream(stream)))

    def dirty_psf(self, image_out, beam_out, stream=None):
        self._ck(lib().muser_dirty_psf(self._h, _ptr(image_out), _ptr(beam_out), _stream(stream)))

    def frame_host(self, uvw_m, freq_hz, vis, weight, grid_id, image_out, beam_out, stream=None):
        """HOST buffers (numpy or pinned CPU tensors) in, HOST images out; synchronises the stream."""
        self._ck(lib().muser_frame_host(self._h, _ptr(uvw_m), _ptr(freq_hz), _ptr(vis), _ptr(weight), _ptr(grid_id),
                                        int(vis.shape[0]), _ptr(image_out), _ptr(beam_out), _stream(stream)))

    def frame_host_async(self, uvw_m, freq_hz, vis, weight, grid_id, image_out, beam_out, stream=None):
        """As frame_host without the final synchronisation (pinned buffers; synchronise the stream before reading)."""
        self._ck(lib().muser_frame_host_async(self._h, _ptr(uvw_m), _ptr(freq_hz), _ptr(vis), _ptr(weight), _ptr(grid_id),
                                              int(vis.shape[0]), _ptr(image_out), _ptr(beam_out), _stream(stream)))

    # ---- inspection
    def get_grid(self, grid_out, wgrid_out, stream=None):
        self._ck(lib().muser_get_grid(self._h, _ptr(grid_out), _ptr(wgrid_out), _stream(stream)))

    def get_counts(self, counts_out, stream=None):
        self._ck(lib().muser_get_counts(self._h, _ptr(counts_out), _stream(stream)))

    def get_weighted_grid(self, grid_out, wgrid_out, stream=None):
        self._ck(lib().muser_get_weighted_grid(self._h, _ptr(grid_out), _ptr(wgrid_out), _stream(stream)))

    def get_table(self, plane=0):
        import numpy as np
        n = ctypes.c_int(0)
        self._ck(lib().muser_get_table(self._h, plane, None, ctypes.byref(n)))
        out = np.empty(n.value, np.float32)
        self._ck(lib().muser_get_table(self._h, plane, out.ctypes.data, ctypes.byref(n)))
        return out

    def get_stats(self):
        sw, a, b, c = ctypes.c_double(), ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
        self._ck(lib().muser_get_stats(self._h, ctypes.byref(sw), ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
        return dict(sum_weights=sw.value, n_gridded=a.value, n_dropped=b.value, n_flagged=c.value)

    def set_profiling(self, enabled):
        self._ck(lib().muser_set_profiling(self._h, 1 if enabled else 0))

    def get_profile(self):
        ms = (ctypes.c_double * len(STAGES))()
        n = (ctypes.c_longlong * len(STAGES))()
        self._ck(lib().muser_get_profile(self._h, ms, n))
        return {s: (ms[i], n[i]) for i, s in enumerate(STAGES)}


    def get_launch_count(self):
        return int(lib().muser_get_launch_count(self._h))


# ---- host-only helpers (no GPU): the library's own fp64 generators
def host_table(kind, support, oversample, param=0.0):
    import numpy as np
    out = np.empty(support * oversample + 1, np.float64)
    rc = lib().muser_host_table(kind, support, oversample, float(param), out.ctypes.data)
    if rc:
        raise MuserError(rc, "muser_host_table")
    return out


def host_wtable(support, oversample, w_lambda, fov_rad):
    import numpy as np
    out = np.empty(2 * (support * oversample + 1), np.float64)
    rc = lib().muser_host_wtable(support, oversample, float(w_lambda), float(fov_rad), out.ctypes.data)
    if rc:
        raise MuserError(rc, "muser_host_wtable")
    return out.view(np.complex128)


def host_corrector(table, support, oversample, n):
    import numpy as np
    t = np.ascontiguousarray(table, np.float64)
    out = np.empty(n, np.float64)
    rc = lib().muser_host_corrector(t.ctypes.data, support, oversample, n, out.ctypes.data)
    if rc:
        raise MuserError(rc, "muser_host_corrector")
    return out


MUSER_STATIC_MAX_GRIDS = 1024


def histogram_static(image, nbins, hist_out, stream=None):
    """muser_histogram_static: own-range histograms of `image` (device float [ngrids][...]) into `hist_out` (device
    uint32/int32 [ngrids][nbins]) without a handle and without any device allocation inside the library: for callers that
    cannot cudaMalloc (a steady-state monitoring loop, a process whose HBM belongs to another allocator).  At most
    MUSER_STATIC_MAX_GRIDS images per call; calls share one scratch array per device, so keep them on one stream."""
    ngrids = int(image.shape[0])
    npix = int(image.numel() // max(ngrids, 1))
    err = ctypes.create_string_buffer(256)
    rc = lib().muser_histogram_static(_ptr(image), npix, ngrids, int(nbins), _ptr(hist_out), _stream(stream), err, len(err))
    if rc:
        raise MuserError(rc, err.value.decode())


MICROBENCH = ("fp32_fma_flops", "fp32_ffma2_flops", "shared_int_adds", "shared_f32_cas_adds", "global_f32_red_adds")


def microbench():
    """Measured device limits (per second) the roofline discussion of DESIGN.md refers to."""
    out = {}
    for kind, name in enumerate(MICROBENCH):
        v = ctypes.c_double()
        rc = lib().muser_microbench(kind, ctypes.byref(v))
        if rc:
            raise MuserError(rc, "muser_microbench")
        out[name] = v.value
    return out


def version():
    return lib().muser_version().decode()
