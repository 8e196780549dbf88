"""Thin ctypes binding of libfdas.so (include/fdas.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and
streams.  There is no CPU fallback: importing this module raises if ``libfdas.so`` is missing, and
every call raises ``FdasError`` on a non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdas.so")

FDAS_FP32, FDAS_BF16, FDAS_BF16_PLANE16, FDAS_BF16_TC, FDAS_BF16_TC_PLANE16 = 0, 1, 2, 3, 4
PRECISIONS = {"fp32": FDAS_FP32, "bf16": FDAS_BF16, "bf16_plane16": FDAS_BF16_PLANE16,
              "bf16_tc": FDAS_BF16_TC, "bf16_tc_plane16": FDAS_BF16_TC_PLANE16}
FDAS_HSUM_PLAIN, FDAS_HSUM_NEIGHBOUR_MAX = 0, 1
FDAS_OK, FDAS_EARG, FDAS_EALLOC, FDAS_ECUDA, FDAS_ECUFFT, FDAS_EOVERFLOW, FDAS_EUNSUPPORTED = range(7)

EXPORTS = (
    "fdas_plan", "fdas_plan_info", "fdas_prepare_spectrum", "fdas_convolve_plane",
    "fdas_harmonic_sum_peaks", "fdas_plan_invalidate_plane", "fdas_plan_set_harmonic_mode", "fdas_search_host", "fdas_search_batch", "fdas_thresholds_from_sigma",
    "fdas_whiten_static", "fdas_plan_templates_host", "fdas_plan_debug_maxplane", "fdas_plan_debug_rawspectrum", "fdas_plan_debug_fail_prepare", "fdas_plan_launch_count", "fdas_destroy", "fdas_strerror",
    "fdas_last_error_detail",
)


class FdasInfo(C.Structure):
    _fields_ = [("n_in", C.c_int64), ("nfft", C.c_int64), ("nbins", C.c_int64), ("nz", C.c_int32),
                ("seg_len", C.c_int32), ("halfwidth", C.c_int32), ("valid", C.c_int32),
                ("nseg", C.c_int64), ("plane_pitch", C.c_int64), ("spec_elem_bytes", C.c_int32),
                ("plane_elem_bytes", C.c_int32), ("precision", C.c_int32), ("reserved", C.c_int32),
                ("zmax", C.c_double), ("zstep", C.c_double), ("tsamp", C.c_double), ("tobs", C.c_double)]


CAND_DTYPE = np.dtype([("r", "<u4"), ("zidx", "<i2"), ("h", "<u2"), ("power", "<f4"), ("flags", "<u4")])
assert CAND_DTYPE.itemsize == 16


class FdasError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        detail = _lib.fdas_last_error_detail().decode() if _lib is not None else ""
        msg = _lib.fdas_strerror(status).decode() if _lib is not None else "?"
        super().__init__(f"{where}: status {status} ({msg}) {detail}")


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2211_13517_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, dbl, ci = C.c_void_p, C.c_int64, C.c_double, C.c_int
    L.fdas_plan.argtypes = [C.POINTER(vp), i64, dbl, dbl, dbl, ci, ci]
    L.fdas_plan_info.argtypes = [vp, C.POINTER(FdasInfo)]
    L.fdas_prepare_spectrum.argtypes = [vp, vp, vp, vp]
    L.fdas_convolve_plane.argtypes = [vp, vp, vp, vp]
    L.fdas_harmonic_sum_peaks.argtypes = [vp, vp, ci, C.POINTER(C.c_float), i64, vp, i64, vp, vp]
    L.fdas_plan_invalidate_plane.argtypes = [vp]
    L.fdas_plan_set_harmonic_mode.argtypes = [vp, ci]
    L.fdas_search_host.argtypes = [vp, vp, ci, C.POINTER(C.c_float), i64, vp, i64, C.POINTER(i64), vp]
    L.fdas_search_batch.argtypes = [vp, C.POINTER(vp), ci, ci, ci, C.POINTER(C.c_float), i64, vp, i64,
                                    C.POINTER(i64), vp]
    L.fdas_thresholds_from_sigma.argtypes = [ci, dbl, C.POINTER(C.c_float)]
    L.fdas_plan_templates_host.argtypes = [vp, vp]
    L.fdas_plan_debug_maxplane.argtypes = [vp, C.POINTER(vp), C.POINTER(i64)]
    L.fdas_plan_debug_rawspectrum.argtypes = [vp, C.POINTER(vp), C.POINTER(i64)]
    L.fdas_whiten_static.argtypes = [vp, i64, vp, ci, vp]
    L.fdas_plan_debug_fail_prepare.argtypes = [vp, ci]
    L.fdas_plan_launch_count.argtypes = [vp]
    L.fdas_plan_launch_count.restype = i64
    L.fdas_destroy.argtypes = [vp]
    L.fdas_strerror.argtypes = [ci]
    L.fdas_strerror.restype = C.c_char_p
    L.fdas_last_error_detail.restype = C.c_char_p
    return L


_lib = None
_lib = _load()


def lib():
    return _lib


def _check(status: int, where: str):
    if status != FDAS_OK:
        raise FdasError(status, where)


def thresholds_from_sigma(H: int, nsigma: float) -> np.ndarray:
    out = np.empty(H, dtype=np.float32)
    _check(_lib.fdas_thresholds_from_sigma(H, float(nsigma), out.ctypes.data_as(C.POINTER(C.c_float))),
           "fdas_thresholds_from_sigma")
    return out


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def whiten_static(d_X, nbins: int, d_spec, stream=None):
    """fdas_whiten_static: whitening without a plan and without any allocation, for callers that may not
    call cudaMalloc (see include/fdas.h: a real-time stage whose HBM is all in its own pool, a plug-in that
    may only touch the buffers it is given).  d_X: raw spectrum, a float32 device tensor of >= nbins (re, im)
    pairs or a raw device pointer (int); d_spec: (nbins, 2) float32 or bfloat16 device tensor (output).
    At most 2^24 bins (the fixed scratch array's limit); calls on one device must not overlap on the GPU."""
    import torch
    x_ptr = d_X.data_ptr() if hasattr(d_X, "data_ptr") else int(d_X)
    assert d_spec.is_cuda and d_spec.is_contiguous() and d_spec.numel() >= 2 * int(nbins)
    assert d_spec.dtype in (torch.float32, torch.bfloat16)
    _check(_lib.fdas_whiten_static(x_ptr, int(nbins), d_spec.data_ptr(),
                                   1 if d_spec.dtype == torch.bfloat16 else 0, _stream_ptr(stream)),
           "fdas_whiten_static")


@dataclass
class PeakResult:
    count: int            # true number found (may exceed capacity)
    cands: np.ndarray     # structured array CAND_DTYPE, first min(count, capacity)


class Plan:
    """fdas_plan handle.  Device buffers are torch tensors owned by the caller."""

    def __init__(self, n: int, tsamp: float, zmax: float, zstep: float, seg_len: int = 2048,
                 precision="fp32"):
        prec = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        h = C.c_void_p()
        _check(_lib.fdas_plan(C.byref(h), int(n), float(tsamp), float(zmax), float(zstep),
                              int(seg_len), prec), "fdas_plan")
        self._h = h
        info = FdasInfo()
        _check(_lib.fdas_plan_info(self._h, C.byref(info)), "fdas_plan_info")
        self.info = info

    # ---- sizes -------------------------------------------------------------------------
    @property
    def precision(self) -> int:
        return int(self.info.precision)

    def alloc_spec(self, device="cuda"):
        import torch
        if self.precision == FDAS_FP32:
            return torch.empty((self.info.nbins, 2), dtype=torch.float32, device=device)
        return torch.empty((self.info.nbins, 2), dtype=torch.bfloat16, device=device)

    def alloc_plane(self, device="cuda"):
        import torch
        dt = torch.bfloat16 if self.precision in (FDAS_BF16_PLANE16, FDAS_BF16_TC_PLANE16) else torch.float32
        return torch.empty((self.info.nz, self.info.plane_pitch), dtype=dt, device=device)

    def alloc_cands(self, capacity: int, device="cuda"):
        import torch
        return (torch.empty((capacity, 4), dtype=torch.int32, device=device),
                torch.zeros(1, dtype=torch.int64, device=device))

    # ---- the three per-trial calls (asynchronous on the stream) ------------------------------
    def prepare_spectrum(self, d_series, d_spec, stream=None):
        assert d_series.is_cuda and d_series.dtype.is_floating_point and d_series.element_size() == 4
        assert d_series.numel() >= self.info.nfft and d_series.is_contiguous()
        _check(_lib.fdas_prepare_spectrum(self._h, d_series.data_ptr(), d_spec.data_ptr(),
                                          _stream_ptr(stream)), "fdas_prepare_spectrum")

    def convolve_plane(self, d_spec, d_plane, stream=None):
        _check(_lib.fdas_convolve_plane(self._h, d_spec.data_ptr(), d_plane.data_ptr(),
                                        _stream_ptr(stream)), "fdas_convolve_plane")

    def harmonic_sum_peaks(self, d_plane, H, thresholds, r_lo, d_cands, d_count, stream=None):
        thr = np.ascontiguousarray(thresholds, dtype=np.float32)
        assert thr.size >= H
        cap = int(d_cands.shape[0]) if d_cands is not None else 0
        _check(_lib.fdas_harmonic_sum_peaks(
            self._h, d_plane.data_ptr(), int(H), thr.ctypes.data_as(C.POINTER(C.c_float)), int(r_lo),
            d_cands.data_ptr() if d_cands is not None else None, cap, d_count.data_ptr(),
            _stream_ptr(stream)), "fdas_harmonic_sum_peaks")

    def set_harmonic_mode(self, mode):
        """"plain" (S_h) or "neighbour_max" (S'_h: harmonic k at its maximum within floor(k/2) bins of k r)."""
        m = {"plain": FDAS_HSUM_PLAIN, "neighbour_max": FDAS_HSUM_NEIGHBOUR_MAX}.get(mode, mode)
        _check(_lib.fdas_plan_set_harmonic_mode(self._h, int(m)), "fdas_plan_set_harmonic_mode")

    def invalidate_plane(self):
        """The plane convolve_plane wrote last was modified by the caller: rebuild the block maxima."""
        _check(_lib.fdas_plan_invalidate_plane(self._h), "fdas_plan_invalidate_plane")

    @staticmethod
    def read_cands(d_cands, d_count) -> PeakResult:
        count = int(d_count.cpu().item())
        n = min(count, int(d_cands.shape[0]))
        raw = d_cands[:n].cpu().numpy()
        return PeakResult(count, raw.view(CAND_DTYPE).reshape(-1).copy())

    # ---- end-to-end host entry point ---------------------------------------------------------
    def search_host(self, h_series: np.ndarray, H, thresholds, r_lo, capacity=1 << 16,
                    out: Optional[np.ndarray] = None, stream=None) -> PeakResult:
        """h_series: float32 numpy array (pinned for full-speed copies) of n_in samples."""
        assert h_series.dtype == np.float32 and h_series.size >= self.info.n_in
        thr = np.ascontiguousarray(thresholds, dtype=np.float32)
        if out is None:
            out = np.empty(capacity, dtype=CAND_DTYPE)
        cnt = C.c_int64(0)
        st = _lib.fdas_search_host(self._h, h_series.ctypes.data, int(H),
                                   thr.ctypes.data_as(C.POINTER(C.c_float)), int(r_lo),
                                   out.ctypes.data, int(out.size), C.byref(cnt), _stream_ptr(stream))
        if st not in (FDAS_OK, FDAS_EOVERFLOW):
            raise FdasError(st, "fdas_search_host")
        n = min(cnt.value, out.size)
        return PeakResult(int(cnt.value), out[:n])

    def search_host_raw(self, h_ptr: int, H, thr_c, r_lo, out_ptr: int, capacity: int, stream_ptr: int):
        """Lowest-overhead form for benchmarks: raw host pointers; returns (status, count)."""
        cnt = C.c_int64(0)
        st = _lib.fdas_search_host(self._h, h_ptr, int(H), thr_c, int(r_lo), out_ptr, int(capacity),
                                   C.byref(cnt), stream_ptr)
        return st, cnt.value

    # ---- many trials, pipelined (configs[3], configs[4]) -------------------------------------
    def search_batch(self, series, H, thresholds, r_lo, capacity=1 << 16, out=None, stream=None):
        """series: list of device tensors (all) or of float32 numpy arrays / pinned CPU tensors (all),
        n_in samples each.  Returns (counts[int64 ntrials], cands[ntrials, capacity] CAND_DTYPE, status);
        status is FDAS_OK or FDAS_EOVERFLOW."""
        n = len(series)
        on_host = n == 0 or not (hasattr(series[0], "is_cuda") and series[0].is_cuda)
        ptrs = (C.c_void_p * max(n, 1))()
        for i, x in enumerate(series):
            if hasattr(x, "data_ptr"):
                assert x.is_cuda != on_host and x.numel() >= self.info.n_in and x.element_size() == 4
                ptrs[i] = x.data_ptr()
            else:
                assert on_host and x.dtype == np.float32 and x.size >= self.info.n_in
                ptrs[i] = x.ctypes.data
        thr = np.ascontiguousarray(thresholds, dtype=np.float32)
        if out is None:
            out = np.empty((max(n, 1), capacity), dtype=CAND_DTYPE)
        assert out.shape[0] >= n and out.flags.c_contiguous
        counts = np.zeros(max(n, 1), dtype=np.int64)
        st = _lib.fdas_search_batch(self._h, ptrs, 1 if on_host else 0, n, int(H),
                                    thr.ctypes.data_as(C.POINTER(C.c_float)), int(r_lo), out.ctypes.data,
                                    int(out.shape[1]), counts.ctypes.data_as(C.POINTER(C.c_int64)),
                                    _stream_ptr(stream))
        if st not in (FDAS_OK, FDAS_EOVERFLOW):
            raise FdasError(st, "fdas_search_batch")
        return counts[:n], out, st

    # ---- diagnostics -----------------------------------------------------------------------
    def templates_host(self) -> np.ndarray:
        taps = 2 * self.info.halfwidth + 1
        out = np.empty((self.info.nz, taps), dtype=np.complex128)
        _check(_lib.fdas_plan_templates_host(self._h, out.ctypes.data), "fdas_plan_templates_host")
        return out

    def debug_maxplane(self):
        """(device pointer, pitch) of the plan-owned block-maximum plane (diagnostic)."""
        ptr, pitch = C.c_void_p(), C.c_int64()
        _check(_lib.fdas_plan_debug_maxplane(self._h, C.byref(ptr), C.byref(pitch)), "fdas_plan_debug_maxplane")
        return int(ptr.value), int(pitch.value)

    def debug_rawspectrum(self):
        """(device pointer, complex length) of the plan-owned raw spectrum X of the last prepare (diagnostic)."""
        ptr, n = C.c_void_p(), C.c_int64()
        _check(_lib.fdas_plan_debug_rawspectrum(self._h, C.byref(ptr), C.byref(n)), "fdas_plan_debug_rawspectrum")
        return int(ptr.value), int(n.value)

    def debug_fail_prepare(self, nth: int):
        """Fault injection (diagnostic): the (nth + 1)-th prepare step enqueued from now on fails with FDAS_ECUDA."""
        _check(_lib.fdas_plan_debug_fail_prepare(self._h, int(nth)), "fdas_plan_debug_fail_prepare")

    def launch_count(self) -> int:
        return int(_lib.fdas_plan_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            _lib.fdas_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
