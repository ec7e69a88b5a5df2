"""Thin ctypes binding of the C-ABI library (include/cbmf.h): same names, argument
marshalling only.  Every step of the path runs in the CUDA kernels behind the ABI.

Loading fails loudly if libcbmf.so cannot be built or loaded: there is no CPU fallback,
and this module never imports oracle/.

Arrays may be numpy arrays / CPU torch tensors (host-pointer entry points) or CUDA torch
tensors (the *_dev entry points); torch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

i64_t = C.c_int64

from . import build as _build

OK, EINVAL, ESTATE, ECUDA, ENOMEM, ELIMIT, WTRUNC = 0, -1, -2, -3, -4, -5, 1
NOALLOC_MAX_N = 1 << 20                  # CBMF_NOALLOC_MAX_N of cbmf.h

PEAK_DTYPE = np.dtype([("snr_max", "<f4"), ("idx_peak", "<i4"), ("phase", "<f4"), ("sigma", "<f4")])
TRIG_DTYPE = np.dtype([("template_idx", "<i4"), ("sample_idx", "<i4"), ("snr", "<f4"), ("phase", "<f4")])


class Template(C.Structure):
    _fields_ = [("m1", C.c_double), ("m2", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    """Load (building if needed) libcbmf.so and declare every entry point of cbmf.h."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, i64, dbl, flt = C.c_void_p, C.c_int64, C.c_double, C.c_float
    sig = {
        "cbmf_create": (C.c_int, [C.POINTER(vp), C.c_int, i64, dbl, dbl, vp]),
        "cbmf_destroy": (C.c_int, [vp]),
        "cbmf_set_psd": (C.c_int, [vp, vp, i64]),
        "cbmf_set_psd_dev": (C.c_int, [vp, vp, i64]),
        "cbmf_load_segment": (C.c_int, [vp, vp, i64]),
        "cbmf_load_segment_dev": (C.c_int, [vp, vp, i64]),
        "cbmf_filter_bank": (C.c_int, [vp, vp, i64, flt, vp, vp, i64, C.POINTER(i64)]),
        "cbmf_filter_bank_dev": (C.c_int, [vp, vp, i64, flt, vp, vp, i64, C.POINTER(i64)]),
        "cbmf_cluster_triggers": (C.c_int, [vp, i64, i64, i64, vp, i64, C.POINTER(i64)]),
        "cbmf_filter_bank_clustered": (C.c_int, [vp, vp, i64, flt, i64, vp, vp, i64, C.POINTER(i64), C.POINTER(i64)]),
        "cbmf_filter_stream": (C.c_int, [vp, vp, i64, vp, i64, flt, i64, vp, vp, i64, vp, C.POINTER(i64), C.POINTER(i64)]),
        "cbmf_chisq": (C.c_int, [vp, vp, i64, vp, C.c_int, vp, vp]),
        "cbmf_filter_bank_td": (C.c_int, [vp, vp, i64, flt, vp, vp, i64, C.POINTER(i64)]),
        "cbmf_debug_td_template": (C.c_int, [vp, Template, vp]),
        "cbmf_debug_snr_series": (C.c_int, [vp, Template, vp, vp]),
        "cbmf_debug_template": (C.c_int, [vp, Template, vp]),
        "cbmf_debug_ifft": (C.c_int, [vp, vp, vp, i64, i64]),
        "cbmf_debug_ifft_dev": (C.c_int, [vp, vp, vp, i64, i64]),
        "cbmf_debug_generate_dev": (C.c_int, [vp, vp, i64, vp]),
        "cbmf_ifft_noalloc_dev": (C.c_int, [C.c_int, vp, vp, vp, i64, i64]),
        "cbmf_debug_fp32_peak": (C.c_int, [C.c_int, C.POINTER(dbl), C.POINTER(dbl)]),
        "cbmf_debug_get_prefix": (C.c_int, [vp, vp]),
        "cbmf_debug_get_weights": (C.c_int, [vp, vp]),
        "cbmf_set_pn_order": (C.c_int, [vp, C.c_int]),
        "cbmf_get_pn_order": (C.c_int, [vp]),
        "cbmf_set_sub_batch": (C.c_int, [vp, C.c_int]),
        "cbmf_get_sub_batch": (C.c_int, [vp]),
        "cbmf_set_streams": (C.c_int, [vp, C.c_int]),
        "cbmf_get_streams": (C.c_int, [vp]),
        "cbmf_get_split": (C.c_int, [vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
        "cbmf_last_bad_template": (i64, [vp]),
        "cbmf_launch_count": (i64, [vp]),
        "cbmf_last_pass_time": (C.c_int, [vp, C.c_int, C.POINTER(dbl), C.POINTER(i64)]),
        "cbmf_set_profiling": (C.c_int, [vp, C.c_int]),
        "cbmf_debug_timeline": (C.c_int, [vp, C.c_int, vp, i64, C.POINTER(i64)]),
        "cbmf_strerror": (C.c_char_p, [C.c_int]),
        "cbmf_last_cuda_error": (C.c_char_p, [vp]),
        "cbmf_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)            # AttributeError if the library lacks a declared symbol
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


EXPORTS = ("cbmf_create cbmf_destroy cbmf_set_psd cbmf_set_psd_dev cbmf_load_segment "
           "cbmf_load_segment_dev cbmf_filter_bank cbmf_filter_bank_dev cbmf_cluster_triggers "
           "cbmf_filter_bank_clustered cbmf_filter_stream cbmf_chisq cbmf_filter_bank_td cbmf_debug_td_template cbmf_debug_snr_series "
           "cbmf_debug_template cbmf_debug_ifft cbmf_debug_ifft_dev cbmf_debug_generate_dev cbmf_ifft_noalloc_dev cbmf_debug_fp32_peak "
           "cbmf_debug_get_prefix cbmf_debug_get_weights cbmf_set_pn_order cbmf_get_pn_order cbmf_set_sub_batch cbmf_get_sub_batch "
           "cbmf_set_streams cbmf_get_streams cbmf_get_split cbmf_last_bad_template "
           "cbmf_launch_count cbmf_last_pass_time cbmf_set_profiling cbmf_debug_timeline cbmf_strerror "
           "cbmf_last_cuda_error cbmf_version").split()


class CbmfError(RuntimeError):
    def __init__(self, rc: int, what: str, detail: str = ""):
        msg = lib().cbmf_strerror(rc).decode()
        super().__init__(f"{what}: {msg} (rc={rc})" + (f" [{detail}]" if detail else ""))
        self.rc = rc


def _is_tensor(a) -> bool:
    return hasattr(a, "data_ptr") and hasattr(a, "is_cuda")


_TORCH_NAME = {"float64": "torch.float64", "float32": "torch.float32", "uint8": "torch.uint8",
               "complex64": "torch.complex64"}


def _ptr(a, dtype=None, device=None, itemsize=None):
    """-> (address, on_device).  numpy arrays and tensors must be contiguous and of `dtype` (a numpy dtype
    name; for output records `itemsize` = 16 also admits raw uint8 buffers); a CUDA tensor must live on
    device index `device`.  A wrong dtype would be misread by the kernels, so it is an error here."""
    if a is None:
        return None, False
    if _is_tensor(a):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None:
            ok = str(a.dtype) == _TORCH_NAME.get(dtype, "torch." + dtype)
            if not ok and itemsize is not None:
                ok = str(a.dtype) == "torch.uint8" and a.numel() % itemsize == 0
            if not ok:
                raise ValueError(f"expected a {dtype} tensor, got {a.dtype}")
        if a.is_cuda and device is not None and a.device.index != device:
            raise ValueError(f"tensor lives on cuda:{a.device.index}, the context on cuda:{device}")
        return a.data_ptr(), bool(a.is_cuda)
    if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
        raise ValueError("expected a C-contiguous numpy array or a torch tensor")
    if dtype is not None:
        ok = a.dtype == np.dtype(dtype) if dtype in ("float64", "float32", "uint8", "complex64") else a.dtype == dtype
        if not ok and itemsize is not None:
            ok = a.dtype.itemsize == itemsize or (a.dtype == np.uint8 and a.size % itemsize == 0)
        if not ok:
            raise ValueError(f"expected dtype {dtype}, got {a.dtype}")
    return a.ctypes.data, False


def _nbytes(a) -> int:
    return int(a.numel() * a.element_size()) if _is_tensor(a) else int(a.nbytes)


# Calls that return only after the context's stream has drained (cbmf.h: "every call that returns results is
# synchronous"; the host-pointer set / load wait too).  Matched as prefixes of the name handed to Context._check;
# the two stream-ordered calls are named cbmf_set_psd_dev / cbmf_load_segment_dev there and are excluded below.
_WAITING = ("cbmf_filter_", "cbmf_chisq", "cbmf_debug_snr_series", "cbmf_debug_template", "cbmf_debug_td_template",
            "cbmf_debug_ifft", "cbmf_debug_generate_dev", "cbmf_debug_get_")


class Context:
    """cbmf_ctx: one segment length / sample rate / lower cutoff on one device and stream."""

    def __init__(self, n: int, fs: float, f_low: float, device: int = 0, stream: int | None = None):
        self.n, self.fs, self.f_low, self.device = int(n), float(fs), float(f_low), int(device)
        self._h = C.c_void_p()
        # CUDA tensors handed to the stream-ordered calls (cbmf_set_psd_dev, cbmf_load_segment_dev): those return
        # before the device has read their input, so the binding keeps the tensors alive until a call that waits
        # for the context's stream has returned.  Otherwise a temporary (g.load_segment(x.cuda())) would go back to
        # torch's caching allocator at once and, with the context on another stream than the one the tensor was
        # allocated on, could be handed out again and overwritten before the kernel reads it.
        self._held = []
        rc = lib().cbmf_create(C.byref(self._h), self.device, self.n, self.fs, self.f_low,
                               C.c_void_p(stream or 0))
        if rc:
            self._h = C.c_void_p()
            raise CbmfError(rc, "cbmf_create")

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            lib().cbmf_destroy(self._h)          # waits for the context's stream
            self._h = C.c_void_p()
        if getattr(self, "_held", None):
            self._held.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc: int, what: str) -> int:
        if rc >= 0 and (what in ("cbmf_set_psd", "cbmf_load_segment") or what.startswith(_WAITING)):
            self._held.clear()                   # the context's stream has been waited for: the device is done with them
        if rc < 0:
            detail = lib().cbmf_last_cuda_error(self._h).decode() if rc == ECUDA else ""
            if rc == EINVAL and what == "cbmf_filter_bank":
                bad = int(lib().cbmf_last_bad_template(self._h))
                if bad >= 0:
                    detail = f"first invalid template: index {bad}"
            raise CbmfError(rc, what, detail)
        return rc

    # -- the three calls of the path
    def set_psd(self, psd):
        if isinstance(psd, np.ndarray):
            psd = np.ascontiguousarray(psd, dtype=np.float64)
        p, dev = _ptr(psd, "float64", self.device)
        n_bins = int(psd.numel() if _is_tensor(psd) else psd.size)
        if dev:
            self._held.append(psd)
            self._check(lib().cbmf_set_psd_dev(self._h, p, n_bins), "cbmf_set_psd_dev")
        else:
            self._check(lib().cbmf_set_psd(self._h, p, n_bins), "cbmf_set_psd")

    def load_segment(self, samples):
        if isinstance(samples, np.ndarray):
            samples = np.ascontiguousarray(samples, dtype=np.float32)
        p, dev = _ptr(samples, "float32", self.device)
        n = int(samples.numel() if _is_tensor(samples) else samples.size)
        if dev:
            self._held.append(samples)
            self._check(lib().cbmf_load_segment_dev(self._h, p, n), "cbmf_load_segment_dev")
        else:
            self._check(lib().cbmf_load_segment(self._h, p, n), "cbmf_load_segment")

    def filter_bank(self, bank, snr_threshold: float, trig_capacity: int = 1 << 16):
        """Host arrays in, host arrays out: -> (peaks[PEAK_DTYPE], triggers[TRIG_DTYPE], n_found, rc)."""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        peaks = np.zeros(nt, dtype=PEAK_DTYPE)
        trig = np.zeros(max(int(trig_capacity), 1), dtype=TRIG_DTYPE)
        nf = C.c_int64(0)
        rc = lib().cbmf_filter_bank(self._h, b.ctypes.data if nt else None, nt, float(snr_threshold),
                                    peaks.ctypes.data if nt else None,
                                    trig.ctypes.data if trig_capacity else None, int(trig_capacity),
                                    C.byref(nf))
        self._check(rc, "cbmf_filter_bank")
        return peaks, trig[:min(nf.value, int(trig_capacity))], nf.value, rc

    def filter_bank_td(self, bank, snr_threshold: float, trig_capacity: int = 1 << 16):
        """cbmf_filter_bank_td (the paper's own path: time-domain templates, two polarisations): same results layout
        as filter_bank.  -> (peaks[PEAK_DTYPE], triggers[TRIG_DTYPE], n_found, rc)."""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        peaks = np.zeros(nt, dtype=PEAK_DTYPE)
        trig = np.zeros(max(int(trig_capacity), 1), dtype=TRIG_DTYPE)
        nf = C.c_int64(0)
        rc = lib().cbmf_filter_bank_td(self._h, b.ctypes.data if nt else None, nt, float(snr_threshold),
                                       peaks.ctypes.data if nt else None,
                                       trig.ctypes.data if trig_capacity else None, int(trig_capacity), C.byref(nf))
        self._check(rc, "cbmf_filter_bank_td")
        return peaks, trig[:min(nf.value, int(trig_capacity))], nf.value, rc

    def filter_bank_into(self, bank, snr_threshold: float, peaks_out, trig_out, trig_capacity: int):
        """Caller-owned buffers (all host -- numpy / pinned tensors -- or all CUDA tensors):
        bank float64 [B,2], peaks_out 16 B/template, trig_out 16 B/entry.  -> (n_found, rc)."""
        pb, dev = _ptr(bank, "float64", self.device)
        pp, devp = _ptr(peaks_out, "peak records", self.device, itemsize=16)
        pt, devt = _ptr(trig_out, "trigger records", self.device, itemsize=16)
        if devp != dev or (trig_out is not None and devt != dev):
            raise ValueError("bank, peaks_out and trig_out must all be host or all be device arrays")
        nt = int((bank.numel() if _is_tensor(bank) else bank.size) // 2)
        if _nbytes(peaks_out) < 16 * nt:
            raise ValueError("peaks_out is smaller than 16 bytes per template")
        if trig_out is not None and _nbytes(trig_out) < 16 * int(trig_capacity):
            raise ValueError("trig_out is smaller than 16 bytes per trigger of trig_capacity")
        nf = C.c_int64(0)
        f = lib().cbmf_filter_bank_dev if dev else lib().cbmf_filter_bank
        rc = f(self._h, pb, nt, float(snr_threshold), pp, pt, int(trig_capacity), C.byref(nf))
        self._check(rc, "cbmf_filter_bank")
        return nf.value, rc

    def filter_bank_clustered(self, bank, snr_threshold: float, window_samples: int, event_capacity: int = 1 << 16):
        """Host arrays in, host arrays out: -> (peaks[PEAK_DTYPE], events[TRIG_DTYPE], n_events, n_trig_found, rc).
        The host clusters each sub-batch's triggers while the GPU filters the next ones."""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        peaks = np.zeros(nt, dtype=PEAK_DTYPE)
        ev = np.zeros(max(int(event_capacity), 1), dtype=TRIG_DTYPE)
        ne, nf = C.c_int64(0), C.c_int64(0)
        rc = lib().cbmf_filter_bank_clustered(self._h, b.ctypes.data if nt else None, nt, float(snr_threshold),
                                              int(window_samples), peaks.ctypes.data if nt else None,
                                              ev.ctypes.data if event_capacity else None, int(event_capacity),
                                              C.byref(ne), C.byref(nf))
        self._check(rc, "cbmf_filter_bank")
        return peaks, ev[:min(ne.value, int(event_capacity))], ne.value, nf.value, rc

    def filter_bank_clustered_into(self, bank, snr_threshold: float, window_samples: int, peaks_out, events_out,
                                   event_capacity: int):
        """Caller-owned HOST buffers (numpy / pinned tensors).  -> (n_events, n_trig_found, rc)"""
        pb, dev = _ptr(bank, "float64")
        pp, devp = _ptr(peaks_out, "peak records", itemsize=16)
        pe, deve = _ptr(events_out, "trigger records", itemsize=16)
        if dev or devp or deve:
            raise ValueError("cbmf_filter_bank_clustered takes host arrays (the clustering runs on the host)")
        nt = int((bank.numel() if _is_tensor(bank) else bank.size) // 2)
        if _nbytes(peaks_out) < 16 * nt or (events_out is not None and _nbytes(events_out) < 16 * int(event_capacity)):
            raise ValueError("output buffer too small")
        ne, nf = C.c_int64(0), C.c_int64(0)
        rc = lib().cbmf_filter_bank_clustered(self._h, pb, nt, float(snr_threshold), int(window_samples), pp, pe,
                                              int(event_capacity), C.byref(ne), C.byref(nf))
        self._check(rc, "cbmf_filter_bank")
        return ne.value, nf.value, rc

    def filter_stream(self, samples, bank, snr_threshold: float, discard: int, trig_capacity: int = 1 << 16):
        """cbmf_filter_stream on a host float32 stream (numpy or pinned tensor).
        -> (peaks[S, B] PEAK_DTYPE, triggers TRIG_DTYPE, seg_offsets int64[S + 1], n_found, rc)"""
        if isinstance(samples, np.ndarray):
            samples = np.ascontiguousarray(samples, dtype=np.float32)
        ps, dev = _ptr(samples, "float32")
        if dev:
            raise ValueError("cbmf_filter_stream takes a host stream")
        n_total = int(samples.numel() if _is_tensor(samples) else samples.size)
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        hop = self.n - int(discard)
        n_seg = (n_total - self.n) // hop + 1 if (0 < hop <= self.n and n_total >= self.n) else 1
        peaks = np.zeros((max(n_seg, 1), nt), dtype=PEAK_DTYPE)
        trig = np.zeros(max(int(trig_capacity), 1), dtype=TRIG_DTYPE)
        offs = np.zeros(max(n_seg, 1) + 1, dtype=np.int64)
        nf, ns = C.c_int64(0), C.c_int64(0)
        rc = lib().cbmf_filter_stream(self._h, ps, n_total, b.ctypes.data if nt else None, nt, float(snr_threshold),
                                      int(discard), peaks.ctypes.data if nt else None,
                                      trig.ctypes.data if trig_capacity else None, int(trig_capacity),
                                      offs.ctypes.data, C.byref(nf), C.byref(ns))
        self._check(rc, "cbmf_filter_bank")
        return peaks[:ns.value], trig[:int(offs[ns.value])], offs[:ns.value + 1], nf.value, rc

    def chisq(self, bank, sample_idx, p_bands: int, want_bands: bool = False):
        """cbmf_chisq: chi^2 of every template at its own sample.  -> chisq float32[B] (, z_l complex128[B, p])"""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        idx = np.ascontiguousarray(sample_idx, dtype=np.int32)
        if len(idx) != len(b):
            raise ValueError("one sample index per template")
        chi = np.zeros(len(b), dtype=np.float32)
        zl = np.zeros((len(b), int(p_bands)), dtype=np.complex128) if want_bands else None
        rc = lib().cbmf_chisq(self._h, b.ctypes.data if len(b) else None, len(b), idx.ctypes.data if len(b) else None,
                              int(p_bands), chi.ctypes.data if len(b) else None, zl.ctypes.data if want_bands else None)
        self._check(rc, "cbmf_filter_bank")
        return (chi, zl) if want_bands else chi

    # -- diagnostics
    def debug_snr_series(self, m1: float, m2: float, want_z: bool = True):
        snr = np.empty(self.n, dtype=np.float32)
        z = np.empty(self.n, dtype=np.complex64) if want_z else None
        rc = lib().cbmf_debug_snr_series(self._h, Template(m1, m2), snr.ctypes.data,
                                         z.ctypes.data if want_z else None)
        self._check(rc, "cbmf_debug_snr_series")
        return snr, z

    def debug_td_template(self, m1: float, m2: float):
        """-> (h_plus[n], h_cross[n]) float32: the time-domain polarisations of cbmf_filter_bank_td."""
        h = np.empty((self.n, 2), dtype=np.float32)
        self._check(lib().cbmf_debug_td_template(self._h, Template(m1, m2), h.ctypes.data), "cbmf_debug_td_template")
        return h[:, 0].copy(), h[:, 1].copy()

    def debug_template(self, m1: float, m2: float) -> np.ndarray:
        h = np.empty(self.n // 2 + 1, dtype=np.complex64)
        self._check(lib().cbmf_debug_template(self._h, Template(m1, m2), h.ctypes.data), "cbmf_debug_template")
        return h

    def debug_ifft(self, x, out=None):
        """Unnormalised inverse DFT of `batch` vectors [batch, n] complex64 (numpy or CUDA tensor;
        `out`: optional preallocated CUDA tensor of the same shape)."""
        if _is_tensor(x) and x.is_cuda:
            import torch
            if out is None:
                out = torch.empty_like(x)
            batch = x.numel() // self.n
            self._check(lib().cbmf_debug_ifft_dev(self._h, x.data_ptr(), out.data_ptr(), self.n, batch),
                        "cbmf_debug_ifft_dev")
            return out
        a = np.ascontiguousarray(x, dtype=np.complex64)
        out = np.empty_like(a)
        self._check(lib().cbmf_debug_ifft(self._h, a.ctypes.data, out.ctypes.data, self.n, a.size // self.n),
                    "cbmf_debug_ifft")
        return out

    def debug_generate_dev(self, bank_dev, q_out_dev):
        nt = bank_dev.numel() // 2
        self._check(lib().cbmf_debug_generate_dev(self._h, bank_dev.data_ptr(), nt, q_out_dev.data_ptr()),
                    "cbmf_debug_generate_dev")

    def debug_get_prefix(self) -> np.ndarray:
        p = np.empty(self.n // 2, dtype=np.float64)
        self._check(lib().cbmf_debug_get_prefix(self._h, p.ctypes.data), "cbmf_debug_get_prefix")
        return p

    def debug_get_weights(self) -> np.ndarray:
        w = np.empty(self.n // 2, dtype=np.complex64)
        self._check(lib().cbmf_debug_get_weights(self._h, w.ctypes.data), "cbmf_debug_get_weights")
        return w

    def set_pn_order(self, half_order: int):
        """4 = 2PN phase (default), 5 = 2.5PN (the paper's stated order, NEXT-3)."""
        self._check(lib().cbmf_set_pn_order(self._h, int(half_order)), "cbmf_set_pn_order")

    def get_pn_order(self) -> int:
        return int(lib().cbmf_get_pn_order(self._h))

    # -- tuning / introspection
    def set_sub_batch(self, k: int):
        self._check(lib().cbmf_set_sub_batch(self._h, int(k)), "cbmf_set_sub_batch")

    def get_sub_batch(self) -> int:
        return int(lib().cbmf_get_sub_batch(self._h))

    def set_streams(self, k: int):
        self._check(lib().cbmf_set_streams(self._h, int(k)), "cbmf_set_streams")

    def get_streams(self) -> int:
        return int(lib().cbmf_get_streams(self._h))

    def get_split(self):
        """-> (log2 N1, log2 N2): pass 1 = column FFTs of N1 points, pass 2 = row FFTs of N2 points."""
        a, b = C.c_int(0), C.c_int(0)
        self._check(lib().cbmf_get_split(self._h, C.byref(a), C.byref(b)), "cbmf_get_split")
        return int(a.value), int(b.value)

    def last_bad_template(self) -> int:
        return int(lib().cbmf_last_bad_template(self._h))

    def launch_count(self) -> int:
        return int(lib().cbmf_launch_count(self._h))

    def set_profiling(self, mode: int):
        """0 off, 1 every pass launch alone on the context's stream, 2 in the real overlapped schedule."""
        self._check(lib().cbmf_set_profiling(self._h, int(mode)), "cbmf_set_profiling")

    def debug_timeline(self, which: int) -> np.ndarray:
        """[launches, 2] float32: start / end (ms since the first pass-1 launch) of every launch of pass `which`."""
        out = np.zeros((4096, 2), dtype=np.float32)
        n = C.c_int64(0)
        self._check(lib().cbmf_debug_timeline(self._h, int(which), out.ctypes.data, 4096, C.byref(n)), "cbmf_debug_timeline")
        return out[:min(int(n.value), 4096)]

    def last_pass_time(self, which: int):
        ms, nl = C.c_double(0), C.c_int64(0)
        self._check(lib().cbmf_last_pass_time(self._h, int(which), C.byref(ms), C.byref(nl)), "cbmf_last_pass_time")
        return ms.value, nl.value


def cluster_triggers(trig, n_samples: int, window_samples: int, event_capacity: int | None = None):
    """cbmf_cluster_triggers (host only): trig = TRIG_DTYPE records sorted by (template, sample).
    -> (events[TRIG_DTYPE], n_events, rc)"""
    t = np.ascontiguousarray(trig, dtype=TRIG_DTYPE)
    cap = len(t) if event_capacity is None else int(event_capacity)
    ev = np.zeros(max(cap, 1), dtype=TRIG_DTYPE)
    n = C.c_int64(0)
    rc = lib().cbmf_cluster_triggers(t.ctypes.data if len(t) else None, len(t), int(n_samples), int(window_samples),
                                     ev.ctypes.data if cap else None, cap, C.byref(n))
    if rc < 0:
        raise CbmfError(rc, "cbmf_cluster_triggers")
    return ev[:min(n.value, cap)], n.value, rc


def ifft_noalloc_dev(x, out, n: int, stream: int | None = None) -> int:
    """cbmf_ifft_noalloc_dev: unnormalised inverse DFT of the vectors of `x` ([batch, n] complex64 CUDA tensor) into
    `out` (same shape, same device, preallocated by the caller), for callers that must not allocate device memory
    (a guest of a framework that owns the GPU's memory, a loop that may not stall in cudaMalloc, code running while
    a stream is being captured): no context, the scratch buffer is a fixed 8 MiB array inside the library, hence
    n <= NOALLOC_MAX_N.  This wrapper allocates nothing either and only marshals; the work is enqueued on `stream`
    (a cudaStream_t handle, default stream if None) and NOT waited for.  Calls that may overlap on one GPU share
    the scratch array and race: keep them on one stream.  Returns the raw code (OK, or ELIMIT / EINVAL / ECUDA:
    no exception, so that a caller can probe the limit)."""
    xp, xdev = _ptr(x, "complex64")
    op, odev = _ptr(out, "complex64")
    if not (xdev and odev) or x.device != out.device:
        raise ValueError("x and out must be CUDA tensors on the same device")
    if x.numel() % int(n) or out.numel() != x.numel():
        raise ValueError("x must hold whole vectors of n values and out must match it")
    return int(lib().cbmf_ifft_noalloc_dev(x.device.index, C.c_void_p(stream or 0), xp, op, int(n), x.numel() // int(n)))


def debug_fp32_peak(device: int = 0):
    """cbmf_debug_fp32_peak -> (FFMA TFLOP/s, packed FFMA2 TFLOP/s) measured on dependent FMA chains."""
    a, b = C.c_double(0), C.c_double(0)
    rc = lib().cbmf_debug_fp32_peak(int(device), C.byref(a), C.byref(b))
    if rc < 0:
        raise CbmfError(rc, "cbmf_debug_fp32_peak")
    return a.value, b.value


def version() -> str:
    return lib().cbmf_version().decode()
