"""ctypes binding of the CPU oracle (oracle/mf_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
imports nothing from paper_1006_4644_b200: the oracle and the CUDA path share no
code.

The oracle follows SURVEY.md §8(c) "Definition" (eq. 2.1,
PAPER.md:96-103 steps 1-4); see the header of mf_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mf_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

OK, EINVAL, ESTATE, ENOMEM, WTRUNC = 0, -1, -2, -4, 1


def build(force: bool = False) -> str:
    """Compile mf_oracle.c with gcc -O2 (as it stands, never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Peak(C.Structure):
    _fields_ = [("snr_max", C.c_double), ("idx_peak", C.c_int64),
                ("phase", C.c_double), ("sigma", C.c_double)]


class Trigger(C.Structure):
    _fields_ = [("template_idx", C.c_int64), ("sample_idx", C.c_int64),
                ("snr", C.c_double), ("phase", C.c_double)]


PEAK_DTYPE = np.dtype([("snr_max", "f8"), ("idx_peak", "i8"), ("phase", "f8"), ("sigma", "f8")])
TRIG_DTYPE = np.dtype([("template_idx", "i8"), ("sample_idx", "i8"), ("snr", "f8"), ("phase", "f8")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_fft.argtypes = [dp, C.c_int64, C.c_int]
        L.orc_f_isco.argtypes = [C.c_double, C.c_double]
        L.orc_f_isco.restype = C.c_double
        L.orc_psi.argtypes = [C.c_double] * 3
        L.orc_psi.restype = C.c_double
        L.orc_psi_pn.argtypes = [C.c_double] * 3 + [C.c_int]
        L.orc_psi_pn.restype = C.c_double
        L.orc_set_pn_order.argtypes = [C.c_void_p, C.c_int]
        L.orc_band.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                               C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.orc_create.argtypes = [C.POINTER(C.c_void_p), C.c_int64, C.c_double, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_psd.argtypes = [C.c_void_p, dp, C.c_int64]
        L.orc_load_segment.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int64]
        L.orc_template.argtypes = [C.c_void_p, C.c_double, C.c_double, dp]
        L.orc_sigma2.argtypes = [C.c_void_p, C.c_double, C.c_double, dp]
        L.orc_snr_series.argtypes = [C.c_void_p, C.c_double, C.c_double, dp, dp, dp]
        L.orc_filter_bank.argtypes = [C.c_void_p, dp, C.c_int64, C.c_double, C.POINTER(Peak),
                                      C.POINTER(Trigger), C.c_int64, C.POINTER(C.c_int64)]
        L.orc_chisq.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int64, C.c_int, dp, dp, C.POINTER(C.c_int64)]
        L.orc_cluster_triggers.argtypes = [C.POINTER(Trigger), C.c_int64, C.c_int64, C.c_int64,
                                           C.POINTER(Trigger), C.c_int64, C.POINTER(C.c_int64)]
        L.orc_td_phase.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, dp, dp]
        L.orc_td_extent.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, dp, dp, dp]
        L.orc_td_template.argtypes = [C.c_void_p, C.c_double, C.c_double, dp, dp]
        L.orc_td_snr_series.argtypes = [C.c_void_p, C.c_double, C.c_double, dp, dp, dp, dp, dp]
        L.orc_td_filter_bank.argtypes = [C.c_void_p, dp, C.c_int64, C.c_double, C.POINTER(Peak),
                                         C.POINTER(Trigger), C.c_int64, C.POINTER(C.c_int64)]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, rc, what):
        super().__init__(f"oracle {what} failed: rc={rc}")
        self.rc = rc


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def fft(x: np.ndarray, sign: int) -> np.ndarray:
    """Radix-2 FFT of a complex128 vector; sign=-1 forward, +1 unnormalised inverse."""
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    rc = lib().orc_fft(_dp(a.view(np.float64)), a.size, int(sign))
    if rc:
        raise OracleError(rc, "orc_fft")
    return a


def psi(m1: float, m2: float, f: float) -> float:
    return lib().orc_psi(float(m1), float(m2), float(f))


def psi_pn(m1: float, m2: float, f: float, half_order: int) -> float:
    """SPA phase at 2PN (half_order 4) or 2.5PN (5): NEXT-3."""
    return lib().orc_psi_pn(float(m1), float(m2), float(f), int(half_order))


def f_isco(m1: float, m2: float) -> float:
    return lib().orc_f_isco(float(m1), float(m2))


def band(n: int, fs: float, f_low: float, m1: float, m2: float):
    klo, khi = C.c_int64(), C.c_int64()
    rc = lib().orc_band(n, fs, f_low, m1, m2, C.byref(klo), C.byref(khi))
    if rc:
        raise OracleError(rc, "orc_band")
    return klo.value, khi.value


def td_phase(m1: float, m2: float, tau: float, half_order: int):
    """NEXT-3 (time domain): -> (phi_gw [rad], F [Hz]) at tau = t_c - t seconds before coalescence."""
    phi, f = C.c_double(), C.c_double()
    rc = lib().orc_td_phase(float(m1), float(m2), float(tau), int(half_order), C.byref(phi), C.byref(f))
    if rc:
        raise OracleError(rc, "orc_td_phase")
    return phi.value, f.value


def td_extent(m1: float, m2: float, f_low: float, half_order: int):
    """-> (tau_start, tau_end, f_end): the time-domain template lives on tau_end <= t_c - t <= tau_start."""
    a, b, f = C.c_double(), C.c_double(), C.c_double()
    rc = lib().orc_td_extent(float(m1), float(m2), float(f_low), int(half_order), C.byref(a), C.byref(b), C.byref(f))
    if rc:
        raise OracleError(rc, "orc_td_extent")
    return a.value, b.value, f.value


def cluster_triggers(trig: np.ndarray, n_samples: int, window: int, capacity: int | None = None):
    """NEXT-1 twin: -> (events[TRIG_DTYPE], n_events, rc).  trig: TRIG_DTYPE records."""
    t = np.ascontiguousarray(trig, dtype=TRIG_DTYPE)
    cap = len(t) if capacity is None else int(capacity)
    out = np.zeros(max(cap, 1), dtype=TRIG_DTYPE)
    n = C.c_int64()
    rc = lib().orc_cluster_triggers(t.ctypes.data_as(C.POINTER(Trigger)), len(t), int(n_samples), int(window),
                                    out.ctypes.data_as(C.POINTER(Trigger)), cap, C.byref(n))
    if rc < 0:
        raise OracleError(rc, "orc_cluster_triggers")
    return out[:min(n.value, cap)], n.value, rc


def stream_segments(n_total: int, n: int, discard: int):
    """Segment starts of NEXT-2 (reading A25): hop = n - discard, as many whole segments as fit."""
    if not (0 <= discard < n) or n_total < n:
        raise ValueError("bad stream geometry")
    hop = n - discard
    return [s * hop for s in range((n_total - n) // hop + 1)]


def filter_stream(n: int, fs: float, f_low: float, psd: np.ndarray, stream: np.ndarray, bank: np.ndarray,
                  snr_threshold: float, discard: int):
    """NEXT-2 twin (PAPER.md:247-255 table 4.1, :157): a continuous float32 stream is cut into segments of n samples
    that overlap by `discard` samples; every segment is matched-filtered on its own (circular, as orc_snr_series
    defines it) and the first `discard` output samples, which the wrap-around of templates up to that length
    corrupts, are left out of the peak and of the trigger list.  Written as the definition: per segment and template
    the full series from orc_snr_series, then numpy's argmax / comparison on the slice [discard, n).
    -> (peaks[S, B] PEAK_DTYPE with idx_peak relative to the segment start, triggers TRIG_DTYPE (sample_idx relative
        to the segment start, sorted by (template, sample) inside each segment), seg_offsets int64[S + 1],
        seg_starts list)"""
    starts = stream_segments(len(stream), n, discard)
    b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
    o = Oracle(n, fs, f_low)
    o.set_psd(psd)
    peaks = np.zeros((len(starts), len(b)), dtype=PEAK_DTYPE)
    trig, offs = [], [0]
    for si, s0 in enumerate(starts):
        o.load_segment(np.ascontiguousarray(stream[s0:s0 + n], dtype=np.float32))
        for ti, (m1, m2) in enumerate(b):
            rho, z, sigma = o.snr_series(m1, m2)
            if not sigma > 0:
                peaks[si, ti] = (0.0, -1, 0.0, 0.0)
                continue
            j = discard + int(np.argmax(rho[discard:]))               # first maximum = smallest index
            peaks[si, ti] = (rho[j], j, np.angle(z[j]), sigma)
            for jj in discard + np.nonzero(rho[discard:] > snr_threshold)[0]:
                trig.append((ti, int(jj), rho[jj], np.angle(z[jj])))
        offs.append(len(trig))
    o.close()
    return peaks, np.array(trig, dtype=TRIG_DTYPE), np.array(offs, dtype=np.int64), starts


def num_threads() -> int:
    return lib().orc_num_threads()


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


class Oracle:
    """Context mirroring the product's C ABI (create / set_psd / load_segment / filter_bank)."""

    def __init__(self, n: int, fs: float, f_low: float):
        self.n, self.fs, self.f_low = int(n), float(fs), float(f_low)
        self._h = C.c_void_p()
        rc = lib().orc_create(C.byref(self._h), self.n, self.fs, self.f_low)
        if rc:
            raise OracleError(rc, "orc_create")

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_pn_order(self, half_order: int):
        rc = lib().orc_set_pn_order(self._h, int(half_order))
        if rc:
            raise OracleError(rc, "orc_set_pn_order")

    def set_psd(self, psd: np.ndarray):
        p = np.ascontiguousarray(psd, dtype=np.float64)
        rc = lib().orc_set_psd(self._h, _dp(p), p.size)
        if rc:
            raise OracleError(rc, "orc_set_psd")

    def load_segment(self, samples: np.ndarray):
        s = np.ascontiguousarray(samples, dtype=np.float32)
        rc = lib().orc_load_segment(self._h, s.ctypes.data_as(C.POINTER(C.c_float)), s.size)
        if rc:
            raise OracleError(rc, "orc_load_segment")

    def template(self, m1: float, m2: float) -> np.ndarray:
        h = np.empty(self.n // 2 + 1, dtype=np.complex128)
        rc = lib().orc_template(self._h, m1, m2, _dp(h.view(np.float64)))
        if rc:
            raise OracleError(rc, "orc_template")
        return h

    def sigma2(self, m1: float, m2: float) -> float:
        s = C.c_double()
        rc = lib().orc_sigma2(self._h, m1, m2, C.byref(s))
        if rc:
            raise OracleError(rc, "orc_sigma2")
        return s.value

    def snr_series(self, m1: float, m2: float):
        """-> (rho[n], z[n] complex128, sigma)"""
        rho = np.empty(self.n, dtype=np.float64)
        z = np.empty(self.n, dtype=np.complex128)
        s = C.c_double()
        rc = lib().orc_snr_series(self._h, m1, m2, _dp(rho), _dp(z.view(np.float64)), C.byref(s))
        if rc:
            raise OracleError(rc, "orc_snr_series")
        return rho, z, s.value

    def chisq(self, m1: float, m2: float, j: int, p: int):
        """NEXT-4 twin (ref. [24]): -> (chi^2, z_l complex128[p], band edges int64[p + 1])"""
        chi = C.c_double()
        zl = np.zeros(p, dtype=np.complex128)
        edges = np.zeros(p + 1, dtype=np.int64)
        rc = lib().orc_chisq(self._h, m1, m2, int(j), int(p), C.byref(chi), _dp(zl.view(np.float64)),
                             edges.ctypes.data_as(C.POINTER(C.c_int64)))
        if rc:
            raise OracleError(rc, "orc_chisq")
        return chi.value, zl, edges

    def td_template(self, m1: float, m2: float):
        """NEXT-3 (time domain): -> (h_plus[n], h_cross[n]), coalescence at sample 0 (= n)."""
        hp, hc = np.empty(self.n), np.empty(self.n)
        rc = lib().orc_td_template(self._h, m1, m2, _dp(hp), _dp(hc))
        if rc:
            raise OracleError(rc, "orc_td_template")
        return hp, hc

    def td_snr_series(self, m1: float, m2: float):
        """-> (rho[n], c_plus/sigma_plus [n], c_cross/sigma_cross [n], sigma_plus, sigma_cross)"""
        rho, cp, cc = np.empty(self.n), np.empty(self.n), np.empty(self.n)
        sp, sc = C.c_double(), C.c_double()
        rc = lib().orc_td_snr_series(self._h, m1, m2, _dp(rho), _dp(cp), _dp(cc), C.byref(sp), C.byref(sc))
        if rc:
            raise OracleError(rc, "orc_td_snr_series")
        return rho, cp, cc, sp.value, sc.value

    def td_filter_bank(self, bank: np.ndarray, snr_threshold: float, trig_capacity: int = 1 << 20):
        """-> (peaks[PEAK_DTYPE], triggers[TRIG_DTYPE], n_found, rc) with the time-domain templates"""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        peaks = np.zeros(max(nt, 1), dtype=PEAK_DTYPE)
        trig = np.zeros(max(trig_capacity, 1), dtype=TRIG_DTYPE)
        nf = C.c_int64()
        rc = lib().orc_td_filter_bank(self._h, _dp(b), nt, float(snr_threshold),
                                      peaks.ctypes.data_as(C.POINTER(Peak)),
                                      trig.ctypes.data_as(C.POINTER(Trigger)), trig_capacity, C.byref(nf))
        if rc < 0:
            raise OracleError(rc, "orc_td_filter_bank")
        return peaks[:nt], trig[:min(nf.value, trig_capacity)], nf.value, rc

    def filter_bank(self, bank: np.ndarray, snr_threshold: float, trig_capacity: int = 1 << 20):
        """-> (peaks[PEAK_DTYPE], triggers[TRIG_DTYPE], n_found, rc)"""
        b = np.ascontiguousarray(bank, dtype=np.float64).reshape(-1, 2)
        nt = b.shape[0]
        peaks = np.zeros(max(nt, 1), dtype=PEAK_DTYPE)
        trig = np.zeros(max(trig_capacity, 1), dtype=TRIG_DTYPE)
        nf = C.c_int64()
        rc = lib().orc_filter_bank(self._h, _dp(b), nt, float(snr_threshold),
                                   peaks.ctypes.data_as(C.POINTER(Peak)),
                                   trig.ctypes.data_as(C.POINTER(Trigger)), trig_capacity,
                                   C.byref(nf))
        if rc < 0:
            raise OracleError(rc, "orc_filter_bank")
        return peaks[:nt], trig[:min(nf.value, trig_capacity)], nf.value, rc
