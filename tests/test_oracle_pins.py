"""Pins for the CPU oracle (oracle/mf_oracle.c): what the paper and the mathematics fix.

No test here compares the oracle with itself or with the CUDA path.  The pins are P1-P13 of
SURVEY.md §8(c): brute-force DFT, Parseval, quoted 40-digit phase values, the textbook
chirp-time expansion, closed forms of the normalisation (noise-free injection recovers its
optimal SNR at t_c with phase phi_c; self-match = 1), adaptive quadrature of sigma^2, noise
statistics, covariances, Cauchy-Schwarz, the prefix-sum identity, and an O(N n_b) brute-force
evaluation of the filter definition (eq. 2.1).
"""
import os

import numpy as np
import pytest

import oracle
from testsupport import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _survey_values():
    out = {}
    for line in open(os.path.join(GOLD, "survey_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


SV = _survey_values()


def _direct_dft(x, sign):
    n = x.size
    jk = np.outer(np.arange(n), np.arange(n)) % n
    return (np.exp(sign * 2j * np.pi * jk / n) * x[None, :]).sum(axis=1)


# ------------------------------------------------------------------ P1, P2: the FFT

@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 128, 256])
def test_p1_fft_equals_direct_dft(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        got = oracle.fft(x, sign)
        ref = _direct_dft(x, sign)
        assert np.max(np.abs(got - ref)) < 1e-12 * np.linalg.norm(x) * np.sqrt(n)


def test_p1_fft_roundtrip_delta_linearity():
    n = 4096
    rng = np.random.default_rng(0)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    y = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert np.allclose(oracle.fft(oracle.fft(x, -1), +1), n * x, rtol=0, atol=1e-9)
    j0 = 37
    d = np.zeros(n, complex)
    d[j0] = 1.0
    k = np.arange(n)
    assert np.allclose(oracle.fft(d, -1), np.exp(-2j * np.pi * k * j0 / n), atol=1e-12)
    assert np.allclose(oracle.fft(d, +1), np.exp(+2j * np.pi * k * j0 / n), atol=1e-12)
    a, b = 0.3 - 1.1j, 2.0 + 0.5j
    assert np.allclose(oracle.fft(a * x + b * y, -1), a * oracle.fft(x, -1) + b * oracle.fft(y, -1), atol=1e-9)


def test_p1_fft_rejects_non_power_of_two():
    with pytest.raises(oracle.OracleError):
        oracle.fft(np.zeros(12, complex), -1)


def test_p2_parseval():
    n = 1 << 14
    rng = np.random.default_rng(1)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = oracle.fft(x, -1)
    assert abs(np.sum(np.abs(x) ** 2) - np.sum(np.abs(X) ** 2) / n) < 1e-12 * np.sum(np.abs(x) ** 2)


# ------------------------------------------------------------------ P3, P4, P5: the phase

def _psi_rows():
    rows = []
    for line in open(os.path.join(GOLD, "psi_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 4:
            rows.append(tuple(float(v) for v in line))
    return rows


@pytest.mark.parametrize("m1,m2,f,want", _psi_rows())
def test_p3_psi_quoted_values(m1, m2, f, want):
    assert oracle.psi(m1, m2, f) == pytest.approx(want, rel=2e-13, abs=1e-11)


def test_p3_brackets_at_eta_quarter():
    # recover the 1PN and 2PN brackets from the oracle's Psi by solving for them at three v
    # (eta = 1/4): Psi + pi/4 = 3/(32 v^5) [1 + B1 v^2 - 16 pi v^3 + B2 v^4]
    m = 1.4
    M = 2 * m * W.T_SUN_S
    vs = np.array([0.10, 0.16, 0.22])
    fs_ = vs ** 3 / (np.pi * M)
    lhs = np.array([(oracle.psi(m, m, f) + np.pi / 4) * 32 * v ** 5 / 3 - 1 + 16 * np.pi * v ** 3
                    for f, v in zip(fs_, vs)])
    A = np.stack([vs ** 2, vs ** 4], axis=1)
    b1, b2 = np.linalg.lstsq(A, lhs, rcond=None)[0]
    assert b1 == pytest.approx(SV["bracket_1pn_eta_quarter"], rel=1e-8)
    assert b2 == pytest.approx(SV["bracket_2pn_eta_quarter"], rel=1e-7)


def test_p4_scaling_law_and_symmetry():
    # Psi_T(f; lam m1, lam m2) = Psi_T(lam f; m1, m2); symmetric in m1 <-> m2
    for (m1, m2, f, lam) in [(1.0, 1.0, 100.0, 10.0), (1.4, 2.3, 57.0, 3.5), (2.0, 9.0, 31.0, 0.37)]:
        assert oracle.psi(lam * m1, lam * m2, f) == pytest.approx(oracle.psi(m1, m2, lam * f), rel=1e-13)
        assert oracle.psi(m1, m2, f) == oracle.psi(m2, m1, f) or \
            oracle.psi(m1, m2, f) == pytest.approx(oracle.psi(m2, m1, f), rel=1e-15)


def _chirp_time_textbook(m1, m2, f):
    """Chirp times tau0 + tau1 - tau1.5 + tau2 of the 2PN inspiral (the published
    "chirp time" parametrisation of the restricted 2PN waveform), a different set of rational
    coefficients from those of the phase: 743/336, 11/4, 3058673/1016064, 5429/1008, 617/144."""
    M = (m1 + m2) * W.T_SUN_S
    eta = m1 * m2 / (m1 + m2) ** 2
    x = np.pi * M * f
    t0 = 5.0 / (256.0 * np.pi * f * eta) * x ** (-5.0 / 3.0)
    t1 = 5.0 / (192.0 * np.pi * f * eta) * (743.0 / 336.0 + 11.0 * eta / 4.0) / x
    t15 = 1.0 / (8.0 * f * eta) * x ** (-2.0 / 3.0)
    t2 = 5.0 / (128.0 * np.pi * f * eta) * (3058673.0 / 1016064.0 + 5429.0 * eta / 1008.0
                                           + 617.0 * eta ** 2 / 144.0) * x ** (-1.0 / 3.0)
    return t0, t0 + t1 - t15 + t2


@pytest.mark.parametrize("m1,m2,f,key", [(1.4, 1.4, 40.0, "chirp_s_1p4_40hz"), (1.0, 1.0, 40.0, "chirp_s_1_1_40hz"),
                                        (3.0, 3.0, 40.0, "chirp_s_3_3_40hz"), (10.0, 10.0, 40.0, "chirp_s_10_10_40hz"),
                                        (1.4, 1.4, 10.0, "chirp_s_1p4_10hz")])
def test_p5_stationary_phase_time_equals_chirp_time(m1, m2, f, key):
    # stationary phase: the time before coalescence at which the chirp passes f is
    # tau(f) = -(1/2pi) dPsi/df.  Central difference of the oracle's Psi vs the textbook series.
    h = f * 1e-4
    tau = -(oracle.psi(m1, m2, f + h) - oracle.psi(m1, m2, f - h)) / (2 * h) / (2 * np.pi)
    t0, tsum = _chirp_time_textbook(m1, m2, f)
    assert tau == pytest.approx(tsum, rel=1e-7)
    assert tau == pytest.approx(SV[key], rel=2e-3)          # value printed in SURVEY.md P5
    if key == "chirp_s_1p4_40hz":
        assert t0 == pytest.approx(SV["chirp_newt_s_1p4_40hz"], rel=1e-3)


def test_p5_sign_convention_chirp_sweeps_up_and_ends_at_tc():
    # Reading A3: h~ ~ e^{-i Psi} with the forward transform e^{-2 pi i f t} gives a chirp whose
    # frequency RISES with time and whose energy ends at t_c = 0 (mod T).
    n, fs, f_low = 1 << 16, 2048.0, 40.0
    o = oracle.Oracle(n, fs, f_low)
    h = o.template(3.0, 3.0)                       # 7.1 s long from 40 Hz, fits the 32 s segment
    full = np.zeros(n, complex)
    full[: n // 2 + 1] = h
    ht = oracle.fft(full, +1)                      # analytic signal h(t) + i H[h](t), t_c at j = 0 = n
    p = np.abs(ht) ** 2
    one_s = int(fs)
    assert p[-one_s:].sum() > 50 * p[:one_s].sum()            # energy just before t_c, none after
    assert p[-8 * one_s:].sum() > 0.97 * p.sum()
    # instantaneous frequency from the phase increments, 6 s and 0.05 s before coalescence
    def inst_f(j0):
        seg = ht[j0: j0 + 64]
        return np.angle(seg[1:] * np.conj(seg[:-1])).mean() * fs / (2 * np.pi)
    f_early, f_late = inst_f(n - 6 * one_s), inst_f(n - int(0.05 * fs))
    assert 40.0 < f_early < 50.0 and f_late > 150.0 and f_late > f_early
    # and the early frequency is the one the chirp-time series predicts at tau = 6 s
    lo, hi = 40.0, 60.0
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if _chirp_time_textbook(3.0, 3.0, mid)[1] > 6.0 - 32 / fs else (lo, mid)
    assert f_early == pytest.approx(lo, rel=5e-3)


# ------------------------------------------------------------------ band, f_ISCO, sigma

def test_band_edges_and_fisco_quoted_values():
    assert oracle.f_isco(1.0, 1.0) * 2.0 == pytest.approx(SV["f_isco_times_mtot_hz"], rel=1e-8)
    assert oracle.f_isco(3.0, 7.0) * 10.0 == pytest.approx(SV["f_isco_times_mtot_hz"], rel=1e-8)
    assert oracle.band(1 << 16, 2048.0, 40.0, 1.4, 1.4)[0] == SV["k_lo_cfg0"]
    assert oracle.band(1 << 20, 4096.0, 40.0, 1.4, 1.4)[0] == SV["k_lo_cfg1"]
    assert oracle.band(1 << 22, 4096.0, 10.0, 1.4, 1.4)[0] == SV["k_lo_cfg1"]
    # Nyquist cap (A7): a light system at fs = 2048 is cut at N/2 - 1, never at N/2
    assert oracle.band(1 << 16, 2048.0, 40.0, 1.0, 1.0)[1] == (1 << 15) - 1
    # ISCO cut: floor(f_ISCO / df), inclusive
    klo, khi = oracle.band(1 << 16, 2048.0, 40.0, 10.0, 10.0)
    df = 2048.0 / (1 << 16)
    assert khi * df <= oracle.f_isco(10, 10) < (khi + 1) * df
    # empty band: f_ISCO <= f_low
    klo, khi = oracle.band(1 << 12, 2048.0, 40.0, 60.0, 60.0)
    assert khi < klo


@pytest.mark.parametrize("log2n,fs,f_low,kind,key,tol", [
    (16, 2048.0, 40.0, "A", "sigma_1p4_cfg0", 3e-6), (20, 4096.0, 40.0, "A", "sigma_1p4_cfg1", 3e-6),
    (22, 4096.0, 10.0, "B", "sigma_1p4_cfg3", 3e-6)])
def test_sigma_quoted_values(log2n, fs, f_low, kind, key, tol):
    n = 1 << log2n
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(W.onesided_psd(kind, n, fs, f_low))
    assert np.sqrt(o.sigma2(1.4, 1.4)) == pytest.approx(SV[key], rel=tol)


@pytest.mark.parametrize("log2n,fs,f_low,kind,tol", [(16, 2048.0, 40.0, "A", 3e-5), (20, 4096.0, 40.0, "A", 4e-6)])
def test_p7_sigma_vs_adaptive_quadrature(log2n, fs, f_low, kind, tol):
    from scipy.integrate import quad
    n = 1 << log2n
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(W.onesided_psd(kind, n, fs, f_low))
    m1, m2 = 1.4, 1.4
    klo, khi = oracle.band(n, fs, f_low, m1, m2)
    df = fs / n
    # the rectangle rule over bins [klo, khi] is the midpoint rule on [ (klo-1/2) df, (khi+1/2) df ]
    a, b = (klo - 0.5) * df, (khi + 0.5) * df
    val, _ = quad(lambda f: 4.0 * f ** (-7.0 / 3.0) / W.psd_A(f), a, b, epsabs=0, epsrel=1e-12, limit=400)
    assert o.sigma2(m1, m2) == pytest.approx(val, rel=tol)


def test_p11_prefix_table_equals_direct_sum():
    n, fs, f_low = 1 << 16, 2048.0, 40.0
    psd = W.onesided_psd("A", n, fs, f_low)
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(psd)
    df = fs / n
    k = np.arange(n // 2 + 1)
    with np.errstate(divide="ignore"):
        term = np.where(k >= 1280, (np.maximum(k, 1) * df) ** (-7.0 / 3.0) / psd, 0.0)
    P = 4.0 * df * np.cumsum(term)
    for m1, m2 in [(1.4, 1.4), (1.0, 1.0), (3.0, 9.0), (10.0, 10.0), (2.2, 1.1)]:
        khi = oracle.band(n, fs, f_low, m1, m2)[1]
        assert o.sigma2(m1, m2) == pytest.approx(P[khi], rel=1e-13)


# ------------------------------------------------------------------ P6: closed forms

def _oracle_for(w):
    o = oracle.Oracle(w.n, w.fs, w.f_low)
    o.set_psd(w.psd)
    o.load_segment(w.samples)
    return o


def test_p6_noise_free_injection_recovers_snr_time_phase():
    w = W.config0(noise=False)
    o = _oracle_for(w)
    pk, trig, nf, rc = o.filter_bank(w.bank, w.threshold)
    inj = w.injections[0]
    p = pk[inj.template_idx]
    # samples are rounded to float32 (A21): 6e-8 per sample, ~1e-9 on the peak
    assert p["snr_max"] == pytest.approx(inj.snr, rel=1e-8)
    assert p["idx_peak"] == inj.sample(w.fs) == 40960
    assert p["phase"] == pytest.approx(inj.phi_c, abs=1e-8)
    assert p["sigma"] == pytest.approx(SV["sigma_1p4_cfg0"], rel=3e-6)
    # P10 Cauchy-Schwarz: no other template reaches the exact one
    others = np.delete(pk["snr_max"], inj.template_idx)
    assert np.all(others < inj.snr * (1 - 1e-6))


def test_p6_normalised_self_match_is_one():
    n, fs, f_low = 1 << 14, 2048.0, 40.0
    psd = W.onesided_psd("A", n, fs, f_low)
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(psd)
    m1, m2 = 2.0, 1.3
    h = o.template(m1, m2)
    sigma = np.sqrt(o.sigma2(m1, m2))
    shift = 5000
    k = np.arange(n // 2 + 1)
    d = W.to_time_domain(h / sigma * np.exp(-2j * np.pi * k * shift / n) * np.exp(1j * 1.1), n, fs)
    o.load_segment(d)
    pk, *_ = o.filter_bank(np.array([[m1, m2]]), 6.0)
    assert pk[0]["snr_max"] == pytest.approx(1.0, rel=1e-7)
    assert pk[0]["idx_peak"] == shift
    assert pk[0]["phase"] == pytest.approx(1.1, abs=1e-7)


def test_p13_bruteforce_definition():
    # direct O(N n_b) evaluation of z[j] = 4 df sum_k d~[k] h~*[k]/S_n[k] e^{+2 pi i jk/N}
    # with d~ from a direct DFT (no FFT anywhere), vs the oracle's FFT route
    w = W.small_case(log2n=10, fs=1024.0, f_low=40.0, n_templates=3, seed=5)
    n, df, dt = w.n, w.fs / w.n, 1.0 / w.fs
    o = _oracle_for(w)
    j = np.arange(n)
    for (m1, m2) in w.bank:
        klo, khi = oracle.band(n, w.fs, w.f_low, m1, m2)
        k = np.arange(klo, khi + 1)
        dtil = dt * (w.samples.astype(np.float64)[None, :] * np.exp(-2j * np.pi * np.outer(k, j) / n)).sum(axis=1)
        f = k * df
        hconj = f ** (-7.0 / 6.0) * np.exp(1j * np.array([oracle.psi(m1, m2, x) for x in f]))
        q = 4.0 * df * dtil * hconj / w.psd[k]
        z_ref = (q[None, :] * np.exp(2j * np.pi * np.outer(j, k) / n)).sum(axis=1)
        sigma_ref = np.sqrt(4.0 * df * np.sum(f ** (-7.0 / 3.0) / w.psd[k]))
        rho, z, sigma = o.snr_series(m1, m2)
        assert sigma == pytest.approx(sigma_ref, rel=1e-13)
        assert np.max(np.abs(z - z_ref)) < 1e-11 * np.max(np.abs(z_ref))
        assert np.max(np.abs(rho - np.abs(z_ref) / sigma_ref)) < 1e-10


# ------------------------------------------------------------------ P8: noise statistics

def test_p8_pure_noise_statistics():
    w = W.sweep_point(16, 4)            # noise only, N = 2^16
    o = _oracle_for(w)
    m2s, var_re, var_im, tail = [], [], [], []
    for (m1, m2) in w.bank:
        rho, z, sigma = o.snr_series(m1, m2)
        m2s.append(np.mean(rho ** 2))
        var_re.append(np.var(z.real / sigma))
        var_im.append(np.var(z.imag / sigma))
        tail.append(np.mean(rho > 2.5))
    assert np.mean(m2s) == pytest.approx(2.0, rel=0.03)        # <rho^2> = 2 (A4)
    assert np.mean(var_re) == pytest.approx(1.0, rel=0.04)
    assert np.mean(var_im) == pytest.approx(1.0, rel=0.04)
    assert np.mean(tail) == pytest.approx(np.exp(-2.5 ** 2 / 2), rel=0.15)   # Rayleigh tail


# ------------------------------------------------------------------ P9: covariances

def test_p9_linearity_shift_phase_scale():
    w = W.small_case(log2n=13, n_templates=3, seed=21)
    n = w.n
    m1, m2 = w.bank[1]
    o = _oracle_for(w)
    rho, z, sigma = o.snr_series(m1, m2)
    # circular shift of the data by s samples shifts the output by s
    s = 1234
    o.load_segment(np.roll(w.samples, s))
    rho_s, z_s, _ = o.snr_series(m1, m2)
    assert np.max(np.abs(np.roll(z, s) - z_s)) < 1e-12 * np.max(np.abs(z))
    # d -> a d scales rho by |a|
    o.load_segment((w.samples * np.float32(2.0)))
    rho_a, *_ = o.snr_series(m1, m2)
    assert np.allclose(rho_a, 2.0 * rho, rtol=1e-12)
    # S_n -> c S_n (data fixed) scales rho by 1/sqrt(c); sigma by 1/sqrt(c)
    o.set_psd(4.0 * w.psd)
    o.load_segment(w.samples)
    rho_c, _, sigma_c = o.snr_series(m1, m2)
    assert np.allclose(rho_c, rho / 2.0, rtol=1e-12) and sigma_c == pytest.approx(sigma / 2.0, rel=1e-13)
    # linearity in the data: z(a + b) = z(a) + z(b)
    o.set_psd(w.psd)
    a = w.samples.copy()
    b = np.roll(w.samples, 77) * np.float32(0.5)
    o.load_segment(a)
    za = o.snr_series(m1, m2)[1]
    o.load_segment(b)
    zb = o.snr_series(m1, m2)[1]
    ab = a.astype(np.float64) + b.astype(np.float64)
    o.load_segment(ab.astype(np.float32))
    zab = o.snr_series(m1, m2)[1]
    assert np.max(np.abs(zab - (za + zb))) < 1e-6 * np.max(np.abs(za))   # float32 rounding of a+b


def test_p9_coalescence_phase_rotates_z():
    n, fs, f_low = 1 << 13, 2048.0, 40.0
    psd = W.onesided_psd("A", n, fs, f_low)
    m1, m2 = 1.7, 2.4
    outs = []
    for phi in (0.0, 0.9):
        spec = W.source_spectrum(n, fs, f_low, psd, m1, m2, 2.0, phi, 10.0)
        o = oracle.Oracle(n, fs, f_low)
        o.set_psd(psd)
        o.load_segment(W.to_time_domain(spec, n, fs))
        outs.append(o.snr_series(m1, m2))
    (rho0, z0, _), (rho1, z1, _) = outs
    assert np.max(np.abs(rho0 - rho1)) < 1e-6 * rho0.max()
    j = int(np.argmax(rho0))
    assert np.angle(z1[j] / z0[j]) == pytest.approx(0.9, abs=1e-6)


# ------------------------------------------------------------------ P12: injections in noise

def test_p12_injection_in_noise_cfg0():
    w = W.config0()
    o = _oracle_for(w)
    inj = w.injections[0]
    pk, trig, nf, rc = o.filter_bank(w.bank, w.threshold)
    p = pk[inj.template_idx]
    assert abs(p["snr_max"] - inj.snr) < 3.0
    assert abs(p["idx_peak"] - inj.sample(w.fs)) <= 2
    # the exact template is the loudest of the bank
    assert int(np.argmax(pk["snr_max"])) == inj.template_idx
    # linearity: z(noise + signal) - z(noise) = z(signal)
    z_ns = o.snr_series(inj.m1, inj.m2)[1]
    w_s = W.config0(noise=False)
    o.load_segment(w_s.samples)
    z_s = o.snr_series(inj.m1, inj.m2)[1]
    noise_only = (w.samples.astype(np.float64) - w_s.samples.astype(np.float64)).astype(np.float32)
    o.load_segment(noise_only)
    z_n = o.snr_series(inj.m1, inj.m2)[1]
    assert np.max(np.abs(z_ns - z_n - z_s)) < 1e-5 * np.max(np.abs(z_s))   # float32 sample rounding


# ------------------------------------------------------------------ peaks and triggers

def test_triggers_are_exactly_the_samples_above_threshold():
    w = W.config0()
    o = _oracle_for(w)
    thr = 5.0
    pk, trig, nf, rc = o.filter_bank(w.bank, thr)
    assert rc == oracle.OK and nf == len(trig) and nf > 20
    keys = list(zip(trig["template_idx"], trig["sample_idx"]))
    assert keys == sorted(keys)                                # sorted by (template, sample)
    want = []
    for t, (m1, m2) in enumerate(w.bank):
        rho, z, _ = o.snr_series(m1, m2)
        js = np.nonzero(rho > thr)[0]
        want += [(t, int(j)) for j in js]
        assert pk[t]["idx_peak"] == int(np.argmax(rho)) and pk[t]["snr_max"] == rho.max()
        assert pk[t]["phase"] == pytest.approx(np.angle(z[int(np.argmax(rho))]), abs=1e-14)
        sel = trig[trig["template_idx"] == t]
        assert np.array_equal(sel["snr"], rho[js]) and np.allclose(sel["phase"], np.angle(z[js]), atol=1e-15)
    assert keys == want
    # strict '>' (A14): a threshold equal to a trigger's own SNR drops it
    snr0 = float(trig["snr"].max())
    _, trig2, nf2, _ = o.filter_bank(w.bank, snr0)
    assert nf2 == 0
    # capacity: list truncated, full count still returned, warning code
    _, trig3, nf3, rc3 = o.filter_bank(w.bank, thr, trig_capacity=7)
    assert rc3 == oracle.WTRUNC and nf3 == nf and len(trig3) == 7
    assert list(zip(trig3["template_idx"], trig3["sample_idx"])) == keys[:7]


def test_peak_tie_takes_lowest_index():
    # a periodic input makes the output periodic: the maximum is attained (at least) twice, to
    # within rounding; construct an exact tie instead with all-zero data
    n, fs, f_low = 1 << 10, 1024.0, 40.0
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(W.onesided_psd("A", n, fs, f_low))
    o.load_segment(np.zeros(n, np.float32))
    pk, trig, nf, rc = o.filter_bank(np.array([[1.4, 1.4]]), 6.0)
    assert pk[0]["snr_max"] == 0.0 and pk[0]["idx_peak"] == 0 and nf == 0


def test_empty_band_template_and_errors():
    w = W.small_case(log2n=12, n_templates=4, seed=3)
    o = oracle.Oracle(w.n, w.fs, w.f_low)
    with pytest.raises(oracle.OracleError) as e:      # segment before PSD
        o.load_segment(w.samples)
    assert e.value.rc == oracle.ESTATE
    o.set_psd(w.psd)
    with pytest.raises(oracle.OracleError) as e:      # filter before segment
        o.filter_bank(w.bank, 6.0)
    assert e.value.rc == oracle.ESTATE
    o.load_segment(w.samples)
    bank = np.vstack([w.bank, [[60.0, 60.0]]])          # f_ISCO = 36.6 Hz < f_low: empty band
    pk, trig, nf, rc = o.filter_bank(bank, 6.0)
    assert tuple(pk[-1]) == (0.0, -1, 0.0, 0.0)
    for bad in ([[0.0, 1.0]], [[1.0, -2.0]], [[np.nan, 1.0]], [[np.inf, 1.0]]):
        with pytest.raises(oracle.OracleError) as e:
            o.filter_bank(np.array(bad), 6.0)
        assert e.value.rc == oracle.EINVAL
    with pytest.raises(oracle.OracleError):
        o.filter_bank(w.bank, -1.0)
    bad_psd = w.psd.copy()
    bad_psd[w.n // 4] = 0.0
    with pytest.raises(oracle.OracleError):
        o.set_psd(bad_psd)
    bad_psd[w.n // 4] = np.nan
    with pytest.raises(oracle.OracleError):
        o.set_psd(bad_psd)
    s = w.samples.copy()
    s[5] = np.inf
    with pytest.raises(oracle.OracleError):
        o.load_segment(s)
    with pytest.raises(oracle.OracleError):
        oracle.Oracle(1000, 2048.0, 40.0)
    with pytest.raises(oracle.OracleError):
        oracle.Oracle(1024, 2048.0, 2000.0)
    # changing the PSD invalidates the segment
    o.set_psd(w.psd)
    with pytest.raises(oracle.OracleError) as e:
        o.filter_bank(w.bank, 6.0)
    assert e.value.rc == oracle.ESTATE


def test_psd_infinite_weight_zero():
    # A9: +inf PSD bins carry weight 0 -- making some in-band bins infinite must equal removing them
    w = W.small_case(log2n=12, n_templates=2, seed=8)
    psd = w.psd.copy()
    psd[300:340] = np.inf
    o = oracle.Oracle(w.n, w.fs, w.f_low)
    o.set_psd(psd)
    o.load_segment(w.samples)
    m1, m2 = w.bank[0]
    rho, z, sigma = o.snr_series(m1, m2)
    klo, khi = oracle.band(w.n, w.fs, w.f_low, m1, m2)
    k = np.array([kk for kk in range(klo, khi + 1) if not 300 <= kk < 340])
    df = w.fs / w.n
    assert sigma ** 2 == pytest.approx(4 * df * np.sum((k * df) ** (-7 / 3) / psd[k]), rel=1e-13)
    assert np.all(np.isfinite(rho))


def test_oracle_under_sanitizers(tmp_path):
    """the oracle built with -fsanitize=address,undefined runs two pins (P1 and the bank
    loop with an empty band and a truncated list) without a report (tests/asan_driver.c)."""
    import subprocess
    exe = str(tmp_path / "asan_driver")
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", "-o", exe, os.path.join(ROOT, "tests", "asan_driver.c"),
           os.path.join(ROOT, "oracle", "mf_oracle.c"), "-lm"]
    subprocess.run(cmd, check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="2")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and "asan driver ok" in r.stdout, (r.returncode, r.stdout, r.stderr[-2000:])


# ------------------------------------------------------------------ NEXT-1: trigger clustering
# Pins: hand-built trigger lists whose events follow from the definition (reading A24) by inspection.

def _tr(rows):
    a = np.zeros(len(rows), dtype=oracle.TRIG_DTYPE)
    for i, (t, j, r) in enumerate(rows):
        a[i] = (t, j, r, 0.1 * i)
    return a


def _ev(ev):
    return [(int(e["template_idx"]), int(e["sample_idx"]), float(e["snr"])) for e in ev]


def test_cluster_single_run_keeps_its_maximum():
    tr = _tr([(0, 100, 6.5), (0, 101, 7.5), (0, 102, 9.0), (0, 103, 8.0), (0, 104, 6.1)])
    ev, n, rc = oracle.cluster_triggers(tr, 1 << 12, 2)
    assert rc == 0 and n == 1 and _ev(ev) == [(0, 102, 9.0)]
    assert ev[0]["phase"] == tr[2]["phase"]                        # the whole record of the maximum is kept


def test_cluster_gap_rule_is_inclusive_at_window():
    base = [(0, 10, 7.0), (0, 15, 8.0)]                            # 5 samples apart
    assert oracle.cluster_triggers(_tr(base), 4096, 5)[1] == 1     # gap == window: one event
    ev, n, _ = oracle.cluster_triggers(_tr(base), 4096, 4)         # gap > window: two events
    assert n == 2 and _ev(ev) == [(0, 10, 7.0), (0, 15, 8.0)]
    assert oracle.cluster_triggers(_tr(base), 4096, 0)[1] == 2     # window 0: every sample its own event


def test_cluster_chain_links_far_ends():
    """Samples 0, 3, 6, 9 with window 3 are one event although 0 and 9 are 9 apart (chain rule)."""
    tr = _tr([(2, 0, 6.1), (2, 3, 6.2), (2, 6, 6.9), (2, 9, 6.3), (2, 20, 7.7)])
    ev, n, _ = oracle.cluster_triggers(tr, 4096, 3)
    assert n == 2 and _ev(ev) == [(2, 6, 6.9), (2, 20, 7.7)]


def test_cluster_wraps_around_the_segment_end():
    """The filter output is circular (A11): N-2 and 1 are 3 samples apart."""
    n_s = 1024
    tr = _tr([(0, 1, 6.5), (0, 500, 7.0), (0, n_s - 2, 8.5)])
    ev, n, _ = oracle.cluster_triggers(tr, n_s, 3)
    assert n == 2 and _ev(ev) == [(0, 500, 7.0), (0, n_s - 2, 8.5)]
    ev, n, _ = oracle.cluster_triggers(tr, n_s, 2)
    assert n == 3
    # a ring of triggers that closes on itself is ONE event
    ring = _tr([(0, j, 6.0 + 0.001 * j) for j in range(0, n_s, 4)])
    ev, n, _ = oracle.cluster_triggers(ring, n_s, 4)
    assert n == 1 and _ev(ev) == [(0, n_s - 4, 6.0 + 0.001 * (n_s - 4))]


def test_cluster_ties_take_the_smallest_sample():
    tr = _tr([(0, 40, 7.0), (0, 41, 9.0), (0, 42, 9.0), (0, 43, 8.0)])
    ev, n, _ = oracle.cluster_triggers(tr, 4096, 1)
    assert _ev(ev) == [(0, 41, 9.0)]
    n_s = 256                                                      # tie across the wrap: sample 0 < sample N-1
    tr = _tr([(0, n_s - 1, 9.0), (0, 0, 9.0)])
    assert _ev(oracle.cluster_triggers(tr, n_s, 1)[0]) == [(0, 0, 9.0)]


def test_cluster_templates_never_merge_and_order_is_template_then_sample():
    tr = _tr([(3, 100, 6.5), (1, 100, 7.0), (1, 101, 7.5), (3, 101, 6.6), (0, 4000, 8.0), (1, 900, 6.2)])   # unsorted input
    ev, n, rc = oracle.cluster_triggers(tr, 4096, 8)
    assert rc == 0 and _ev(ev) == [(0, 4000, 8.0), (1, 101, 7.5), (1, 900, 6.2), (3, 101, 6.6)]


def test_cluster_empty_count_only_truncation_and_errors():
    ev, n, rc = oracle.cluster_triggers(_tr([]), 1024, 5)
    assert n == 0 and rc == 0 and len(ev) == 0
    tr = _tr([(0, 10, 7.0), (0, 100, 8.0), (1, 5, 6.5)])
    ev, n, rc = oracle.cluster_triggers(tr, 1024, 5, capacity=2)
    assert n == 3 and rc == oracle.WTRUNC and _ev(ev) == [(0, 10, 7.0), (0, 100, 8.0)]
    ev, n, rc = oracle.cluster_triggers(tr, 1024, 5, capacity=0)
    assert n == 3 and len(ev) == 0
    with pytest.raises(oracle.OracleError):
        oracle.cluster_triggers(_tr([(0, 2000, 7.0)]), 1024, 5)    # sample outside the segment
    with pytest.raises(oracle.OracleError):
        oracle.cluster_triggers(tr, 1024, -1)


def test_cluster_of_a_real_trigger_list_cfg0():
    """configs[0] through the oracle: the SNR-12 injection gives a run of adjacent above-threshold samples in
    the matching template; with a window of 16 samples it is ONE event at the peak sample, and the number of
    events equals the number of runs counted directly from the series."""
    w = W.config0()
    o = oracle.Oracle(w.n, w.fs, w.f_low)
    o.set_psd(w.psd)
    o.load_segment(w.samples)
    pk, tr, nf, _ = o.filter_bank(w.bank, w.threshold)
    ev, n, rc = oracle.cluster_triggers(tr, w.n, 16)
    mine = ev[ev["template_idx"] == 16]
    assert len(mine) == 1 and int(mine[0]["sample_idx"]) == int(pk[16]["idx_peak"]) and mine[0]["snr"] == pk[16]["snr_max"]
    # count runs directly: per template, sorted samples, a new run where the circular gap exceeds the window
    runs = 0
    for t in np.unique(tr["template_idx"]):
        s = np.sort(tr["sample_idx"][tr["template_idx"] == t])
        gaps = np.diff(np.concatenate([s, [s[0] + w.n]]))
        runs += max(1, int(np.sum(gaps > 16)))
    assert n == runs


# ------------------------------------------------------------------ NEXT-2: segment streaming

def _stream_case(n=1 << 14, fs=2048.0, f_low=40.0, n_seg_hops=3, snr=11.0, m=(2.5, 2.0), noise_seed=None):
    """A stream of n + n_seg_hops * n/2 samples: one chirp whose whole duration (1.8 s from 40 Hz for 2.5 + 2.0)
    lies inside the valid half of segment 1, optionally on coloured noise."""
    hop = n // 2
    n_total = n + n_seg_hops * hop
    big = 1 << int(np.ceil(np.log2(n_total)))
    psd_big = W.onesided_psd("A", big, fs, f_low)
    t_c = (hop + n // 2 + n // 4) / fs                         # global sample 1.25 n: segment 1, local sample 0.75 n
    spec = W.source_spectrum(big, fs, f_low, psd_big, m[0], m[1], t_c, 0.4, snr)
    if noise_seed is not None:
        spec = spec + W.noise_spectrum(big, fs, f_low, psd_big, noise_seed)
    stream = W.to_time_domain(spec, big, fs)[:n_total]
    return n, fs, f_low, W.onesided_psd("A", n, fs, f_low), stream, hop, int(round(t_c * fs))


def test_stream_geometry():
    assert oracle.stream_segments(4096, 1024, 512) == [0, 512, 1024, 1536, 2048, 2560, 3072]
    assert oracle.stream_segments(1024, 1024, 512) == [0]
    assert oracle.stream_segments(4000, 1024, 0) == [0, 1024, 2048]
    with pytest.raises(ValueError):
        oracle.stream_segments(1000, 1024, 0)


def test_stream_no_discard_equals_independent_segments():
    """discard = 0: the stream call is the bank call on consecutive disjoint segments."""
    n, fs, f_low, psd, stream, hop, _ = _stream_case(n=1 << 12, noise_seed=5)
    bank = np.array([[2.5, 2.0], [1.4, 1.4]])
    pk, tr, offs, starts = oracle.filter_stream(n, fs, f_low, psd, stream, bank, 4.0, 0)
    assert starts == [0, n]
    o = oracle.Oracle(n, fs, f_low); o.set_psd(psd)
    for s, s0 in enumerate(starts):
        o.load_segment(stream[s0:s0 + n])
        pk1, tr1, _, _ = o.filter_bank(bank, 4.0)
        assert np.array_equal(pk[s]["idx_peak"], pk1["idx_peak"]) and np.allclose(pk[s]["snr_max"], pk1["snr_max"], rtol=1e-14)
        seg = tr[offs[s]:offs[s + 1]]
        assert np.array_equal(seg["template_idx"], tr1["template_idx"]) and np.array_equal(seg["sample_idx"], tr1["sample_idx"])


def test_stream_recovers_injection_in_the_segment_that_holds_it():
    """Noise-free stream: the chirp lies wholly inside segment 1 and ends in its valid half, so segment 1 recovers
    SNR, global time and phase as the one-segment closed form does (P6); in segments 0 and 2 its coalescence time
    falls outside the valid half, so their valid-half maxima stay well below it; every reported index is >= discard."""
    n, fs, f_low, psd, stream, hop, j_glob = _stream_case()
    bank = np.array([[2.5, 2.0]])
    pk, tr, offs, starts = oracle.filter_stream(n, fs, f_low, psd, stream, bank, 6.0, hop)
    assert starts == [0, hop, 2 * hop, 3 * hop]
    assert int(pk[1, 0]["idx_peak"]) + starts[1] == j_glob
    # the band-limited SPA chirp has long low-frequency tails in the time domain (sharp 40 Hz edge): the 8 s segment
    # cuts ~1.5 % of its SNR; the full-length buffer recovers 11.0000 (P6)
    assert abs(pk[1, 0]["snr_max"] - 11.0) < 0.03 * 11.0
    assert abs(pk[1, 0]["phase"] - 0.4) < 2e-2
    assert np.all(pk["idx_peak"] >= hop)
    assert pk[0, 0]["snr_max"] < 0.8 * 11.0 and pk[3, 0]["snr_max"] < 0.8 * 11.0
    # segment 2 holds the coalescence time at local sample n/4 < discard: not reported there
    seg2 = tr[offs[2]:offs[3]]
    assert not np.any(seg2["sample_idx"] + starts[2] == j_glob)
    seg1 = tr[offs[1]:offs[2]]
    assert np.any(seg1["sample_idx"] + starts[1] == j_glob) and np.all(seg1["sample_idx"] >= hop)


def test_stream_valid_half_is_free_of_wrap_around():
    """Overlap-save: for a template shorter than the discarded part, the valid-half outputs of a segment depend only
    on that segment's data in the right place: the series of segment 1 on [discard, n) equals, sample for sample, the
    series of a segment twice as long that holds the same data at those times -- up to the slowly decaying tails of the
    band-limited template and whitening responses."""
    n, fs, f_low, psd, stream, hop, j_glob = _stream_case(noise_seed=9)
    m1, m2 = 2.5, 2.0
    o1 = oracle.Oracle(n, fs, f_low); o1.set_psd(psd); o1.load_segment(stream[hop:hop + n])
    rho1 = o1.snr_series(m1, m2)[0]
    # the long segment covers global samples [0, 2n); segment 1 covers [hop, hop + n), its valid half is [n, 1.5 n)
    o2 = oracle.Oracle(2 * n, fs, f_low); o2.set_psd(W.onesided_psd("A", 2 * n, fs, f_low)); o2.load_segment(stream[:2 * n])
    rho2 = o2.snr_series(m1, m2)[0]
    a, b = rho1[hop:], rho2[n:n + hop]
    # not exact: S_n is a hard wall at f_low (configs[0]: "else infinite"), so template and 1/S_n ring for seconds
    # and a little of the wrapped data leaks into the valid half: a few per cent of the peak at worst, 1 % typically
    assert np.max(np.abs(a - b)) < 0.08 * rho1.max() and np.median(np.abs(a - b)) < 0.02 * rho1.max()
    assert int(np.argmax(a)) == int(np.argmax(b))
    # while the discarded part IS corrupted by what wraps around from the segment's end (the chirp itself)
    assert np.max(np.abs(rho1[:hop // 4] - rho2[hop:hop + hop // 4])) > 3 * np.max(np.abs(a - b))


# ------------------------------------------------------------------ NEXT-4: chi-squared veto (ref. [24])

def _orc(w):
    o = oracle.Oracle(w.n, w.fs, w.f_low)
    o.set_psd(w.psd)
    o.load_segment(w.samples)
    return o


def test_chisq_bands_sum_to_the_filter_output_and_have_equal_power():
    w = W.config0()
    o = _orc(w)
    m1, m2 = 1.4, 1.4
    rho, z, sigma = o.snr_series(m1, m2)
    klo, khi = oracle.band(w.n, w.fs, w.f_low, m1, m2)
    f = np.arange(w.n // 2 + 1) * (w.fs / w.n)
    for p in (1, 2, 8, 16):
        for j in (0, 40960, 12345, w.n - 1):
            chi, zl, edges = o.chisq(m1, m2, j, p)
            assert abs(zl.sum() - z[j]) <= 1e-9 * abs(z).max()            # sum_l z_l = z[j] (pinned series, P13)
            assert edges[0] == klo and edges[p] == khi + 1 and np.all(np.diff(edges) > 0)
        # equal expected SNR^2 per band, to the granularity of one bin
        term = 4.0 * (w.fs / w.n) * f[klo:khi + 1] ** (-7.0 / 3.0) / w.psd[klo:khi + 1]
        s2 = np.array([term[edges[l] - klo:edges[l + 1] - klo].sum() for l in range(p)])
        assert abs(s2.sum() - sigma ** 2) <= 1e-12 * sigma ** 2
        assert np.max(np.abs(s2 - sigma ** 2 / p)) <= term.max() * 1.0000001
    assert o.chisq(m1, m2, 40960, 1)[0] == 0.0                            # p = 1: identically zero


def test_chisq_vanishes_for_data_proportional_to_the_template():
    w = W.config0(noise=False)                                            # noise-free exact-parameter injection
    o = _orc(w)
    j = w.injections[0].sample(w.fs)
    for p in (2, 8, 16):
        chi, zl, _ = o.chisq(1.4, 1.4, j, p)
        assert chi < 1e-9                                                 # against rho^2 = 144
    # another template on the same data: the bands disagree
    assert o.chisq(2.2, 1.1, j, 8)[0] > 1.0


def test_chisq_has_2p_minus_2_degrees_of_freedom_in_noise():
    w = W.sweep_point(16, 4)                                              # noise only, N = 2^16
    o = _orc(w)
    p = 8
    js = np.arange(0, w.n, 97)[:400]
    chis = np.array([o.chisq(w.bank[0, 0], w.bank[0, 1], int(j), p)[0] for j in js])
    assert abs(chis.mean() - (2 * p - 2)) < 0.08 * (2 * p - 2)            # mean of a chi^2_14: 14 +- 0.26 over 400
    assert abs(chis.var() - 2 * (2 * p - 2)) < 0.35 * 2 * (2 * p - 2)


def test_chisq_rejects_a_glitch_that_rings_the_template():
    """A loud impulse gives a large SNR in every template but its power is spread evenly over frequency, not as
    f^-7/3: chi^2 per degree of freedom is far above 1, while the chirp of configs[0] in noise stays near 1."""
    w = W.config0()
    o = _orc(w)
    j_inj = w.injections[0].sample(w.fs)
    chi_sig = o.chisq(1.4, 1.4, j_inj, 16)[0]
    assert chi_sig < 2.0 * 30
    s = w.samples.copy(); s[30000] += 4.0e4
    o.load_segment(s)
    pk, _, _, _ = o.filter_bank(w.bank[16:17], 6.0)
    assert pk[0]["snr_max"] > 12.0
    chi_glitch = o.chisq(1.4, 1.4, int(pk[0]["idx_peak"]), 16)[0]
    assert chi_glitch > 10 * 30


# ------------------------------------------------------------------ NEXT-3: the 2.5PN phase term

def _taylorf2_from_energy_balance(eta):
    """Coefficients psi_n, n = 0..5, of Psi(f) = 3/(128 eta v^5) sum_n psi_n v^n (n = 5: the coefficient of ln f,
    i.e. of 3 ln v), DERIVED here from the post-Newtonian energy function and flux by the stationary-phase relation
    d^2 Psi / df^2 = 2 pi dt/df = -(2 pi^2 M^2 / 3) e'(v) / (v^2 F(v)),  v = (pi M f)^(1/3):
    series division of e'(v) by F(v), then two integrations in f term by term (the v^5 term integrates to ln f).
    Energy and flux to 2.5PN (Blanchet, Living Rev. Relativity 9, 4 (2006), eqs. (194) and (231), circular orbits):
      e(v)  = -(eta v^2 / 2) [1 - (9 + eta)/12 v^2 - (81 - 57 eta + eta^2)/24 v^4]
      F(v)  = (32/5) eta^2 v^10 [1 - (1247/336 + 35 eta/12) v^2 + 4 pi v^3
              + (-44711/9072 + 9271 eta/504 + 65 eta^2/18) v^4 - (8191/672 + 583 eta/24) pi v^5]."""
    from fractions import Fraction as Fr
    import math
    pi = math.pi
    a2, a4 = -(9 + eta) / 12.0, -(81 - 57 * eta + eta ** 2) / 24.0
    num = [1.0, 0.0, 2 * a2, 0.0, 3 * a4, 0.0]                                  # -e'(v) / (eta v)
    den = [1.0, 0.0, -(1247 / 336 + 35 * eta / 12), 4 * pi,
           -44711 / 9072 + 9271 * eta / 504 + 65 * eta ** 2 / 18, -(8191 / 672 + 583 * eta / 24) * pi]
    s = []                                                                      # S(v) = num / den, power series
    for n in range(6):
        s.append(num[n] - sum(s[k] * den[n - k] for k in range(n)))
    # Psi'' = K v^-11 S(v), K = 5 pi^2 M^2 / (48 eta); integrating f^alpha twice, alpha = (n - 11)/3:
    # psi_n = 40 s_n / ((n - 8)(n - 5)) for n != 5, and the ln f coefficient is -(40/9) s_5 (see DESIGN.md §3 A27)
    out = [40.0 * s[n] / ((n - 8) * (n - 5)) for n in range(5)]
    out.append(-(40.0 / 9.0) * s[5])
    return out


@pytest.mark.parametrize("m1,m2", [(1.4, 1.4), (1.0, 3.0), (10.0, 1.2)])
def test_p3b_phase_coefficients_follow_from_energy_balance(m1, m2):
    """Pins BOTH the 2PN coefficients of orc_psi (already fixed by the survey's 40-digit values) and the 2.5PN term of
    orc_psi_pn: extract the oracle's coefficients numerically and compare with the energy-balance derivation."""
    eta = m1 * m2 / (m1 + m2) ** 2
    want = _taylorf2_from_energy_balance(eta)
    assert abs(want[0] - 1.0) < 1e-14 and abs(want[1]) < 1e-14
    assert abs(want[2] - (3715 / 756 + 55 * eta / 9)) < 1e-12
    assert abs(want[3] + 16 * np.pi) < 1e-12
    assert abs(want[4] - (15293365 / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72)) < 1e-11
    assert abs(want[5] - np.pi * (38645 / 756 - 65 * eta / 9)) < 1e-11
    # the oracle's 2.5PN term, extracted as a function: [Psi_2.5 - Psi_2] * 128 eta / 3 = C (1 + ln(f / f_isco))
    M = (m1 + m2) * 4.925490947641267e-6
    fi = oracle.f_isco(m1, m2)
    for f in (10.0, 40.0, 133.0, 900.0):
        extra = (oracle.psi_pn(m1, m2, f, 5) - oracle.psi_pn(m1, m2, f, 4)) * 128 * eta / 3
        assert abs(extra - want[5] * (1 + np.log(f / fi))) < 1e-9 * abs(want[5]) * 10
        assert oracle.psi_pn(m1, m2, f, 4) == oracle.psi(m1, m2, f)
    # and the full oracle phase against the derived series, evaluated independently
    for f in (20.0, 100.0, 400.0):
        v = (np.pi * M * f) ** (1 / 3)
        series = -np.pi / 4 + 3 / (128 * eta * v ** 5) * (sum(want[n] * v ** n for n in range(5))
                                                         + want[5] * v ** 5 * (1 + 3 * np.log(v * np.sqrt(6.0))))
        assert abs(series - oracle.psi_pn(m1, m2, f, 5)) < 1e-9 * abs(series)


def test_p3b_chirp_time_with_the_25pn_term():
    """-(1/2 pi) dPsi/df = time to coalescence: the 2.5PN term adds C/(2 pi f) * 3/(128 eta), a few tenths of a second
    at 40 Hz for 1.4 + 1.4 (the 2.5PN chirp-time term is negative in tau, i.e. the chirp is shorter)."""
    m1 = m2 = 1.4
    eta = 0.25
    f, h = 40.0, 1e-3
    tau = lambda order: -(oracle.psi_pn(m1, m2, f + h, order) - oracle.psi_pn(m1, m2, f - h, order)) / (2 * h) / (2 * np.pi)
    c5 = np.pi * (38645 / 756 - 65 * eta / 9)
    assert abs((tau(5) - tau(4)) + 3 / (128 * eta) * c5 / (2 * np.pi * f)) < 1e-6
    assert -0.25 < tau(5) - tau(4) < -0.05


# ------------------------------------------------------------------ NEXT-3, second part: the time-domain generator
# (PAPER.md:173-179).  Pins of orc_td_phase / orc_td_extent / orc_td_template / orc_td_snr_series / orc_td_filter_bank.

def _energy_balance_dvdt(M, eta, v, half_order):
    """dv/dt = -Flux(v) / (M e'(v)) with the energy function and flux quoted in _taylorf2_from_energy_balance
    (Blanchet, Living Rev. Relativity 9, 4 (2006), eqs. (194), (231)), the flux cut at the same order as the phase."""
    pi = np.pi
    a2, a4 = -(9 + eta) / 12.0, -(81 - 57 * eta + eta ** 2) / 24.0
    eprime = -eta * v * (1 + 2 * a2 * v ** 2 + 3 * a4 * v ** 4)
    series = (1 - (1247 / 336 + 35 * eta / 12) * v ** 2 + 4 * pi * v ** 3
              + (-44711 / 9072 + 9271 * eta / 504 + 65 * eta ** 2 / 18) * v ** 4)
    if half_order >= 5:
        series -= (8191 / 672 + 583 * eta / 24) * pi * v ** 5
    flux = 32 / 5 * eta ** 2 * v ** 10 * series
    return -flux / (M * eprime)


def _tau_at_v(m1, m2, v, order):
    M = (m1 + m2) * 4.925490947641267e-6
    target = v ** 3 / (np.pi * M)
    lo, hi = 1e-6, 1e9                                   # F decreases with tau on the branch that sweeps upward
    for _ in range(200):
        mid = np.sqrt(lo * hi)
        if oracle.td_phase(m1, m2, mid, order)[1] > target:
            lo = mid
        else:
            hi = mid
    return np.sqrt(lo * hi)


@pytest.mark.parametrize("m1,m2", [(1.4, 1.4), (1.0, 3.0), (10.0, 1.2)])
@pytest.mark.parametrize("order", [4, 5])
def test_td_frequency_obeys_energy_balance(m1, m2, order):
    """The explicit-in-time series is the inversion of t(v) from dE/dt = -Flux, so v(t) = (pi M F)^(1/3) of
    orc_td_phase satisfies dv/dt = -Flux/(M e'(v)) up to the first neglected order: a relative residual c v^(n+1)
    with c nearly constant (n = 4: 2PN, n = 5: 2.5PN).  A wrong coefficient at order m <= n leaves a residual
    ~ v^m instead: the ratio residual / v^(n+1) would then change by (0.15/0.05)^(n+1-m) >= 3 over the range."""
    M = (m1 + m2) * 4.925490947641267e-6
    eta = m1 * m2 / (m1 + m2) ** 2
    ratios = []
    for v in (0.05, 0.07, 0.10, 0.15):
        tau = _tau_at_v(m1, m2, v, order)
        h = tau * 1e-5
        v_hi = (np.pi * M * oracle.td_phase(m1, m2, tau - h, order)[1]) ** (1 / 3)
        v_lo = (np.pi * M * oracle.td_phase(m1, m2, tau + h, order)[1]) ** (1 / 3)
        dvdt = (v_hi - v_lo) / (2 * h)
        want = _energy_balance_dvdt(M, eta, v, order)
        ratios.append((dvdt - want) / want / v ** (order + 1))
    ratios = np.array(ratios)
    assert np.all(np.abs(ratios) < 250) and np.all(np.abs(ratios) > 20)
    assert np.max(np.abs(ratios)) / np.min(np.abs(ratios)) < 1.35, ratios
    assert np.all(np.sign(ratios) == np.sign(ratios[0]))


@pytest.mark.parametrize("order", [4, 5])
def test_td_frequency_is_the_phase_derivative(order):
    """F = (1/2 pi) d phi_gw / dt = -(1/2 pi) d phi_gw / d tau; the phase grows with time; to leading order F is the
    textbook Newtonian chirp F = (1/pi) (5/(256 tau))^(3/8) Mc^(-5/8), the corrections being of relative order v^2."""
    m1, m2 = 1.4, 1.4
    Mc = (m1 * m2) ** 0.6 / (m1 + m2) ** 0.2 * 4.925490947641267e-6
    for tau in (30.0, 3.0, 0.3, 0.03):
        h = tau * 1e-6
        p_late, f = oracle.td_phase(m1, m2, tau - h, order)[0], oracle.td_phase(m1, m2, tau, order)[1]
        p_early = oracle.td_phase(m1, m2, tau + h, order)[0]
        assert p_late > p_early
        assert (p_late - p_early) / (2 * h) / (2 * np.pi) == pytest.approx(f, rel=2e-6)
        newton = (5.0 / (256.0 * tau)) ** 0.375 * Mc ** -0.625 / np.pi
        assert f == pytest.approx(newton, rel=0.02 + 2.0 * (np.pi * (m1 + m2) * 4.925490947641267e-6 * f) ** (2 / 3))


def test_td_extent_end_points():
    """The template starts where F = f_low and ends at f_ISCO (2PN, comparable masses) or at the maximum of F where
    the series stops sweeping upward first (2.5PN); 1.4 + 1.4 Msun from 40 Hz lasts 25 s (Newtonian chirp time 24.9 s
    plus post-Newtonian corrections of a few per cent)."""
    m1 = m2 = 1.4
    ts, te, fe = oracle.td_extent(m1, m2, 40.0, 4)
    assert oracle.td_phase(m1, m2, ts, 4)[1] == pytest.approx(40.0, rel=1e-12)
    assert fe == pytest.approx(oracle.f_isco(m1, m2), rel=1e-12)
    assert oracle.td_phase(m1, m2, te, 4)[1] == pytest.approx(fe, rel=1e-12)
    Mc = (m1 * m2) ** 0.6 / (m1 + m2) ** 0.2 * 4.925490947641267e-6
    t_newton = 5.0 / 256.0 * (np.pi * 40.0) ** (-8.0 / 3.0) * Mc ** (-5.0 / 3.0)
    assert 24.5 < t_newton < 25.5 and ts == pytest.approx(t_newton, rel=0.06)
    ts5, te5, fe5 = oracle.td_extent(m1, m2, 40.0, 5)
    assert 300.0 < fe5 < oracle.f_isco(m1, m2)                    # stops early: F has a maximum there
    for sgn in (-1, 1):
        assert oracle.td_phase(m1, m2, te5 * (1 + sgn * 1e-3), 5)[1] < fe5 * (1 + 1e-12)
    assert ts5 == pytest.approx(ts, rel=0.02) and ts5 != ts
    # a system whose f_ISCO lies below the cut-off has no template
    assert oracle.td_extent(60.0, 60.0, 40.0, 4)[:2] == (0.0, 0.0)


def _td_case(n=1 << 15, fs=2048.0, f_low=40.0, order=4):
    psd = W.onesided_psd("A", n, fs, f_low)
    o = oracle.Oracle(n, fs, f_low)
    o.set_pn_order(order)
    o.set_psd(psd)
    return o, psd


def test_td_template_layout():
    n, fs = 1 << 15, 2048.0
    o, _ = _td_case(n, fs)
    m1, m2 = 3.0, 2.5
    ts, te, fe = oracle.td_extent(m1, m2, 40.0, 4)
    hp, hc = o.td_template(m1, m2)
    nz = np.nonzero(hp ** 2 + hc ** 2)[0]
    assert nz[0] == n - int(np.floor(ts * fs)) and nz[-1] == n - int(np.ceil(te * fs))
    amp = np.sqrt(hp ** 2 + hc ** 2)[nz]
    assert amp[0] == pytest.approx(1.0, rel=1e-3)                  # (F / f_low)^(2/3) at F = f_low
    assert np.all(np.diff(amp) > 0)                                # Newtonian amplitude grows with F
    assert amp[-1] == pytest.approx((oracle.td_phase(m1, m2, (n - nz[-1]) / fs, 4)[1] / 40.0) ** (2 / 3), rel=1e-9)
    assert 0.9 * (fe / 40.0) ** (2 / 3) < amp[-1] <= (fe / 40.0) ** (2 / 3)
    # the instantaneous frequency read off the samples equals F
    j = nz[len(nz) // 2]
    dphi = np.angle((hp[j + 1] + 1j * hc[j + 1]) / (hp[j - 1] + 1j * hc[j - 1]))
    assert dphi * fs / (4 * np.pi) == pytest.approx(oracle.td_phase(m1, m2, (n - j) / fs, 4)[1], rel=1e-4)
    # too long for the segment
    with pytest.raises(oracle.OracleError):
        oracle.Oracle(1 << 12, fs, 40.0).td_template(1.0, 1.0)


def test_td_template_amplitude_law_by_stationary_phase():
    """The amplitude law (F / f_low)^(2/3) of orc_td_template, pinned by something other than its own formula:
    for a chirp A(t) cos phi(t) the stationary-phase spectrum is |H(f)| = A(t_f) / (2 sqrt(dF/dt)) at F(t_f) = f, so
    with dF/dt ~ F^(11/3) the spectrum must fall as f^(-7/6) (an exponent 1/3 would give f^(-3/2), an exponent 1
    f^(-5/6)), and its absolute level must equal the prediction built from A and from dF/dt read off orc_td_phase by
    a finite difference.  The spectrum is numpy's FFT of the samples, averaged over 6 % bands to smooth the ripple of
    the sharp start at f_low."""
    n, fs, f_low = 1 << 16, 2048.0, 40.0
    o, _ = _td_case(n, fs)
    m1 = m2 = 1.4
    hp, _hc = o.td_template(m1, m2)
    H = np.abs(np.fft.rfft(hp))
    f = np.fft.rfftfreq(n, 1.0 / fs)
    ts, te, _fe = oracle.td_extent(m1, m2, f_low, 4)

    def band_rms(F):
        m = (f >= 0.97 * F) & (f < 1.03 * F)
        return np.sqrt(np.mean(H[m] ** 2))

    def tau_of(F):                                       # F(tau) falls with tau = t_c - t: bisection
        lo, hi = te, ts
        for _ in range(100):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if oracle.td_phase(m1, m2, mid, 4)[1] > F else (lo, mid)
        return 0.5 * (lo + hi)

    freqs = np.array([60.0, 100.0, 200.0, 400.0])        # a decade, away from both ends of the chirp
    meas = np.array([band_rms(F) for F in freqs])
    slope = np.polyfit(np.log(freqs), np.log(meas), 1)[0]
    # -3/2 or -5/6 for a wrong exponent; the post-Newtonian terms of dF/dt steepen the Newtonian -7/6 by a few per cent
    assert abs(slope + 7.0 / 6.0) < 0.06, slope
    for F, got in zip(freqs, meas):
        tau = tau_of(F)
        d = 1e-4 * tau
        f_dot = (oracle.td_phase(m1, m2, tau - d, 4)[1] - oracle.td_phase(m1, m2, tau + d, 4)[1]) / (2 * d)
        want = fs * (F / f_low) ** (2.0 / 3.0) / (2.0 * np.sqrt(f_dot))       # numpy's FFT carries no dt: times fs
        assert got == pytest.approx(want, rel=1e-2), (F, got, want)


@pytest.mark.parametrize("order", [4, 5])
def test_td_noise_free_injection_closed_forms(order):
    """Data = A h_+ of the same template, shifted circularly by t0: c_+(t0) = A sigma_+, c_x(t0) = A (h_+|h_x)/sigma_x
    with the two polarisations in quadrature, so rho_max = A sigma_+ at sample t0 with phase 0; injecting h_x gives
    phase pi/2; sigma_+ = sigma_x to the accuracy of the quadrature."""
    n, fs = 1 << 15, 2048.0
    o, psd = _td_case(n, fs, order=order)
    m1, m2 = 3.0, 2.5
    hp, hc = o.td_template(m1, m2)
    t0, A = 9000, 0.37
    for h, want_phase in ((hp, 0.0), (hc, np.pi / 2)):
        o.load_segment(np.roll(A * h, t0).astype(np.float32))
        rho, cp, cc, sp, sc = o.td_snr_series(m1, m2)
        assert int(np.argmax(rho)) == t0
        assert sp == pytest.approx(sc, rel=2e-3)
        assert rho[t0] == pytest.approx(A * (sp if h is hp else sc), rel=2e-4)
        assert np.arctan2(cc[t0], cp[t0]) == pytest.approx(want_phase, abs=2e-2)
    # the definition of sigma_+ by hand: 4 df sum |H_+|^2 / S_n with numpy's FFT
    H = np.fft.rfft(hp) / fs
    klo = int(np.ceil(40.0 * n / fs))
    k = np.arange(klo, n // 2)
    assert sp == pytest.approx(np.sqrt(4 * fs / n * np.sum(np.abs(H[k]) ** 2 / psd[k])), rel=1e-10)
    # and the correlator at one lag by a direct time-frequency sum
    D = np.fft.rfft(np.roll(A * hc, t0).astype(np.float32).astype(np.float64)) / fs
    j = t0 - 3
    cdir = 4 * fs / n * np.real(np.sum(D[k] * np.conj(H[k]) / psd[k] * np.exp(2j * np.pi * j * k / n))) / sp
    assert cp[j] == pytest.approx(cdir, rel=1e-8, abs=1e-10)


def test_td_filter_agrees_with_the_spa_filter():
    """The same binary in the two domains: a noise-free time-domain injection filtered with the stationary-phase
    template of the same masses (orc_snr_series) peaks at the injected coalescence sample (within the few samples by
    which the two approximants' end points differ) and recovers most of its SNR -- pins the placement of t_c, the sign
    of the phase and the sweep direction of the time-domain generator against the independently pinned SPA one."""
    n, fs = 1 << 16, 2048.0
    o, psd = _td_case(n, fs, order=4)
    m1 = m2 = 1.4
    hp, hc = o.td_template(m1, m2)
    t0 = 40960
    o.load_segment(np.roll(hp, t0).astype(np.float32))
    rho_td, *_ , sp, sc = o.td_snr_series(m1, m2)
    rho, z, sigma = o.snr_series(m1, m2)
    assert abs(int(np.argmax(rho)) - t0) <= 3
    assert rho.max() > 0.95 * rho_td.max()
    # a time-REVERSED chirp (sweeping down) is not found
    o.load_segment(np.roll(hp[::-1], t0).astype(np.float32))
    assert o.snr_series(m1, m2)[0].max() < 0.2 * rho_td.max()


def test_td_noise_statistics_and_bank():
    w = W.small_case(log2n=15, fs=2048.0, f_low=40.0, n_templates=3, seed=11)
    o = _oracle_for(w)
    bank = np.array([[2.4, 2.2], [3.0, 2.9], [80.0, 70.0]])
    rhos = [o.td_snr_series(m1, m2) for m1, m2 in bank[:2]]
    for rho, cp, cc, sp, sc in rhos:
        assert np.mean(cp ** 2) == pytest.approx(1.0, rel=0.15) and np.mean(cc ** 2) == pytest.approx(1.0, rel=0.15)
    pk, tr, nf, rc = o.td_filter_bank(bank, 2.5)
    assert rc == 0 and pk[2]["idx_peak"] == -1 and pk[2]["snr_max"] == 0.0          # f_ISCO < f_low
    want = []
    for t, (rho, cp, cc, sp, sc) in enumerate(rhos):
        j = int(np.argmax(rho))
        assert pk[t]["idx_peak"] == j and pk[t]["snr_max"] == rho[j] and pk[t]["sigma"] == sp
        assert pk[t]["phase"] == pytest.approx(np.arctan2(cc[j], cp[j]), abs=1e-12)
        want += [(t, int(jj)) for jj in np.nonzero(rho > 2.5)[0]]
    assert nf == len(want) > 0
    assert [(int(a), int(b)) for a, b in zip(tr["template_idx"], tr["sample_idx"])] == want
    pk2, tr2, nf2, rc2 = o.td_filter_bank(bank, 2.5, trig_capacity=5)
    assert rc2 == oracle.WTRUNC and nf2 == nf and len(tr2) == 5 and np.array_equal(tr2, tr[:5])
