"""Seeded synthetic workloads (SURVEY.md §8(d) "Synthetic inputs"; BASELINE.json configs[0..4]).

TEST SUPPORT, NOT PRODUCT: this module lives outside the product package and is the ONE piece
that serves both the CPU oracle (tests) and the CUDA path (tests, bench.py, smoke()).  It holds none of the filter's arithmetic: no matched
filter, no FFT of the product, no template generator of the product, no sigma
table.  What it does hold is the *source model* used to simulate the detector
data -- coloured Gaussian noise plus injected chirps -- written in numpy
(float64, numpy's FFT as a library primitive).  The injected chirp is a third,
independent statement of the 2PN SPA phase of BASELINE.json configs[0] ("v form");
neither oracle/ nor csrc/ imports it.

The paper measures on "a given input" and a uniform template grid
for one [1.4,1.4] Msun source at 4 kHz, N = 2^20; there is no
public data set, so these seeded recipes stand in for it.

Random numbers: a counter-based generator (splitmix64 of seed/stream/index ->
53-bit uniforms -> Box-Muller), so every value is a pure function of
(seed, stream, index) and does not depend on numpy's generator streams.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# G M_sun / c^3 in seconds (G M_sun = 1.3271244e20 m^3 s^-2, c = 299792458 m/s); SURVEY.md A8.
T_SUN_S = 4.925490947641267e-6

_U64 = np.uint64


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = (x + _U64(0x9E3779B97F4A7C15)).astype(np.uint64)
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        return z ^ (z >> _U64(31))


def _bits(seed: int, stream: int, n: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        key = _splitmix64(np.array([(seed & 0xFFFFFFFF) | ((stream & 0xFFFFFFFF) << 32)], dtype=np.uint64))
        key = _splitmix64(key)
        idx = np.arange(n, dtype=np.uint64)
        return _splitmix64(key + idx * _U64(0xD1342543DE82EF95))


def uniform01(seed: int, stream: int, n: int) -> np.ndarray:
    """n uniforms in [0,1), a pure function of (seed, stream, index)."""
    return (_bits(seed, stream, n) >> _U64(11)).astype(np.float64) * 2.0 ** -53


def normal_pairs(seed: int, stream: int, n: int):
    """n independent pairs (g1, g2) of standard normals (Box-Muller)."""
    u1 = ((_bits(seed, 2 * stream, n) >> _U64(11)).astype(np.float64) + 1.0) * 2.0 ** -53  # (0,1]
    u2 = uniform01(seed, 2 * stream + 1, n)
    r = np.sqrt(-2.0 * np.log(u1))
    return r * np.cos(2.0 * np.pi * u2), r * np.sin(2.0 * np.pi * u2)


# ----------------------------------------------------------------- PSDs (inputs)

def psd_A(f: np.ndarray) -> np.ndarray:
    """BASELINE.json configs[0]: S_n(f) = (f/215)^-4 + 2 + 2 (f/215)^2."""
    x = np.asarray(f, dtype=np.float64) / 215.0
    with np.errstate(divide="ignore"):
        return x ** -4 + 2.0 + 2.0 * x ** 2


def psd_B(f: np.ndarray) -> np.ndarray:
    """BASELINE.json configs[3]: S_n(f) = (f/50)^-6 + (f/50)^-2 + 1 + (f/50)^2."""
    x = np.asarray(f, dtype=np.float64) / 50.0
    with np.errstate(divide="ignore"):
        return x ** -6 + x ** -2 + 1.0 + x ** 2


def onesided_psd(kind: str, n: int, fs: float, f_low: float) -> np.ndarray:
    """S_n on the DFT grid k = 0..n/2; +inf below f_low ("else infinite", configs[0])."""
    f = np.arange(n // 2 + 1, dtype=np.float64) * (fs / n)
    s = {"A": psd_A, "B": psd_B}[kind](f)
    s[f < f_low] = np.inf
    return s


# ------------------------------------------------------- source model (injections)

def _source_phase(m1: float, m2: float, f: np.ndarray) -> np.ndarray:
    """2PN SPA phase of the simulated source, BASELINE.json configs[0] (t_c = phi_c = 0)."""
    M = (m1 + m2) * T_SUN_S
    eta = m1 * m2 / (m1 + m2) ** 2
    v = np.cbrt(np.pi * M * f)
    br = (1.0 + (3715.0 / 756.0 + 55.0 * eta / 9.0) * v ** 2 - 16.0 * np.pi * v ** 3
          + (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta ** 2 / 72.0) * v ** 4)
    return -np.pi / 4.0 + 3.0 / (128.0 * eta * v ** 5) * br


def source_spectrum(n: int, fs: float, f_low: float, psd: np.ndarray, m1: float, m2: float,
                    t_c: float, phi_c: float, snr: float) -> np.ndarray:
    """h~_inj[k], k = 0..n/2: A f^-7/6 exp(-i(2 pi f t_c - phi_c + Psi(f))) on
    f_low <= f <= min(f_ISCO, below Nyquist), scaled to optimal SNR `snr` (reading A20)."""
    df = fs / n
    k = np.arange(n // 2 + 1)
    f = k * df
    f_isco = 1.0 / (6.0 ** 1.5 * np.pi * (m1 + m2) * T_SUN_S)
    k_lo = int(np.ceil(f_low * (n / fs)))
    k_hi = min(int(np.floor(f_isco * (n / fs))), n // 2 - 1)
    h = np.zeros(n // 2 + 1, dtype=np.complex128)
    if k_hi < k_lo:
        return h
    sl = slice(k_lo, k_hi + 1)
    amp = f[sl] ** (-7.0 / 6.0)
    sigma2 = 4.0 * df * np.sum(amp ** 2 / psd[sl])
    a = snr / np.sqrt(sigma2)
    h[sl] = a * amp * np.exp(-1j * (2.0 * np.pi * f[sl] * t_c - phi_c + _source_phase(m1, m2, f[sl])))
    return h


def noise_spectrum(n: int, fs: float, f_low: float, psd: np.ndarray, seed: int) -> np.ndarray:
    """n~[k] = sqrt(T S_n(f_k)/4) (g1 + i g2) for f_k >= f_low, k = 1..n/2-1; DC = Nyquist = 0
    (so that <|n~|^2> = T S_n / 2, one-sided; reading A5)."""
    T = n / fs
    x = np.zeros(n // 2 + 1, dtype=np.complex128)
    g1, g2 = normal_pairs(seed, 0, n // 2 - 1)
    k = np.arange(1, n // 2)
    ok = (k * (fs / n) >= f_low) & np.isfinite(psd[1:n // 2])
    amp = np.zeros(n // 2 - 1)
    amp[ok] = np.sqrt(T * psd[1:n // 2][ok] / 4.0)
    x[1:n // 2] = amp * (g1 + 1j * g2)
    return x


def to_time_domain(spec: np.ndarray, n: int, fs: float) -> np.ndarray:
    """d[j] = df sum_k (Hermitian-extended spec)[k] e^{+2 pi i jk/n}, rounded to float32."""
    return (fs * np.fft.irfft(spec, n)).astype(np.float32)


# ------------------------------------------------------------------- workloads

@dataclass
class Injection:
    m1: float
    m2: float
    t_c: float
    phi_c: float
    snr: float
    template_idx: int  # bank index of the exact-parameter template

    def sample(self, fs: float) -> int:
        return int(round(self.t_c * fs))


@dataclass
class Workload:
    name: str
    n: int
    fs: float
    f_low: float
    psd_kind: str
    threshold: float
    psd: np.ndarray            # float64 [n/2+1]
    samples: np.ndarray        # float32 [n]
    bank: np.ndarray           # float64 [B, 2]
    injections: list = field(default_factory=list)

    @property
    def n_templates(self) -> int:
        return int(self.bank.shape[0])


def draw_bank(seed: int, n_templates: int, lo: float, hi: float) -> np.ndarray:
    u = uniform01(seed, 0, 2 * n_templates).reshape(n_templates, 2)   # m1 then m2, template by template
    return lo + (hi - lo) * u


def _build(name, n, fs, f_low, psd_kind, bank, noise_seed, inj, threshold=6.0, noise=True):
    psd = onesided_psd(psd_kind, n, fs, f_low)
    spec = noise_spectrum(n, fs, f_low, psd, noise_seed) if noise else np.zeros(n // 2 + 1, np.complex128)
    for i in inj:
        spec = spec + source_spectrum(n, fs, f_low, psd, i.m1, i.m2, i.t_c, i.phi_c, i.snr)
    return Workload(name, n, fs, f_low, psd_kind, threshold, psd, to_time_domain(spec, n, fs), bank, list(inj))


def _snap(t: float, fs: float) -> float:
    return round(t * fs) / fs


def config0(noise: bool = True) -> Workload:
    """configs[0] "Tiny": N=2^16, fs=2048, f_low=40, PSD A, noise seed 1, one (1.4,1.4)
    injection at t_c=20 s, phi_c=0.3, SNR 12; 16 templates U[1,3]^2 (seed 2) + the exact one."""
    n, fs = 1 << 16, 2048.0
    bank = np.vstack([draw_bank(2, 16, 1.0, 3.0), [[1.4, 1.4]]])
    inj = [Injection(1.4, 1.4, 20.0, 0.3, 12.0, 16)]
    return _build("cfg0", n, fs, 40.0, "A", bank, 1, inj, noise=noise)


def config1(n_templates: int = 1024) -> Workload:
    """configs[1]: N=2^20, fs=4096, 1024 templates U[1,3]^2 (seed 3), 4 injections at SNR 8-15."""
    n, fs = 1 << 20, 4096.0
    bank = draw_bank(3, 1024, 1.0, 3.0)
    u = uniform01(3 + 200, 0, 8)
    T = n / fs
    inj = []
    for r, (ti, frac) in enumerate(zip((128, 384, 640, 896), (0.2, 0.4, 0.6, 0.8))):
        inj.append(Injection(float(bank[ti, 0]), float(bank[ti, 1]), _snap(frac * T, fs),
                             float(2 * np.pi * u[2 * r] - np.pi), float(8.0 + 7.0 * u[2 * r + 1]), ti))
    w = _build("cfg1", n, fs, 40.0, "A", bank, 3 + 100, inj)
    if n_templates != 1024:
        w.bank = w.bank[:n_templates]
    return w


def config2(n_templates: int = 65536) -> Workload:
    """configs[2] bank throughput: N=2^20, fs=4096, 65536 templates U[1,10]^2 (seed 4),
    noise + 1 injection (= bank template 32768) at SNR 10."""
    n, fs = 1 << 20, 4096.0
    bank = draw_bank(4, 65536, 1.0, 10.0)
    u = uniform01(4 + 200, 0, 1)
    ti = 32768
    inj = [Injection(float(bank[ti, 0]), float(bank[ti, 1]), _snap(0.5 * n / fs, fs),
                     float(2 * np.pi * u[0] - np.pi), 10.0, ti)]
    w = _build("cfg2", n, fs, 40.0, "A", bank, 4 + 100, inj)
    if n_templates != 65536:
        w.bank = w.bank[:n_templates]
    return w


def config3(n_templates: int = 4096) -> Workload:
    """configs[3] long segment: N=2^22, fs=4096, f_low=10, PSD B, 4096 templates U[1,5]^2
    (seed 5), 2 injections (= bank templates 1024, 3072) at SNR 10."""
    n, fs = 1 << 22, 4096.0
    bank = draw_bank(5, 4096, 1.0, 5.0)
    u = uniform01(5 + 200, 0, 2)
    T = n / fs
    inj = [Injection(float(bank[ti, 0]), float(bank[ti, 1]), _snap(frac * T, fs),
                     float(2 * np.pi * u[r] - np.pi), 10.0, ti)
           for r, (ti, frac) in enumerate(((1024, 0.3), (3072, 0.7)))]
    w = _build("cfg3", n, fs, 10.0, "B", bank, 5 + 100, inj)
    if n_templates != 4096:
        w.bank = w.bank[:n_templates]
    return w


def sweep_point(log2n: int, batch: int, seed: int = 6) -> Workload:
    """configs[4] kernel sweep: N = 2^log2n, fs=4096, f_low=40, PSD A, `batch` templates
    U[1,3]^2, noise only."""
    n, fs = 1 << log2n, 4096.0
    bank = draw_bank(seed + log2n, batch, 1.0, 3.0)
    return _build(f"sweep_2^{log2n}_b{batch}", n, fs, 40.0, "A", bank, seed + 100 + log2n, [])


def small_case(log2n: int = 12, fs: float = 2048.0, f_low: float = 40.0, n_templates: int = 5,
               seed: int = 11, psd_kind: str = "A", snr: float = 9.0, heavy: bool = False) -> Workload:
    """A small noise+injection case for fast tests (not a BASELINE config).  heavy=True draws
    masses high enough that f_ISCO cuts the band (and some bands are empty)."""
    n = 1 << log2n
    lo, hi = (3.0, 60.0) if heavy else (1.0, 3.0)
    bank = draw_bank(seed, n_templates, lo, hi)
    ti = n_templates // 2
    inj = [Injection(float(bank[ti, 0]), float(bank[ti, 1]), _snap(0.625 * n / fs, fs), 0.7, snr, ti)]
    return _build(f"small_2^{log2n}", n, fs, f_low, psd_kind, bank, seed + 100, inj)


def by_name(name: str, n_templates: int | None = None) -> Workload:
    if name == "cfg0":
        return config0()
    f = {"cfg1": config1, "cfg2": config2, "cfg3": config3}[name]
    return f() if n_templates is None else f(n_templates)
