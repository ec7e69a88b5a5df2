"""NEXT-3, second part: the paper's own template path -- time-domain
generation of the two polarisations, forward FFT, normalisation by a reduction, two correlators, quadrature sum --
the product (cbmf_filter_bank_td, cbmf_debug_td_template) against the oracle (orc_td_*)."""
import numpy as np
import pytest

import oracle
from testsupport import workloads as W
from parity import check_peaks, check_triggers

pytestmark = pytest.mark.gpu


def _pair(n, fs, f_low, psd, order, samples=None):
    from paper_1006_4644_b200 import cbmf
    g = cbmf.Context(n, fs, f_low)
    g.set_psd(psd)
    g.set_pn_order(order)
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(psd)
    o.set_pn_order(order)
    if samples is not None:
        g.load_segment(samples); o.load_segment(samples)
    return g, o


@pytest.mark.parametrize("log2n,fs,f_low", [(16, 2048.0, 40.0), (20, 4096.0, 40.0), (22, 4096.0, 15.0)])
@pytest.mark.parametrize("order", [4, 5])
def test_td_template_vs_oracle(log2n, fs, f_low, order):
    """The generated polarisations sample by sample: same extent (a boundary sample may differ where tau_start or
    tau_end falls within rounding of a sample), mismatch 1 - <a,b>/<a,a> in the time domain <= 1e-6 (the paper's own
    GPU-single vs CPU-double figure is 3e-4), pointwise error <= 3e-5 of the largest amplitude."""
    n = 1 << log2n
    psd = W.onesided_psd("A", n, fs, f_low)
    g, o = _pair(n, fs, f_low, psd, order)
    for m1, m2 in ((1.4, 1.4), (1.0, 3.0), (4.0, 2.5), (9.0, 1.1)):
        hp_g, hc_g = g.debug_td_template(m1, m2)
        hp_o, hc_o = o.td_template(m1, m2)
        nz_g, nz_o = (hp_g != 0) | (hc_g != 0), (hp_o != 0) | (hc_o != 0)
        assert np.count_nonzero(nz_g != nz_o) <= 2
        a = hp_o + 1j * hc_o
        b = hp_g.astype(np.float64) + 1j * hc_g.astype(np.float64)
        both = nz_g & nz_o
        assert np.max(np.abs(a[both] - b[both])) <= 3e-5 * np.max(np.abs(a))
        delta = 1.0 - np.sum((a[both] * np.conj(b[both])).real) / np.sum(np.abs(a[both]) ** 2)
        assert abs(delta) <= 1e-6, delta
    g.close(); o.close()


def _td_workload(log2n, fs, f_low, bank, inj, order, seed, snr=11.0):
    """Seeded coloured noise plus one time-domain injection (the oracle's own generator supplies the waveform: inputs
    may come from the input generators or the oracle, never from the CUDA path)."""
    n = 1 << log2n
    psd = W.onesided_psd("A", n, fs, f_low)
    noise = W.to_time_domain(W.noise_spectrum(n, fs, f_low, psd, seed), n, fs).astype(np.float64)
    o = oracle.Oracle(n, fs, f_low)
    o.set_psd(psd); o.set_pn_order(order)
    hp, hc = o.td_template(*inj)
    o.load_segment(hp.astype(np.float32))
    _, _, _, sp, _ = o.td_snr_series(*inj)            # sigma_+ of the injected template
    o.close()
    t0 = int(0.6 * n)
    d = noise + snr / sp * np.roll(np.cos(0.4) * hp + np.sin(0.4) * hc, t0)
    return n, psd, d.astype(np.float32), t0


@pytest.mark.parametrize("log2n,fs,order", [(15, 2048.0, 4), (16, 2048.0, 5), (18, 4096.0, 4)])
def test_filter_bank_td_vs_oracle(log2n, fs, order):
    f_low = 40.0
    lo = 2.2 if log2n == 15 else 1.3                   # the chirp must fit the segment
    bank = np.vstack([W.draw_bank(70 + log2n, 5, lo, lo + 2.0), [[2.6, 2.4]], [[90.0, 80.0]]])
    n, psd, samples, t0 = _td_workload(log2n, fs, f_low, bank, (2.6, 2.4), order, 300 + log2n)
    g, o = _pair(n, fs, f_low, psd, order, samples)
    thr = 3.8
    pk_g, tr_g, nf_g, rc_g = g.filter_bank_td(bank, thr, trig_capacity=1 << 18)
    pk_o, tr_o, nf_o, rc_o = o.td_filter_bank(bank, thr, trig_capacity=1 << 18)
    assert rc_g == 0 and rc_o == 0
    series = {}

    def rho_at(t, j):
        if t not in series:
            series[t] = o.td_snr_series(*bank[t])[0]
        return series[t][j]
    check_peaks(pk_g, pk_o, rho_at)
    assert pk_g[5]["idx_peak"] == t0 and pk_g[5]["snr_max"] > 8.0                 # the injection is found
    assert abs(pk_g[5]["phase"] - 0.4) < 0.4
    assert pk_g[6]["idx_peak"] == -1                                               # f_ISCO below the cut-off
    n_g, n_o = check_triggers(tr_g, tr_o, thr)
    assert n_o > 20 and abs(nf_g - nf_o) <= max(3, nf_o // 100)
    # pointwise series through the product epilogue: threshold 0 makes every sample a trigger
    pk1, tr1, nf1, rc1 = g.filter_bank_td(bank[5:6], 0.0, trig_capacity=n)
    assert nf1 == n and np.array_equal(tr1["sample_idx"], np.arange(n))
    rho_o = rho_at(5, slice(None))
    assert np.max(np.abs(tr1["snr"] - rho_o)) <= 1e-3 * rho_o.max()
    # truncation keeps the first triggers in (template, sample) order
    pk2, tr2, nf2, rc2 = g.filter_bank_td(bank, thr, trig_capacity=7)
    assert rc2 == 1 and nf2 == nf_g and np.array_equal(tr2, tr_g[:7])
    g.close(); o.close()


def test_filter_bank_td_errors_and_state():
    from paper_1006_4644_b200 import cbmf
    n, fs, f_low = 1 << 13, 2048.0, 40.0
    psd = W.onesided_psd("A", n, fs, f_low)
    g = cbmf.Context(n, fs, f_low)
    with pytest.raises(cbmf.CbmfError) as e:
        g.filter_bank_td(np.array([[5.0, 5.0]]), 6.0)
    assert e.value.rc == -2                                                        # ESTATE
    g.set_psd(psd)
    g.load_segment(np.zeros(n, dtype=np.float32))
    # 1.4 + 1.4 from 40 Hz lasts 25 s: longer than the 4 s segment
    with pytest.raises(cbmf.CbmfError) as e:
        g.filter_bank_td(np.array([[6.0, 6.0], [1.4, 1.4], [-1.0, 2.0]]), 6.0)
    assert e.value.rc == -1 and g.last_bad_template() == 1
    pk, tr, nf, rc = g.filter_bank_td(np.array([[6.0, 6.0]]), 6.0)                 # all-zero data
    assert rc == 0 and nf == 0 and pk[0]["snr_max"] == 0.0 and pk[0]["idx_peak"] == 0 and pk[0]["sigma"] > 0
    # the SPA path still works on the same context afterwards
    pk, tr, nf, rc = g.filter_bank(np.array([[6.0, 6.0]]), 6.0)
    assert rc == 0 and pk[0]["sigma"] > 0
    g.close()


def test_filter_bank_td_full_size_sample():
    """N = 2^20 (the metric's size): three templates of the cfg1 mass range against the oracle."""
    n, fs, f_low = 1 << 20, 4096.0, 40.0
    bank = np.array([[1.4, 1.4], [2.9, 1.1], [2.0, 2.0]])
    n, psd, samples, t0 = _td_workload(20, fs, f_low, bank, (1.4, 1.4), 5, 777, snr=12.0)
    g, o = _pair(n, fs, f_low, psd, 5, samples)
    pk_g, tr_g, nf_g, rc_g = g.filter_bank_td(bank, 5.0, trig_capacity=1 << 16)
    pk_o, tr_o, nf_o, rc_o = o.td_filter_bank(bank, 5.0, trig_capacity=1 << 16)
    check_peaks(pk_g, pk_o, lambda t, j: o.td_snr_series(*bank[t])[0][j])
    check_triggers(tr_g, tr_o, 5.0)
    assert pk_g[0]["idx_peak"] == t0
    g.close(); o.close()
