"""NEXT-3: templates at the paper's stated order, 2.5PN in phase -- the product
(cbmf_set_pn_order(5)) against the oracle (orc_set_pn_order(5)) through every generator path."""
import numpy as np
import pytest

import oracle
from testsupport import workloads as W
from parity import SERIES_TOL_OF_PEAK, check_peaks, check_triggers, mismatch

pytestmark = pytest.mark.gpu


def _pair(wl, load=True):
    from paper_1006_4644_b200 import cbmf
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    g.set_psd(wl.psd)
    g.set_pn_order(5)
    assert g.get_pn_order() == 5
    o = oracle.Oracle(wl.n, wl.fs, wl.f_low)
    o.set_psd(wl.psd)
    o.set_pn_order(5)
    if load:
        g.load_segment(wl.samples); o.load_segment(wl.samples)
    return g, o


@pytest.mark.parametrize("log2n,fs,f_low,kind", [(20, 4096.0, 40.0, "A"), (16, 2048.0, 40.0, "A"), (22, 4096.0, 10.0, "B"), (13, 2048.0, 40.0, "A")])
def test_template_25pn_vs_oracle(log2n, fs, f_low, kind):
    """debug_template reads the PRODUCT generator: by rows at 2^20, per-bin table path at 2^16 / 2^13, per-bin series at
    2^22.  Mismatch <= 1e-6 (the paper's metric), pointwise phase error <= 2e-5; and the 2.5PN template differs from
    the 2PN one by whole radians, so the term is really there."""
    n = 1 << log2n
    wl_psd = W.onesided_psd(kind, n, fs, f_low)
    from paper_1006_4644_b200 import cbmf
    g = cbmf.Context(n, fs, f_low); g.set_psd(wl_psd)
    o = oracle.Oracle(n, fs, f_low); o.set_psd(wl_psd)
    wgt = np.where(np.isfinite(wl_psd), 1.0 / wl_psd, 0.0)
    for m1, m2 in ((1.4, 1.4), (1.0, 3.0), (4.0, 2.5)):
        h4 = g.debug_template(m1, m2)
        g.set_pn_order(5); o.set_pn_order(5)
        hg, ho = g.debug_template(m1, m2), o.template(m1, m2)
        g.set_pn_order(4); o.set_pn_order(4)
        nz = ho != 0
        assert np.array_equal(hg == 0, ho == 0)
        assert abs(mismatch(hg, ho, wgt)) <= 1e-6
        assert np.max(np.abs(hg[nz] - ho[nz]) / np.abs(ho[nz])) <= 2e-5
        assert np.max(np.abs(hg[nz] - h4[nz]) / np.abs(ho[nz])) > 1.0
    g.close(); o.close()


@pytest.mark.parametrize("name", ["cfg0", "small15", "small19", "cfg1x64"])
def test_filter_bank_25pn_vs_oracle(name):
    # cfg1x64: the first 64 templates of configs[1] at its full size, N = 2^20 (the by-rows ln k path of the bench split)
    wl = {"cfg0": W.config0, "small15": lambda: W.small_case(log2n=15, n_templates=6, seed=88),
          "small19": lambda: W.small_case(log2n=19, fs=4096.0, n_templates=4, seed=89),
          "cfg1x64": lambda: W.config1(64)}[name]()
    g, o = _pair(wl)
    for (m1, m2) in wl.bank[:3]:
        rho_g, z_g = g.debug_snr_series(m1, m2)
        rho_o, z_o, sig = o.snr_series(m1, m2)
        assert np.max(np.abs(rho_g - rho_o)) <= SERIES_TOL_OF_PEAK * rho_o.max()
        assert np.max(np.abs(z_g - z_o)) <= SERIES_TOL_OF_PEAK * rho_o.max() * sig
    pk_g, tr_g, nf, rc = g.filter_bank(wl.bank, 5.0, trig_capacity=1 << 18)
    pk_o, tr_o, _, _ = o.filter_bank(wl.bank, 5.0)
    cache = {}

    def rho_at(t, j):
        if t not in cache:
            cache[t] = o.snr_series(*wl.bank[t])[0]
        return cache[t][j]

    near = check_peaks(pk_g, pk_o, rho_at)
    check_triggers(tr_g, tr_o, 5.0)
    assert len(near) <= 1
    # chi^2 and the stream call use the same constants
    chi = g.chisq(wl.bank, pk_g["idx_peak"], 8)
    for t in range(min(3, len(wl.bank))):
        chi_o = o.chisq(wl.bank[t, 0], wl.bank[t, 1], int(pk_g[t]["idx_peak"]), 8)[0]
        assert abs(chi[t] - chi_o) <= 2e-3 * chi_o + 2e-2
    g.close(); o.close()


def test_pn_order_arguments():
    from paper_1006_4644_b200 import cbmf
    wl = W.small_case(log2n=12, n_templates=2)
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    assert g.get_pn_order() == 4
    for bad in (0, 3, 6, 7):
        with pytest.raises(cbmf.CbmfError):
            g.set_pn_order(bad)
    g.set_psd(wl.psd); g.load_segment(wl.samples)
    a = g.filter_bank(wl.bank, 6.0)
    g.set_pn_order(5)
    b = g.filter_bank(wl.bank, 6.0)                    # PSD and segment stay loaded; results change
    g.set_pn_order(4)
    c = g.filter_bank(wl.bank, 6.0)
    assert np.array_equal(a[0], c[0]) and not np.array_equal(a[0]["phase"], b[0]["phase"])
    assert np.array_equal(a[0]["sigma"], b[0]["sigma"])
    g.close()
