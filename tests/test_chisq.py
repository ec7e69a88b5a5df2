"""NEXT-4 (ref. [24]): cbmf_chisq against the oracle's twin (orc_chisq)."""
import numpy as np
import pytest

import oracle
from testsupport import workloads as W

pytestmark = pytest.mark.gpu


def _pair(wl):
    from paper_1006_4644_b200 import cbmf
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    g.set_psd(wl.psd); g.load_segment(wl.samples)
    o = oracle.Oracle(wl.n, wl.fs, wl.f_low)
    o.set_psd(wl.psd); o.load_segment(wl.samples)
    return g, o


@pytest.mark.parametrize("name,p", [("cfg0", 1), ("cfg0", 4), ("cfg0", 16), ("cfg1_64", 8), ("heavy", 16)])
def test_chisq_vs_oracle(name, p):
    wl = {"cfg0": W.config0, "cfg1_64": lambda: W.config1(64),
          "heavy": lambda: W.small_case(log2n=15, n_templates=9, heavy=True, seed=31)}[name]()
    if name == "heavy":
        wl.bank[0] = (80.0, 90.0)                                  # empty band
    g, o = _pair(wl)
    pk, _, _, _ = g.filter_bank(wl.bank, wl.threshold)
    idx = pk["idx_peak"].copy()
    chi, zl = g.chisq(wl.bank, idx, p, want_bands=True)
    for t, (m1, m2) in enumerate(wl.bank):
        if idx[t] < 0:
            assert chi[t] == 0
            continue
        chi_o, zl_o, edges_o = o.chisq(m1, m2, int(idx[t]), p)
        sig = float(pk[t]["sigma"])
        scale = float(pk[t]["snr_max"]) * sig                      # |z| at the peak
        assert np.max(np.abs(zl[t] - zl_o)) <= 2e-4 * scale, (t, p)          # a boundary bin may sit on the other side
        assert abs(zl[t].sum() - zl_o.sum()) <= 2e-5 * scale
        assert abs(chi[t] - chi_o) <= 2e-3 * chi_o + 2e-3 * p, (t, chi[t], chi_o)
    if p == 1:
        assert np.all(chi == 0)
    g.close(); o.close()


def test_chisq_separates_chirp_from_glitch():
    """configs[0]: the injected chirp has chi^2 / (2p - 2) ~ 1 in its own template; a loud impulse rings every
    template to a large SNR but fails the test by orders of magnitude (what the veto is for)."""
    from paper_1006_4644_b200 import cbmf
    wl = W.config0()
    p = 16
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    g.set_psd(wl.psd); g.load_segment(wl.samples)
    pk, _, _, _ = g.filter_bank(wl.bank, 6.0)
    chi = g.chisq(wl.bank, pk["idx_peak"], p)
    assert chi[16] < 2.0 * (2 * p - 2) and pk[16]["snr_max"] > 10
    s = wl.samples.copy(); s[30000] += 4.0e4
    g.load_segment(s)
    pk2, _, _, _ = g.filter_bank(wl.bank, 6.0)
    chi2 = g.chisq(wl.bank, pk2["idx_peak"], p)
    loud = pk2["snr_max"] > 12
    assert loud.sum() >= 10 and np.all(chi2[loud] > 10 * (2 * p - 2))
    # arguments
    with pytest.raises(cbmf.CbmfError):
        g.chisq(wl.bank, np.full(len(wl.bank), wl.n, dtype=np.int32), p)
    with pytest.raises(cbmf.CbmfError):
        g.chisq(wl.bank, pk2["idx_peak"], 0)
    assert np.all(g.chisq(wl.bank, np.full(len(wl.bank), -1, dtype=np.int32), p) == 0)
    g.close()
