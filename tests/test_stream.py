"""NEXT-2: cbmf_filter_stream against the oracle's twin
(oracle.filter_stream) on the same seeded stream, segment by segment."""
import numpy as np
import pytest

import oracle
from testsupport import workloads as W
from parity import check_peaks, check_triggers

pytestmark = pytest.mark.gpu


def _stream(n, fs, f_low, n_hops, hop, seed, inj):
    """Coloured noise + chirps, generated in one long buffer and cut to n + n_hops * hop samples."""
    n_total = n + n_hops * hop
    big = 1 << int(np.ceil(np.log2(n_total)))
    psd_big = W.onesided_psd("A", big, fs, f_low)
    spec = W.noise_spectrum(big, fs, f_low, psd_big, seed)
    for (m1, m2, j_glob, phi, snr) in inj:
        spec = spec + W.source_spectrum(big, fs, f_low, psd_big, m1, m2, j_glob / fs, phi, snr)
    return W.to_time_domain(spec, big, fs)[:n_total]


def _compare_with_oracle(n, fs, f_low, psd, stream, bank, thr, discard, pk, tr, offs):
    """Segment by segment against oracle.filter_stream; -> the segment starts."""
    pk_o, tr_o, offs_o, starts = oracle.filter_stream(n, fs, f_low, psd, stream, bank, thr, discard)
    assert pk.shape == pk_o.shape == (len(starts), len(bank)) and len(offs) == len(starts) + 1
    o = oracle.Oracle(n, fs, f_low); o.set_psd(psd)
    for s, s0 in enumerate(starts):
        o.load_segment(stream[s0:s0 + n])
        rho_cache = {}

        def rho_at(t, j):
            if t not in rho_cache:
                rho_cache[t] = o.snr_series(*bank[t])[0]
            return rho_cache[t][j]

        near = check_peaks(pk[s], pk_o[s], rho_at)
        assert len(near) <= 1 and np.all(pk[s]["idx_peak"] >= discard)
        seg_g, seg_o = tr[offs[s]:offs[s + 1]], tr_o[offs_o[s]:offs_o[s + 1]]
        assert np.all(seg_g["sample_idx"] >= discard)
        check_triggers(seg_g, seg_o, thr)
    o.close()
    return starts


@pytest.mark.parametrize("log2n,discard_frac,sub_batch", [(14, 0.5, 3), (16, 0.5, 64), (14, 0.25, 64), (13, 0.0, 2)])
def test_filter_stream_vs_oracle(log2n, discard_frac, sub_batch):
    from paper_1006_4644_b200 import cbmf
    n, fs, f_low = 1 << log2n, 2048.0, 40.0
    discard = int(discard_frac * n)
    hop = n - discard
    bank = np.vstack([W.draw_bank(50 + log2n, 6, 1.5, 4.0), [[2.5, 2.0]]])
    j_inj = hop + discard + (n - discard) // 2                   # inside the valid part of segment 1
    stream = _stream(n, fs, f_low, 3, hop, 60 + log2n, [(2.5, 2.0, j_inj, 0.4, 10.0)])
    psd = W.onesided_psd("A", n, fs, f_low)
    thr = 5.0
    g = cbmf.Context(n, fs, f_low)
    g.set_psd(psd)
    g.set_sub_batch(sub_batch)
    pk, tr, offs, nf, rc = g.filter_stream(stream, bank, thr, discard, trig_capacity=1 << 18)
    assert rc == 0 and nf == len(tr) == offs[-1]
    starts = _compare_with_oracle(n, fs, f_low, psd, stream, bank, thr, discard, pk, tr, offs)
    # the injection is found in segment 1 at its global time
    assert abs(int(pk[1, 6]["idx_peak"]) + starts[1] - j_inj) <= 1 and pk[1, 6]["snr_max"] > 7.0
    # a plain load_segment + filter_bank afterwards needs a new segment (the stream used the slot), then works
    with pytest.raises(cbmf.CbmfError) as e:
        g.filter_bank(bank, thr)
    assert e.value.rc == cbmf.ESTATE
    g.load_segment(stream[:n])
    pk0, tr0, _, _ = g.filter_bank(bank, thr)
    if discard == 0:
        assert np.array_equal(pk0, pk[0]) and np.array_equal(tr0, tr[offs[0]:offs[1]])
    g.close()


@pytest.mark.parametrize("log2n,n_hops,n_templates", [(18, 2, 8), (19, 2, 8), (20, 2, 8), (21, 1, 4)])
def test_filter_stream_vs_oracle_table_sizes(log2n, n_hops, n_templates):
    """The segment lengths of the paper's online table (table 4.1: 2^18 ... 2^21), discard = n/2
    (reading A25): these run the 512- and 1024-point masked pass-2 kernels (and, at 2^21, the 2048 x 1024 split) that
    bench.py's online_capacity rows time.  Two injections: A coalesces in the valid half of segment 1; B coalesces
    one second after the end of segment 0, so its chirp straddles that boundary -- segment 1 holds it in its valid
    half and must find it, while in segment 2 (where there is one) it falls one second after the segment start,
    inside the discarded half, and must appear in neither the peak nor the trigger list of that segment."""
    from paper_1006_4644_b200 import cbmf
    n, fs, f_low = 1 << log2n, 2048.0, 40.0
    discard = n // 2
    hop = n - discard
    inj_a, inj_b = (2.5, 2.0), (1.6, 1.45)
    bank = np.vstack([W.draw_bank(70 + log2n, n_templates - 2, 1.5, 4.0), [inj_a], [inj_b]])
    ia, ib = n_templates - 2, n_templates - 1
    j_a = hop + discard + hop // 3
    j_b = n + int(fs)
    stream = _stream(n, fs, f_low, n_hops, hop, 80 + log2n, [(*inj_a, j_a, 0.4, 11.0), (*inj_b, j_b, -1.1, 12.0)])
    psd = W.onesided_psd("A", n, fs, f_low)
    thr = 5.5
    g = cbmf.Context(n, fs, f_low)
    g.set_psd(psd)
    pk, tr, offs, nf, rc = g.filter_stream(stream, bank, thr, discard, trig_capacity=1 << 18)
    assert rc == 0 and nf == len(tr) == offs[-1]
    starts = _compare_with_oracle(n, fs, f_low, psd, stream, bank, thr, discard, pk, tr, offs)
    assert len(starts) == n_hops + 1
    assert abs(int(pk[1, ia]["idx_peak"]) + starts[1] - j_a) <= 1 and pk[1, ia]["snr_max"] > 8.0
    assert abs(int(pk[1, ib]["idx_peak"]) + starts[1] - j_b) <= 1 and pk[1, ib]["snr_max"] > 8.0
    seg1 = tr[offs[1]:offs[2]]
    assert np.any((seg1["template_idx"] == ib) & (np.abs(seg1["sample_idx"] + starts[1] - j_b) <= 1))
    if n_hops >= 2:
        assert j_b - starts[2] < discard                          # B sits in the discarded half of segment 2 ...
        assert pk[2, ib]["snr_max"] < 8.0                          # ... and is not what that segment reports
        seg2 = tr[offs[2]:offs[3]]
        assert not np.any((seg2["template_idx"] == ib) & (np.abs(seg2["sample_idx"] + starts[2] - j_b) <= 64))
    g.close()


def test_filter_stream_truncation_and_errors():
    from paper_1006_4644_b200 import cbmf
    n, fs, f_low = 1 << 12, 2048.0, 40.0
    stream = _stream(n, fs, f_low, 4, n // 2, 5, [])
    bank = W.draw_bank(3, 3, 1.5, 3.0)
    g = cbmf.Context(n, fs, f_low)
    with pytest.raises(cbmf.CbmfError) as e:
        g.filter_stream(stream, bank, 3.0, n // 2)
    assert e.value.rc == cbmf.ESTATE                              # no PSD yet
    g.set_psd(W.onesided_psd("A", n, fs, f_low))
    full = g.filter_stream(stream, bank, 3.0, n // 2, trig_capacity=1 << 16)
    assert full[4] == 0 and len(full[0]) == 5 and full[3] > 40
    cap = int(full[2][2]) + 3                                     # capacity runs out inside segment 2
    pk, tr, offs, nf, rc = g.filter_stream(stream, bank, 3.0, n // 2, trig_capacity=cap)
    assert rc == cbmf.WTRUNC and nf == full[3] and len(tr) == cap
    assert np.array_equal(tr, full[1][:cap]) and np.array_equal(pk, full[0])
    assert list(offs[:3]) == list(full[2][:3]) and np.all(offs[3:] == cap)
    for bad_discard in (-1, n):
        with pytest.raises(cbmf.CbmfError):
            g.filter_stream(stream, bank, 3.0, bad_discard)
    with pytest.raises(cbmf.CbmfError):
        g.filter_stream(stream[:n - 1], bank, 3.0, 0)
    s2 = stream.copy(); s2[n + 7] = np.nan                        # a NaN in the part only segment 1+ sees
    with pytest.raises(cbmf.CbmfError) as e:
        g.filter_stream(s2, bank, 3.0, n // 2)
    assert e.value.rc == cbmf.EINVAL
    with pytest.raises(cbmf.CbmfError):
        g.filter_stream(stream, np.array([[1.4, -1.0]]), 3.0, n // 2)
    assert g.last_bad_template() == 0
    g.close()
