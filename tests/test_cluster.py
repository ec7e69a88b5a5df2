"""NEXT-1: the product's host-side clustering (csrc/cluster.h, one scan of a
sorted list) against the oracle's twin (pairwise definition, transitive closure).  The host function needs no GPU;
the pipelined bank call is a -m gpu test."""
import numpy as np
import pytest

import oracle
from testsupport import workloads as W


def _rand_list(rng, n_templates, n_samples, n_trig, clumpy):
    """Random sorted trigger list: `clumpy` puts most triggers in short runs so that windows matter."""
    keys = set()
    n_trig = min(n_trig, n_templates * n_samples // 3)
    while len(keys) < n_trig:
        t = int(rng.integers(n_templates))
        if clumpy and rng.random() < 0.8:
            c0 = int(rng.integers(n_samples))
            for d in range(int(rng.integers(1, 12))):
                keys.add((t, (c0 + d * int(rng.integers(1, 4))) % n_samples))
        else:
            keys.add((t, int(rng.integers(n_samples))))
    keys = sorted(keys)[:n_trig]
    a = np.zeros(len(keys), dtype=oracle.TRIG_DTYPE)
    for i, (t, j) in enumerate(keys):
        a[i] = (t, j, 6.0 + float(rng.integers(0, 40)) * 0.125, rng.uniform(-3, 3))       # coarse SNR grid: ties happen
    return a


def _to_product(tr):
    from paper_1006_4644_b200 import cbmf
    p = np.zeros(len(tr), dtype=cbmf.TRIG_DTYPE)
    for f in ("template_idx", "sample_idx", "snr", "phase"):
        p[f] = tr[f]
    return p


def _same(ev_p, ev_o):
    assert len(ev_p) == len(ev_o)
    assert np.array_equal(ev_p["template_idx"], ev_o["template_idx"])
    assert np.array_equal(ev_p["sample_idx"], ev_o["sample_idx"])
    assert np.array_equal(ev_p["snr"], ev_o["snr"].astype(np.float32))
    assert np.array_equal(ev_p["phase"], ev_o["phase"].astype(np.float32))


@pytest.mark.parametrize("seed", range(12))
def test_cluster_matches_oracle_on_random_lists(seed):
    from paper_1006_4644_b200 import cbmf
    rng = np.random.default_rng(seed)
    n_samples = int(rng.choice([64, 256, 1024, 4096]))
    tr = _rand_list(rng, int(rng.integers(1, 6)), n_samples, int(rng.integers(1, 300)), clumpy=seed % 2 == 0)
    for window in (0, 1, 2, 5, 17, n_samples // 4, n_samples):
        ev_o, n_o, _ = oracle.cluster_triggers(tr, n_samples, window)
        ev_p, n_p, rc = cbmf.cluster_triggers(_to_product(tr), n_samples, window)
        assert rc == 0 and n_p == n_o, (seed, window)
        _same(ev_p, ev_o)


def test_cluster_wrap_and_ties_match_oracle():
    from paper_1006_4644_b200 import cbmf
    n_s = 512
    cases = [
        [(0, 0, 9.0), (0, n_s - 1, 9.0)],                                   # tie across the wrap -> sample 0
        [(0, 1, 6.5), (0, 300, 7.0), (0, n_s - 2, 8.5)],                    # tail beats head: event sorts last
        [(0, 1, 8.5), (0, 300, 7.0), (0, n_s - 2, 6.5)],                    # head beats tail
        [(0, j, 6.0 + (j % 7)) for j in range(0, n_s, 3)],                  # a closed ring: one event
        [(1, 5, 7.0), (1, 6, 7.0), (1, 7, 7.0), (4, 5, 7.5)],               # plateau: first sample
    ]
    for rows in cases:
        tr = np.zeros(len(rows), dtype=oracle.TRIG_DTYPE)
        for i, (t, j, r) in enumerate(rows):
            tr[i] = (t, j, r, 0.01 * i)
        for window in (1, 3, 4):
            ev_o, n_o, _ = oracle.cluster_triggers(tr, n_s, window)
            ev_p, n_p, _ = cbmf.cluster_triggers(_to_product(tr), n_s, window)
            assert n_p == n_o
            _same(ev_p, ev_o)


def test_cluster_arguments():
    from paper_1006_4644_b200 import cbmf
    good = np.zeros(3, dtype=cbmf.TRIG_DTYPE)
    good["template_idx"] = [0, 0, 1]; good["sample_idx"] = [3, 9, 2]; good["snr"] = [7, 8, 9]
    ev, n, rc = cbmf.cluster_triggers(good, 16, 2, event_capacity=2)
    assert n == 3 and rc == cbmf.WTRUNC and list(ev["sample_idx"]) == [3, 9]
    ev, n, rc = cbmf.cluster_triggers(good[:0], 16, 2)
    assert n == 0 and rc == 0
    for bad in (good[::-1].copy(), ):                                        # not sorted
        with pytest.raises(cbmf.CbmfError):
            cbmf.cluster_triggers(bad, 16, 2)
    dup = good.copy(); dup["sample_idx"][1] = 3                              # repeated key
    with pytest.raises(cbmf.CbmfError):
        cbmf.cluster_triggers(dup, 16, 2)
    with pytest.raises(cbmf.CbmfError):
        cbmf.cluster_triggers(good, 8, 2)                                    # sample 9 outside the segment
    with pytest.raises(cbmf.CbmfError):
        cbmf.cluster_triggers(good, 16, -1)


@pytest.mark.gpu
@pytest.mark.parametrize("name,window,sub_batch", [("cfg0", 16, 5), ("cfg0", 0, 64), ("cfg1_256", 64, 16)])
def test_filter_bank_clustered_vs_oracle(name, window, sub_batch):
    """The pipelined call (raw triggers copied behind every launch pair, clustered on the host while the next pairs
    run): bit for bit the clustering of the plain call's trigger list, and the oracle's events end to end."""
    from paper_1006_4644_b200 import cbmf
    from parity import SNR_RTOL
    wl = W.config0() if name == "cfg0" else W.config1(256)
    thr = 5.0 if name == "cfg0" else wl.threshold           # cfg0 at 5: a few hundred noise triggers as well
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    g.set_psd(wl.psd); g.load_segment(wl.samples)
    g.set_sub_batch(sub_batch)
    pk, tr, nf, rc = g.filter_bank(wl.bank, thr, trig_capacity=1 << 18)
    assert rc == 0
    pk_c, ev, n_ev, nf_c, rc_c = g.filter_bank_clustered(wl.bank, thr, window)
    g.close()
    assert rc_c == 0 and nf_c == nf and np.array_equal(pk_c, pk)
    want, n_want, _ = cbmf.cluster_triggers(tr, wl.n, window)
    assert n_ev == n_want and np.array_equal(ev, want)
    # end to end against the oracle: its own triggers, its own clustering
    o = oracle.Oracle(wl.n, wl.fs, wl.f_low); o.set_psd(wl.psd); o.load_segment(wl.samples)
    pk_o, tr_o, _, _ = o.filter_bank(wl.bank, thr)
    ev_o, _, _ = oracle.cluster_triggers(tr_o, wl.n, window)
    o.close()
    # events well above threshold must agree one to one (an event whose members straddle the 1e-3 threshold band can
    # split or vanish on one side: reading A15)
    strong_o = {(int(e["template_idx"]), int(e["sample_idx"])): e for e in ev_o if e["snr"] > 1.02 * thr}
    strong_g = {(int(e["template_idx"]), int(e["sample_idx"])): e for e in ev if e["snr"] > 1.02 * thr}
    all_o = {(int(e["template_idx"]), int(e["sample_idx"])) for e in ev_o}
    all_g = {(int(e["template_idx"]), int(e["sample_idx"])) for e in ev}
    assert set(strong_o) <= all_g and set(strong_g) <= all_o
    for k, e in strong_g.items():
        if k in strong_o:
            assert abs(e["snr"] - strong_o[k]["snr"]) <= SNR_RTOL * strong_o[k]["snr"]
    for inj in wl.injections:
        if inj.template_idx < wl.n_templates and window > 0:
            mine = ev[ev["template_idx"] == inj.template_idx]
            assert any(abs(int(m["sample_idx"]) - inj.sample(wl.fs)) <= 2 for m in mine)


@pytest.mark.gpu
@pytest.mark.parametrize("log2n,n_templates,sub_batch", [(13, 5, 2), (20, 6, 6)])
def test_filter_bank_clustered_overflow_path(log2n, n_templates, sub_batch):
    """threshold 0: every sample of every template is a trigger, far more than a launch pair's region holds; the call
    filters the overflowed pairs again through the plain path, in runs of templates whose triggers fit one list
    (at 2^20 the single pair of 6 templates holds 6 M triggers: a run of 4 and a run of 2).  With a window of one
    sample every template is one closed ring of triggers: one event, its global maximum.  The call is not profiled:
    the per-pass record of an earlier profiled call does not survive it."""
    from paper_1006_4644_b200 import cbmf
    wl = W.small_case(log2n=log2n, n_templates=n_templates, seed=77)
    g = cbmf.Context(wl.n, wl.fs, wl.f_low)
    g.set_psd(wl.psd); g.load_segment(wl.samples)
    g.set_sub_batch(sub_batch)
    g.set_profiling(2)
    g.filter_bank(wl.bank, wl.threshold)
    assert g.last_pass_time(0)[1] > 0
    pk, ev, n_ev, nf, rc = g.filter_bank_clustered(wl.bank, 0.0, 1)
    assert g.last_pass_time(0) == (0.0, 0) and g.last_pass_time(1) == (0.0, 0) and len(g.debug_timeline(0)) == 0
    g.set_profiling(0)
    pk_plain = g.filter_bank(wl.bank, 0.0, trig_capacity=0)[0]
    g.close()
    assert rc == 0 and nf == n_templates * wl.n and n_ev == n_templates
    assert np.array_equal(pk, pk_plain)
    assert np.array_equal(ev["template_idx"], np.arange(n_templates)) and np.array_equal(ev["sample_idx"], pk["idx_peak"])
    assert np.array_equal(ev["snr"], pk["snr_max"])
