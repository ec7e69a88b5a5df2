"""Multi-GPU host logic on CPU: bank slices and the gloo gather of per-rank results
(bank sharding, no data-path collective)."""
import os
import socket

import numpy as np
import pytest

from paper_1006_4644_b200.sharding import gather_results, globalise_triggers, shard_range

PEAK = np.dtype([("snr_max", "<f4"), ("idx_peak", "<i4"), ("phase", "<f4"), ("sigma", "<f4")])
TRIG = np.dtype([("template_idx", "<i4"), ("sample_idx", "<i4"), ("snr", "<f4"), ("phase", "<f4")])


@pytest.mark.parametrize("n,world", [(0, 1), (1, 4), (7, 2), (1024, 8), (65536, 3), (5, 8)])
def test_shard_range_partitions_the_bank(n, world):
    edges = [shard_range(n, r, world) for r in range(world)]
    assert edges[0][0] == 0 and edges[-1][1] == n
    for (a0, b0), (a1, b1) in zip(edges, edges[1:]):
        assert b0 == a1 and b0 >= a0 and b1 >= a1
    sizes = [b - a for a, b in edges]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_shard_range_rejects_bad_arguments():
    for args in [(4, -1, 2), (4, 2, 2), (4, 0, 0), (-1, 0, 1)]:
        with pytest.raises(ValueError):
            shard_range(*args)


def test_globalise_triggers_offsets_only_the_template_index():
    t = np.zeros(3, dtype=TRIG)
    t["template_idx"] = [0, 0, 2]
    t["sample_idx"] = [5, 9, 1]
    g = globalise_triggers(t, 100)
    assert list(g["template_idx"]) == [100, 100, 102] and list(g["sample_idx"]) == [5, 9, 1]
    assert list(t["template_idx"]) == [0, 0, 2]


def _fake_slice(a, b):
    """Deterministic stand-in results for bank slice [a, b) with rank-local trigger indices."""
    pk = np.zeros(b - a, dtype=PEAK)
    pk["snr_max"] = np.arange(a, b) * 0.5
    pk["idx_peak"] = np.arange(a, b) * 3
    tr = np.zeros(2 * (b - a), dtype=TRIG)
    tr["template_idx"] = np.repeat(np.arange(b - a), 2)
    tr["sample_idx"] = np.tile([4, 8], b - a)
    return pk, tr


def _worker(rank, world, port, n, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = shard_range(n, rank, world)
        pk, tr = _fake_slice(a, b)
        allp, allt = gather_results(pk, tr, n)
        if rank == 0:
            q.put((allp.tobytes(), allt.tobytes()))
        else:
            assert allp is None and allt is None
            q.put(None)
    finally:
        dist.destroy_process_group()


def test_gather_results_gloo_world2():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    n, world = 11, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    outs = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    got = [o for o in outs if o is not None]
    assert len(got) == 1
    allp = np.frombuffer(got[0][0], dtype=PEAK)
    allt = np.frombuffer(got[0][1], dtype=TRIG)
    want_p, want_t = _fake_slice(0, n)                  # one rank owning the whole bank
    assert np.array_equal(allp, want_p)
    assert np.array_equal(allt, want_t)
    keys = allt["template_idx"].astype(np.int64) * (1 << 32) + allt["sample_idx"]
    assert np.all(np.diff(keys) > 0)


def test_gather_results_without_process_group_is_identity():
    pk, tr = _fake_slice(0, 4)
    p2, t2 = gather_results(pk, tr, 4)
    assert p2 is pk and t2 is tr
