"""Bank sharding for more than one GPU.

Templates are independent ("loop over the bank"), so the path shards with no
exchange inside it: every rank holds the whole segment (w[k], <= 64 MiB) and filters one
contiguous slice of the bank; the host concatenates the per-rank results.  The paper only
announces a multi-GPU version.  Nothing here does filter arithmetic: it is
index bookkeeping plus an optional torch.distributed gather of the 16-byte result records.
"""
from __future__ import annotations

import numpy as np


def shard_range(n_templates: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice [a, b) of the bank owned by `rank`; sizes differ by at most one,
    earlier ranks take the larger slices."""
    if world < 1 or not (0 <= rank < world) or n_templates < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(n_templates, world)
    a = rank * q + min(rank, r)
    return a, a + q + (1 if rank < r else 0)


def globalise_triggers(trig: np.ndarray, first_template: int) -> np.ndarray:
    """Rank-local template indices -> bank indices (order is kept: still sorted)."""
    out = trig.copy()
    out["template_idx"] += np.int32(first_template)
    return out


def gather_results(peaks: np.ndarray, trig: np.ndarray, n_templates: int, group=None):
    """All ranks call this with the results of their slice (template_idx rank-local); rank 0
    gets (peaks of the whole bank in bank order, all triggers sorted by (template, sample)),
    the others (None, None).  Uses torch.distributed object collectives (host side, outside
    any timed region); with no process group initialised it is the identity."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return peaks, trig
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    a, _ = shard_range(n_templates, rank, world)
    payload = (peaks, globalise_triggers(trig, a))
    box = [None] * world if rank == 0 else None
    dist.gather_object(payload, box, dst=0, group=group)
    if rank != 0:
        return None, None
    all_peaks = np.concatenate([p for p, _ in box])
    all_trig = np.concatenate([t for _, t in box])
    assert len(all_peaks) == n_templates
    return all_peaks, all_trig
