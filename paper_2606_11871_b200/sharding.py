"""Multi-GPU layout of the check path: one process per GPU, policy and key replicated, the
event stream split into contiguous ranges, NO collective on the hot loop.  The only exchange is at read-out:
one sum all-reduce over the counter words (global + per-site) and one min all-reduce for the first-violation
key.  Events are independent given the read-only policy ("This property is site-local"), so the
union of the ranks' verdicts is the single-GPU result and the reduced counters equal the single-GPU counters.

Host logic only (no method arithmetic); covered by world_size-2 gloo tests on CPU.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from .binding import COUNTER_FIELDS

_IDX = {k: i for i, k in enumerate(COUNTER_FIELDS)}
_MIN_WORDS = (_IDX["first_violation_key"],)                    # min over ranks (R12)
_KEEP_WORDS = (_IDX["policy_digest"], _IDX["last_mode"])       # identical on every rank: not summed


def shard_range(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range [lo, hi) of rank `rank`: sizes differ by at most one, ranges tile [0, n)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(int(n_events), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def globalise_first_violation(key: int, shard_lo: int) -> int:
    """A rank numbers its events from 0; the global key adds the shard's start to the sequence part."""
    if key == (1 << 64) - 1:
        return key
    return (((key >> 5) + shard_lo) << 5) | (key & 31)


def reduce_counters(glob: dict, per_site: np.ndarray | None, shard_lo: int = 0, group=None,
                    device: torch.device | str = "cpu"):
    """All-reduce what wg_read_counters returned on each rank.  `device` is where the collective runs
    ("cuda" under NCCL, "cpu" under gloo).  Returns (global dict, per-site array) valid on every rank."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        out = dict(glob)
        out["first_violation_key"] = globalise_first_violation(glob["first_violation_key"], shard_lo)
        return out, per_site
    words = np.array([glob[k] for k in COUNTER_FIELDS], dtype=np.uint64)
    words[_IDX["first_violation_key"]] = globalise_first_violation(int(words[_IDX["first_violation_key"]]), shard_lo)
    # int64 carriers: sums stay far below 2^63; the min word is compared as unsigned by flipping the top bit
    s = torch.from_numpy(words.view(np.int64).copy()).to(device)
    m = s[list(_MIN_WORDS)] ^ torch.iinfo(torch.int64).min
    keep = s[list(_KEEP_WORDS)].clone()
    s[list(_MIN_WORDS)] = 0
    s[list(_KEEP_WORDS)] = 0
    dist.all_reduce(s, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(m, op=dist.ReduceOp.MIN, group=group)
    s[list(_MIN_WORDS)] = m ^ torch.iinfo(torch.int64).min
    s[list(_KEEP_WORDS)] = keep
    out_words = s.cpu().numpy().view(np.uint64)
    out = {k: int(v) for k, v in zip(COUNTER_FIELDS, out_words)}
    site = None
    if per_site is not None:
        t = torch.from_numpy(np.ascontiguousarray(per_site).view(np.int64).copy()).to(device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        site = t.cpu().numpy().view(np.uint64)
    return out, site
