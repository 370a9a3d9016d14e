"""Multi-GPU layout of the check path: one process per GPU, policy and key replicated, the
event stream split into contiguous ranges, NO collective on the hot loop.  The only exchange is at read-out:
one sum all-reduce over the counter words (global + per-site) and one min all-reduce for the first-violation
key.  Events are independent given the read-only policy ("This property is site-local"), so the
union of the ranks' verdicts is the single-GPU result and the reduced counters equal the single-GPU counters.

Each rank tells its engine where its slice starts (``wg_set_sequence_base(lo)``), so first-violation keys, the
first-violation record and ring records carry the stream's own sequence numbers and need no fixing up afterwards
(``shard_lo`` stays 0 in ``reduce_counters``; the argument remains for callers whose ranks number from 0).

Host logic only (no method arithmetic); covered by world_size-2 gloo tests on CPU (tests/test_sharding_gloo.py) and, on
the real engine, by two processes sharing cuda:0 (tests/test_gpu_sharding.py).
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


def reduce_first_record(key: int, record, group=None, device: torch.device | str = "cpu"):
    """The first-violation RECORD of the whole stream on every rank: the record of the rank that holds the smallest
    key (``key`` = this rank's first_violation_key with global sequence numbers, ``record`` = its wg_violation_rec as a
    numpy structured scalar, or None).  One all-gather of 56 bytes per rank.  Returns (key, record or None)."""
    none = (1 << 64) - 1
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return key, record
    mine = np.zeros(7, dtype=np.uint64)
    mine[0] = key if record is not None else none
    if record is not None:
        mine[1:] = np.frombuffer(np.asarray(record).tobytes(), dtype=np.uint64)
    t = torch.from_numpy(mine.view(np.int64).copy()).to(device)
    world = dist.get_world_size(group)
    parts = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(parts, t, group=group)
    rows = np.stack([p_.cpu().numpy().view(np.uint64) for p_ in parts])
    best = int(np.argmin(rows[:, 0]))
    if rows[best, 0] == none:
        return none, None
    rec = np.frombuffer(rows[best, 1:].tobytes(), dtype=np.asarray(record).dtype if record is not None else _REC_DTYPE)[0]
    return int(rows[best, 0]), rec


from .binding import VIOLATION_DTYPE as _REC_DTYPE  # noqa: E402  (48 bytes = six u64 words)
