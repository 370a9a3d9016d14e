"""N > 1 host logic on CPU: two gloo ranks each run the ORACLE on their contiguous shard of one
stream; the reduced counters and the concatenated verdicts must equal the single-process result.  (The GPU path
uses the same shard_range / reduce_counters with the engine's counters; here the oracle stands in for the
engine because this box has no GPU — what is under test is the sharding and the read-out exchange.)"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2606_11871_b200 import sharding  # noqa: E402
from paper_2606_11871_b200 import streams as S  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_range_tiles_the_stream():
    for n in (0, 1, 7, 100, 58_000_000):
        for w in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(10, 2, 2)


def test_first_violation_key_globalises_by_shard_start():
    assert sharding.globalise_first_violation((1 << 64) - 1, 123) == (1 << 64) - 1
    assert sharding.globalise_first_violation((5 << 5) | 17, 1000) == (1005 << 5) | 17


def _worker(rank: int, world: int, port: int, n_events: int, q):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        st = S.make_stream(4, "cpu", n_events=n_events)
        pol = st.policy
        orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
        hdr = st.hdr.numpy().view(np.uint64)
        tag_t = torch.from_numpy(orc.sign(hdr, st.val.numpy().view(np.uint64)).view(np.int64).copy())
        st.apply_return_tamper(tag_t)
        orc.reset_counters()
        lo, hi = sharding.shard_range(n_events, rank, world)
        val, tag = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
        orc.set_sequence_base(lo)  # the rank's events keep the stream's own sequence numbers
        out = orc.verify(hdr[lo:hi], val[lo:hi], tag[lo:hi], st.mode)
        g, s = orc.read_counters()
        gr, sr = sharding.reduce_counters(g, s, 0)
        key, rec = sharding.reduce_first_record(g["first_violation_key"], orc.read_first_violation())
        q.put((rank, lo, hi, out, gr, sr, key, None if rec is None else np.asarray(rec).tobytes()))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_equal_one_process():
    import oracle
    n = 40_003
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # single-process truth
    st = S.make_stream(4, "cpu", n_events=n)
    pol = st.policy
    orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
    hdr = st.hdr.numpy().view(np.uint64)
    tag_t = torch.from_numpy(orc.sign(hdr, st.val.numpy().view(np.uint64)).view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    orc.reset_counters()
    out = orc.verify(hdr, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64), st.mode)
    g, s = orc.read_counters()
    assert np.array_equal(np.concatenate([res[0][3], res[1][3]]), out)
    assert g["first_violation_key"] != (1 << 64) - 1
    first = orc.read_first_violation()
    for _, _, _, _, gr, sr, key, rec in res:  # every rank holds the reduced result
        assert gr == g, {k: (gr[k], g[k]) for k in g if gr[k] != g[k]}
        assert np.array_equal(sr, s)
        assert key == g["first_violation_key"] and rec == np.asarray(first).tobytes()
