"""N > 1 on the REAL engine ("This property is site-local"): two
processes, each with its own engine over its shard_range slice of ONE config-4 stream, sequence base = slice start,
counters reduced with sharding.reduce_counters, first record with sharding.reduce_first_record.  Verdicts, reduced
counters (global + per site) and the first-violation record must equal the single-engine run AND the oracle.
Both ranks share cuda:0 over gloo (this box has one GPU; nothing here makes one rank's kernel wait for the other's);
with two or more GPUs the same test also runs over NCCL, one device per rank."""
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

pytestmark = pytest.mark.gpu
N_EVENTS = 300_007
RING = 1 << 12


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _prepare():
    """The stream, signed by the oracle and corrupted as planned (same on every process: seeded)."""
    import oracle
    st = S.make_stream(4, "cpu", n_events=N_EVENTS)
    pol = st.policy
    orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
    hdr = st.hdr.numpy().view(np.uint64)
    tag_t = torch.from_numpy(orc.sign(hdr, st.val.numpy().view(np.uint64)).view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    orc.reset_counters()
    return st, orc, tag_t


def _worker(rank: int, world: int, port: int, backend: str, q):
    from paper_2606_11871_b200 import binding as B
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    devno = rank if backend == "nccl" else 0
    torch.cuda.set_device(devno)
    dev = torch.device("cuda", devno)
    dist.init_process_group(backend, rank=rank, world_size=world)
    try:
        st, _, tag_t = _prepare()
        lo, hi = sharding.shard_range(N_EVENTS, rank, world)
        eng = B.Engine(devno).load(st.policy)
        eng.wg_set_ring_capacity(RING)
        eng.wg_set_sequence_base(lo)
        out = eng.wg_verify_continuations(st.hdr[lo:hi].to(dev), st.val[lo:hi].to(dev), tag_t[lo:hi].to(dev), st.mode)
        g, s = eng.wg_read_counters()
        t, first, ring = eng.wg_read_telemetry(RING)
        cdev = dev if backend == "nccl" else "cpu"
        gr, sr = sharding.reduce_counters(g, s, 0, device=cdev)
        key, rec = sharding.reduce_first_record(g["first_violation_key"], first, device=cdev)
        q.put((rank, lo, hi, out.cpu().numpy().view(np.uint32), gr, sr, key, None if rec is None else rec.tobytes(),
               ring.tobytes()))
        eng.close()
    finally:
        dist.destroy_process_group()


def _run(world: int, backend: str):
    from paper_2606_11871_b200 import binding as B
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, backend, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0

    # the oracle and ONE engine over the whole stream
    st, orc, tag_t = _prepare()
    hdr, val, tag = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
    orc.set_ring_capacity(RING)
    o_out = orc.verify(hdr, val, tag, st.mode)
    og, os_ = orc.read_counters()
    dev = torch.device("cuda", 0)
    eng = B.Engine(0).load(st.policy)
    eng.wg_set_ring_capacity(RING)
    e_out = eng.wg_verify_continuations(st.hdr.to(dev), st.val.to(dev), tag_t.to(dev), st.mode).cpu().numpy().view(np.uint32)
    eg, es = eng.wg_read_counters()
    _, e_first, e_ring = eng.wg_read_telemetry(RING)
    eng.close()
    assert np.array_equal(e_out, o_out) and eg == og and np.array_equal(es, os_)

    sharded = np.concatenate([r[3] for r in res])
    assert np.array_equal(sharded, o_out) and o_out[:, 0].any()
    o_first = orc.read_first_violation()
    assert og["first_violation_key"] != (1 << 64) - 1
    for _, lo, hi, _, gr, sr, key, rec, _ in res:  # every rank holds the reduced result
        assert gr == og, {k: (gr[k], og[k]) for k in og if gr[k] != og[k]}
        assert np.array_equal(sr, os_)
        assert key == og["first_violation_key"]
        assert rec == np.asarray(o_first).tobytes() == np.asarray(e_first).tobytes()
    # the ranks' rings together are the single engine's ring (global sequence numbers), in any order
    rings = np.concatenate([np.frombuffer(r[8], dtype=B.VIOLATION_DTYPE) for r in res])
    key_of = lambda a: sorted(tuple(int(x[f]) for f in B.VIOLATION_DTYPE.names) for x in a)  # noqa: E731
    assert key_of(rings) == key_of(e_ring) == key_of(orc.read_violations(RING))


def test_two_engines_on_one_gpu_over_gloo_equal_one_engine_and_the_oracle():
    _run(2, "gloo")


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs")
def test_two_engines_on_two_gpus_over_nccl_equal_one_engine_and_the_oracle():
    _run(2, "nccl")
