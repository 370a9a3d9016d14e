"""The synthetic policies / streams have the shapes BASELINE.json and SURVEY.md §8(d) state.  CPU only."""
import numpy as np
import torch

from paper_2606_11871_b200 import streams as S
from tests.util import popc


def _sizes(p):
    return np.diff(p.tgt_off.astype(np.int64))


def test_policy_shapes():
    p1 = S.make_policy(1)
    assert p1.n_sites == 72 and (p1.kind == 0).sum() == 64 and (p1.kind == 1).sum() == 8
    s = _sizes(p1)[p1.kind == 1]
    assert s.min() >= 1 and s.max() <= 4
    p2 = S.make_policy(2)
    assert p2.n_sites == 1343 and (p2.kind == 0).all() and p2.tgts.size == 0
    p3 = S.make_policy(3)
    assert p3.n_sites == 40 and p3.tgts.size == 154 and _sizes(p3).min() >= 1 and _sizes(p3).max() <= 16
    p4 = S.make_policy(4)
    assert p4.n_sites == 51621
    assert [(p4.kind == k).sum() for k in range(7)] == [1343, 154, 45000, 15, 99, 10, 5000]
    s4 = np.sort(_sizes(p4)[p4.kind == 1])
    assert np.median(s4) == 1 and s4[int(0.9 * 154)] == 3 and s4.max() == 10 and s4.sum() == 248
    assert (s4 == 1).sum() == 109 and (s4 > 1).sum() == 45 and (s4 - 1).sum() == 94
    p5 = S.make_policy(5, n_sites=4000, max_set=4096)
    s5 = _sizes(p5)[p5.kind == 1]
    assert (p5.kind == 1).sum() == 2000 and s5.min() >= 1 and s5.max() <= 4096 and s5.max() > 1000
    for p in (p1, p3, p4, p5):  # sorted, unique, 16-byte aligned, inside the window
        for site in np.nonzero(p.kind == 1)[0][:200]:
            t = p.tgts[p.tgt_off[site]:p.tgt_off[site + 1]].astype(np.int64)
            assert (np.diff(t) > 0).all() and (t % 16 == 0).all()
            assert t.min() >= S.CODE_BASE and t.max() < S.CODE_BASE + 16 * p.window_slots
    assert p1.k0 != p2.k0 and 0 <= p1.k0 < 1 << 64


def test_streams_are_deterministic():
    a, b = S.make_stream(1, n_events=3000), S.make_stream(1, n_events=3000)
    assert torch.equal(a.hdr, b.hdr) and torch.equal(a.val, b.val)
    assert torch.equal(a.ret_tamper.arg, b.ret_tamper.arg)


def test_config4_proportions_and_masks():
    st = S.make_stream(4, n_events=116_000)
    kind = st.policy.kind[st.site_id().numpy()]
    assert (kind == 0).sum() == 76_600 and (kind == 1).sum() == 27_800 and (kind > 1).sum() == 11_600
    dens = popc(st.active_mask().numpy()).mean() / 32
    assert 0.89 < dens < 0.91
    ctx = st.hdr[:, 1].numpy()
    assert (ctx & 31 == 0).all() and (ctx >> 48 == 1).all()
    # Zipf: the hottest return site takes a large share
    ret_sites = st.site_id().numpy()[kind == 0]
    assert np.bincount(ret_sites).max() / ret_sites.size > 0.10
    assert abs(len(st.ret_tamper) - 38) <= 1 and abs(len(st.fwd_tamper) - 14) <= 1
    # uniform / divergent mix
    u = st.uniform.numpy()
    assert 0.67 < u[kind == 0].mean() < 0.73 and 0.87 < u[kind == 1].mean() < 0.93


def test_config5_masks_span_single_lane_to_full():
    st = S.make_stream(5, n_events=20_000, n_sites=2000, max_set=64)
    pc = popc(st.active_mask().numpy())
    assert pc.min() == 1 and pc.max() == 32 and 15.5 < pc.mean() < 17.5
    assert st.mode == S.DETECT and S.make_stream(5, n_events=10, n_sites=2000, max_set=64, batch_index=1).mode == S.ENFORCE


def test_public_code_shaped_configs_have_the_reported_shapes():
    """Configs 6 and 7: one 38-target site; a contiguous 64-check wrong-callback burst."""
    import numpy as np
    from paper_2606_11871_b200 import streams as S
    from tests import witness
    from tests.util import oracle_for

    st = S.make_stream(6, "cpu")
    sizes = np.diff(st.policy.tgt_off.astype(np.int64))
    assert sorted(sizes[sizes > 0].tolist()) == [38] and st.hdr.shape[0] == 50_000
    st = S.make_stream(7, "cpu")
    orc = oracle_for(st.policy)
    hdr, val = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    out = orc.verify(hdr, val, orc.sign(hdr, val), st.mode)
    b0 = st.meta["burst_start"]
    assert np.array_equal(out[:, 0], witness.expected_viol(st))
    assert int((out[:, 0] != 0).sum()) == 64 and out[b0:b0 + 64, 0].all()
    g, _ = orc.read_counters()
    assert g["fwd_viol_events"] == 64 and g["blocked_events"] == 64
