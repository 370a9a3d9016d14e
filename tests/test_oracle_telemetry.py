"""Pins for the oracle's profiles and telemetry (R26-R29; PAPER.md:196, 264-266,
Table A2).  Nothing here re-calls the oracle to check the oracle: expectations are rebuilt in Python from the
headers, the policy's kind array, the verdict masks and the recorded tamper plan."""
import numpy as np
import torch

import oracle
from paper_2606_11871_b200 import streams as S
from tests import witness
from tests.util import oracle_for, popc

DET, ENF = 0, 1
RET, FWD = 0, 1


def signed_stream(config=4, n=30_011, mode=None):
    st = S.make_stream(config, "cpu", n_events=n, mode=mode)
    orc = oracle_for(st.policy)
    hdr = st.hdr.numpy().view(np.uint64)
    tag = orc.sign(hdr, st.val.numpy().view(np.uint64))
    tag_t = torch.from_numpy(tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    return st, orc, hdr, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)


def fields(hdr):
    site = (hdr[:, 0] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    active = (hdr[:, 0] >> np.uint64(32)).astype(np.uint32)
    return site, active


def ctz(x: int) -> int:
    return (x & -x).bit_length() - 1


def test_ring_holds_exactly_the_violating_events_in_order_with_their_operands():
    st, orc, hdr, val, tag = signed_stream()
    orc.set_ring_capacity(1 << 16)
    out = orc.verify(hdr, val, tag, ENF)
    site, active = fields(hdr)
    bad = np.nonzero(out[:, 0])[0]
    assert bad.size == len(st.ret_tamper) + len(st.fwd_tamper) and bad.size > 5
    assert np.array_equal(out[:, 0], witness.expected_viol(st))
    r = orc.read_violations()
    assert np.array_equal(r["seq"], bad.astype(np.uint64))              # event order, nothing else
    assert np.array_equal(r["viol_mask"], out[bad, 0]) and np.array_equal(r["active_mask"], active[bad])
    assert np.array_equal(r["site_id"], site[bad].astype(np.uint32))
    assert np.array_equal(r["kind"], st.policy.kind[site[bad]].astype(np.uint32))
    lanes = np.array([ctz(int(v)) for v in out[bad, 0]], dtype=np.uint32)
    assert np.array_equal(r["lane"], lanes) and (r["mode"] == ENF).all()
    assert np.array_equal(r["observed"], val[bad, lanes])
    is_ret = st.policy.kind[site[bad]] == RET
    assert np.array_equal(r["stored"][is_ret], tag[bad[is_ret], lanes[is_ret]]) and (r["stored"][~is_ret] == 0).all()
    t = orc.read_telemetry()
    assert t["ring_recorded"] == bad.size and t["ring_dropped"] == 0
    # first record = the record of the smallest (seq, lane); the key says the same
    g, _ = orc.read_counters()
    f = orc.read_first_violation()
    assert f is not None and f == r[0] and g["first_violation_key"] == (int(f["seq"]) << 5 | int(f["lane"]))


def test_bounded_ring_drops_and_counts_and_the_first_record_survives():
    st, orc, hdr, val, tag = signed_stream()
    orc.set_ring_capacity(3)
    out = orc.verify(hdr, val, tag, DET)
    bad = np.nonzero(out[:, 0])[0]
    r, t = orc.read_violations(), orc.read_telemetry()
    assert len(r) == 3 and t["ring_recorded"] == 3 and t["ring_dropped"] == bad.size - 3
    assert set(r["seq"].tolist()) <= set(bad.tolist())
    assert int(orc.read_first_violation()["seq"]) == int(bad[0])
    # reset clears the ring and the first record, keeps the capacity
    orc.reset_counters()
    assert len(orc.read_violations()) == 0 and orc.read_first_violation() is None
    orc.verify(hdr[:bad[0] + 1], val[:bad[0] + 1], tag[:bad[0] + 1], DET)
    assert len(orc.read_violations()) == 1
    # capacity 0 = ring off: nothing recorded, nothing "dropped"
    orc2 = oracle_for(st.policy)
    orc2.verify(hdr, val, tag, DET)
    assert len(orc2.read_violations()) == 0 and orc2.read_telemetry()["ring_dropped"] == 0
    assert orc2.read_first_violation() is not None


def test_unknown_site_and_misrouted_records():
    kind = np.array([RET, FWD], dtype=np.uint8)
    off = np.array([0, 0, 1], dtype=np.uint32)
    tg = np.array([0x40], dtype=np.uint64)
    orc = oracle.Oracle(kind, off, tg, 5, 6, 0)
    orc.set_ring_capacity(8)
    hdr = np.zeros((3, 2), dtype=np.uint64)
    hdr[:, 0] = [77 | (0b1100 << 32), 0 | (0b10 << 32), 1 | (0b1 << 32)]
    val = np.arange(96, dtype=np.uint64).reshape(3, 32)
    val[2, 0] = 65  # 0x40 = 64 would be a member of site 1's set
    orc.check_forward(hdr, val, ENF)
    r = orc.read_violations()
    assert r["kind"].tolist() == [7, RET, FWD] and r["lane"].tolist() == [2, 1, 0]
    assert r["observed"].tolist() == [2, 33, 65] and (r["stored"] == 0).all()


def test_backward_only_and_forward_only_profiles_use_separate_denominators():
    st, orc, hdr, val, tag = signed_stream()
    site, active = fields(hdr)
    kind = st.policy.kind[site]
    full = orc.verify(hdr, val, tag, ENF)
    g_full, s_full = orc.read_counters()
    for flag, skipped_kind, pre in ((oracle.PROFILE_SKIP_FORWARD, FWD, "fwd"), (oracle.PROFILE_SKIP_BACKWARD, RET, "ret")):
        o = oracle_for(st.policy)
        o.set_profile(flag)
        out = o.verify(hdr, val, tag, ENF)
        sk = (kind == skipped_kind)
        assert (out[sk, 0] == 0).all() and np.array_equal(out[sk, 1], active[sk])       # not judged, released
        assert np.array_equal(out[~sk], full[~sk])                                       # everything else unchanged
        g, s = o.read_counters()
        t = o.read_telemetry()
        nonempty = sk & (active != 0)
        assert t[f"skipped_{pre}_events"] == int(nonempty.sum())
        assert t[f"skipped_{pre}_lanes"] == int(popc(active[nonempty]).sum())
        other = "ret" if pre == "fwd" else "fwd"
        assert t[f"skipped_{other}_events"] == 0
        assert g[f"{pre}_checks"] == 0 and g[f"{pre}_lanes"] == 0 and g[f"{pre}_viol"] == 0
        assert g[f"{other}_checks"] == g_full[f"{other}_checks"] and g[f"{other}_viol"] == g_full[f"{other}_viol"]
        assert g["events_total"] == g_full["events_total"]
        assert all(g[f"events_by_kind_{k}"] == g_full[f"events_by_kind_{k}"] for k in range(7))
        assert np.array_equal(s[:, 0], s_full[:, 0])                                     # site.events still counts them
        assert (s[st.policy.kind == skipped_kind, 1:] == 0).all()
    # forward-only at the forward entry point: a return event is skipped, not misrouted
    o = oracle_for(st.policy)
    o.set_profile(oracle.PROFILE_SKIP_BACKWARD)
    out = o.check_forward(hdr, val, ENF)
    g, _ = o.read_counters()
    assert g["events_misrouted"] == 0 and (out[kind == RET, 0] == 0).all()


def test_low_telemetry_changes_no_verdict_and_no_global_counter():
    st, orc, hdr, val, tag = signed_stream()
    full = orc.verify(hdr, val, tag, ENF)
    g_full, _ = orc.read_counters()
    o = oracle_for(st.policy)
    o.set_profile(oracle.PROFILE_LOW_TELEMETRY)
    o.set_ring_capacity(1 << 16)
    out = o.verify(hdr, val, tag, ENF)
    g, s = o.read_counters()
    sign_only = ("signed_lanes", "sign_skipped_events")  # `orc` also signed the stream, `o` did not
    assert np.array_equal(out, full) and {k: v for k, v in g.items() if k not in sign_only} == \
        {k: v for k, v in g_full.items() if k not in sign_only}
    assert (s == 0).all() and len(o.read_violations()) == 0
    f = o.read_first_violation()
    assert f is not None and (int(f["seq"]) << 5 | int(f["lane"])) == g["first_violation_key"]


def test_telemetry_settings_never_change_a_verdict():
    st, orc, hdr, val, tag = signed_stream(config=1, n=20_000)
    a = orc.verify(hdr, val, tag, ENF)
    for cap in (0, 1, 1 << 12):
        o = oracle_for(st.policy)
        o.set_ring_capacity(cap)
        assert np.array_equal(o.verify(hdr, val, tag, ENF), a)


def test_coverage_reduced_profile_leaves_skipped_sites_unjudged_under_their_own_denominator():
    """DESIGN.md R40 ("profiles that skip kernels, sites, counters, or a CFI direction change the protected
    set and are reported under separate denominators"; Table A2).  Expectations are rebuilt from the
    headers, the policy kinds, the skip set and a FULL-profile run's verdict masks (themselves pinned by the witness):
    events at skipped protected sites lose their verdict and move from ret_* / fwd_* to skipped_site_*; nothing else
    changes; without the profile flag the skip set means nothing."""
    st, orc, hdr, val, tag = signed_stream(4, 40_009, mode=ENF)
    site, active = fields(hdr)
    kind = st.policy.kind
    full = orc.verify(hdr, val, tag, ENF)
    assert np.array_equal(full[:, 0], witness.expected_viol(st))
    g_full, s_full = orc.read_counters()
    rng = np.random.default_rng(7)
    skip = (rng.random(kind.size) < 0.3).astype(np.uint8)
    hot = np.bincount(site[site < kind.size], minlength=kind.size)
    skip[np.argsort(-hot)[:3]] = 1  # the three busiest sites too, so that violations fall into the skip set
    in_range = site < kind.size
    k_ev = np.where(in_range, kind[np.minimum(site, kind.size - 1)], 7)
    skipped = in_range & (active != 0) & ((k_ev == RET) | (k_ev == FWD)) & (skip[np.minimum(site, kind.size - 1)] != 0)
    assert skipped.sum() > 1000 and (full[skipped, 0] != 0).any()

    # the flag off: the skip set is ignored
    o1 = oracle_for(st.policy)
    o1.set_skip_sites(skip)
    assert np.array_equal(o1.verify(hdr, val, tag, ENF), full)

    o2 = oracle_for(st.policy)
    o2.set_skip_sites(skip)
    o2.set_profile(oracle.PROFILE_COVERAGE_REDUCED)
    out = o2.verify(hdr, val, tag, ENF)
    exp_viol = np.where(skipped, 0, full[:, 0]).astype(np.uint32)
    assert np.array_equal(out[:, 0], exp_viol) and np.array_equal(out[:, 1], active & ~exp_viol)
    g, s = o2.read_counters()
    t = o2.read_telemetry()
    pc = popc(active)
    assert t["skipped_site_events"] == int(skipped.sum()) and t["skipped_site_lanes"] == int(pc[skipped].sum())
    sk_ret, sk_fwd = skipped & (k_ev == RET), skipped & (k_ev == FWD)
    assert g["ret_checks"] == g_full["ret_checks"] - int(sk_ret.sum())
    assert g["fwd_checks"] == g_full["fwd_checks"] - int(sk_fwd.sum())
    assert g["ret_lanes"] == g_full["ret_lanes"] - int(pc[sk_ret].sum())
    assert g["fwd_lanes"] == g_full["fwd_lanes"] - int(pc[sk_fwd].sum())
    assert g["ret_viol"] == int(popc(exp_viol[k_ev == RET]).sum()) and g["fwd_viol"] == int(popc(exp_viol[k_ev == FWD]).sum())
    assert g["blocked_lanes"] == int(popc(exp_viol).sum())
    for k in ("events_total", "events_empty", "events_unknown_site", "events_misrouted") + tuple(f"events_by_kind_{i}" for i in range(7)):
        assert g[k] == g_full[k], k
    # per site: events unchanged; a skipped site checks no lane and has no violation
    assert np.array_equal(s[:, 0], s_full[:, 0])
    prot_skip = (skip != 0) & ((kind == RET) | (kind == FWD))
    assert (s[prot_skip, 1:] == 0).all() and np.array_equal(s[~prot_skip], s_full[~prot_skip])
    viols = np.nonzero(exp_viol)[0]
    assert g["first_violation_key"] == ((int(viols[0]) << 5) | ctz(int(exp_viol[viols[0]])))

    # a skipped return site at the FORWARD entry point is skipped, not misrouted; an unskipped one still fails closed
    o3 = oracle_for(st.policy)
    o3.set_skip_sites(skip)
    o3.set_profile(oracle.PROFILE_COVERAGE_REDUCED)
    f = o3.check_forward(hdr, val, DET)
    ret_ev = in_range & (k_ev == RET) & (active != 0)
    assert (f[sk_ret, 0] == 0).all() and np.array_equal(f[ret_ev & ~skipped, 0], active[ret_ev & ~skipped])
    assert o3.read_counters()[0]["events_misrouted"] == int((ret_ev & ~skipped).sum())

    # a direction skip takes precedence over the site skip
    o4 = oracle_for(st.policy)
    o4.set_skip_sites(skip)
    o4.set_profile(oracle.PROFILE_COVERAGE_REDUCED | oracle.PROFILE_SKIP_BACKWARD)
    o4.verify(hdr, val, tag, ENF)
    t4 = o4.read_telemetry()
    all_ret = in_range & (k_ev == RET) & (active != 0)
    assert t4["skipped_ret_events"] == int(all_ret.sum()) and t4["skipped_site_events"] == int(sk_fwd.sum())


def test_sequence_base_shifts_keys_and_records_and_nothing_else():
    """DESIGN.md R12 / SURVEY.md §8(e): a rank that checks the slice [lo, hi) of a sharded stream sets its sequence base
    to lo; first-violation key and ring records then carry the stream's own sequence numbers."""
    st, orc, hdr, val, tag = signed_stream(4, 20_011)
    whole = orc.verify(hdr, val, tag, ENF)
    g_whole, _ = orc.read_counters()
    lo = 7_003
    o2 = oracle_for(st.policy)
    o2.set_ring_capacity(1 << 12)
    o2.set_sequence_base(lo)
    part = o2.verify(hdr[lo:], val[lo:], tag[lo:], ENF)
    assert np.array_equal(part, whole[lo:])
    bad = np.nonzero(whole[lo:, 0])[0] + lo
    assert bad.size > 2
    g2, _ = o2.read_counters()
    assert g2["first_violation_key"] == ((int(bad[0]) << 5) | ctz(int(whole[bad[0], 0])))
    assert np.array_equal(o2.read_violations()["seq"], bad.astype(np.uint64))
    assert int(o2.read_first_violation()["seq"]) == int(bad[0])
    assert g2["events_total"] == hdr.shape[0] - lo
