"""Parity of profiles and telemetry (R26-R29): CUDA path through the C-ABI against the
oracle.  Verdicts, counters, telemetry counters and the first-violation record are unique and compared bit for
bit; the ring's ORDER is unspecified, so records are compared sorted by seq, and when the ring overflows only
what is unique (counts) is compared and the kept records are checked to be valid ones."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests.util import oracle_for

pytestmark = pytest.mark.gpu
DET, ENF = 0, 1


def dev():
    return torch.device("cuda", 0)


def prepared(config, n, mode=None):
    st = S.make_stream(config, "cpu", n_events=n, mode=mode)
    orc = oracle_for(st.policy)
    hdr = st.hdr.numpy().view(np.uint64)
    tag = orc.sign(hdr, st.val.numpy().view(np.uint64))
    tag_t = torch.from_numpy(tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    orc.reset_counters()
    eng = B.Engine(0).load(st.policy)
    return st, orc, eng, hdr, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64), \
        (st.hdr.to(dev()), st.val.to(dev()), tag_t.to(dev()))


def same_counters(eng, orc):
    gg, gs = eng.wg_read_counters()
    og, os_ = orc.read_counters()
    assert gg == og, {k: (gg[k], og[k]) for k in og if gg[k] != og[k]}
    assert np.array_equal(gs, os_)


def as_tuple(r):
    return tuple(int(r[f]) for f in B.VIOLATION_DTYPE.names)


@pytest.mark.parametrize("config,n", [(4, 250_003), (1, 65_536), (5, 40_001), (3, 120_007)])  # (3: no return site in the policy: the verify runs the forward kernel)
def test_ring_and_first_record_equal_the_oracle(config, n):
    if config == 5:
        pol = S.make_policy(5, "cpu", n_sites=5_000, max_set=512)
        st = S.make_stream(5, "cpu", n_events=n, policy=pol, batch_index=1)
        orc = oracle_for(pol)
        hdr = st.hdr.numpy().view(np.uint64)
        tag = orc.sign(hdr, st.val.numpy().view(np.uint64))
        tag_t = torch.from_numpy(tag.view(np.int64).copy())
        st.apply_return_tamper(tag_t)
        orc.reset_counters()
        eng = B.Engine(0).load(pol)
        val, tagn = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
        d = (st.hdr.to(dev()), st.val.to(dev()), tag_t.to(dev()))
    else:
        st, orc, eng, hdr, val, tagn, d = prepared(config, n)
    cap = 1 << 15
    orc.set_ring_capacity(cap)
    eng.wg_set_ring_capacity(cap)
    for mode in (ENF, DET):  # two calls: seq runs on, the first record stays the first call's
        o = orc.verify(hdr, val, tagn, mode)
        g = eng.wg_verify_continuations(*d, mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
    same_counters(eng, orc)
    t, first, ring = eng.wg_read_telemetry(cap)
    assert t == orc.read_telemetry() and t["ring_dropped"] == 0 and t["ring_recorded"] > 4
    o_ring = orc.read_violations(cap)
    assert sorted(map(as_tuple, ring)) == sorted(map(as_tuple, o_ring))
    assert first is not None and as_tuple(first) == as_tuple(orc.read_first_violation())
    # reset empties ring and first record; capacity stays
    eng.wg_reset_counters()
    t, first, ring = eng.wg_read_telemetry(cap)
    assert first is None and len(ring) == 0 and t["ring_recorded"] == 0
    eng.close()


def test_full_ring_drops_and_counts_and_keeps_valid_records():
    st, orc, eng, hdr, val, tag, d = prepared(4, 300_007)
    orc.set_ring_capacity(1 << 15)
    eng.wg_set_ring_capacity(5)
    o = orc.verify(hdr, val, tag, ENF)
    g = eng.wg_verify_continuations(*d, ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    valid = set(map(as_tuple, orc.read_violations(1 << 15)))
    t, first, ring = eng.wg_read_telemetry(16)
    assert len(ring) == 5 and t["ring_recorded"] == 5 and t["ring_dropped"] == len(valid) - 5
    kept = list(map(as_tuple, ring))
    assert len(set(kept)) == 5 and set(kept) <= valid
    assert as_tuple(first) == as_tuple(orc.read_first_violation())  # survives the overflow
    eng.close()


@pytest.mark.parametrize("flags", [B.WG_PROFILE_SKIP_FORWARD, B.WG_PROFILE_SKIP_BACKWARD, B.WG_PROFILE_LOW_TELEMETRY,
                                   B.WG_PROFILE_SKIP_FORWARD | B.WG_PROFILE_LOW_TELEMETRY,
                                   B.WG_PROFILE_SKIP_FORWARD | B.WG_PROFILE_SKIP_BACKWARD])
@pytest.mark.parametrize("config", [4, 1, 3])
def test_profiles_match_the_oracle(flags, config):
    st, orc, eng, hdr, val, tag, d = prepared(config, 120_011)
    orc.set_profile(flags)
    eng.wg_set_profile(flags)
    cap = 1 << 18  # the forward entry point fails closed on every return event: the ring must hold them all
    orc.set_ring_capacity(cap)
    eng.wg_set_ring_capacity(cap)
    o = orc.verify(hdr, val, tag, ENF)
    g = eng.wg_verify_continuations(*d, ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    o = orc.check_forward(hdr, val, DET)
    g = eng.wg_check_forward(d[0], d[1], DET).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    same_counters(eng, orc)
    t, first, ring = eng.wg_read_telemetry(cap)
    assert t == orc.read_telemetry() and t["ring_dropped"] == 0
    assert sorted(map(as_tuple, ring)) == sorted(map(as_tuple, orc.read_violations(cap)))
    of = orc.read_first_violation()
    assert (first is None) == (of is None) and (first is None or as_tuple(first) == as_tuple(of))
    # the flags are configuration: they survive a reset; FULL restores the ordinary behaviour
    eng.wg_reset_counters(); orc.reset_counters()
    eng.wg_set_profile(B.WG_PROFILE_FULL); orc.set_profile(0)
    assert np.array_equal(eng.wg_verify_continuations(*d, ENF).cpu().numpy().view(np.uint32), orc.verify(hdr, val, tag, ENF))
    same_counters(eng, orc)
    eng.close()


def test_bad_profile_flags_are_rejected():
    st, orc, eng, hdr, val, tag, d = prepared(1, 1000)
    with pytest.raises(B.WgError) as e:
        eng.wg_set_profile(32)
    assert e.value.status == B.WG_ERR_INVALID_ARG
    eng.close()


# ---------------------------------------------------------------------------------------------------------
# metadata-integrity profile (R37-R38)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,n", [(4, 150_003), (3, 90_001), (5, 30_011)])
def test_metadata_integrity_matches_the_oracle_with_and_without_corruption(config, n):
    rng = np.random.default_rng(config)
    if config == 5:
        pol = S.make_policy(5, "cpu", n_sites=4_000, max_set=300)   # > 2,048 targets: the global-memory search path
        st = S.make_stream(5, "cpu", n_events=n, policy=pol, batch_index=0)
    else:
        st = S.make_stream(config, "cpu", n_events=n)
        pol = st.policy
    orc = oracle_for(pol)
    hdr = st.hdr.numpy().view(np.uint64)
    tag = orc.sign(hdr, st.val.numpy().view(np.uint64))
    tag_t = torch.from_numpy(tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    orc.reset_counters()
    val, tagn = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
    eng = B.Engine(0).load(pol)
    d = (st.hdr.to(dev()), st.val.to(dev()), tag_t.to(dev()))
    flags = B.WG_PROFILE_METADATA_INTEGRITY
    orc.set_profile(flags)
    eng.wg_set_profile(flags)
    # intact records: same verdicts as the ordinary profile
    o = orc.verify(hdr, val, tagn, ENF)
    g = eng.wg_verify_continuations(*d, ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    assert eng.wg_read_telemetry()[0]["fwd_meta_fail_events"] == 0
    # corrupt a few forward records (targets and tokens), the same way on both sides
    fwd_sites = np.nonzero(pol.kind == 1)[0]
    site_of_event = (hdr[:, 0] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    hot = [int(s) for s in fwd_sites if (site_of_event == s).any()][:6]
    for k, s in enumerate(hot):
        if k % 2 == 0:
            idx = int(pol.tgt_off[s]) + int(rng.integers(0, pol.tgt_off[s + 1] - pol.tgt_off[s]))
            x = 1 << int(rng.integers(4, 28))
            orc.policy_poke(0, idx, x)
            eng.wg_policy_poke(0, idx, x)
        else:
            x = int(rng.integers(1, 1 << 63))
            orc.policy_poke(1, s, x)
            eng.wg_policy_poke(1, s, x)
    o = orc.verify(hdr, val, tagn, DET)
    g = eng.wg_verify_continuations(*d, DET).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    o = orc.check_forward(hdr, val, ENF)
    g = eng.wg_check_forward(d[0], d[1], ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    same_counters(eng, orc)
    t = eng.wg_read_telemetry()[0]
    assert t == orc.read_telemetry() and t["fwd_meta_fail_events"] > 0
    eng.close()


# ---------------------------------------------------------------------------------------------------------
# policy-digest binding (second half; R39)
# ---------------------------------------------------------------------------------------------------------
def test_bound_load_refuses_a_mismatch_and_binds_the_tokens():
    st = S.make_stream(4, "cpu", n_events=60_007)
    pol = st.policy
    d = B.wg_policy_digest(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1)
    assert d == oracle.policy_digest(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1)
    eng = B.Engine(0).load(pol)                       # an ordinary engine first
    with pytest.raises(B.WgError) as e:               # wrong digest: refused, the previous policy stays
        eng.wg_load_policy(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, d ^ 4, bound=True)
    assert e.value.status == B.WG_ERR_BAD_POLICY
    hdr, val = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    d_hdr, d_val = st.hdr.to(dev()), st.val.to(dev())
    plain_orc = oracle_for(pol)
    plain_tag = plain_orc.sign(hdr, val)
    assert np.array_equal(eng.wg_sign_continuations(d_hdr, d_val).cpu().numpy().view(np.uint64), plain_tag)
    # bound load: tokens, verdicts and counters equal the bound oracle's; plain tokens no longer verify
    eng.wg_load_policy(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, d, bound=True)
    orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, d, bound=True)
    o_tag = orc.sign(hdr, val)
    g_tag = eng.wg_sign_continuations(d_hdr, d_val)
    assert np.array_equal(g_tag.cpu().numpy().view(np.uint64), o_tag) and not np.array_equal(o_tag, plain_tag)
    tag_t = torch.from_numpy(o_tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    tagn = tag_t.numpy().view(np.uint64)
    val = st.val.numpy().view(np.uint64)
    for tags in (tagn, plain_tag):
        o = orc.verify(hdr, val, tags, ENF)
        g = eng.wg_verify_continuations(d_hdr, st.val.to(dev()), torch.from_numpy(tags.view(np.int64).copy()).to(dev()), ENF)
        assert np.array_equal(g.cpu().numpy().view(np.uint32), o)
    same_counters(eng, orc)
    g, _ = eng.wg_read_counters()
    assert g["ret_viol_events"] > g["ret_checks"] // 2          # the whole plain-token pass violated
    # the shadow stack and the inline form use the same bound token
    orc.shadow_configure(64, 2)
    eng.wg_shadow_configure(64, 2)
    sh = np.zeros((8, 2), dtype=np.uint64)
    ret_site = int(np.nonzero(pol.kind == 0)[0][0])
    sh[:, 0] = np.uint64(ret_site) | (np.uint64(0xFFFF) << np.uint64(32))
    sh[:, 1] = (np.uint64(1) << np.uint64(48)) | (np.arange(8, dtype=np.uint64) << np.uint64(5))
    sv = np.full((8, 32), 0x7F5A40000040, dtype=np.uint64)
    to = lambda a: torch.from_numpy(a.view(np.int64)).to(dev())
    assert np.array_equal(eng.wg_shadow_push(to(sh), to(sv), ENF).cpu().numpy().view(np.uint32), orc.shadow_push(sh, sv, ENF))
    assert np.array_equal(eng.wg_shadow_check_ret(to(sh), to(sv), ENF).cpu().numpy().view(np.uint32), orc.shadow_check_ret(sh, sv, ENF))
    assert eng.wg_shadow_read_counters() == orc.shadow_read_counters() and orc.shadow_read_counters()["viol_lanes"] == 0
    # an ordinary load drops the binding again
    eng.load(pol)
    assert np.array_equal(eng.wg_sign_continuations(d_hdr, d_val).cpu().numpy().view(np.uint64), plain_tag)
    eng.close()


def test_host_path_first_record_and_ring_over_many_chunks():
    """VERDICT r1 weak #8 / ADVICE: the *_host calls alternate chunks between two streams; the first-violation-record
    kernels of consecutive chunks are chained by an event, so the record read back is the record OF
    first_violation_key (wg_read_telemetry returns WG_ERR_INTERNAL otherwise).  > 4 chunks of 256 Ki events, violations
    in every chunk, ring on; against the oracle's ring and first record."""
    n = 5 * (1 << 18) + 12_345
    st, orc, eng, hdr, val, tagn, d = prepared(2, n)
    assert len(np.unique(st.ret_tamper.ev.numpy() // (1 << 18))) == 6  # every chunk holds violations
    cap = 1 << 14
    orc.set_ring_capacity(cap)
    eng.wg_set_ring_capacity(cap)
    h_hdr, h_val, h_tag = st.hdr.pin_memory(), st.val.pin_memory(), torch.from_numpy(tagn.view(np.int64)).pin_memory()
    for mode in (DET, ENF):
        o = orc.verify(hdr, val, tagn, mode)
        g = eng.wg_verify_continuations_host(h_hdr, h_val, h_tag, mode).numpy().view(np.uint32)
        assert np.array_equal(g, o)
    same_counters(eng, orc)
    t, first, ring = eng.wg_read_telemetry(cap)
    assert t == orc.read_telemetry() and t["ring_dropped"] == 0
    assert as_tuple(first) == as_tuple(orc.read_first_violation())
    assert sorted(as_tuple(r) for r in ring) == sorted(as_tuple(r) for r in orc.read_violations())
    eng.close()


@pytest.mark.parametrize("config,n,extra", [(4, 200_003, 0), (4, 120_011, B.WG_PROFILE_SKIP_BACKWARD), (5, 60_007, 0),
                                            (1, 65_536, B.WG_PROFILE_LOW_TELEMETRY)])
def test_coverage_reduced_profile_matches_the_oracle(config, n, extra):
    """DESIGN.md R40 (Table A2): a per-site skip set under its own denominator; the
    oracle side is pinned by reconstruction in tests/test_oracle_telemetry.py."""
    if config == 5:
        pol = S.make_policy(5, "cpu", n_sites=5_000, max_set=512)
        st = S.make_stream(5, "cpu", n_events=n, policy=pol, batch_index=2)
        orc = oracle_for(pol)
        hdr = st.hdr.numpy().view(np.uint64)
        tag_t = torch.from_numpy(orc.sign(hdr, st.val.numpy().view(np.uint64)).view(np.int64).copy())
        st.apply_return_tamper(tag_t)
        orc.reset_counters()
        eng = B.Engine(0).load(pol)
        val, tag = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
        d = (st.hdr.to(dev()), st.val.to(dev()), tag_t.to(dev()))
    else:
        st, orc, eng, hdr, val, tag, d = prepared(config, n)
    pol = st.policy
    rng = np.random.default_rng(11 + config)
    skip = (rng.random(pol.n_sites) < 0.35).astype(np.uint8)
    site = (hdr[:, 0] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    hot = np.bincount(site[site < pol.n_sites], minlength=pol.n_sites)
    skip[np.argsort(-hot)[:2]] = 1
    cap = 1 << 18
    for e_ in (orc, ):
        e_.set_skip_sites(skip); e_.set_profile(oracle.PROFILE_COVERAGE_REDUCED | extra); e_.set_ring_capacity(cap)
    eng.wg_set_skip_sites(skip); eng.wg_set_profile(B.WG_PROFILE_COVERAGE_REDUCED | extra); eng.wg_set_ring_capacity(cap)
    for mode in (ENF, DET):
        o = orc.verify(hdr, val, tag, mode)
        g = eng.wg_verify_continuations(*d, mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
    o = orc.check_forward(hdr, val, ENF)
    g = eng.wg_check_forward(d[0], d[1], ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    same_counters(eng, orc)
    t, first, ring = eng.wg_read_telemetry(cap)
    ot = orc.read_telemetry()
    assert t == ot and t["skipped_site_events"] > 0 and t["ring_dropped"] == 0
    assert sorted(map(as_tuple, ring)) == sorted(map(as_tuple, orc.read_violations(cap)))
    of = orc.read_first_violation()
    assert (first is None) == (of is None) and (first is None or as_tuple(first) == as_tuple(of))
    # sign is unaffected; clearing the set or dropping the flag restores the full profile
    assert np.array_equal(eng.wg_sign_continuations(d[0], d[1]).cpu().numpy().view(np.uint64), orc.sign(hdr, val))
    eng.wg_reset_counters(); orc.reset_counters()
    eng.wg_set_skip_sites(None); orc.set_skip_sites(None)
    assert np.array_equal(eng.wg_verify_continuations(*d, ENF).cpu().numpy().view(np.uint32), orc.verify(hdr, val, tag, ENF))
    same_counters(eng, orc)
    assert eng.wg_read_telemetry()[0]["skipped_site_events"] == 0
    eng.close()


def test_sequence_base_gives_a_slice_the_streams_own_sequence_numbers():
    """wg_set_sequence_base (R12): verdicts of a slice equal the whole stream's; key, first record and
    ring records carry global sequence numbers."""
    st, orc, eng, hdr, val, tag, d = prepared(4, 150_001)
    lo = 61_234
    cap = 1 << 12
    orc.set_ring_capacity(cap); eng.wg_set_ring_capacity(cap)
    orc.set_sequence_base(lo); eng.wg_set_sequence_base(lo)
    o = orc.verify(hdr[lo:], val[lo:], tag[lo:], ENF)
    g = eng.wg_verify_continuations(d[0][lo:], d[1][lo:], d[2][lo:], ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o) and o[:, 0].any()
    same_counters(eng, orc)
    t, first, ring = eng.wg_read_telemetry(cap)
    assert as_tuple(first) == as_tuple(orc.read_first_violation()) and int(first["seq"]) >= lo
    assert sorted(map(as_tuple, ring)) == sorted(map(as_tuple, orc.read_violations(cap)))
    eng.close()
