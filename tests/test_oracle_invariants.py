"""Invariants that pin the oracle's sign / verify / verdict / accounting rules.
Each maps to a protocol or attack shape of the paper.  CPU only."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_11871_b200 import streams as S
from tests import witness
from tests.util import mk_hdr, oracle_for, popc, sign_and_tamper_with_oracle

RET, FWD = oracle.KIND_PROTECTED_RETURN, oracle.KIND_PROTECTED_FORWARD
DET, ENF = oracle.MODE_DETECT, oracle.MODE_ENFORCE
FULL = 0xFFFFFFFF
PROTECTED_KEYS = ["ret_checks", "fwd_checks", "ret_lanes", "fwd_lanes", "ret_viol", "fwd_viol",
                  "ret_viol_events", "fwd_viol_events"]


def small_policy():
    """sites: 0,1 return; 2 forward {0x1000,0x2000,0x3000}; 3 forward {0x4000}; 4..8 the five non-protected kinds."""
    kind = np.array([RET, RET, FWD, FWD, 2, 3, 4, 5, 6], dtype=np.uint8)
    off = np.array([0, 0, 0, 3, 4, 4, 4, 4, 4, 4], dtype=np.uint32)
    tg = np.array([0x1000, 0x2000, 0x3000, 0x4000], dtype=np.uint64)
    return kind, off, tg


def new_oracle(k0=0x1122334455667788, k1=0x99AABBCCDDEEFF00, digest=42):
    return oracle.Oracle(*small_policy(), k0, k1, digest)


def rand_vals(rng, n):
    return rng.integers(0, 1 << 64, size=(n, 32), dtype=np.uint64)


# ---------------------------------------------------------------------------------------------
# sign <-> verify
# ---------------------------------------------------------------------------------------------

def test_untampered_continuations_always_verify():
    """Benign protected transfers pass with no false violation."""
    rng = np.random.default_rng(0)
    orc = new_oracle()
    n = 500
    hdr = mk_hdr(rng.integers(0, 2, n), rng.integers(0, 1 << 32, n), rng.integers(0, 1 << 64, n, dtype=np.uint64))
    val = rand_vals(rng, n)
    tag = orc.sign(hdr, val)
    for mode in (DET, ENF):
        out = orc.verify(hdr, val, tag, mode)
        assert (out[:, 0] == 0).all()
        assert (out[:, 1] == (hdr[:, 0] >> np.uint64(32))).all()
    g, _ = orc.read_counters()
    assert g["ret_viol"] == 0 and g["blocked_lanes"] == 0 and g["first_violation_key"] == (1 << 64) - 1


def test_sign_writes_zero_for_inactive_lanes_and_non_return_sites():
    rng = np.random.default_rng(1)
    orc = new_oracle()
    hdr = mk_hdr([0, 2, 4, 8, 99, 1], [0x0000FFFF, FULL, FULL, FULL, FULL, 0], 0x40)
    val = rand_vals(rng, 6)
    tag = orc.sign(hdr, val)
    assert (tag[0, 16:] == 0).all() and (tag[0, :16] != 0).all()
    assert (tag[1:] == 0).all()
    g, _ = orc.read_counters()
    assert g["signed_lanes"] == 16 and g["sign_skipped_events"] == 4
    assert g["events_total"] == 0  # sign is not a check


def test_every_single_bit_flip_of_tag_or_continuation_is_detected_on_that_lane_only():
    """Return hijack / token tamper (Table 5; §6.7 398-404)."""
    rng = np.random.default_rng(2)
    orc = new_oracle()
    hdr = mk_hdr([1], [0xFFFF0FFF], [0x0001000300000BE0])
    val = rand_vals(rng, 1)
    tag = orc.sign(hdr, val)
    for lane in (0, 7, 31):
        for bit in range(64):
            for which in ("tag", "val"):
                v, t = val.copy(), tag.copy()
                (t if which == "tag" else v)[0, lane] ^= np.uint64(1 << bit)
                out = orc.verify(hdr, v, t, ENF)
                assert out[0, 0] == 1 << lane, (lane, bit, which)
                assert out[0, 1] == 0xFFFF0FFF & ~(1 << lane)
    # a flip in an INACTIVE lane (12..15) is never judged
    t = tag.copy()
    t[0, 13] ^= np.uint64(1)
    assert orc.verify(hdr, val, t, ENF)[0].tolist() == [0, 0xFFFF0FFF]


def test_multi_bit_forgeries_detected():
    rng = np.random.default_rng(3)
    orc = new_oracle()
    hdr = mk_hdr([0] * 64, FULL, 0x20)
    val = rand_vals(rng, 64)
    tag = orc.sign(hdr, val)
    lanes = rng.integers(0, 32, 64)
    for e in range(64):
        k = 1 + e % 8
        bits = rng.choice(64, size=k, replace=False)
        tag[e, lanes[e]] ^= np.uint64(sum(1 << int(b) for b in bits))
    out = orc.verify(hdr, val, tag, DET)
    assert (out[:, 0] == (1 << lanes).astype(np.uint32)).all()


def test_token_replay_fails():
    """A valid tag replayed in another lane, another context (depth / epoch / slot) or at another site
    violates (258 'bind ... callsite identifier, depth, logical thread slot')."""
    orc = new_oracle()
    val = np.full((1, 32), 0x00007F5A40001230, dtype=np.uint64)  # warp-uniform continuation
    hdr = mk_hdr([0], FULL, [0x0001002000000040])
    tag = orc.sign(hdr, val)
    assert len(set(tag[0].tolist())) == 32  # same value, 32 different lane contexts -> 32 different tokens
    # other lane
    t = tag.copy()
    t[0, 3], t[0, 4] = tag[0, 4], tag[0, 3]
    assert orc.verify(hdr, val, t, DET)[0, 0] == (1 << 3) | (1 << 4)
    # other context_base (next depth, next epoch, neighbouring warp slot)
    for ctx in (0x0001004000000040, 0x0002002000000040, 0x0001002000000060):
        assert orc.verify(mk_hdr([0], FULL, [ctx]), val, tag, DET)[0, 0] == FULL
    # other site
    assert orc.verify(mk_hdr([1], FULL, [0x0001002000000040]), val, tag, DET)[0, 0] == FULL
    # low five bits of context_base are ignored (reserved for the lane)
    assert orc.verify(mk_hdr([0], FULL, [0x000100200000005F]), val, tag, DET)[0, 0] == 0


def test_one_corrupted_lane_cannot_hide_in_a_uniform_warp():
    """Divergent-lane backward hijack (Table 5 386)."""
    orc = new_oracle()
    val = np.full((32, 32), 0x00007F5A40000100, dtype=np.uint64)
    hdr = mk_hdr([0] * 32, FULL, 0x80)
    tag = orc.sign(hdr, val)
    for lane in range(32):
        val[lane, lane] = 0x00007F5A40000110
    out = orc.verify(hdr, val, tag, ENF)
    assert (out[:, 0] == (1 << np.arange(32)).astype(np.uint32)).all()


def test_wrong_key_rejects_everything():
    """Writable-shadow baseline contrast: tokens are keyed."""
    rng = np.random.default_rng(4)
    a, b = new_oracle(), new_oracle(k0=0x1122334455667789)
    hdr = mk_hdr([0] * 8, FULL, 0)
    val = rand_vals(rng, 8)
    assert (b.verify(hdr, val, a.sign(hdr, val), DET)[:, 0] == FULL).all()


# ---------------------------------------------------------------------------------------------
# guards, modes
# ---------------------------------------------------------------------------------------------

def test_inactive_lanes_are_never_judged():
    """@P0 RET: predicate-false lanes are not checked."""
    st = S.make_stream(1, n_events=4096)
    orc = oracle_for(st.policy)
    tag = sign_and_tamper_with_oracle(st, orc).numpy()
    hdr, val = st.hdr.numpy(), st.val.numpy().copy()
    orc.reset_counters()
    out1 = orc.verify(hdr, val, tag, ENF)
    g1, s1 = orc.read_counters()
    active = S._unpack32(st.active_mask()).numpy()
    rng = np.random.default_rng(5)
    val2 = np.where(active, val, rng.integers(-(1 << 63), 1 << 63, size=val.shape))
    tag2 = np.where(active, tag, rng.integers(-(1 << 63), 1 << 63, size=val.shape))
    orc.reset_counters()
    out2 = orc.verify(hdr, val2, tag2, ENF)
    g2, s2 = orc.read_counters()
    assert (out1 == out2).all() and g1 == g2 and (s1 == s2).all()
    assert (out1[:, 0] != 0).sum() > 10


def test_detect_never_blocks_enforce_blocks_exactly_the_violating_lanes():
    """Three-run protocol: detect and enforce see the same violations."""
    st = S.make_stream(1, n_events=8192)
    orc = oracle_for(st.policy)
    tag = sign_and_tamper_with_oracle(st, orc).numpy()
    hdr, val = st.hdr.numpy(), st.val.numpy()
    active = (hdr.view(np.uint64)[:, 0] >> np.uint64(32)).astype(np.uint32)
    orc.reset_counters()
    d = orc.verify(hdr, val, tag, DET)
    gd, _ = orc.read_counters()
    orc.reset_counters()
    e = orc.verify(hdr, val, tag, ENF)
    ge, se = orc.read_counters()
    assert (d[:, 0] == e[:, 0]).all()
    assert (d[:, 1] == active).all()
    assert (e[:, 1] == (active & ~e[:, 0])).all()
    assert ((e[:, 0] & ~active) == 0).all() and ((e[:, 1] & ~active) == 0).all()
    assert gd["blocked_lanes"] == 0 and gd["blocked_events"] == 0 and gd["last_mode"] == DET
    assert ge["blocked_lanes"] == int(popc(e[:, 0]).sum()) == ge["ret_viol"] + ge["fwd_viol"]
    assert ge["blocked_events"] == int((e[:, 0] != 0).sum()) and ge["last_mode"] == ENF
    assert int(se[:, 3].sum()) == ge["blocked_lanes"]
    for k in PROTECTED_KEYS + ["events_total", "first_violation_key"]:
        assert gd[k] == ge[k], k


def test_counters_never_feed_verdicts():
    """Telemetry tamper only changes diagnostics."""
    st = S.make_stream(1, n_events=2048)
    orc = oracle_for(st.policy)
    tag = sign_and_tamper_with_oracle(st, orc).numpy()
    hdr, val = st.hdr.numpy(), st.val.numpy()
    a = orc.verify(hdr, val, tag, ENF)
    b = orc.verify(hdr, val, tag, ENF)      # counters now hold the first pass
    orc.reset_counters()
    c = orc.verify(hdr, val, tag, ENF)
    assert (a == b).all() and (a == c).all()


# ---------------------------------------------------------------------------------------------
# accounting
# ---------------------------------------------------------------------------------------------

def test_non_protected_kinds_are_only_counted():
    """Unsupported / fallback / no-surface / fixed-edge / profile-excluded stay outside the protected
    denominator."""
    rng = np.random.default_rng(6)
    orc = new_oracle()
    n = 200
    sites = rng.integers(4, 9, n)
    masks = rng.integers(0, 1 << 32, n)
    hdr = mk_hdr(sites, masks, 0)
    val = rand_vals(rng, n)
    tag = rand_vals(rng, n)
    for entry, mode in ((orc.verify, ENF), (lambda h, v, t, m: orc.check_forward(h, v, m), DET)):
        orc.reset_counters()
        out = entry(hdr, val, tag, mode)
        assert (out[:, 0] == 0).all() and (out[:, 1] == masks.astype(np.uint32)).all()
        g, s = orc.read_counters()
        assert all(g[k] == 0 for k in PROTECTED_KEYS + ["blocked_lanes", "blocked_events"])
        assert g["events_total"] == n
        for k in range(2, 7):
            assert g[f"events_by_kind_{k}"] == int((sites == k + 2).sum())
        assert (s[:, 0] == np.bincount(sites, minlength=9)).all() and (s[:, 1:] == 0).all()
        assert g["first_violation_key"] == (1 << 64) - 1


def test_unknown_site_fails_closed_outside_every_denominator():
    """Out-of-range site id (PAPER.md:135, 154, 242 'fails closed instead of wrapping'); R13."""
    orc = new_oracle()
    hdr = mk_hdr([9, 1 << 31, FULL, 9], [0x0000F00F, FULL, 1, 0], 0)
    val = np.zeros((4, 32), dtype=np.uint64)
    out = orc.verify(hdr, val, val, ENF)
    assert out[:, 0].tolist() == [0x0000F00F, FULL, 1, 0]
    assert out[:, 1].tolist() == [0, 0, 0, 0]
    g, s = orc.read_counters()
    assert g["events_unknown_site"] == 4 and g["events_total"] == 4 and g["events_empty"] == 0
    assert sum(g[f"events_by_kind_{k}"] for k in range(7)) == 0 and (s == 0).all()
    assert all(g[k] == 0 for k in PROTECTED_KEYS)
    assert g["blocked_lanes"] == 8 + 32 + 1 and g["blocked_events"] == 3
    assert g["first_violation_key"] == 0  # seq 0, lane 0


def test_protected_return_event_given_to_forward_entry_is_misrouted():
    """DESIGN.md R14: no tag, cannot authenticate, fail closed; not a check."""
    orc = new_oracle()
    hdr = mk_hdr([0, 2], [0xFF, 0xFF], 0)
    val = np.full((2, 32), 0x1000, dtype=np.uint64)
    out = orc.check_forward(hdr, val, DET)
    assert out.tolist() == [[0xFF, 0xFF], [0, 0xFF]]
    g, s = orc.read_counters()
    assert g["events_misrouted"] == 1 and g["ret_checks"] == 0 and g["ret_lanes"] == 0 and g["ret_viol"] == 0
    assert g["fwd_checks"] == 1 and g["events_by_kind_0"] == 1 and s[0].tolist() == [1, 0, 0, 0]
    assert g["first_violation_key"] == 0


def test_forward_events_inside_verify_ignore_the_tag_row():
    rng = np.random.default_rng(7)
    orc = new_oracle()
    hdr = mk_hdr([2, 3], FULL, 0)
    val = np.full((2, 32), 0x2000, dtype=np.uint64)
    out = orc.verify(hdr, val, rand_vals(rng, 2), ENF)
    assert out.tolist() == [[0, FULL], [FULL, 0]]


def test_empty_active_mask_is_an_event_but_not_a_check():
    """DESIGN.md R22."""
    orc = new_oracle()
    hdr = mk_hdr([0, 2, 4], 0, 0)
    z = np.zeros((3, 32), dtype=np.uint64)
    out = orc.verify(hdr, z, z, ENF)
    assert (out == 0).all()
    g, s = orc.read_counters()
    assert g["events_empty"] == 3 and g["events_total"] == 3
    assert g["ret_checks"] == 0 and g["fwd_checks"] == 0
    assert s[[0, 2, 4], 0].tolist() == [1, 1, 1]


def test_first_violation_key_is_min_seq_lane_over_engine_lifetime():
    """PAPER.md:264-266; R12: seq runs over check calls, sign does not advance it."""
    orc = new_oracle()
    ok = np.full((3, 32), 0x4000, dtype=np.uint64)
    bad = ok.copy()
    bad[2, 9] = 0x4001
    bad[2, 20] = 0x4002
    hdr = mk_hdr([3, 3, 3], FULL, 0)
    orc.check_forward(hdr, ok, DET)                 # seq 0..2, clean
    orc.sign(hdr, ok)                               # does not advance seq
    orc.check_forward(hdr, bad, DET)                # seq 3..5, violation at seq 5 lanes 9 and 20
    orc.check_forward(hdr, bad, DET)                # seq 6..8
    g, _ = orc.read_counters()
    assert g["first_violation_key"] == (5 << 5) | 9
    orc.reset_counters()
    orc.check_forward(hdr, bad, DET)
    assert orc.read_counters()[0]["first_violation_key"] == (2 << 5) | 9


@pytest.mark.parametrize("config,n", [(1, 20000), (4, 60000), (5, 20000)])
def test_accounting_identities_and_generator_witness(config, n):
    """Σ identities of SURVEY.md §8(c) + the constructed expectation equals the oracle's masks."""
    kw = dict(n_sites=2000, max_set=256) if config == 5 else {}
    st = S.make_stream(config, n_events=n, **kw)
    orc = oracle_for(st.policy)
    tag = sign_and_tamper_with_oracle(st, orc).numpy()
    hdr, val = st.hdr.numpy(), st.val.numpy()
    orc.reset_counters()
    out = orc.verify(hdr, val, tag, st.mode)
    g, s = orc.read_counters()
    want = witness.expected_viol(st)
    assert (out[:, 0] == want).all()
    assert (want != 0).sum() >= 5

    site = st.site_id().numpy()
    active = st.active_mask().numpy().astype(np.uint32)
    kind = st.policy.kind[site]
    prot = kind <= 1
    nz = active != 0
    assert g["events_total"] == n == sum(g[f"events_by_kind_{k}"] for k in range(7)) + g["events_unknown_site"]
    assert int(s[:, 0].sum()) == n
    for k in range(7):
        assert g[f"events_by_kind_{k}"] == int((kind == k).sum())
    assert g["ret_checks"] == int(((kind == 0) & nz).sum()) and g["fwd_checks"] == int(((kind == 1) & nz).sum())
    assert g["ret_lanes"] + g["fwd_lanes"] == int(s[:, 1].sum()) == int(popc(active[prot]).sum())
    assert g["ret_viol"] + g["fwd_viol"] == int(s[:, 2].sum()) == int(popc(out[:, 0]).sum())
    assert g["ret_viol"] == int(popc(out[kind == 0, 0]).sum())
    assert g["ret_viol_events"] + g["fwd_viol_events"] == int((out[:, 0] != 0).sum())
    assert (out[~prot, 0] == 0).all() and (s[st.policy.kind > 1, 1:] == 0).all()
    assert ((out[:, 0] & ~active) == 0).all() and ((out[:, 1] & ~active) == 0).all()
    v = np.nonzero(out[:, 0])[0]
    low = int(out[v[0], 0])
    assert g["first_violation_key"] == (int(v[0]) << 5) | ((low & -low).bit_length() - 1)
    assert g["policy_digest"] == st.policy.policy_digest


# ---------------------------------------------------------------------------------------------
# load-time policy validation
# ---------------------------------------------------------------------------------------------

def test_bad_policies_are_rejected_and_load_nothing():
    """PAPER.md:186, 260, 174; R16."""
    kind, off, tg = small_policy()
    assert oracle.validate_policy(kind, off, tg) == 0
    k = kind.copy(); k[4] = 7
    assert oracle.validate_policy(k, off, tg) == 1
    o = off.copy(); o[0] = 1
    assert oracle.validate_policy(kind, o, tg) == 2
    o = off.copy(); o[3], o[4] = 4, 3
    assert oracle.validate_policy(kind, o, tg) == 2
    t = tg.copy(); t[1] = t[0]                       # duplicate
    assert oracle.validate_policy(kind, off, t) == 3
    t = tg.copy(); t[0], t[1] = tg[1], tg[0]         # unsorted
    assert oracle.validate_policy(kind, off, t) == 3
    k = kind.copy(); k[5] = FWD                      # forward site without target evidence
    assert oracle.validate_policy(k, off, tg) == 4
    k = kind.copy(); k[3] = 3                        # unsupported site that owns a set
    assert oracle.validate_policy(k, off, tg) == 5
    with pytest.raises(ValueError):
        oracle.Oracle(k, off, tg, 0, 0)
