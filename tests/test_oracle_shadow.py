"""Pins for the oracle's stateful shadow stack (DESIGN.md
R30-R36).  The token formula is pinned through the OpenSSL-pinned stateless MAC (an entry re-forged with
oracle.mac under the documented context must verify); the stack discipline is pinned against a MAC-free Python
model (lists per thread slot) on random call / return sequences; every fail-closed case has its own test."""
import numpy as np

import oracle
from tests.util import mk_hdr, popc

DET, ENF = 0, 1
RET, FWD, FIXED = 0, 1, 2
FULL = 0xFFFFFFFF
K0, K1 = 0x0123456789ABCDEF, 0xFEDCBA9876543210


def make(n_slots=8, max_depth=4):
    kind = np.array([RET, RET, FWD, FIXED, RET], dtype=np.uint8)
    off = np.array([0, 0, 0, 1, 1, 1], dtype=np.uint32)
    tg = np.array([0x5000], dtype=np.uint64)
    o = oracle.Oracle(kind, off, tg, K0, K1, 0)
    o.shadow_configure(n_slots, max_depth)
    return o


def ctx_base(epoch, slot, depth_field=0):
    return (epoch << 48) | (depth_field << 37) | (slot << 5)


def ev(site, mask, slot, epoch=1, depth_field=0):
    return mk_hdr([site], [mask], [ctx_base(epoch, slot, depth_field)])


def vals(x):
    return np.full((1, 32), x, dtype=np.uint64)


def test_call_return_pairs_verify_in_lifo_order_only():
    o = make()
    a, b = vals(0x7F5A40000010), vals(0x7F5A40000020)
    assert not o.shadow_push(ev(0, FULL, 3), a, ENF)[:, 0].any()
    assert not o.shadow_push(ev(1, FULL, 3), b, ENF)[:, 0].any()
    assert o.shadow_depth(3, 0) == 2 and o.shadow_depth(3, 31) == 2 and o.shadow_depth(2, 0) == 0
    assert not o.shadow_check_ret(ev(1, FULL, 3), b, ENF)[:, 0].any()
    assert not o.shadow_check_ret(ev(0, FULL, 3), a, ENF)[:, 0].any()
    assert o.shadow_depth(3, 7) == 0
    # wrong order: the inner return presented first does not match the outer frame... and vice versa
    o.shadow_push(ev(0, FULL, 3), a, ENF)
    o.shadow_push(ev(1, FULL, 3), b, ENF)
    out = o.shadow_check_ret(ev(0, FULL, 3), a, ENF)
    assert out[0, 0] == FULL and out[0, 1] == 0
    c = o.shadow_read_counters()
    assert c["target_mismatch_lanes"] == 32 and c["token_mismatch_lanes"] == 0 and c["blocked_lanes"] == 32


def test_the_depth_field_of_the_header_is_ignored_and_inactive_lanes_keep_their_state():
    o = make()
    o.shadow_push(ev(0, 0x0000FFFF, 1, depth_field=5), vals(0x10), DET)
    assert o.shadow_depth(1, 0) == 1 and o.shadow_depth(1, 16) == 0
    out = o.shadow_check_ret(ev(0, 0x00FF00FF, 1, depth_field=2), vals(0x10), DET)
    assert out[0, 0] == 0x00FF0000 and out[0, 1] == 0x00FF00FF  # lanes 16-23 never called: underflow; detect releases
    assert o.shadow_depth(1, 0) == 0 and o.shadow_depth(1, 8) == 1 and o.shadow_depth(1, 16) == 0
    assert o.shadow_read_counters()["underflow_lanes"] == 8


def test_token_formula_a_reforged_entry_verifies():
    """Entry (site 4, value A) at depth 1 of thread slot (5, lane 9), epoch 3.  XOR-ing expected_return with A^B and
    the token with MAC(A)^MAC(B) under context (epoch<<48 | depth<<37 | slot<<5 | lane) must give a valid entry for
    B: pins which fields the token binds and how the context word is packed (oracle.mac is pinned by OpenSSL)."""
    o = make()
    A, B, slot, lane, epoch = 0x7F5A40001230, 0x7F5A4000BEE0, 5, 9, 3
    o.shadow_push(ev(0, FULL, slot, epoch), vals(0x111), ENF)   # depth 0
    o.shadow_push(ev(4, FULL, slot, epoch), vals(A), ENF)       # depth 1
    ctx = (epoch << 48) | (1 << 37) | (slot << 5) | lane
    o.shadow_poke(slot, lane, 1, oracle.POKE_EXPECTED, A ^ B)
    o.shadow_poke(slot, lane, 1, oracle.POKE_TOKEN, oracle.mac(K0, K1, 4, A, ctx) ^ oracle.mac(K0, K1, 4, B, ctx))
    v = vals(A)
    v[0, lane] = B
    assert o.shadow_check_ret(ev(4, FULL, slot, epoch), v, ENF)[0, 0] == 0
    # the same forgery computed for a neighbouring lane, slot, depth, epoch or site does not verify
    for d_lane, d_slot, d_depth, d_epoch, d_site in ((1, 0, 0, 0, 0), (0, 1, 0, 0, 0), (0, 0, 1, 0, 0), (0, 0, 0, 1, 0), (0, 0, 0, 0, 1)):
        o2 = make()
        o2.shadow_push(ev(0, FULL, slot, epoch), vals(0x111), ENF)
        o2.shadow_push(ev(4, FULL, slot, epoch), vals(A), ENF)
        wrong = ((epoch + d_epoch) << 48) | ((1 + d_depth) << 37) | ((slot + d_slot) << 5) | (lane + d_lane)
        site = 4 - 3 * d_site  # site 1 is a return site too
        o2.shadow_poke(slot, lane, 1, oracle.POKE_EXPECTED, A ^ B)
        o2.shadow_poke(slot, lane, 1, oracle.POKE_TOKEN, oracle.mac(K0, K1, 4, A, ctx) ^ oracle.mac(K0, K1, site, B, wrong))
        assert o2.shadow_check_ret(ev(4, FULL, slot, epoch), v, ENF)[0, 0] == 1 << lane
        assert o2.shadow_read_counters()["token_mismatch_lanes"] == 1


def test_every_corruption_of_the_writable_shadow_memory_is_caught_on_its_lane_only():
    for field, cause in ((oracle.POKE_EXPECTED, "token_mismatch_lanes"), (oracle.POKE_TOKEN, "token_mismatch_lanes"),
                         (oracle.POKE_CALLSITE, "token_mismatch_lanes"), (oracle.POKE_ENTRY_DEPTH, "depth_mismatch_lanes")):
        for bit in (0, 17, 31) if field in (oracle.POKE_CALLSITE, oracle.POKE_ENTRY_DEPTH) else (0, 33, 63):
            o = make()
            o.shadow_push(ev(0, FULL, 2), vals(0x40), ENF)
            o.shadow_poke(2, 13, 0, field, 1 << bit)
            out = o.shadow_check_ret(ev(0, FULL, 2), vals(0x40), ENF)
            assert out[0, 0] == 1 << 13 and out[0, 1] == FULL & ~(1 << 13)
            c = o.shadow_read_counters()
            assert c[cause] == 1 and c["viol_lanes"] == 1 and c["viol_events"] == 1
    # hijacked continuation: record intact, observed value differs
    o = make()
    o.shadow_push(ev(0, FULL, 2), vals(0x40), ENF)
    v = vals(0x40)
    v[0, 4] ^= np.uint64(0x10)
    assert o.shadow_check_ret(ev(0, FULL, 2), v, ENF)[0, 0] == 1 << 4
    assert o.shadow_read_counters()["target_mismatch_lanes"] == 1
    # depth counter pushed up by the attacker: the next return reads a never-written entry
    o = make()
    o.shadow_push(ev(0, FULL, 2), vals(0x40), ENF)
    o.shadow_poke(2, 6, 0, oracle.POKE_DEPTH_COUNTER, 1 ^ 3)  # depth 1 -> 3
    out = o.shadow_check_ret(ev(0, FULL, 2), vals(0x40), ENF)
    assert out[0, 0] == 1 << 6 and o.shadow_read_counters()["depth_mismatch_lanes"] == 1
    # ... or far past the bounded array: no such entry, still a depth mismatch, and a push there overflows
    o = make(max_depth=4)
    o.shadow_push(ev(0, FULL, 2), vals(0x40), ENF)
    o.shadow_poke(2, 6, 0, oracle.POKE_DEPTH_COUNTER, 1 ^ 0x80000000)
    assert o.shadow_push(ev(0, 1 << 6, 2), vals(0x41), ENF)[0, 0] == 1 << 6
    out = o.shadow_check_ret(ev(0, FULL, 2), vals(0x40), ENF)
    c = o.shadow_read_counters()
    assert out[0, 0] == 1 << 6 and c["depth_mismatch_lanes"] == 1 and c["overflow_lanes"] == 1


def test_replay_across_epochs_fails():
    o = make()
    o.shadow_push(ev(0, FULL, 1, epoch=7), vals(0x99), ENF)
    out = o.shadow_check_ret(ev(0, FULL, 1, epoch=8), vals(0x99), ENF)
    assert out[0, 0] == FULL and o.shadow_read_counters()["token_mismatch_lanes"] == 32


def test_overflow_underflow_fail_closed_without_wrapping():
    o = make(max_depth=3)
    for i in range(3):
        assert o.shadow_push(ev(0, 0xF, 0), vals(0x100 + i), ENF)[0, 0] == 0
    out = o.shadow_push(ev(0, 0xFF, 0), vals(0x200), ENF)
    assert out[0, 0] == 0xF and out[0, 1] == 0xF0                       # lanes 0-3 are full, lanes 4-7 push
    assert o.shadow_depth(0, 0) == 3 and o.shadow_depth(0, 4) == 1
    assert o.shadow_read_counters()["overflow_lanes"] == 4
    for i in (2, 1, 0):                                                  # the three real frames are intact
        assert o.shadow_check_ret(ev(0, 0xF, 0), vals(0x100 + i), ENF)[0, 0] == 0
    assert o.shadow_check_ret(ev(0, 0xF, 0), vals(0x100), ENF)[0, 0] == 0xF  # a fourth return underflows
    assert o.shadow_depth(0, 0) == 0


def test_event_level_failures_touch_no_state():
    o = make(n_slots=4)
    o.shadow_push(ev(0, FULL, 1), vals(0x40), ENF)
    hdr = np.concatenate([ev(2, 0xF, 1), ev(3, 0xF, 1), ev(99, 0xF, 1), ev(0, 0xF, 4), ev(0, 0xF, 0xFFFFFFFF), ev(0, 0, 2)])
    # each of these alone: forward site, fixed-edge site, unknown site, slot == n_slots, huge slot, empty mask
    for i in range(len(hdr)):
        out = o.shadow_push(hdr[i:i + 1], vals(0x1), ENF)
        assert out[0, 0] == (0xF if i < 5 else 0)
        out = o.shadow_check_ret(hdr[i:i + 1], vals(0x1), DET)
        assert out[0, 0] == (0xF if i < 5 else 0) and out[0, 1] == (0xF if i < 5 else 0)
    c = o.shadow_read_counters()
    assert c["non_return_events"] == 6 and c["slot_overflow_events"] == 4 and c["empty_events"] == 2
    assert o.shadow_depth(1, 0) == 1 and o.shadow_depth(2, 0) == 0
    # slot conflict: warp slot 1 twice in one call -> both fail closed, slot 3 proceeds
    hdr = np.concatenate([ev(0, FULL, 1), ev(0, FULL, 3), ev(1, 0xFF, 1)])
    out = o.shadow_push(hdr, np.full((3, 32), 0x70, dtype=np.uint64), ENF)
    assert out[:, 0].tolist() == [FULL, 0, 0xFF]
    assert o.shadow_depth(1, 0) == 1 and o.shadow_depth(3, 0) == 1
    assert o.shadow_read_counters()["slot_conflict_events"] == 2
    assert o.shadow_check_ret(ev(0, FULL, 1), vals(0x40), ENF)[0, 0] == 0  # the frame pushed before is untouched


def test_random_call_return_sequences_against_a_mac_free_model():
    """Untampered runs: violations can only come from the stack discipline (underflow, overflow, returning to
    something else than what was pushed).  A list per thread slot predicts them without computing any MAC."""
    rng = np.random.default_rng(11)
    n_slots, max_depth = 16, 3
    o = make(n_slots, max_depth)
    model = {}
    exp_c = dict(overflow=0, underflow=0, target=0, viol_lanes=0, viol_events=0)
    for step in range(300):
        push = rng.random() < 0.55
        slots = rng.permutation(n_slots)[: rng.integers(1, n_slots + 1)]   # distinct warps per call
        n = len(slots)
        sites = rng.choice([0, 1, 4], n)
        masks = rng.integers(0, 1 << 32, n, dtype=np.uint64)
        hdr = mk_hdr(sites, masks, [ctx_base(1, int(s)) for s in slots])
        val = rng.integers(0, 4, size=(n, 32)).astype(np.uint64) + np.uint64(0x7F5A40000000)
        exp = np.zeros(n, dtype=np.uint32)
        for i in range(n):
            for lane in range(32):
                if not (int(masks[i]) >> lane) & 1:
                    continue
                st = model.setdefault((int(slots[i]), lane), [])
                if push:
                    if len(st) == max_depth:
                        exp[i] |= np.uint32(1 << lane); exp_c["overflow"] += 1
                    else:
                        st.append((int(sites[i]), int(val[i, lane])))
                else:
                    if not st:
                        exp[i] |= np.uint32(1 << lane); exp_c["underflow"] += 1
                    elif st.pop() != (int(sites[i]), int(val[i, lane])):
                        exp[i] |= np.uint32(1 << lane); exp_c["target"] += 1
        mode = int(rng.integers(0, 2))
        out = (o.shadow_push if push else o.shadow_check_ret)(hdr, val, mode)
        assert np.array_equal(out[:, 0], exp), step
        act = masks.astype(np.uint32)
        assert np.array_equal(out[:, 1], act & ~exp if mode == ENF else act)
        exp_c["viol_lanes"] += int(popc(exp).sum()); exp_c["viol_events"] += int((exp != 0).sum())
    c = o.shadow_read_counters()
    assert (c["overflow_lanes"], c["underflow_lanes"], c["target_mismatch_lanes"]) == (exp_c["overflow"], exp_c["underflow"], exp_c["target"])
    assert c["token_mismatch_lanes"] == 0 and c["depth_mismatch_lanes"] == 0
    assert c["viol_lanes"] == exp_c["viol_lanes"] and c["viol_events"] == exp_c["viol_events"]
    assert exp_c["overflow"] > 0 and exp_c["underflow"] > 0 and exp_c["target"] > 0
    for (slot, lane), st in model.items():
        assert o.shadow_depth(slot, lane) == len(st)


def test_known_limit_a_popped_frame_replayed_in_the_same_epoch_at_the_same_depth_still_verifies():
    """DESIGN.md R41: the token binds (callsite, expected_return, epoch, depth, slot, lane) — PAPER.md:258
    "bind the expected return, callsite identifier, depth, logical thread slot, and key material; some helper profiles
    also bind a launch epoch" — and nothing that changes when a frame is popped.  The depth counter is ordinary
    (attacker-writable) memory, so a writer who bumps it back after a return makes the stale frame, whose bytes and
    valid token are still in the array, authenticate again: a return to a continuation that WAS legal for this thread
    slot at this depth in this epoch.  The paper's remedy is the epoch / monotonic counter the caller packs into
    context_base ("profiles may also bind a launch epoch or monotonic counter"): under a new epoch the
    same replay fails.  This test pins both halves so the limit cannot change silently."""
    A = 0x7F5A40000040
    for new_epoch, expect_viol in ((False, 0), (True, 1 << 9)):
        o = make()
        o.shadow_push(ev(0, FULL, 5, epoch=7), vals(A), ENF)
        assert o.shadow_check_ret(ev(0, FULL, 5, epoch=7), vals(A), ENF)[0, 0] == 0  # the legitimate return pops it
        assert o.shadow_depth(5, 9) == 0
        o.shadow_poke(5, 9, 0, oracle.POKE_DEPTH_COUNTER, 1)  # the attacker's write: depth counter 0 -> 1
        out = o.shadow_check_ret(ev(0, 1 << 9, 5, epoch=8 if new_epoch else 7), vals(A), ENF)
        assert out[0, 0] == expect_viol
        c = o.shadow_read_counters()
        assert c["token_mismatch_lanes"] == (1 if new_epoch else 0) and c["underflow_lanes"] == 0
