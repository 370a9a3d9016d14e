"""Parity of the stateful shadow stack (R30-R36): CUDA path through the C-ABI against
the oracle, verdict masks, counters and per-slot depths bit for bit, on random call / return sequences with every
fail-closed case and with the attacker's writes (wg_shadow_poke) mirrored on both sides."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests.util import mk_hdr, oracle_for

pytestmark = pytest.mark.gpu
DET, ENF = 0, 1


def dev():
    return torch.device("cuda", 0)


def to_dev(a):
    a = np.ascontiguousarray(a)
    return torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a).to(dev())


def pair(n_slots, max_depth, config=1):
    pol = S.make_policy(config, "cpu")
    orc, eng = oracle_for(pol), B.Engine(0).load(pol)
    orc.shadow_configure(n_slots, max_depth)
    eng.wg_shadow_configure(n_slots, max_depth)
    return pol, orc, eng


def step(orc, eng, push, hdr, val, mode):
    o = (orc.shadow_push if push else orc.shadow_check_ret)(hdr, val, mode)
    g = (eng.wg_shadow_push if push else eng.wg_shadow_check_ret)(to_dev(hdr), to_dev(val), mode)
    g = g.cpu().numpy().view(np.uint32)
    bad = np.nonzero((g != o).any(1))[0]
    assert bad.size == 0, (push, bad[:5], g[bad[:5]], o[bad[:5]])
    return o


def random_call(rng, pol, n_slots, n, *, slot_span=None, dup=0.0, bad_site=0.02):
    """n events of one lock-step call: distinct warp slots (a fraction `dup` repeated on purpose), mostly return
    sites, a few other / unknown sites, slots partly beyond n_slots, masks from empty to full."""
    span = slot_span or n_slots + n_slots // 8
    slots = rng.permutation(span)[:n].astype(np.uint64)
    k = int(dup * n)
    if k:
        slots[rng.integers(0, n, k)] = slots[rng.integers(0, n, k)]
    ret_sites = np.nonzero(pol.kind == 0)[0]
    sites = ret_sites[rng.integers(0, len(ret_sites), n)].astype(np.uint64)
    odd = rng.random(n) < bad_site
    sites[odd] = rng.choice(np.array([int(np.nonzero(pol.kind == 1)[0][0]), pol.n_sites + 5, 0xFFFFFFFF], dtype=np.uint64), int(odd.sum()))
    masks = rng.integers(0, 1 << 32, n, dtype=np.uint64)
    masks[rng.random(n) < 0.05] = 0
    masks[rng.random(n) < 0.3] = 0xFFFFFFFF
    epoch = np.uint64(3)
    ctx = (epoch << np.uint64(48)) | (rng.integers(0, 8, n, dtype=np.uint64) << np.uint64(37)) | (slots << np.uint64(5))
    return mk_hdr(sites, masks, ctx), slots


def same_state(orc, eng, rng, n_slots):
    assert eng.wg_shadow_read_counters() == orc.shadow_read_counters()
    for _ in range(40):
        s, l = int(rng.integers(0, n_slots)), int(rng.integers(0, 32))
        assert eng.wg_shadow_depth(s, l) == orc.shadow_depth(s, l)


@pytest.mark.parametrize("n_slots,max_depth,n", [(4096, 4, 3000), (257, 1, 200), (50_000, 8, 40_003)])
def test_random_call_return_sequences(n_slots, max_depth, n):
    rng = np.random.default_rng(n_slots)
    pol, orc, eng = pair(n_slots, max_depth)
    pushed = []  # (hdr, val) of earlier pushes, to return to (mostly) the right continuations
    for it in range(14):
        push = rng.random() < 0.55 or not pushed
        hdr, slots = random_call(rng, pol, n_slots, n, dup=0.01 if it % 3 == 0 else 0.0)
        if push:
            val = rng.integers(0, 1 << 16, size=(n, 32)).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000)
            if rng.random() < 0.7:
                val[:] = val[:, :1]  # warp-uniform continuations
            pushed.append((hdr, val))
        else:
            hdr, val = pushed.pop()  # the matching returns ...
            val = val.copy()
            flip = rng.random(n) < 0.01
            val[flip, rng.integers(0, 32, int(flip.sum()))] ^= np.uint64(0x40)  # ... some hijacked
            keep = rng.random(n) < 0.95
            hdr, val = hdr[keep], val[keep]  # ... and some warps do not return in this step
        step(orc, eng, push, hdr, val, ENF if it % 2 else DET)
    same_state(orc, eng, rng, n_slots)
    c = orc.shadow_read_counters()
    assert c["target_mismatch_lanes"] > 0 and c["slot_overflow_events"] > 0 and c["non_return_events"] > 0
    assert c["slot_conflict_events"] > 0 and c["empty_events"] > 0 and c["token_mismatch_lanes"] == 0
    eng.close()


@pytest.mark.parametrize("n", [1, 2, 3, 7, 33])
def test_calls_shorter_than_the_kernels_pipeline(n):
    """The shadow kernels keep three events in flight per warp: calls with fewer events than that (and than one
    block's warps) must still match the oracle, push then return, twice over."""
    rng = np.random.default_rng(100 + n)
    pol, orc, eng = pair(64, 2)
    for rnd in range(3):  # the third push overflows the depth-2 stacks
        hdr, _ = random_call(rng, pol, 64, n, slot_span=64, bad_site=0.0)
        val = rng.integers(0, 1 << 16, size=(n, 32)).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000)
        step(orc, eng, True, hdr, val, ENF)
        if rnd == 1:
            val = val.copy()
            val[0, 5] ^= np.uint64(0x10)
            step(orc, eng, False, hdr, val, DET)
    same_state(orc, eng, rng, 64)
    eng.close()


def test_attacker_writes_and_replay_are_caught_like_the_oracle_says():
    rng = np.random.default_rng(5)
    n_slots, max_depth, n = 1024, 4, 900
    pol, orc, eng = pair(n_slots, max_depth)
    hdr, slots = random_call(rng, pol, n_slots, n, slot_span=n_slots, bad_site=0.0)
    hdr[:, 0] |= np.uint64(0xFFFFFFFF) << np.uint64(32)  # full masks: every thread slot has frames
    val = rng.integers(0, 1 << 40, size=(n, 32)).astype(np.uint64)
    step(orc, eng, True, hdr, val, ENF)
    step(orc, eng, True, hdr, val + np.uint64(16), ENF)
    for i in range(60):  # corrupt random fields of random entries, the same way on both sides
        s, l, d = int(slots[rng.integers(0, n)]), int(rng.integers(0, 32)), int(rng.integers(0, 2))
        field = int(rng.integers(0, 5))
        x = int(rng.integers(1, 1 << 31)) if field >= 2 else int(rng.integers(1, 1 << 63))
        if field == 4:
            x = int(rng.integers(1, 8))
        orc.shadow_poke(s, l, d, field, x)
        eng.wg_shadow_poke(s, l, d, field, x)
    o1 = step(orc, eng, False, hdr, val + np.uint64(16), ENF)
    # second return under another epoch: every surviving frame is a replay
    hdr2 = hdr.copy()
    hdr2[:, 1] += np.uint64(1) << np.uint64(48)
    o2 = step(orc, eng, False, hdr2, val, DET)
    same_state(orc, eng, rng, n_slots)
    c = orc.shadow_read_counters()
    assert o1[:, 0].any() and c["token_mismatch_lanes"] > 0 and c["depth_mismatch_lanes"] > 0
    assert (o2[:, 1] == 0xFFFFFFFF).all()  # detect mode releases
    eng.close()


def test_warp_uniform_returns_with_attacker_writes():
    """check_ret computes the MAC prefix of a warp-uniform return address once per event and falls
    back to the per-lane prefix when any MAC-computing lane's entry disagrees with the first active lane's observed
    value or with the event's site.  Uniform pushes, then every way of breaking that agreement — a hijacked first
    active lane, a hijacked other lane, poked expected_return / token / callsite / depth / depth counter, a replay
    under another epoch — against the oracle."""
    rng = np.random.default_rng(77)
    n_slots, max_depth, n = 2048, 3, 1500
    pol, orc, eng = pair(n_slots, max_depth)
    hdr, slots = random_call(rng, pol, n_slots, n, slot_span=n_slots, bad_site=0.0)
    val = np.repeat(rng.integers(0, 1 << 20, size=(n, 1)).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000), 32, 1)
    step(orc, eng, True, hdr, val, ENF)
    step(orc, eng, True, hdr, val + np.uint64(32), ENF)
    for i in range(200):
        s, l, d = int(slots[rng.integers(0, n)]), int(rng.integers(0, 32)), int(rng.integers(0, 2))
        field = int(rng.integers(0, 5))
        x = int(rng.integers(1, 1 << 31)) if field >= 2 else int(rng.integers(1, 1 << 63))
        if field == 4:
            x = int(rng.integers(1, 4))
        orc.shadow_poke(s, l, d, field, x)
        eng.wg_shadow_poke(s, l, d, field, x)
    obs = val + np.uint64(32)
    masks = (hdr[:, 0] >> np.uint64(32)).astype(np.uint64)
    first = np.array([(int(m) & -int(m)).bit_length() - 1 if m else 0 for m in masks])
    hij = rng.random(n) < 0.05
    obs[hij, first[hij]] ^= np.uint64(0x100)           # the first active lane returns somewhere else
    hij2 = rng.random(n) < 0.05
    obs[hij2, rng.integers(0, 32, int(hij2.sum()))] ^= np.uint64(0x80)  # some other lane does
    o1 = step(orc, eng, False, hdr, obs, ENF)
    hdr2 = hdr.copy()
    hdr2[:, 1] += np.uint64(1) << np.uint64(48)       # the older frames replayed under another epoch
    step(orc, eng, False, hdr2, val, DET)
    same_state(orc, eng, rng, n_slots)
    c = orc.shadow_read_counters()
    assert o1[:, 0].any() and c["token_mismatch_lanes"] > 0 and c["target_mismatch_lanes"] > 0
    assert c["depth_mismatch_lanes"] > 0
    eng.close()


def test_errors_and_reconfigure():
    pol, orc, eng = pair(8, 2)
    with pytest.raises(B.WgError):
        eng.wg_shadow_configure(8, 0)
    with pytest.raises(B.WgError):
        eng.wg_shadow_configure(8, 65)
    with pytest.raises(B.WgError):
        eng.wg_shadow_poke(8, 0, 0, 0, 1)
    hdr = mk_hdr([int(np.nonzero(pol.kind == 0)[0][0])], [0xF], [3 << 5])
    val = np.full((1, 32), 0x50, dtype=np.uint64)
    step(orc, eng, True, hdr, val, ENF)
    assert eng.wg_shadow_depth(3, 0) == 1
    eng.wg_shadow_configure(8, 2)   # reconfiguring zeroes the state and the counters
    orc.shadow_configure(8, 2)
    assert eng.wg_shadow_depth(3, 0) == 0 and eng.wg_shadow_read_counters() == orc.shadow_read_counters()
    step(orc, eng, False, hdr, val, ENF)  # underflow on both sides
    assert eng.wg_shadow_read_counters()["underflow_lanes"] == 4
    eng.close()


def test_known_limit_same_epoch_replay_of_a_popped_frame_matches_the_oracle():
    """DESIGN.md R41: a popped frame replayed by bumping the (attacker-writable) depth counter verifies again under the
    same epoch and fails under a new one; the engine and the oracle agree on both (pinned on the oracle side in
    tests/test_oracle_shadow.py)."""
    pol, orc, eng = pair(16, 4)
    site = int(np.nonzero(pol.kind == 0)[0][0])
    A = np.full((1, 32), 0x7F5A40000040, dtype=np.uint64)
    full = 0xFFFFFFFF

    def hdr(mask, epoch):
        return mk_hdr([site], [mask], [(epoch << 48) | (5 << 5)])

    step(orc, eng, True, hdr(full, 7), A, ENF)
    assert not step(orc, eng, False, hdr(full, 7), A, ENF)[0, 0]
    for lane, epoch, expect in ((9, 7, 0), (11, 8, 1 << 11)):
        orc.shadow_poke(5, lane, 0, oracle.POKE_DEPTH_COUNTER, 1)
        eng.wg_shadow_poke(5, lane, 0, 4, 1)
        assert step(orc, eng, False, hdr(1 << lane, epoch), A, ENF)[0, 0] == expect
    assert eng.wg_shadow_read_counters() == orc.shadow_read_counters()
    eng.close()
