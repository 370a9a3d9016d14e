"""Parity proper: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU oracle, element by
element and bit for bit, on the same seeded inputs (every output is an integer function of
(policy, key, events, mode, call order) — tolerance 0).  Sizes span many CTAs, several grid strides and a ragged
tail.  Run with ``-m gpu`` on the B200 box."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests import witness
from tests.util import mk_hdr, oracle_for

pytestmark = pytest.mark.gpu

DET, ENF = 0, 1
FULL = 0xFFFFFFFF
U64MAX = (1 << 64) - 1


def dev():
    return torch.device("cuda", 0)


def to_dev(a: np.ndarray) -> torch.Tensor:
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint64:
        a = a.view(np.int64)
    if a.dtype == np.uint32:
        a = a.view(np.int32)
    return torch.from_numpy(a).to(dev())


def engine_for(policy) -> B.Engine:
    return B.Engine(0).load(policy)


def assert_counters_equal(eng: B.Engine, orc: "oracle.Oracle"):
    gg, gs = eng.wg_read_counters()
    og, os_ = orc.read_counters()
    diff = {k: (gg[k], og[k]) for k in og if gg[k] != og[k]}
    assert not diff, f"global counters differ (gpu, oracle): {diff}"
    assert np.array_equal(gs, os_), f"per-site counters differ at sites {np.nonzero((gs != os_).any(1))[0][:10]}"


def run_config(config, n_events, mode=None, **kw):
    """Oracle and engine on one seeded stream: sign parity, then check parity, then counters."""
    st = S.make_stream(config, "cpu", n_events=n_events, mode=mode, **kw)
    pol = st.policy
    orc, eng = oracle_for(pol), engine_for(pol)
    hdr_np, val_push = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64).copy()
    d_hdr = st.hdr.to(dev())
    # sign: every tag bit-exact, zeros for inactive lanes and non-return sites
    o_tag = orc.sign(hdr_np, val_push)
    g_tag = eng.wg_sign_continuations(d_hdr, st.val.to(dev()))
    assert np.array_equal(g_tag.cpu().numpy().view(np.uint64), o_tag)
    # corrupt, then check
    tag_t = torch.from_numpy(o_tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    val_np, tag_np = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
    o_out = orc.verify(hdr_np, val_np, tag_np, st.mode)
    g_out = eng.wg_verify_continuations(d_hdr, st.val.to(dev()), tag_t.to(dev()), st.mode)
    g_out = g_out.cpu().numpy().view(np.uint32)
    bad = np.nonzero((g_out != o_out).any(1))[0]
    assert bad.size == 0, f"{bad.size} verdicts differ, first at event {bad[:5]}: gpu {g_out[bad[:5]]} oracle {o_out[bad[:5]]}"
    assert_counters_equal(eng, orc)
    return st, orc, eng, o_out


def test_config1_tiny_full_size_both_modes():
    for mode in (DET, ENF):
        st, orc, eng, out = run_config(1, None, mode=mode)
        assert np.array_equal(out[:, 0], witness.expected_viol(st))  # third, independent derivation
        assert out[:, 0].any()
        eng.close()


def test_config2_backward_only_ragged():
    st, orc, eng, out = run_config(2, 200_003)
    g, _ = eng.wg_read_counters()
    assert g["ret_checks"] > 0 and g["fwd_checks"] == 0 and g["ret_viol_events"] == len(st.ret_tamper)
    assert g["blocked_lanes"] == g["ret_viol"]


def test_config3_forward_only_ragged_detect():
    st, orc, eng, out = run_config(3, 300_001)
    g, _ = eng.wg_read_counters()
    assert g["fwd_checks"] > 0 and g["ret_checks"] == 0 and g["blocked_lanes"] == 0 and g["fwd_viol"] > 0
    assert (out[:, 1] == (st.hdr.numpy().view(np.uint64)[:, 0] >> np.uint64(32))).all()  # detect never blocks


def test_config4_mixed_paper_shaped():
    st, orc, eng, out = run_config(4, 400_007)
    assert np.array_equal(out[:, 0], witness.expected_viol(st))
    g, _ = eng.wg_read_counters()
    # only protected sites are in the denominator
    assert g["ret_checks"] + g["fwd_checks"] <= st.meta["n_ret"] + st.meta["n_fwd"]
    assert sum(g[f"events_by_kind_{k}"] for k in range(2, 7)) == st.meta["n_non"]


def test_config5_stress_alternating_modes_accumulate():
    pol = S.make_policy(5, "cpu", n_sites=20_000, max_set=4096)
    orc, eng = oracle_for(pol), engine_for(pol)
    orc.set_binary_search(True)  # proven equal to the linear scan in test_oracle_membership.py
    for b in range(3):
        st = S.make_stream(5, "cpu", n_events=60_001, policy=pol, batch_index=b)
        assert st.mode == (DET if b % 2 == 0 else ENF)
        hdr_np = st.hdr.numpy().view(np.uint64)
        o_tag = orc.sign(hdr_np, st.val.numpy().view(np.uint64))
        d_hdr = st.hdr.to(dev())
        g_tag = eng.wg_sign_continuations(d_hdr, st.val.to(dev()))
        assert np.array_equal(g_tag.cpu().numpy().view(np.uint64), o_tag)
        tag_t = torch.from_numpy(o_tag.view(np.int64).copy())
        st.apply_return_tamper(tag_t)
        o_out = orc.verify(hdr_np, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64), st.mode)
        g_out = eng.wg_verify_continuations(d_hdr, st.val.to(dev()), tag_t.to(dev()), st.mode)
        assert np.array_equal(g_out.cpu().numpy().view(np.uint32), o_out)
        assert np.array_equal(o_out[:, 0], witness.expected_viol(st))
    assert_counters_equal(eng, orc)  # counters and the event sequence run on across calls and modes


def test_forward_entry_point_matches_oracle_and_fails_closed_on_return_sites():
    st = S.make_stream(1, "cpu", n_events=50_001)
    orc, eng = oracle_for(st.policy), engine_for(st.policy)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    for mode in (DET, ENF):
        o_out = orc.check_forward(hdr_np, val_np, mode)
        g_out = eng.wg_check_forward(st.hdr.to(dev()), st.val.to(dev()), mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g_out, o_out)
    assert_counters_equal(eng, orc)
    g, _ = eng.wg_read_counters()
    assert g["events_misrouted"] > 0 and g["ret_checks"] == 0


def small_policy():
    kind = np.array([0, 0, 1, 1, 2, 3, 4, 5, 6], dtype=np.uint8)
    off = np.array([0, 0, 0, 3, 4, 4, 4, 4, 4, 4], dtype=np.uint32)
    tg = np.array([0x1000, 0x2000, 0x3000, 0x4000], dtype=np.uint64)
    return kind, off, tg


def small_pair(k0=0x1122334455667788, k1=0x99AABBCCDDEEFF00, digest=42):
    kind, off, tg = small_policy()
    eng = B.Engine(0)
    eng.wg_load_policy(kind, off, tg, k0, k1, digest)
    return oracle.Oracle(kind, off, tg, k0, k1, digest), eng


def test_edge_cases_unknown_site_empty_mask_every_kind_single_lanes():
    rng = np.random.default_rng(7)
    orc, eng = small_pair()
    sites = [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 1000, 0xFFFFFFFF, 0, 2, 5, 0, 0, 2, 3, 3]
    masks = [FULL, 1, FULL, 0x80000000, FULL, 5, 6, 7, 8, FULL, 0xF0, 1, 0, 0, 0, 0x80000001, 2, 0x10, FULL, 1]
    n = len(sites)
    hdr = mk_hdr(sites, masks, rng.integers(0, 1 << 64, n, dtype=np.uint64))
    val = rng.integers(0, 1 << 64, size=(n, 32), dtype=np.uint64)
    val[2, :] = 0x2000
    val[2, 5] = 0x2001          # one lane out of set
    val[3, 31] = 0x4000
    val[17, 4] = 0x3000
    val[18, :] = 0x4000
    val[18, 9] = 0x3000         # legal for site 2, not for site 3 (wrong-site-valid-target)
    val[19, 0] = 0
    o_tag = orc.sign(hdr, val)
    g_tag = eng.wg_sign_continuations(to_dev(hdr), to_dev(val)).cpu().numpy().view(np.uint64)
    assert np.array_equal(g_tag, o_tag)
    tag = o_tag.copy()
    tag[15, 31] ^= np.uint64(1 << 63)  # forged token in the last lane
    val[16, 1] ^= np.uint64(1)         # hijacked continuation in lane 1
    for mode in (DET, ENF):
        o = orc.verify(hdr, val, tag, mode)
        g = eng.wg_verify_continuations(to_dev(hdr), to_dev(val), to_dev(tag), mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o), (g, o)
        o = orc.check_forward(hdr, val, mode)
        g = eng.wg_check_forward(to_dev(hdr), to_dev(val), mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
    assert_counters_equal(eng, orc)
    g, _ = eng.wg_read_counters()
    assert g["events_unknown_site"] == 12 and g["events_empty"] == 12 and g["policy_digest"] == 42


def test_inactive_lanes_never_influence_any_output():
    rng = np.random.default_rng(8)
    orc, eng = small_pair()
    n = 4099
    hdr = mk_hdr(rng.integers(0, 9, n), rng.integers(0, 1 << 32, n), rng.integers(0, 1 << 64, n, dtype=np.uint64))
    val = rng.integers(0, 1 << 64, size=(n, 32), dtype=np.uint64)
    tag = orc.sign(hdr, val)
    a = eng.wg_verify_continuations(to_dev(hdr), to_dev(val), to_dev(tag), ENF).cpu()
    ca, sa = eng.wg_read_counters()
    inactive = ((hdr[:, 0:1] >> np.uint64(32)) >> np.arange(32, dtype=np.uint64)[None, :]) & np.uint64(1) == 0
    val2, tag2 = val.copy(), tag.copy()
    val2[inactive] = rng.integers(0, 1 << 64, size=int(inactive.sum()), dtype=np.uint64)
    tag2[inactive] = rng.integers(0, 1 << 64, size=int(inactive.sum()), dtype=np.uint64)
    eng.wg_reset_counters()
    b = eng.wg_verify_continuations(to_dev(hdr), to_dev(val2), to_dev(tag2), ENF).cpu()
    cb, sb = eng.wg_read_counters()
    assert torch.equal(a, b) and ca == cb and np.array_equal(sa, sb)


def test_first_violation_key_is_the_smallest_seq_lane_across_calls_and_resets():
    orc, eng = small_pair()
    rng = np.random.default_rng(9)
    n = 70_001
    hdr = mk_hdr(np.zeros(n, dtype=np.int64), np.full(n, FULL), np.full(n, 0x40))
    val = rng.integers(0, 1 << 64, size=(n, 32), dtype=np.uint64)
    tag = orc.sign(hdr, val)
    d_hdr, d_val = to_dev(hdr), to_dev(val)
    eng.wg_verify_continuations(d_hdr, d_val, to_dev(tag), DET)       # clean call: seq advances by n
    assert eng.wg_read_counters()[0]["first_violation_key"] == U64MAX
    bad = tag.copy()
    for e, lane in ((69_999, 0), (40_000, 17), (40_000, 30), (55_555, 3)):
        bad[e, lane] ^= np.uint64(2)
    eng.wg_verify_continuations(d_hdr, d_val, to_dev(bad), ENF)
    orc.verify(hdr, val, tag, DET)
    orc.verify(hdr, val, bad, ENF)
    g, _ = eng.wg_read_counters()
    assert g["first_violation_key"] == ((n + 40_000) << 5 | 17) == orc.read_counters()[0]["first_violation_key"]
    assert g["last_mode"] == ENF
    eng.wg_reset_counters()
    eng.wg_verify_continuations(d_hdr, d_val, to_dev(bad), DET)
    g, _ = eng.wg_read_counters()
    assert g["first_violation_key"] == (40_000 << 5 | 17) and g["blocked_lanes"] == 0


def test_n_zero_is_a_noop_and_errors_are_status_codes():
    orc, eng = small_pair()
    z_hdr = torch.zeros((0, 2), dtype=torch.int64, device=dev())
    z_val = torch.zeros((0, 32), dtype=torch.int64, device=dev())
    eng.wg_sign_continuations(z_hdr, z_val)
    eng.wg_verify_continuations(z_hdr, z_val, z_val, ENF)
    eng.wg_check_forward(z_hdr, z_val, ENF)
    g, _ = eng.wg_read_counters()
    assert g["events_total"] == 0 and g["last_mode"] == 0
    hdr = to_dev(mk_hdr([0], [FULL], [0]))
    val = torch.zeros((1, 32), dtype=torch.int64, device=dev())
    with pytest.raises(B.WgError) as ei:
        eng.wg_verify_continuations(hdr, val, val, 2)
    assert ei.value.status == B.WG_ERR_INVALID_ARG
    with pytest.raises(B.WgError) as ei:  # misaligned value pointer
        eng.wg_check_forward(hdr, torch.zeros(33, dtype=torch.int64, device=dev())[1:].view(1, 32), DET)
    assert ei.value.status == B.WG_ERR_INVALID_ARG
    with pytest.raises(B.WgError) as ei:
        B.Engine(0).wg_check_forward(hdr, val, DET)
    assert ei.value.status == B.WG_ERR_NO_POLICY


@pytest.mark.parametrize("mutate,why", [
    (lambda k, o, t: k.__setitem__(4, 7), "kind >= 7"),
    (lambda k, o, t: o.__setitem__(0, 1), "tgt_off[0] != 0"),
    (lambda k, o, t: o.__setitem__(3, 5), "offsets decrease"),
    (lambda k, o, t: t.__setitem__(1, 0x1000), "duplicate target"),
    (lambda k, o, t: t.__setitem__(2, 0x1800), "unsorted set"),
    (lambda k, o, t: k.__setitem__(0, 1), "forward site with no targets"),
    (lambda k, o, t: k.__setitem__(3, 0), "return site owning targets"),
])
def test_bad_policy_loads_nothing_and_keeps_the_previous_one(mutate, why):
    orc, eng = small_pair()
    kind, off, tg = small_policy()
    mutate(kind, off, tg)
    assert oracle.validate_policy(kind, off, tg) != 0, why
    with pytest.raises(B.WgError) as ei:
        eng.wg_load_policy(kind, off, tg, 1, 2, 3)
    assert ei.value.status == B.WG_ERR_BAD_POLICY
    fresh = B.Engine(0)
    with pytest.raises(B.WgError):
        fresh.wg_load_policy(kind, off, tg, 1, 2, 3)
    assert not fresh._h  # nothing was created
    # the engine still answers with its previous policy and key
    hdr = mk_hdr([2, 0], [FULL, FULL], [0, 0])
    val = np.full((2, 32), 0x3000, dtype=np.uint64)
    tag = orc.sign(hdr, val)
    g = eng.wg_verify_continuations(to_dev(hdr), to_dev(val), to_dev(tag), ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, orc.verify(hdr, val, tag, ENF)) and (g[:, 0] == 0).all()
    assert eng.wg_read_counters()[0]["policy_digest"] == 42


def test_replacing_the_policy_resets_counters_and_rekeys():
    orc, eng = small_pair()
    hdr = mk_hdr([0], [FULL], [0x20])
    val = np.arange(32, dtype=np.uint64).reshape(1, 32)
    t1 = eng.wg_sign_continuations(to_dev(hdr), to_dev(val)).cpu().numpy().view(np.uint64)
    eng.wg_verify_continuations(to_dev(hdr), to_dev(val), to_dev(t1), ENF)
    kind, off, tg = small_policy()
    eng.wg_load_policy(kind, off, tg, 5, 6, 7)
    g, s = eng.wg_read_counters()
    assert g["events_total"] == 0 and g["signed_lanes"] == 0 and g["policy_digest"] == 7 and not s.any()
    out = eng.wg_verify_continuations(to_dev(hdr), to_dev(val), to_dev(t1), ENF).cpu().numpy().view(np.uint32)
    assert out[0, 0] == FULL and out[0, 1] == 0  # tags of the old key no longer verify (wrong key)
    o2 = oracle.Oracle(kind, off, tg, 5, 6, 7)
    assert np.array_equal(o2.verify(hdr, val, t1, ENF), out)


def test_host_buffer_entry_points_equal_the_device_ones():
    st = S.make_stream(4, "cpu", n_events=600_011)  # > 2 staging chunks of 256 Ki events, ragged
    orc, eng = oracle_for(st.policy), engine_for(st.policy)
    hdr_np = st.hdr.numpy().view(np.uint64)
    h_hdr, h_val = st.hdr.pin_memory(), st.val.pin_memory()
    g_tag = eng.wg_sign_continuations_host(h_hdr, h_val)
    o_tag = orc.sign(hdr_np, st.val.numpy().view(np.uint64))
    assert np.array_equal(g_tag.numpy().view(np.uint64), o_tag)
    st.apply_return_tamper(g_tag)
    h_val = st.val.pin_memory()
    o_out = orc.verify(hdr_np, st.val.numpy().view(np.uint64), g_tag.numpy().view(np.uint64), ENF)
    g_out = eng.wg_verify_continuations_host(h_hdr, h_val, g_tag, ENF)
    assert np.array_equal(g_out.numpy().view(np.uint32), o_out)
    o_f = orc.check_forward(hdr_np, st.val.numpy().view(np.uint64), DET)
    g_f = eng.wg_check_forward_host(h_hdr, h_val, DET)  # pageable or pinned both work
    assert np.array_equal(g_f.numpy().view(np.uint32), o_f)
    assert_counters_equal(eng, orc)


def test_work_runs_on_the_callers_stream():
    st = S.make_stream(2, "cpu", n_events=100_000)
    orc, eng = oracle_for(st.policy), engine_for(st.policy)
    s = torch.cuda.Stream()
    d_hdr, d_val = st.hdr.to(dev()), st.val.to(dev())
    torch.cuda.synchronize()
    before = eng.wg_kernel_launches()
    with torch.cuda.stream(s):
        tag = eng.wg_sign_continuations(d_hdr, d_val)
        out = eng.wg_verify_continuations(d_hdr, d_val, tag, ENF)
    s.synchronize()
    assert eng.wg_kernel_launches() - before == 3  # sign; check + its one-thread first-violation-record kernel
    assert not out[:, 0].any()
    assert np.array_equal(tag.cpu().numpy().view(np.uint64), orc.sign(st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)))


# ---------------------------------------------------------------------------------------------------------
# tile structure of the v2 kernels: every ragged length around the 16-event tile and the 20-warp CTA
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 15, 16, 17, 31, 32, 33, 319, 320, 321, 16 * 20 * 148 - 1, 16 * 20 * 148 + 17])
def test_ragged_lengths_around_tile_and_grid_boundaries(n):
    st = S.make_stream(4, "cpu", n_events=n)
    run = run_config(4, n)
    run[2].close()
    # the forward entry point walks the same tiles without tag rows
    orc, eng = oracle_for(st.policy), engine_for(st.policy)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    o = orc.check_forward(hdr_np, val_np, ENF)
    g = eng.wg_check_forward(st.hdr.to(dev()), st.val.to(dev()), ENF).cpu().numpy().view(np.uint32)
    assert np.array_equal(g, o)
    assert_counters_equal(eng, orc)
    eng.close()


def test_wrong_key_on_a_small_policy_counts_in_shared_memory():
    """Same attack on config 1's 72-site policy: per-site counters (violations and blocked lanes included) take the
    shared-memory path of the kernel; every counter must still equal the oracle's."""
    st = S.make_stream(1, "cpu", n_events=30_011)
    pol = st.policy
    orc, eng = oracle_for(pol), engine_for(pol)
    other = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1 ^ (1 << 63), pol.policy_digest)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    tag = other.sign(hdr_np, val_np)
    for mode in (ENF, DET, ENF):
        o = orc.verify(hdr_np, val_np, tag, mode)
        g = eng.wg_verify_continuations(st.hdr.to(dev()), st.val.to(dev()), to_dev(tag), mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
    assert_counters_equal(eng, orc)
    _, gs = eng.wg_read_counters()
    assert gs[:, 3].sum() > 0 and gs[:, 2].sum() > gs[:, 3].sum()  # blocked only in the two enforce passes
    eng.close()


def test_every_lane_violates_under_the_wrong_key():
    """Tags signed under another key: every active lane of every return event must be blocked (the violation
    path of the kernels is normally rare; here it runs on every tile)."""
    st = S.make_stream(2, "cpu", n_events=40_003)
    pol = st.policy
    orc, eng = oracle_for(pol), engine_for(pol)
    other = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0 ^ 1, pol.k1, pol.policy_digest)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    tag = other.sign(hdr_np, val_np)
    for mode in (ENF, DET):
        o = orc.verify(hdr_np, val_np, tag, mode)
        g = eng.wg_verify_continuations(st.hdr.to(dev()), st.val.to(dev()), to_dev(tag), mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
        assert (o[:, 0] == (hdr_np[:, 0] >> np.uint64(32)).astype(np.uint32)).all()  # viol == active everywhere
    assert_counters_equal(eng, orc)
    g, _ = eng.wg_read_counters()
    first = int(np.nonzero(hdr_np[:, 0] >> np.uint64(32))[0][0])           # first event with an active lane
    mask = int(hdr_np[first, 0] >> np.uint64(32))
    assert g["first_violation_key"] == (first << 5) | ((mask & -mask).bit_length() - 1)
    eng.close()


@pytest.mark.parametrize("config", [6, 7])
def test_public_code_shaped_streams(config):
    """a 38-target family at one indirect site and a wrong-callback burst that
    records 64 forward-violation checks — shapes only."""
    st, orc, eng, out = run_config(config, None)
    assert np.array_equal(out[:, 0], witness.expected_viol(st))
    g, _ = eng.wg_read_counters()
    if config == 6:
        sizes = np.diff(st.policy.tgt_off.astype(np.int64))
        assert sizes.max() == 38 and (sizes > 0).sum() == 1 and g["fwd_viol_events"] == len(st.fwd_tamper) > 50
    else:
        b0 = st.meta["burst_start"]
        assert g["fwd_viol_events"] == S.BURST_CHECKS == 64 and g["ret_viol"] == 0
        assert out[b0:b0 + 64, 0].all() and not out[:b0, 0].any() and not out[b0 + 64:, 0].any()
        assert (out[b0:b0 + 64, 1] == 0).all()                      # enforce: the whole burst is blocked
        assert g["first_violation_key"] >> 5 == b0
    eng.close()


def test_two_engines_on_two_streams_share_no_state():
    """Two engines (different policies, keys, modes) fed from two streams with no synchronisation in between: each
    one's verdicts and accumulated counters are the oracle's, i.e. nothing in the library is process-global."""
    st_a, st_b = S.make_stream(2, "cpu", n_events=200_003), S.make_stream(3, "cpu", n_events=150_001)
    orc_a, eng_a = oracle_for(st_a.policy), engine_for(st_a.policy)
    orc_b, eng_b = oracle_for(st_b.policy), engine_for(st_b.policy)
    hdr_a, val_a = st_a.hdr.numpy().view(np.uint64), st_a.val.numpy().view(np.uint64)
    hdr_b, val_b = st_b.hdr.numpy().view(np.uint64), st_b.val.numpy().view(np.uint64)
    tag_a = oracle_for(st_a.policy).sign(hdr_a, val_a)  # a second oracle: signing counts, and eng_a signs nothing
    tag_t = torch.from_numpy(tag_a.view(np.int64).copy())
    st_a.apply_return_tamper(tag_t)
    tag_a = tag_t.numpy().view(np.uint64)
    d = [t.to(dev()) for t in (st_a.hdr, st_a.val, tag_t, st_b.hdr, st_b.val)]
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for it in range(4):
        outs.append((eng_a.wg_verify_continuations(d[0], d[1], d[2], ENF if it % 2 else DET, stream=s1),
                     eng_b.wg_check_forward(d[3], d[4], DET if it % 2 else ENF, stream=s2)))
    torch.cuda.synchronize()
    for it, (ga, gb) in enumerate(outs):
        oa = orc_a.verify(hdr_a, val_a, tag_a, ENF if it % 2 else DET)
        ob = orc_b.check_forward(hdr_b, val_b, DET if it % 2 else ENF)
        assert np.array_equal(ga.cpu().numpy().view(np.uint32), oa)
        assert np.array_equal(gb.cpu().numpy().view(np.uint32), ob)
    assert_counters_equal(eng_a, orc_a)
    assert_counters_equal(eng_b, orc_b)
    eng_a.close()
    eng_b.close()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs")
def test_reloading_an_engine_onto_another_device_moves_everything_it_owns():
    """a reload onto a different device once freed only the staging buffers, leaving the
    first-violation record, the ring and the shadow arrays on the old device.  Now the engine is moved whole: tables,
    record and ring are re-created on the new device, the shadow state is dropped."""
    st = S.make_stream(4, "cpu", n_events=50_003)
    orc = oracle_for(st.policy)
    hdr, val = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    tag_t = torch.from_numpy(orc.sign(hdr, val).view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    orc.reset_counters()
    orc.set_ring_capacity(4096)
    eng = B.Engine(0).load(st.policy)
    eng.wg_set_ring_capacity(4096)
    eng.wg_shadow_configure(64, 2)
    d0 = torch.device("cuda", 0)
    eng.wg_verify_continuations(st.hdr.to(d0), st.val.to(d0), tag_t.to(d0), ENF)
    eng.device = 1
    eng.load(st.policy)  # same handle, other device: counters restart
    d1 = torch.device("cuda", 1)
    with torch.cuda.device(1):
        out = eng.wg_verify_continuations(st.hdr.to(d1), st.val.to(d1), tag_t.to(d1), ENF).cpu().numpy().view(np.uint32)
        assert np.array_equal(out, orc.verify(hdr, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64), ENF))
        assert_counters_equal(eng, orc)
        t, first, ring = eng.wg_read_telemetry(4096)
        assert first is not None and len(ring) == t["ring_recorded"] > 0
        with pytest.raises(B.WgError):  # the shadow state did not move: it has to be configured again
            eng.wg_shadow_read_counters()
    eng.close()


@pytest.mark.parametrize("n_big", [8, 3000])
def test_a_target_equal_to_the_all_ones_word_is_an_ordinary_member(n_big):
    """Degenerate case of the large-policy encoding: the hash index of the target sets (wg_check.cu) marks a free slot
    with the all-ones word, so a set that CONTAINS 0xFFFF_FFFF_FFFF_FFFF cannot store it and carries a flag instead.
    Membership must still be exactly the set's: all-ones is allowed at the site that lists it and
    nowhere else, as a warp-uniform target and as one lane's target, before and after wg_policy_poke rewrites that
    element (the index is rebuilt, the flag follows).  n_big = 8: the staged table (no hash index); 3000: the hash
    index (more than 2,048 targets)."""
    rng = np.random.default_rng(77 + n_big)
    # sites: 0 return, 1 forward with all-ones as its last element, 2 forward without, 3 forward with one element
    base = np.uint64(0x7F5A40000000)
    set1 = np.concatenate([np.sort(rng.choice(1 << 20, n_big, replace=False).astype(np.uint64)) * np.uint64(16) + base,
                           np.array([U64MAX], dtype=np.uint64)])
    set2 = np.sort(rng.choice(1 << 20, 5, replace=False).astype(np.uint64)) * np.uint64(16) + base + np.uint64(8)
    set3 = np.array([0x1234], dtype=np.uint64)
    kind = np.array([0, 1, 1, 1], dtype=np.uint8)
    off = np.array([0, 0, len(set1), len(set1) + len(set2), len(set1) + len(set2) + 1], dtype=np.uint32)
    tg = np.concatenate([set1, set2, set3])
    k0, k1 = 0x0123456789ABCDEF, 0x0FEDCBA987654321
    orc = oracle.Oracle(kind, off, tg, k0, k1, 5)
    eng = B.Engine(0)
    eng.wg_load_policy(kind, off, tg, k0, k1, 5)

    n = 4096 + 7
    site = rng.integers(1, 4, n).astype(np.uint64)
    mask = rng.integers(1, 1 << 32, n, dtype=np.uint64)
    ctx = rng.integers(0, 1 << 63, n, dtype=np.uint64)
    val = np.empty((n, 32), dtype=np.uint64)
    sets = {1: set1, 2: set2, 3: set3}
    for e in range(n):
        members = sets[int(site[e])]
        val[e, :] = members[rng.integers(0, len(members))] if rng.random() < 0.5 else members[rng.integers(0, len(members), 32)]
        r = rng.random()
        if r < 0.3:
            val[e, :] = U64MAX              # warp-uniform all-ones: legal at site 1 only
        elif r < 0.6:
            val[e, rng.integers(0, 32)] = U64MAX  # one lane all-ones
    hdr = mk_hdr(site, mask, ctx)
    d_hdr, d_val = to_dev(hdr), to_dev(val)

    def compare():
        for mode in (DET, ENF):
            o = orc.check_forward(hdr, val, mode)
            g = eng.wg_check_forward(d_hdr, d_val, mode).cpu().numpy().view(np.uint32)
            bad = np.nonzero((g != o).any(1))[0]
            assert bad.size == 0, (mode, bad[:5], g[bad[:5]], o[bad[:5]], site[bad[:5]])
        return o

    o = compare()
    at1 = (site == 1) & (val == U64MAX).all(1)
    assert at1.any() and not o[at1, 0].any(), "all-ones is a member of site 1's set"
    at2 = (site != 1) & (val == U64MAX).all(1)
    assert at2.any() and (o[at2, 0] == (mask[at2] & np.uint64(FULL)).astype(np.uint32)).all(), "and of no other set"
    # the attacker-write hook turns the all-ones element into another address (still ascending) and back
    idx = len(set1) - 1
    x = int(U64MAX) ^ int(set1[-2] + np.uint64(1))
    for _ in range(2):
        orc.policy_poke(0, idx, x)
        eng.wg_policy_poke(0, idx, x)
        compare()
    assert_counters_equal(eng, orc)
    eng.close()


def test_a_policy_without_sites_fails_every_event_closed():
    """Degenerate policy: no site at all (what the policy does not list is not authorised).  Every event
    names an unknown site: verify and the forward entry point fail its active lanes closed (R13), sign writes zero rows,
    nothing enters a protected-site denominator, and the per-site array is empty."""
    kind, off, tg = np.zeros(0, dtype=np.uint8), np.zeros(1, dtype=np.uint32), np.zeros(0, dtype=np.uint64)
    orc = oracle.Oracle(kind, off, tg, 11, 12, 13)
    eng = B.Engine(0)
    eng.wg_load_policy(kind, off, tg, 11, 12, 13)
    rng = np.random.default_rng(3)
    n = 20 * 32 * 5 + 3
    site = rng.choice(np.array([0, 1, 7, 0xFFFFFFFF], dtype=np.uint64), n)
    mask = rng.integers(0, 1 << 32, n, dtype=np.uint64)
    mask[::7] = 0
    hdr = mk_hdr(site, mask, rng.integers(0, 1 << 63, n, dtype=np.uint64))
    val = rng.integers(0, 1 << 63, size=(n, 32), dtype=np.uint64)
    tag = rng.integers(0, 1 << 63, size=(n, 32), dtype=np.uint64)
    d_hdr, d_val, d_tag = to_dev(hdr), to_dev(val), to_dev(tag)
    g_tag = eng.wg_sign_continuations(d_hdr, d_val).cpu().numpy().view(np.uint64)
    assert np.array_equal(g_tag, orc.sign(hdr, val)) and not g_tag.any()
    for mode in (ENF, DET):
        o = orc.verify(hdr, val, tag, mode)
        g = eng.wg_verify_continuations(d_hdr, d_val, d_tag, mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o) and np.array_equal(g[:, 0], mask.astype(np.uint32))
        o = orc.check_forward(hdr, val, mode)
        g = eng.wg_check_forward(d_hdr, d_val, mode).cpu().numpy().view(np.uint32)
        assert np.array_equal(g, o)
    gg, gs = eng.wg_read_counters()
    og, os_ = orc.read_counters()
    assert gg == og and gs.shape == os_.shape == (0, 4)
    assert gg["ret_checks"] == gg["fwd_checks"] == 0 and gg["events_unknown_site"] == 4 * n
    eng.close()
