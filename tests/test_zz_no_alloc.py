"""wg_verify_continuations_static (include/warpguard.h, "allocation-free verify"): the verify kernel with its scratch
memory (group ticket, counter words, first-violation key, per-site counters) in the library's static device array.
Checked against the existing path, wg_verify_continuations + wg_read_counters on a second engine with the same
policy, bit for bit (verdicts, counters, per-site counters), on two calls in a row whose second is smaller, runs in the
other mode and therefore shows anything the first call left behind in the shared array.

Collected last on purpose (the name sorts after every other test file); runs alone or after the others."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S

pytestmark = pytest.mark.gpu

NOT_PER_CALL = ("policy_digest", "last_mode")  # documented as 0 in the static call's copy


def _existing_path(ref: B.Engine, st, tag, mode):
    ref.wg_reset_counters()
    out = ref.wg_verify_continuations(st.hdr, st.val, tag, mode)
    g, s = ref.wg_read_counters()
    return out, g, s


def test_static_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    dev = torch.device("cuda", 0)
    st1 = S.make_stream(4, dev, n_events=300_007)  # 51,621 sites (<= WG_STATIC_MAX_SITES), several tiles, ragged tail
    st2 = S.make_stream(4, dev, n_events=100_003, policy=st1.policy, batch_index=1)
    assert st1.policy.n_sites <= B.WG_STATIC_MAX_SITES
    eng = B.Engine(0).load(st1.policy)  # the engine the static calls go through
    ref = B.Engine(0).load(st1.policy)  # the existing path
    # everything the calls write is allocated here, by the caller, before the first call
    n_max = st1.hdr.shape[0]
    out_buf = torch.empty((n_max, 2), dtype=torch.int32, device=dev)
    cnt_buf = torch.empty(26, dtype=torch.int64, device=dev)
    site_buf = torch.empty((eng.n_sites, 4), dtype=torch.int64, device=dev)
    tags = []
    for st in (st1, st2):
        tag = ref.wg_sign_continuations(st.hdr, st.val)
        st.apply_return_tamper(tag)
        tags.append(tag)
    torch.cuda.synchronize()
    free_before = None
    for k, (st, tag, mode) in enumerate(((st1, tags[0], S.ENFORCE), (st2, tags[1], S.DETECT))):
        n = st.hdr.shape[0]
        want_out, want_g, want_s = _existing_path(ref, st, tag, mode)
        if k == 1:  # (the first call may load the module and resolves the array's address; the second does nothing new)
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info(0)[0]
        out_buf.fill_(-1)
        cnt_buf.fill_(-1)
        site_buf.fill_(-1)
        out, cnt, site = eng.wg_verify_continuations_static(st.hdr, st.val, tag, mode, out=out_buf[:n], counters=cnt_buf,
                                                            per_site=site_buf)
        torch.cuda.synchronize()
        if k == 1:
            assert torch.cuda.mem_get_info(0)[0] == free_before  # no device memory was taken or returned
        assert torch.equal(out, want_out)
        assert bool((out_buf[n:] == -1).all())  # nothing written past the call's n verdicts
        g = B.Engine.counter_dict(cnt)
        assert want_g["ret_viol"] > 0 and want_g["fwd_viol"] > 0 and want_g["first_violation_key"] != (1 << 64) - 1
        for name in B.COUNTER_FIELDS:
            if name in NOT_PER_CALL:
                assert g[name] == 0, name
            else:
                assert g[name] == want_g[name], (k, name, g[name], want_g[name])
        assert np.array_equal(site.cpu().numpy().view(np.uint64), want_s)
    # stateless: the engine's own counters and event sequence saw none of it ...
    g, s = eng.wg_read_counters()
    assert g["events_total"] == 0 and g["first_violation_key"] == (1 << 64) - 1 and not s.any()
    # ... and its ordinary path is undisturbed afterwards
    out = eng.wg_verify_continuations(st2.hdr, st2.val, tags[1], S.DETECT)
    want_out, want_g, want_s = _existing_path(ref, st2, tags[1], S.DETECT)
    g, s = eng.wg_read_counters()
    assert torch.equal(out, want_out) and np.array_equal(s, want_s)
    assert all(g[name] == want_g[name] for name in B.COUNTER_FIELDS)
    eng.close()
    ref.close()


def test_static_entry_point_empty_call_and_limits():
    dev = torch.device("cuda", 0)
    st = S.make_stream(1, dev, n_events=1_000)
    eng = B.Engine(0).load(st.policy)
    tag = eng.wg_sign_continuations(st.hdr, st.val)
    # n == 0: zero counters, key all-ones, whatever the previous call left in the array
    eng.wg_verify_continuations_static(st.hdr, st.val, tag, S.ENFORCE)
    out, cnt, site = eng.wg_verify_continuations_static(st.hdr[:0], st.val[:0], tag[:0], S.ENFORCE)
    g = B.Engine.counter_dict(cnt)
    assert out.shape[0] == 0 and not site.cpu().numpy().any()
    assert all(v == ((1 << 64) - 1 if k == "first_violation_key" else 0) for k, v in g.items())
    # more events than one launch covers: refused before anything is touched (no buffer of that size exists here)
    rc = B.lib().wg_verify_continuations_static(eng._h, st.hdr.data_ptr(), st.val.data_ptr(), tag.data_ptr(),
                                                out.data_ptr(), None, None, C.c_uint64(B.WG_STATIC_MAX_EVENTS + 1),
                                                S.ENFORCE, None)
    assert rc == B.WG_ERR_STATIC_LIMIT and "WG_STATIC_MAX" in B.strerror(rc)
    eng.close()
    # more sites than the static per-site counters hold
    big = S.make_policy(5, dev, n_sites=B.WG_STATIC_MAX_SITES + 2, max_set=4)
    stb = S.make_stream(5, dev, policy=big, n_events=2_000)
    engb = B.Engine(0).load(big)
    tagb = engb.wg_sign_continuations(stb.hdr, stb.val)
    with pytest.raises(B.WgError) as ei:
        engb.wg_verify_continuations_static(stb.hdr, stb.val, tagb, S.DETECT)
    assert ei.value.status == B.WG_ERR_STATIC_LIMIT
    engb.wg_verify_continuations(stb.hdr, stb.val, tagb, S.DETECT)  # the ordinary path takes the same policy
    engb.close()
