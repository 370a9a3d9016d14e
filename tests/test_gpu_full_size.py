"""BASELINE.json's configs at their FULL sizes, in the launch configuration bench.py times, against the oracle over the
WHOLE stream: every tag, every verdict pair, the global counters and the full per-site counter
array — the only place the contended per-site counter path (a Zipf(1.1) hot site x 58 M events; PAPER.md:113, 127:
only protected sites in the denominator; Table 3) meets the oracle.  The oracle runs on all host cores
(tests/fullsize.py), chunk by chunk, while the engine runs once over the whole stream on the GPU."""
import numpy as np
import pytest
import torch

from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests import fullsize

pytestmark = [pytest.mark.gpu, pytest.mark.filterwarnings("ignore:This process.*is multi-threaded:DeprecationWarning")]
CHUNK = 4_000_000


def dev():
    return torch.device("cuda", 0)


def whole_stream_parity(st, eng, binary_search=False):
    """sign -> (host: oracle sign, tamper, oracle verify, chunk by chunk) -> tamper on the GPU -> verify -> compare."""
    n = st.hdr.shape[0]
    pol = st.policy
    tag = eng.wg_sign_continuations(st.hdr, st.val)
    gsign, _ = eng.wg_read_counters(per_site=False)
    plan = st.ret_tamper
    p_ev, p_lane, p_what, p_arg = (x.cpu().numpy() for x in (plan.ev, plan.lane, plan.what, plan.arg))
    o_out = np.empty((n, 2), dtype=np.uint32)
    o_glob, o_site, o_signed = None, np.zeros((pol.n_sites, 4), dtype=np.uint64), 0
    for lo in range(0, n, CHUNK):
        hi = min(n, lo + CHUNK)
        hdr = st.hdr[lo:hi].cpu().numpy().view(np.uint64)
        val = st.val[lo:hi].cpu().numpy().view(np.uint64)
        tg = tag[lo:hi].cpu().numpy().view(np.uint64)
        o_tag, gs, _ = fullsize.oracle_chunk(pol, "sign", hdr, val, None, 0, lo, binary_search)
        bad = np.nonzero((o_tag != tg).any(axis=1))[0]
        assert bad.size == 0, ("tags differ from the oracle", lo + bad[:5])
        o_signed += gs["signed_lanes"]
        # the recorded corruption of this chunk (what Stream.apply_return_tamper does on the GPU)
        sel = (p_ev >= lo) & (p_ev < hi)
        for ev, lane, what, arg in zip(p_ev[sel] - lo, p_lane[sel], p_what[sel], p_arg[sel]):
            (tg if what == S.T_TAG_XOR else val)[ev, lane] ^= np.uint64(int(arg) & ((1 << 64) - 1))
        out, g, site = fullsize.oracle_chunk(pol, "verify", hdr, val, tg, st.mode, lo, binary_search)
        o_out[lo:hi] = out
        o_glob = fullsize.add_counters(o_glob, g)
        o_site += site
    assert gsign["signed_lanes"] == o_signed
    st.apply_return_tamper(tag)
    eng.wg_reset_counters()
    out = eng.wg_verify_continuations(st.hdr, st.val, tag, st.mode).cpu().numpy().view(np.uint32)
    bad = np.nonzero((out != o_out).any(axis=1))[0]
    assert bad.size == 0, ("verdicts differ from the oracle", bad[:5], out[bad[:5]], o_out[bad[:5]])
    gg, gs = eng.wg_read_counters()
    for k in ("signed_lanes", "sign_skipped_events"):  # (the oracle's verify-only processes signed nothing)
        gg[k] = o_glob[k] = 0
    assert gg == o_glob, {k: (gg[k], o_glob[k]) for k in o_glob if gg[k] != o_glob[k]}
    bad = np.nonzero((gs != o_site).any(axis=1))[0]
    assert bad.size == 0, ("per-site counters differ from the oracle", bad[:5], gs[bad[:5]], o_site[bad[:5]])
    return gg, gs, out


def test_config4_full_size_whole_stream_against_the_oracle():
    """58.0 M events, 52.2 M checks, 51,621 sites, Zipf(1.1): every output and every per-site counter."""
    st = S.make_stream(4, dev())
    assert st.hdr.shape[0] == S.FULL_EVENTS[4]
    eng = B.Engine(0).load(st.policy)
    g, s, out = whole_stream_parity(st, eng)
    assert g["ret_checks"] == 38_300_000 and g["fwd_checks"] == 13_900_000 and g["events_total"] == S.FULL_EVENTS[4]
    assert g["ret_viol_events"] == len(st.ret_tamper) and g["fwd_viol_events"] == len(st.fwd_tamper)
    assert int(s[:, 0].max()) > 5_000_000  # the hot site really is hot: its counters took the contended path
    eng.close()


@pytest.mark.parametrize("config", [2, 3])
def test_configs_2_and_3_full_size_whole_stream_against_the_oracle(config):
    st = S.make_stream(config, dev())
    assert st.hdr.shape[0] == S.FULL_EVENTS[config]
    eng = B.Engine(0).load(st.policy)
    g, s, out = whole_stream_parity(st, eng)
    assert g["ret_viol_events"] == len(st.ret_tamper) and g["fwd_viol_events"] == len(st.fwd_tamper)
    eng.close()


def test_config5_full_size_policy_one_whole_batch_against_the_oracle():
    """1 M protected sites, log-uniform sets up to 4,096 entries (~246 M targets, searched from L2 / HBM), one whole 8 M
    event batch with 1-32 active lanes per event.  The oracle's membership is std::binary_search here (agreement with
    the linear scan on every set size is pinned in tests/test_oracle_membership.py; SURVEY 8(d) allows it for config 5)."""
    pol = S.make_policy(5, dev())
    assert pol.n_sites == 1_000_000 and pol.tgt_off[-1] > 100_000_000
    st = S.make_stream(5, dev(), policy=pol, batch_index=1)
    eng = B.Engine(0).load(pol)
    g, s, out = whole_stream_parity(st, eng, binary_search=True)
    assert g["ret_viol_events"] == len(st.ret_tamper)
    assert len(st.fwd_tamper) - 20 <= g["fwd_viol_events"] <= len(st.fwd_tamper)  # (a flipped bit can hit another member)
    eng.close()


def test_one_call_longer_than_one_launch_tiles_a_pattern_the_oracle_judged():
    """Maximum sizes: a launch covers at most 2^27 - 32 events (element indices event * 32 + lane stay below 2^32), a CALL
    may be longer and is cut into launches by the C-ABI layer (pointer offsets, sequence base, ticket slots).  The stream
    is a 4,096-event config-4 pattern repeated 32,769.x times (134,221,829 events, 34 GB of values): the oracle judges
    the pattern (and its ragged tail) once; every tag and verdict of the long call must equal the pattern's, the
    counters must be the pattern's times the number of repeats plus the tail's, and the first-violation key the
    pattern's own (sequence numbers run through the call, R12)."""
    P = 4096
    n = (1 << 27) - 32 + P + 5
    full, tail = divmod(n, P)
    free, _ = torch.cuda.mem_get_info(0)
    if free < 90 * (1 << 30):
        pytest.skip("needs ~80 GB of device memory")
    st = S.make_stream(4, "cpu", n_events=P, mode=S.ENFORCE)
    pol = st.policy
    from tests.util import oracle_for
    hdr_p, val_p = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64).copy()
    orc = oracle_for(pol)
    tag_p = orc.sign(hdr_p, val_p)
    tag_t = torch.from_numpy(tag_p.view(np.int64).copy())
    st.apply_return_tamper(tag_t)  # (values and tags, as the recorded plan says)
    val_c, tag_c = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)
    orc = oracle_for(pol)
    out_p = orc.verify(hdr_p, val_c, tag_c, S.ENFORCE)
    g_p, s_p = orc.read_counters()
    first_p = g_p["first_violation_key"]
    orc_t = oracle_for(pol)
    orc_t.verify(hdr_p[:tail], val_c[:tail], tag_c[:tail], S.ENFORCE)
    g_t, s_t = orc_t.read_counters()
    assert out_p[:, 0].any() and first_p != (1 << 64) - 1

    def tiled(a):  # the pattern, repeated to n rows on the device (no temporary of the full size)
        t = a.to(dev())
        big = torch.empty((n, t.shape[1]), dtype=t.dtype, device=dev())
        big[: full * P].view(full, P, -1).copy_(t.view(1, P, -1).expand(full, P, -1))
        big[full * P:].copy_(t[:tail])
        return big

    def equals_pattern(big, pat):
        pat = pat.to(dev())
        ok = bool((big[: full * P].view(full, P, -1) == pat.view(1, P, -1)).all())
        return ok and bool((big[full * P:] == pat[:tail]).all())

    eng = B.Engine(0).load(pol)
    d_hdr = tiled(st.hdr)
    d_val = tiled(torch.from_numpy(val_p.view(np.int64)))
    g_tag = eng.wg_sign_continuations(d_hdr, d_val)
    assert equals_pattern(g_tag, torch.from_numpy(tag_p.view(np.int64))), "tags of the long call differ from the pattern's"
    del g_tag, d_val
    d_val = tiled(st.val)
    d_tag = tiled(tag_t)
    eng.wg_reset_counters()
    out = eng.wg_verify_continuations(d_hdr, d_val, d_tag, S.ENFORCE)
    assert equals_pattern(out, torch.from_numpy(out_p.view(np.int32))), "verdicts of the long call differ from the pattern's"
    gg, gs = eng.wg_read_counters()
    skip = ("first_violation_key", "policy_digest", "last_mode", "signed_lanes", "sign_skipped_events")
    for k in g_p:
        if k not in skip:
            assert gg[k] == full * g_p[k] + g_t[k], (k, gg[k], g_p[k], g_t[k])
    assert gg["first_violation_key"] == first_p
    assert np.array_equal(gs, np.uint64(full) * s_p + s_t)
    eng.close()
    del d_hdr, d_val, d_tag, out
    torch.cuda.empty_cache()  # (the other GPU tests, some of them in child processes, get the 70 GB back)
