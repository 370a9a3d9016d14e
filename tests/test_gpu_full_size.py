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
