"""Out-of-bounds writes and input clobbering, checked without a memory checker (compute-sanitizer is not available
on the GPU pool): every caller-owned buffer of a call sits inside a larger allocation between two bands of a canary
pattern, the output rows themselves start out as canary, and after the call (a) every band still holds the pattern,
(b) every input buffer is byte for byte what it was, (c) every output row was written and equals the oracle's.
Lengths are ragged around the 16-event tile, the 20-warp block and the 148-block grid.  Run with ``-m gpu``."""
import numpy as np
import pytest
import torch

from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests.test_gpu_shadow import pair, random_call
from tests.util import oracle_for

pytestmark = pytest.mark.gpu

DET, ENF = 0, 1
BAND = 67  # rows of canary on either side (odd on purpose: band edges are only 8 / 16 byte aligned)
CANARY64 = 0x5CA1AB1E0DDC0FFE
CANARY32 = 0x5CA1AB1E


def dev():
    return torch.device("cuda", 0)


class Guarded:
    """[BAND | n rows | BAND] in one allocation; `.mid` is the contiguous [n, cols] view handed to the library."""

    def __init__(self, n, cols, dtype, payload=None):
        self.canary = CANARY64 if dtype == torch.int64 else CANARY32
        self.n = n
        self.full = torch.full((n + 2 * BAND, cols), self.canary, dtype=dtype, device=dev())
        self.mid = self.full[BAND:BAND + n]
        assert self.mid.is_contiguous() and self.mid.data_ptr() % 8 == 0
        if payload is not None:
            self.mid.copy_(payload)
        self.before = self.full.clone()

    def bands_intact(self):
        lo, hi = self.full[:BAND], self.full[BAND + self.n:]
        return bool((lo == self.canary).all()) and bool((hi == self.canary).all())

    def unchanged(self):
        return bool(torch.equal(self.full, self.before))


def t64(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int64))


@pytest.mark.parametrize("config,n", [(4, 1), (4, 17), (4, 16 * 20 + 5), (4, 16 * 20 * 148 + 17), (5, 70_001), (3, 4_099)])
def test_stateless_calls_write_exactly_their_output_rows(config, n):
    st = S.make_stream(config, "cpu", n_events=n)
    orc, eng = oracle_for(st.policy), B.Engine(0).load(st.policy)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)

    hdr, val = Guarded(n, 2, torch.int64, st.hdr), Guarded(n, 32, torch.int64, st.val)
    tag = Guarded(n, 32, torch.int64)
    eng.wg_sign_continuations(hdr.mid, val.mid, tag=tag.mid)
    torch.cuda.synchronize()
    o_tag = orc.sign(hdr_np, val_np)
    assert tag.bands_intact() and hdr.unchanged() and val.unchanged()
    assert np.array_equal(tag.mid.cpu().numpy().view(np.uint64), o_tag)  # no canary left: every row was written

    tag_in = Guarded(n, 32, torch.int64, t64(o_tag))
    for mode in (ENF, DET):
        out = Guarded(n, 2, torch.int32)
        eng.wg_verify_continuations(hdr.mid, val.mid, tag_in.mid, mode, out=out.mid)
        torch.cuda.synchronize()
        o = orc.verify(hdr_np, val_np, o_tag, mode)
        assert out.bands_intact() and hdr.unchanged() and val.unchanged() and tag_in.unchanged()
        assert np.array_equal(out.mid.cpu().numpy().view(np.uint32), o)

        out = Guarded(n, 2, torch.int32)
        eng.wg_check_forward(hdr.mid, val.mid, mode, out=out.mid)
        torch.cuda.synchronize()
        o = orc.check_forward(hdr_np, val_np, mode)
        assert out.bands_intact() and hdr.unchanged() and val.unchanged()
        assert np.array_equal(out.mid.cpu().numpy().view(np.uint32), o)
    eng.close()


@pytest.mark.parametrize("n", [1, 3, 33, 32 * 16 + 7, 20_011])
def test_shadow_calls_write_exactly_their_output_rows(n):
    rng = np.random.default_rng(7000 + n)
    n_slots = max(64, 2 * n)
    pol, orc, eng = pair(n_slots, 2)
    hdr_np, _ = random_call(rng, pol, n_slots, n)
    val_np = rng.integers(0, 1 << 16, size=(n, 32)).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000)
    hdr, val = Guarded(n, 2, torch.int64, t64(hdr_np)), Guarded(n, 32, torch.int64, t64(val_np))
    for push, mode in ((True, ENF), (False, DET), (True, DET), (True, ENF), (True, ENF), (False, ENF)):
        out = Guarded(n, 2, torch.int32)
        (eng.wg_shadow_push if push else eng.wg_shadow_check_ret)(hdr.mid, val.mid, mode, out=out.mid)
        torch.cuda.synchronize()
        o = (orc.shadow_push if push else orc.shadow_check_ret)(hdr_np, val_np, mode)
        assert out.bands_intact() and hdr.unchanged() and val.unchanged()
        assert np.array_equal(out.mid.cpu().numpy().view(np.uint32), o)
    assert eng.wg_shadow_read_counters() == orc.shadow_read_counters()
    eng.close()


class GuardedHost(Guarded):
    def __init__(self, n, cols, dtype, payload=None):
        self.canary = CANARY64 if dtype == torch.int64 else CANARY32
        self.n = n
        self.full = torch.full((n + 2 * BAND, cols), self.canary, dtype=dtype).pin_memory()
        self.mid = self.full[BAND:BAND + n]
        if payload is not None:
            self.mid.copy_(payload)
        self.before = self.full.clone()


@pytest.mark.parametrize("n", [5, 262_144 + 13])
def test_host_buffer_calls_write_exactly_their_output_rows(n):
    """The `*_host` entry points stream chunks of 256 Ki events through device staging buffers: the last, ragged chunk
    must copy back n rows and not a row more."""
    st = S.make_stream(4, "cpu", n_events=n)
    orc, eng = oracle_for(st.policy), B.Engine(0).load(st.policy)
    hdr_np, val_np = st.hdr.numpy().view(np.uint64), st.val.numpy().view(np.uint64)
    hdr, val = GuardedHost(n, 2, torch.int64, st.hdr), GuardedHost(n, 32, torch.int64, st.val)
    tag = GuardedHost(n, 32, torch.int64)
    eng.wg_sign_continuations_host(hdr.mid, val.mid, tag=tag.mid)
    o_tag = orc.sign(hdr_np, val_np)
    assert tag.bands_intact() and hdr.unchanged() and val.unchanged()
    assert np.array_equal(tag.mid.numpy().view(np.uint64), o_tag)
    out = GuardedHost(n, 2, torch.int32)
    eng.wg_verify_continuations_host(hdr.mid, val.mid, tag.mid, ENF, out=out.mid)
    assert out.bands_intact() and hdr.unchanged() and val.unchanged()
    assert np.array_equal(out.mid.numpy().view(np.uint32), orc.verify(hdr_np, val_np, o_tag, ENF))
    out = GuardedHost(n, 2, torch.int32)
    eng.wg_check_forward_host(hdr.mid, val.mid, DET, out=out.mid)
    assert out.bands_intact() and hdr.unchanged() and val.unchanged()
    assert np.array_equal(out.mid.numpy().view(np.uint32), orc.check_forward(hdr_np, val_np, DET))
    eng.close()
