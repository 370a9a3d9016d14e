"""The inline device form (include/warpguard_device.cuh) against the oracle: a user kernel
(tests/inline_user_kernel.cu, built with nvcc for sm_100a) calls wg_dev_sign / wg_dev_verify / wg_dev_check_forward
per thread; tags and per-lane verdicts must equal the oracle's on the events of the matching site kind."""
import ctypes as C
import shutil
import subprocess
from pathlib import Path

import numpy as np
import pytest
import torch

from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import streams as S
from tests.util import oracle_for

pytestmark = pytest.mark.gpu
HERE = Path(__file__).resolve().parent
ROOT = HERE.parent
SO = HERE / "libinline_user_kernel.so"


def build_user_kernel():
    src = HERE / "inline_user_kernel.cu"
    deps = [src, ROOT / "include" / "warpguard_device.cuh", ROOT / "include" / "warpguard_sip32.cuh"]
    if SO.exists() and SO.stat().st_mtime >= max(d.stat().st_mtime for d in deps):
        return
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-shared",
                    "-Xcompiler", "-fPIC", "-I", str(ROOT / "include"), "-o", str(SO), str(src), "-lcudart_static",
                    "-lpthread", "-ldl", "-lrt"], check=True)


@pytest.mark.parametrize("config,n", [(4, 120_007), (5, 50_003)])
def test_inline_helpers_equal_the_oracle(config, n):
    build_user_kernel()
    L = C.CDLL(str(SO))
    L.wg_test_run_inline.argtypes = [B.DeviceView, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_uint64, C.c_int, C.c_void_p]
    dev = torch.device("cuda", 0)
    if config == 5:
        pol = S.make_policy(5, "cpu", n_sites=5_000, max_set=512)
        st = S.make_stream(5, "cpu", n_events=n, policy=pol)
    else:
        st = S.make_stream(config, "cpu", n_events=n)
        pol = st.policy
    orc, eng = oracle_for(pol), B.Engine(0).load(pol)
    view = eng.wg_get_device_view()
    hdr = st.hdr.numpy().view(np.uint64)
    site = (hdr[:, 0] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    kind = np.where(site < pol.n_sites, pol.kind[np.minimum(site, pol.n_sites - 1)], 7)
    d_hdr, d_val = st.hdr.to(dev), st.val.to(dev)
    stream = torch.cuda.current_stream().cuda_stream

    # push at the call sites
    o_tag = orc.sign(hdr, st.val.numpy().view(np.uint64))
    d_tag = torch.zeros((n, 32), dtype=torch.int64, device=dev)
    d_viol = torch.zeros(n, dtype=torch.int32, device=dev)
    assert L.wg_test_run_inline(view, d_hdr.data_ptr(), d_val.data_ptr(), None, d_tag.data_ptr(), d_viol.data_ptr(), n, 0, stream) == 0
    assert np.array_equal(d_tag.cpu().numpy().view(np.uint64), o_tag)

    # corrupt, then check_ret at the return sites
    tag_t = torch.from_numpy(o_tag.view(np.int64).copy())
    st.apply_return_tamper(tag_t)
    d_val, d_tag = st.val.to(dev), tag_t.to(dev)
    o_out = orc.verify(hdr, st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64), 1)
    assert L.wg_test_run_inline(view, d_hdr.data_ptr(), d_val.data_ptr(), d_tag.data_ptr(), None, d_viol.data_ptr(), n, 1, stream) == 0
    g = d_viol.cpu().numpy().view(np.uint32)
    is_ret = kind == 0
    assert np.array_equal(g[is_ret], o_out[is_ret, 0]) and o_out[is_ret, 0].any()
    active = (hdr[:, 0] >> np.uint64(32)).astype(np.uint32)
    assert np.array_equal(g[~is_ret], active[~is_ret])  # any other site fails closed at a return check

    # forward checks at the indirect-branch sites
    assert L.wg_test_run_inline(view, d_hdr.data_ptr(), d_val.data_ptr(), None, None, d_viol.data_ptr(), n, 2, stream) == 0
    g = d_viol.cpu().numpy().view(np.uint32)
    is_fwd = kind == 1
    assert np.array_equal(g[is_fwd], o_out[is_fwd, 0]) and is_fwd.any() and o_out[is_fwd, 0].any()
    assert np.array_equal(g[~is_fwd], active[~is_fwd])
    eng.close()


def test_no_key_material_is_reachable_through_the_view():
    """the engine once cached per-site SipHash mid-states in global memory, and a SipRound is a
    bijection, so one 32-byte read gave the key.  Now the only device memory the view points at is the policy image
    itself: every site record must be exactly {kind, set offset, set size, flags = 0} — a function of the policy alone,
    identical under two different keys — and the key-equivalent words travel in the view BY VALUE (kernel parameters,
    PAPER.md:256)."""
    build_user_kernel()
    L = C.CDLL(str(SO))
    L.wg_test_copy_site_recs.argtypes = [B.DeviceView, C.c_void_p]
    pol = S.make_policy(4, "cpu")
    images = []
    for k0, k1 in ((pol.k0, pol.k1), (pol.k0 ^ 0x5555, pol.k1 ^ 0x7777)):
        eng = B.Engine(0)
        eng.wg_load_policy(pol.kind, pol.tgt_off, pol.tgts, k0, k1, pol.policy_digest)
        view = eng.wg_get_device_view()
        raw = np.zeros((pol.n_sites, 4), dtype=np.uint32)
        assert L.wg_test_copy_site_recs(view, raw.ctypes.data) == 0
        images.append(raw)
        M = (1 << 64) - 1
        consts = (0x736f6d6570736575, 0x646f72616e646f6d, 0x6c7967656e657261, 0x7465646279746573)
        assert [int(v) for v in view.v_init] == [(k ^ c) & M for k, c in zip((k0, k1, k0, k1), consts)]
        eng.close()
    expect = np.stack([pol.kind.astype(np.uint32), pol.tgt_off[:-1].astype(np.uint32),
                       np.diff(pol.tgt_off.astype(np.int64)).astype(np.uint32), np.zeros(pol.n_sites, np.uint32)], axis=1)
    assert np.array_equal(images[0], expect) and np.array_equal(images[1], expect)
