"""The C-ABI library loads without a GPU and exports every symbol include/warpguard.h declares; calls that need
a device fail with a status code, never by running anything on the CPU.  CPU only."""
import ctypes as C
import re
from pathlib import Path

import numpy as np

from paper_2606_11871_b200 import binding as B
from paper_2606_11871_b200 import build as wg_build

ROOT = Path(__file__).resolve().parent.parent


def declared_symbols():
    text = (ROOT / "include" / "warpguard.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(wg_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    wg_build.build()
    L = C.CDLL(str(B.LIB_PATH))
    names = declared_symbols()
    assert {"wg_load_policy", "wg_sign_continuations", "wg_verify_continuations", "wg_check_forward",
            "wg_read_counters"} <= set(names)
    for name in names:
        assert hasattr(L, name), f"{name} declared in warpguard.h but not exported"
    assert sorted(B.EXPORTS) == names  # the binding carries the same names, no more, no fewer


def test_no_device_means_an_error_status_not_a_cpu_path():
    import torch
    if torch.cuda.is_available():
        return
    L = B.lib()
    assert L.wg_strerror(0) == b"ok"
    kind = np.zeros(1, dtype=np.uint8)
    off = np.zeros(2, dtype=np.uint32)
    d = B._PolicyDesc()
    d.n_sites, d.kind, d.tgt_off, d.tgts = 1, kind.ctypes.data, off.ctypes.data, None
    h = C.c_void_p(None)
    assert L.wg_load_policy(C.byref(h), 0, C.byref(d)) == B.WG_ERR_CUDA and not h
    off[1] = 3  # a return site owning targets is rejected before any device is looked for
    assert L.wg_load_policy(C.byref(h), 0, C.byref(d)) == B.WG_ERR_BAD_POLICY
    assert L.wg_check_forward(None, None, None, None, 1, 0, None) == B.WG_ERR_NO_POLICY


def test_product_package_never_touches_the_oracle():
    for f in (ROOT / "paper_2606_11871_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            text = f.read_text()
            assert not re.search(r"^\s*(import|from)\s+oracle\b|wg_oracle|wgo_|#include\s+\"[^\"]*oracle", text, re.M), f


def test_policy_digest_runs_on_the_host_and_equals_the_oracle():
    """wg_policy_digest needs no GPU (load-time host code): it must equal the oracle's digest, itself pinned against
    libcrypto in tests/test_oracle_metadata.py."""
    import numpy as np

    import oracle
    from paper_2606_11871_b200 import binding as B
    from paper_2606_11871_b200 import streams as S

    for config in (1, 3):
        pol = S.make_policy(config, "cpu")
        assert B.wg_policy_digest(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1) == \
            oracle.policy_digest(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1)
    kind = np.array([0, 1, 2], dtype=np.uint8)
    off = np.array([0, 0, 2, 2], dtype=np.uint32)
    tg = np.array([16, 32], dtype=np.uint64)
    a = B.wg_policy_digest(kind, off, tg, 1, 2)
    assert a == oracle.policy_digest(kind, off, tg, 1, 2) and a != B.wg_policy_digest(kind, off, tg, 1, 3)
