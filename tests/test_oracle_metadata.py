"""Pins for the metadata-integrity profile of the oracle (R37-R38).
The record token's message format is pinned against libcrypto's SIPHASH: a record re-forged with tokens computed by
OpenSSL over struct.pack('<Q...') must authenticate."""
import struct

import numpy as np
import pytest

import oracle
from tests import openssl_mac
from tests.util import mk_hdr

DET, ENF = 0, 1
FULL = 0xFFFFFFFF
K0, K1 = 0x0706050403020100, 0x0F0E0D0C0B0A0908
KEY = struct.pack("<QQ", K0, K1)


def make():
    kind = np.array([0, 1, 1, 2, 1], dtype=np.uint8)           # sites 1, 2, 4 are protected-forward
    off = np.array([0, 0, 3, 4, 4, 9], dtype=np.uint32)
    tg = np.array([0x1000, 0x2000, 0x3000, 0x7000, 0x10, 0x20, 0x30, 0x40, 0x50], dtype=np.uint64)
    return oracle.Oracle(kind, off, tg, K0, K1, 0), kind, off, tg


def events():
    hdr = mk_hdr([1, 2, 4, 1, 4, 0, 3, 2], [FULL, 0xFF, 0xF0F0, 1, 0, FULL, 3, FULL], [0] * 8)
    val = np.zeros((8, 32), dtype=np.uint64)
    val[0, :] = 0x2000; val[0, 7] = 0x2008
    val[1, :] = 0x7000
    val[2, :] = np.array([0x10, 0x20, 0x30, 0x40, 0x50, 0x60, 0x10, 0x20] * 4, dtype=np.uint64)
    val[3, :] = 0x3000
    val[7, :] = 0x1000
    return hdr, val


def record_msg(site, targets):
    return struct.pack("<QQ", site, len(targets)) + b"".join(struct.pack("<Q", int(t)) for t in targets)


def test_an_intact_record_authenticates_and_changes_nothing():
    o, kind, off, tg = make()
    hdr, val = events()
    plain = o.check_forward(hdr, val, ENF)
    o2, *_ = make()
    o2.set_profile(oracle.PROFILE_METADATA_INTEGRITY)
    assert np.array_equal(o2.check_forward(hdr, val, ENF), plain)
    assert o2.read_telemetry()["fwd_meta_fail_events"] == 0
    assert plain[0, 0] == 1 << 7 and plain[1, 0] == 0 and plain[7, 0] == FULL


@pytest.mark.parametrize("what,index", [(0, 0), (0, 2), (1, 1)])
def test_a_corrupted_record_fails_closed_on_its_site_only(what, index):
    o, kind, off, tg = make()
    hdr, val = events()
    ref = o.check_forward(hdr, val, ENF)
    o2, *_ = make()
    o2.set_profile(oracle.PROFILE_METADATA_INTEGRITY)
    o2.policy_poke(what, index, 1 << 4)                 # site 1's set or token
    out = o2.check_forward(hdr, val, ENF)
    site = (hdr[:, 0] & np.uint64(0xFFFFFFFF)).astype(int)
    active = (hdr[:, 0] >> np.uint64(32)).astype(np.uint32)
    hit = site == 1
    assert np.array_equal(out[hit, 0], active[hit]) and (out[hit, 1] == 0).all()   # every active lane blocked
    assert np.array_equal(out[~hit], ref[~hit])
    assert o2.read_telemetry()["fwd_meta_fail_events"] == int((hit & (active != 0)).sum())
    g, _ = o2.read_counters()
    assert g["fwd_viol"] >= int(np.unpackbits(active[hit].view(np.uint8)).sum())


def test_without_the_profile_a_corrupted_set_is_silently_a_different_policy():
    o, *_ = make()
    hdr, val = events()
    o.policy_poke(0, 1, 0x2000 ^ 0x2008)                # 0x2000 -> 0x2008 in site 1's set
    out = o.check_forward(hdr, val, ENF)
    assert out[0, 0] == FULL & ~(1 << 7)                # now only lane 7 (target 0x2008) passes


def test_record_token_format_against_libcrypto():
    ossl = openssl_mac.get()
    if ossl is None:
        pytest.skip("libcrypto without SIPHASH")
    o, kind, off, tg = make()
    o.set_profile(oracle.PROFILE_METADATA_INTEGRITY)
    hdr, val = events()
    # re-forge site 4's record: target 0x30 -> 0x38, token adjusted with OpenSSL tokens of the old and new record
    old = tg[4:9].copy()
    new = old.copy(); new[2] = 0x38
    o.policy_poke(0, 6, 0x30 ^ 0x38)
    o.policy_poke(1, 4, ossl(KEY, record_msg(4, old)) ^ ossl(KEY, record_msg(4, new)))
    out = o.check_forward(hdr, val, ENF)
    assert o.read_telemetry()["fwd_meta_fail_events"] == 0
    # event 2: site 4, lanes 4-7 and 12-15 active, values 0x50 0x60 0x10 0x20: only 0x60 is out of set
    assert out[2, 0] == (1 << 5) | (1 << 13)
    val2 = val.copy(); val2[2, 4] = 0x30; val2[2, 6] = 0x38
    out = o.check_forward(hdr, val2, ENF)
    assert out[2, 0] == (1 << 4) | (1 << 5) | (1 << 13)   # 0x30 is no longer allowed, 0x38 is
    # the same forgery with a wrong site id, a wrong count or a swapped order does not authenticate
    for msg in (record_msg(5, new), struct.pack("<QQ", 4, 6) + record_msg(4, new)[16:], record_msg(4, new[::-1])):
        o2, *_ = make()
        o2.set_profile(oracle.PROFILE_METADATA_INTEGRITY)
        o2.policy_poke(0, 6, 0x30 ^ 0x38)
        o2.policy_poke(1, 4, ossl(KEY, record_msg(4, old)) ^ ossl(KEY, msg))
        o2.check_forward(hdr, val, ENF)
        assert o2.read_telemetry()["fwd_meta_fail_events"] == 1


# ---------------------------------------------------------------------------------------------------------
# policy-digest binding (second half; R39)
# ---------------------------------------------------------------------------------------------------------
def test_policy_digest_format_and_bound_load_against_libcrypto():
    ossl = openssl_mac.get()
    if ossl is None:
        pytest.skip("libcrypto without SIPHASH")
    o, kind, off, tg = make()
    msg = struct.pack("<QQ", len(kind), len(tg)) + bytes(kind) + b"\0" * (-len(kind) % 8)
    msg += b"".join(struct.pack("<I", int(x)) for x in off) + b"\0" * (-4 * len(off) % 8)
    msg += b"".join(struct.pack("<Q", int(t)) for t in tg)
    d = oracle.policy_digest(kind, off, tg, K0, K1)
    assert d == ossl(KEY, msg)
    # a bound load refuses any other digest, and any other image under the right digest
    with pytest.raises(ValueError):
        oracle.Oracle(kind, off, tg, K0, K1, d ^ 1, bound=True)
    tg2 = tg.copy(); tg2[3] += np.uint64(16)
    with pytest.raises(ValueError):
        oracle.Oracle(kind, off, tg2, K0, K1, d, bound=True)
    ob = oracle.Oracle(kind, off, tg, K0, K1, d, bound=True)
    # tokens of the bound engine: first message word = site | digest32 << 32 (libcrypto over struct.pack)
    hdr = mk_hdr([0], [FULL], [0x0001000000000040])
    val = np.full((1, 32), 0x7F5A40000010, dtype=np.uint64)
    tag = ob.sign(hdr, val)
    for lane in (0, 5, 31):
        w0 = 0 | ((d & 0xFFFFFFFF) << 32)
        assert int(tag[0, lane]) == ossl(KEY, struct.pack("<QQQ", w0, 0x7F5A40000010, 0x0001000000000040 | lane))
    # ... verify under the same binding, and do not carry over to the unbound engine nor to another image
    assert ob.verify(hdr, val, tag, ENF)[0, 0] == 0
    assert o.verify(hdr, val, tag, ENF)[0, 0] == FULL
    d2 = oracle.policy_digest(kind, off, tg2, K0, K1)
    other = oracle.Oracle(kind, off, tg2, K0, K1, d2, bound=True)
    assert d2 != d and other.verify(hdr, val, tag, ENF)[0, 0] == FULL
