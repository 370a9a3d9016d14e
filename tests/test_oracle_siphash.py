"""Pins for the oracle's MAC: published / OpenSSL known answers, live libcrypto cross-check,
encoding and lane-context rules.  CPU only."""
import random
import struct
from pathlib import Path

import pytest

import oracle
from tests import openssl_mac

GOLD = Path(__file__).resolve().parent / "golden"


def _rows(name):
    for line in (GOLD / name).read_text().splitlines():
        if line and not line.startswith("#"):
            yield line.split()


def test_siphash_known_answers():
    """Line 1 is the SipHash paper's Appendix A worked example (a129ca6149be45e5)."""
    rows = list(_rows("siphash24_kat.txt"))
    assert rows[0][2] == "a129ca6149be45e5"
    for key_hex, msg_hex, want in rows:
        key = bytes.fromhex(key_hex)
        k0, k1 = struct.unpack("<QQ", key)
        msg = b"" if msg_hex == "-" else bytes.fromhex(msg_hex)
        assert oracle.siphash24(k0, k1, msg) == int(want, 16), (msg_hex, want)


def test_mac_layout_known_answers():
    """Token = SipHash over LE64(site) || LE64(value) || LE64(ctx) (R2-R4, R20)."""
    n = 0
    for key_hex, site, val, ctx, want in _rows("mac_layout_kat.txt"):
        k0, k1 = struct.unpack("<QQ", bytes.fromhex(key_hex))
        assert oracle.mac(k0, k1, int(site), int(val, 16), int(ctx, 16)) == int(want, 16)
        n += 1
    assert n == 7


def test_known_answers_distinguish_every_field():
    """The KAT rows differ in exactly one field each, so a swapped / dropped field fails one."""
    rows = {(r[1], r[2], r[3]): r[4] for r in _rows("mac_layout_kat.txt") if r[0].startswith("0001")}
    base = rows[("1", "0x00007f5a40000010", "0x0000000000000020")]
    assert rows[("1", "0x00007f5a40000010", "0x0000000000000021")] != base  # context
    assert rows[("2", "0x00007f5a40000010", "0x0000000000000020")] != base  # site
    assert rows[("1", "0x00007f5a40000020", "0x0000000000000020")] != base  # value


@pytest.fixture(scope="module")
def ossl():
    o = openssl_mac.get()
    if o is None:
        pytest.skip("libcrypto SIPHASH not available")
    return o


def test_siphash_vs_openssl_all_lengths(ossl):
    """Every message length 0..63 (all tail-byte cases of the padding rule) and some long ones."""
    rnd = random.Random(1)
    for n in list(range(64)) + [64, 65, 127, 255, 256, 257, 1000]:
        for _ in range(4):
            key = rnd.randbytes(16)
            msg = rnd.randbytes(n)
            k0, k1 = struct.unpack("<QQ", key)
            assert oracle.siphash24(k0, k1, msg) == ossl(key, msg), n


def test_mac_vs_openssl_random_tuples(ossl):
    """10^5 random (key, site, value, ctx): the token is exactly EVP_MAC SIPHASH(size=8) over the
    24-byte message — a library reduction, independent of the oracle's own SipHash."""
    rnd = random.Random(2)
    for i in range(100_000):
        key = rnd.randbytes(16)
        k0, k1 = struct.unpack("<QQ", key)
        site = rnd.getrandbits(32) if i % 3 else rnd.randrange(0, 2000)
        val = rnd.getrandbits(64)
        ctx = rnd.getrandbits(64)
        assert oracle.mac(k0, k1, site, val, ctx) == ossl(key, struct.pack("<QQQ", site, val, ctx))


def test_lane_ctx():
    """Low five bits of context_base are reserved for the lane (R2)."""
    for base in (0, 0x20, 0x3F, 0x0001000300000BE0, 0xFFFFFFFFFFFFFFFF, 0x1F):
        for lane in range(32):
            got = oracle.lane_ctx(base, lane)
            assert got & 31 == lane
            assert got >> 5 == base >> 5
    assert oracle.lane_ctx(0x0001000300000BFF, 3) == 0x0001000300000BE3
