#!/usr/bin/env python3
"""Re-creates siphash24_kat.txt and mac_layout_kat.txt with the `openssl` CLI only.

Independent of oracle/ and of the CUDA path: the message bytes are written to a file and
hashed by `openssl mac ... SIPHASH` (OpenSSL 3.x).  Usage: python tests/golden/regen_openssl_kat.py
"""
import struct
import subprocess
import tempfile
from pathlib import Path

HERE = Path(__file__).resolve().parent


def sip(key: bytes, msg: bytes) -> int:
    with tempfile.NamedTemporaryFile() as f:
        f.write(msg)
        f.flush()
        out = subprocess.run(["openssl", "mac", "-macopt", "hexkey:" + key.hex(), "-macopt", "size:8",
                              "-in", f.name, "SIPHASH"], check=True, capture_output=True, text=True).stdout
    return int.from_bytes(bytes.fromhex(out.strip()), "little")  # openssl prints the output bytes in order


K = bytes(range(16))
with open(HERE / "siphash24_kat.txt", "w") as f:
    f.write("# key_hex msg_hex(- = empty) -> siphash-2-4 as u64 hex (little-endian reading of the 8 output bytes)\n")
    for n in (15, 0, 8, 24):
        m = bytes(range(n))
        f.write(f"{K.hex()} {m.hex() or '-'} {sip(K, m):016x}\n")

CASES = [
    (K, 0, 0x0, 0x0),
    (K, 1, 0x00007F5A40000010, 0x20),
    (K, 1, 0x00007F5A40000010, 0x21),
    (K, 2, 0x00007F5A40000010, 0x20),
    (K, 1, 0x00007F5A40000020, 0x20),
    (struct.pack("<QQ", 0x0123456789ABCDEF, 0xFEDCBA9876543210), 1342, 0x00007F5A400FFFF0, 0x0001000300000BFF),
    (bytes(16), 0xFFFFFFFF, 0xFFFFFFFFFFFFFFFF, 0xFFFFFFFFFFFFFFFF),
]
with open(HERE / "mac_layout_kat.txt", "w") as f:
    f.write("# key_hex(16 bytes; k0,k1 = LE64 halves) site_id value context_id -> token u64 hex; "
            "message = LE64(site_id) || LE64(value) || LE64(context_id)\n")
    for key, site, val, ctx in CASES:
        f.write(f"{key.hex()} {site} {val:#018x} {ctx:#018x} {sip(key, struct.pack('<QQQ', site, val, ctx)):016x}\n")
