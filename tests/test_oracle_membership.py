"""Forward membership pinned by brute force (Python sets) on tiny and small sets.  CPU only."""
import random

import numpy as np

import oracle
from tests.util import mk_hdr

FWD = oracle.KIND_PROTECTED_FORWARD


def _probe_values(members, rnd):
    vals = {0, (1 << 64) - 1, 1, (1 << 63)}
    for m in members:
        vals.update({m, (m - 1) % (1 << 64), (m + 1) % (1 << 64), (m - 16) % (1 << 64), (m + 16) % (1 << 64)})
        for _ in range(3):
            vals.add(m ^ (1 << rnd.randrange(64)))
    vals.update({min(members), max(members), (min(members) - 1) % (1 << 64), (max(members) + 1) % (1 << 64)})
    for _ in range(16):
        vals.add(rnd.getrandbits(64))
    return sorted(vals)


def _run(sizes, rnd, binary):
    sets = []
    for n in sizes:
        s = set()
        while len(s) < n:
            s.add(rnd.choice([rnd.getrandbits(64), 0x7F5A40000000 + 16 * rnd.randrange(1 << 16), rnd.randrange(64)]))
        sets.append(sorted(s))
    kind = np.full(len(sets), FWD, dtype=np.uint8)
    off = np.zeros(len(sets) + 1, dtype=np.uint32)
    off[1:] = np.cumsum([len(s) for s in sets])
    tg = np.array([x for s in sets for x in s], dtype=np.uint64)
    orc = oracle.Oracle(kind, off, tg, 1, 2)
    orc.set_binary_search(binary)
    for site, members in enumerate(sets):
        probes = _probe_values(members, rnd)
        while len(probes) % 32:
            probes.append(rnd.getrandbits(64))
        v = np.array(probes, dtype=np.uint64).reshape(-1, 32)
        hdr = mk_hdr(np.full(v.shape[0], site), 0xFFFFFFFF, 0)
        out = orc.check_forward(hdr, v, oracle.MODE_DETECT)
        mset = set(members)
        for r in range(v.shape[0]):
            want = sum(1 << j for j in range(32) if int(v[r, j]) not in mset)
            assert int(out[r, 0]) == want, (site, r)
            assert int(out[r, 1]) == 0xFFFFFFFF


def test_tiny_sets_brute_force():
    _run([1, 2, 3, 4] * 4, random.Random(3), binary=False)


def test_all_sizes_up_to_64_brute_force():
    _run(list(range(1, 65)), random.Random(4), binary=False)


def test_binary_search_variant_agrees():
    """wgo_set_binary_search(1) (used only to time config 5) gives the same verdicts."""
    _run(list(range(1, 65)) + [257, 1000, 4096], random.Random(5), binary=True)


def test_wrong_site_valid_target_violates_and_same_site_alternative_passes():
    """a target legal at site A presented at site B violates; any member of the
    site's own set passes whichever lane carries it."""
    kind = np.array([FWD, FWD], dtype=np.uint8)
    off = np.array([0, 3, 5], dtype=np.uint32)
    tg = np.array([0x100, 0x200, 0x300, 0x150, 0x250], dtype=np.uint64)
    orc = oracle.Oracle(kind, off, tg, 7, 9)
    v = np.zeros((2, 32), dtype=np.uint64)
    v[0, :] = [[0x100, 0x200, 0x300][j % 3] for j in range(32)]  # legal alternatives at site 0
    v[1, :] = 0x150
    v[1, 5] = 0x200                                               # legal at site 0 only
    out = orc.check_forward(mk_hdr([0, 1], 0xFFFFFFFF, 0), v, oracle.MODE_ENFORCE)
    assert out[0].tolist() == [0, 0xFFFFFFFF]
    assert out[1].tolist() == [1 << 5, 0xFFFFFFFF & ~(1 << 5)]
