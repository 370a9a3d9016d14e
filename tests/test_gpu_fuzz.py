"""Randomised parity: random policies (all seven kinds, set sizes around the staging limits, site counts around the
shared-memory-counter limit), random events (unknown sites, empty to full masks, uniform and divergent values drawn
from the sets or not), every entry point, modes, profiles and tunings — the oracle decides.  Seeds are fixed."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_11871_b200 import binding as B
from tests.util import mk_hdr

pytestmark = pytest.mark.gpu


def dev():
    return torch.device("cuda", 0)


def to_dev(a):
    a = np.ascontiguousarray(a)
    return torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a).to(dev())


def random_policy(rng, n_sites, n_fwd_targets):
    kind = rng.choice(np.arange(7, dtype=np.uint8), n_sites, p=[0.35, 0.25, 0.1, 0.05, 0.1, 0.05, 0.1])
    kind[0], kind[1] = 0, 1  # at least one of each protected kind
    fwd = np.nonzero(kind == 1)[0]
    sizes = np.ones(len(fwd), dtype=np.int64)
    extra = n_fwd_targets - len(fwd)
    if extra > 0:
        sizes += rng.multinomial(extra, rng.dirichlet(np.full(len(fwd), 0.3)))
    cnt = np.zeros(n_sites, dtype=np.int64)
    cnt[fwd] = sizes
    off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.uint32)
    tg = np.empty(int(off[-1]), dtype=np.uint64)
    for s in fwd:
        k = int(cnt[s])
        tg[off[s]:off[s + 1]] = np.sort(rng.choice(1 << 20, k, replace=False).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000))
    return kind, off, tg


def random_events(rng, kind, off, tg, n):
    n_sites = len(kind)
    site = rng.integers(0, n_sites, n).astype(np.uint64)
    site[rng.random(n) < 0.02] = rng.choice(np.array([n_sites, n_sites + 7, 0xFFFFFFFF], dtype=np.uint64), 1)[0]
    mask = rng.integers(0, 1 << 32, n, dtype=np.uint64)
    r = rng.random(n)
    mask[r < 0.08] = 0
    mask[(r >= 0.08) & (r < 0.4)] = 0xFFFFFFFF
    mask[(r >= 0.4) & (r < 0.5)] = np.uint64(1) << rng.integers(0, 32, int(((r >= 0.4) & (r < 0.5)).sum())).astype(np.uint64)
    ctx = rng.integers(0, 1 << 63, n, dtype=np.uint64)
    val = rng.integers(0, 1 << 20, size=(n, 32)).astype(np.uint64) * np.uint64(16) + np.uint64(0x7F5A40000000)
    uniform = rng.random(n) < 0.6
    val[uniform] = val[uniform, :1]
    # forward events: mostly legal targets
    for e in np.nonzero(site < n_sites)[0]:
        s = int(site[e])
        if kind[s] == 1 and rng.random() < 0.9:
            members = tg[off[s]:off[s + 1]]
            if uniform[e]:
                val[e, :] = members[rng.integers(0, len(members))]
            else:
                val[e, :] = members[rng.integers(0, len(members), 32)]
            if rng.random() < 0.1:
                val[e, rng.integers(0, 32)] ^= np.uint64(1) << np.uint64(rng.integers(0, 40))
    return mk_hdr(site, mask, ctx), val


@pytest.mark.parametrize("seed,n_sites,n_tgts,n", [
    (1, 9, 12, 700), (2, 1024, 2048, 5_003), (3, 1025, 2049, 5_003), (4, 300, 1500, 20_017), (5, 5000, 30_000, 20_001),
    (6, 2, 2, 33), (7, 1500, 1500, 16 * 20 * 148 + 5), (8, 64, 4096, 3_001)])
def test_random_policies_and_streams(seed, n_sites, n_tgts, n):
    rng = np.random.default_rng(seed)
    kind, off, tg = random_policy(rng, n_sites, n_tgts)
    k0, k1 = int(rng.integers(0, 1 << 63)), int(rng.integers(0, 1 << 63))
    hdr, val = random_events(rng, kind, off, tg, n)
    d_hdr, d_val = to_dev(hdr), to_dev(val)
    for trial in range(4):
        orc = oracle.Oracle(kind, off, tg, k0, k1, seed)
        eng = B.Engine(0)
        eng.wg_load_policy(kind, off, tg, k0, k1, seed)
        flags = [0, B.WG_PROFILE_LOW_TELEMETRY, B.WG_PROFILE_SKIP_FORWARD | B.WG_PROFILE_METADATA_INTEGRITY,
                 B.WG_PROFILE_SKIP_BACKWARD | B.WG_PROFILE_METADATA_INTEGRITY][trial]
        orc.set_profile(flags)
        eng.wg_set_profile(flags)
        if trial >= 2:
            orc.set_ring_capacity(64)
            eng.wg_set_ring_capacity(64)
        o_tag = orc.sign(hdr, val)
        g_tag = eng.wg_sign_continuations(d_hdr, d_val)
        assert np.array_equal(g_tag.cpu().numpy().view(np.uint64), o_tag)
        tag = o_tag.copy()
        hit = rng.random(n) < 0.03
        lanes = rng.integers(0, 32, n)
        tag[hit, lanes[hit]] ^= np.uint64(1) << rng.integers(0, 64, int(hit.sum())).astype(np.uint64)
        d_tag = to_dev(tag)
        for mode in (1, 0):
            o = orc.verify(hdr, val, tag, mode)
            g = eng.wg_verify_continuations(d_hdr, d_val, d_tag, mode).cpu().numpy().view(np.uint32)
            assert np.array_equal(g, o), (seed, trial, mode, np.nonzero((g != o).any(1))[0][:5])
            o = orc.check_forward(hdr, val, mode)
            g = eng.wg_check_forward(d_hdr, d_val, mode).cpu().numpy().view(np.uint32)
            assert np.array_equal(g, o), (seed, trial, mode)
        gg, gs = eng.wg_read_counters()
        og, os_ = orc.read_counters()
        assert gg == og, {k: (gg[k], og[k]) for k in og if gg[k] != og[k]}
        assert np.array_equal(gs, os_)
        t, first, ring = eng.wg_read_telemetry(64)
        assert t == orc.read_telemetry()
        of = orc.read_first_violation()
        assert (first is None) == (of is None)
        if first is not None:
            assert all(int(first[f]) == int(of[f]) for f in B.VIOLATION_DTYPE.names)
        eng.close()


@pytest.mark.parametrize("seed,n_sites,n_tgts,n", [(21, 300, 900, 20_011), (22, 4000, 9000, 20_011)])
def test_random_policies_without_a_return_site(seed, n_sites, n_tgts, n):
    """No protected-return site in the policy: wg_verify_continuations runs the forward kernel and must
    still decide what the oracle's verify decides — unknown sites and empty masks included, tags ignored — on the staged
    table (900 targets) and on the hash index (9,000), in every profile."""
    rng = np.random.default_rng(seed)
    kind, off, tg = random_policy(rng, n_sites, n_tgts)
    ret = np.nonzero(kind == 0)[0]
    kind[ret] = rng.choice(np.array([2, 3, 4, 5, 6], dtype=np.uint8), len(ret))  # (return sites own no targets: relabel freely)
    assert not (kind == 0).any() and (kind == 1).any()
    k0, k1 = int(rng.integers(0, 1 << 63)), int(rng.integers(0, 1 << 63))
    hdr, val = random_events(rng, kind, off, tg, n)
    tag = rng.integers(0, 1 << 63, size=(n, 32), dtype=np.uint64)
    d_hdr, d_val, d_tag = to_dev(hdr), to_dev(val), to_dev(tag)
    for flags in (0, B.WG_PROFILE_LOW_TELEMETRY, B.WG_PROFILE_SKIP_FORWARD, B.WG_PROFILE_SKIP_BACKWARD | B.WG_PROFILE_METADATA_INTEGRITY):
        orc = oracle.Oracle(kind, off, tg, k0, k1, seed)
        eng = B.Engine(0)
        eng.wg_load_policy(kind, off, tg, k0, k1, seed)
        orc.set_profile(flags)
        eng.wg_set_profile(flags)
        orc.set_ring_capacity(256)
        eng.wg_set_ring_capacity(256)
        assert not eng.wg_sign_continuations(d_hdr, d_val).any() and not orc.sign(hdr, val).any()
        for mode in (1, 0):
            o = orc.verify(hdr, val, tag, mode)
            g = eng.wg_verify_continuations(d_hdr, d_val, d_tag, mode).cpu().numpy().view(np.uint32)
            assert np.array_equal(g, o), (seed, flags, mode, np.nonzero((g != o).any(1))[0][:5])
        gg, gs = eng.wg_read_counters()
        og, os_ = orc.read_counters()
        assert gg == og, {k: (gg[k], og[k]) for k in og if gg[k] != og[k]}
        assert np.array_equal(gs, os_)
        t, first, ring = eng.wg_read_telemetry(256)
        assert t == orc.read_telemetry()
        of = orc.read_first_violation()
        assert (first is None) == (of is None)
        if first is not None:
            assert all(int(first[f]) == int(of[f]) for f in B.VIOLATION_DTYPE.names)
        eng.close()
