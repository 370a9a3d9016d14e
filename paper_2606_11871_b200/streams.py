"""Seeded synthetic policies and per-warp check-event streams (BASELINE.json configs 1-5).

This module is the ONLY code shared by the oracle-side tests and the CUDA-side
tests / bench.  It holds none of the method's arithmetic: no MAC, no membership
test, no verdict or counter rule.  Tags are produced by whichever signer the
caller passes in (the oracle's in parity tests, the engine's in bench.py), and
tampering is applied afterwards from a recorded plan.

The streams stand in for the paper's 77-artifact corpus and attack matrix, which
are not available (Table A7); only the paper's counts and
distributions are used: 51,621 sites, 1,343 returns, 154 supported / 15
unsupported forward entries, 10 fallback entries, target-set sizes with median /
p90 / max = 1 / 3 / 10, and 38.3 M + 13.9 M = 52.2 M dynamic checks
(PAPER.md:333-340, 349-363).  The recipe is written out in DESIGN.md §4.

Everything is torch (int64 bit patterns standing for the u64 / u32 fields) so the
same code runs on the CPU for the oracle tests and on the GPU at full size.
Layouts handed to the engine:

  hdr  int64 [n, 2]   word 0 = site_id | active_mask << 32, word 1 = context_base
                      (little-endian image of {u32 site_id; u32 active_mask; u64 context_base})
  val  int64 [n, 32]  per-lane continuation (return events) or target (forward events)
  tag  int64 [n, 32]  per-lane stored token (signer output, then tampered)
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

# site kinds (Table 2; numbering of include/warpguard.h)
PROTECTED_RETURN, PROTECTED_FORWARD, FIXED_EDGE, UNSUPPORTED, PROFILE_EXCLUDED, FALLBACK, NO_SURFACE = range(7)
DETECT, ENFORCE = 0, 1

CODE_BASE = 0x00007F5A40000000  # code window base; addresses are CODE_BASE + 16 * slot
SLOT_BYTES = 16                 # SASS instructions are 128-bit

# tamper kinds recorded in the plan
T_TAG_XOR = 0       # tag[ev, lane] ^= arg      (return event, after signing)
T_VAL_XOR = 1       # val[ev, lane] ^= arg      (return: after signing; forward: at generation)
T_VAL_SET_LANE = 2  # val[ev, lane]  = arg      (forward, out-of-set address in one lane)
T_VAL_SET_ALL = 3   # val[ev, every active lane] = arg   (forward, warp-uniform event)

_MASK64 = (1 << 64) - 1


def _u64(x: int) -> int:
    return x & _MASK64


@dataclass
class Policy:
    """Host-side policy description, the argument of wg_load_policy."""
    kind: np.ndarray      # uint8  [n_sites]
    tgt_off: np.ndarray   # uint32 [n_sites + 1]
    tgts: np.ndarray      # uint64 [tgt_off[-1]]
    k0: int
    k1: int
    policy_digest: int
    window_slots: int
    free_slots: torch.Tensor | None = None  # int64 slots of the window that hold no target of any site

    @property
    def n_sites(self) -> int:
        return int(self.kind.size)


@dataclass
class TamperPlan:
    ev: torch.Tensor    # int64 [m] event index
    lane: torch.Tensor  # int64 [m] lane (for T_VAL_SET_ALL: the lowest active lane)
    what: torch.Tensor  # int64 [m] T_*
    arg: torch.Tensor   # int64 [m] xor mask or replacement value

    @staticmethod
    def empty(device) -> "TamperPlan":
        z = torch.zeros(0, dtype=torch.int64, device=device)
        return TamperPlan(z, z.clone(), z.clone(), z.clone())

    def __len__(self) -> int:
        return int(self.ev.numel())

    @staticmethod
    def cat(plans) -> "TamperPlan":
        plans = [p for p in plans if len(p)]
        if not plans:
            raise ValueError("no plans")
        return TamperPlan(*(torch.cat([getattr(p, f) for p in plans]) for f in ("ev", "lane", "what", "arg")))


@dataclass
class Stream:
    name: str
    policy: Policy
    mode: int
    hdr: torch.Tensor            # int64 [n, 2]
    val: torch.Tensor            # int64 [n, 32]; return rows hold the values AT PUSH TIME until
                                 # apply_return_tamper() is called
    uniform: torch.Tensor        # bool [n] generator's own note: event was built warp-uniform
    ret_tamper: TamperPlan       # to apply after signing
    fwd_tamper: TamperPlan       # already applied to val; kept as the construction record
    meta: dict = field(default_factory=dict)
    _ret_applied: bool = False

    @property
    def n(self) -> int:
        return int(self.hdr.shape[0])

    def site_id(self) -> torch.Tensor:
        return self.hdr[:, 0] & 0xFFFFFFFF

    def active_mask(self) -> torch.Tensor:
        return (self.hdr[:, 0] >> 32) & 0xFFFFFFFF

    def apply_return_tamper(self, tag: torch.Tensor) -> None:
        """In place: corrupt the signed stream as the plan says (tags and observed continuations)."""
        assert not self._ret_applied, "return tamper already applied"
        p = self.ret_tamper
        if len(p):
            t = p.what == T_TAG_XOR
            tag[p.ev[t], p.lane[t]] ^= p.arg[t]
            v = p.what == T_VAL_XOR
            self.val[p.ev[v], p.lane[v]] ^= p.arg[v]
        self._ret_applied = True


# ----------------------------------------------------------------------------------------------
# random helpers (no method arithmetic)
# ----------------------------------------------------------------------------------------------

def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _rand_u64(shape, g, device) -> torch.Tensor:
    """Uniform 64-bit patterns as int64."""
    hi = torch.randint(0, 1 << 32, shape, generator=g, device=device, dtype=torch.int64)
    lo = torch.randint(0, 1 << 32, shape, generator=g, device=device, dtype=torch.int64)
    return (hi << 32) | lo


def _zipf_ranks(n: int, n_ranks: int, s: float, g, device) -> torch.Tensor:
    """n draws of a bounded Zipf(s) rank in [0, n_ranks): P(r) ~ (r + 1) ** -s."""
    w = torch.arange(1, n_ranks + 1, dtype=torch.float64, device=device).pow_(-s)
    cdf = torch.cumsum(w, 0)
    cdf /= cdf[-1].clone()
    u = torch.rand(n, generator=g, device=device, dtype=torch.float64)
    return torch.searchsorted(cdf, u).clamp_(max=n_ranks - 1)


def _pack_bits(bits: torch.Tensor) -> torch.Tensor:
    """bool [m, w] -> int64 [m] with bit j = bits[:, j]."""
    w = bits.shape[1]
    sh = torch.arange(w, device=bits.device, dtype=torch.int64)
    if w == 64:  # keep bit 63 out of a signed sum
        lo = (bits[:, :32].to(torch.int64) << sh[:32]).sum(1)
        hi = (bits[:, 32:].to(torch.int64) << sh[:32]).sum(1)
        return (hi << 32) | lo
    return (bits.to(torch.int64) << sh).sum(1)


def _unpack32(mask: torch.Tensor) -> torch.Tensor:
    sh = torch.arange(32, device=mask.device, dtype=torch.int64)
    return ((mask[:, None] >> sh) & 1).bool()


def _k_of_w_bits(k: torch.Tensor, w: int, g, device) -> torch.Tensor:
    """For each row a uniformly random subset of exactly k[i] of w positions, as bool [m, w]."""
    r = torch.rand((k.numel(), w), generator=g, device=device)
    kth = torch.sort(r, dim=1).values.gather(1, (k - 1).clamp(min=0)[:, None])
    return (r <= kth) & (k[:, None] > 0)


def _pick_active_lane(mask: torch.Tensor, g, device) -> torch.Tensor:
    """One uniformly chosen set bit of each (non-zero) mask."""
    bits = _unpack32(mask)
    cs = torch.cumsum(bits.to(torch.int64), 1)
    pc = cs[:, -1]
    j = (torch.rand(mask.numel(), generator=g, device=device, dtype=torch.float64) * pc).long().clamp_(max=31)
    j = torch.minimum(j, (pc - 1).clamp(min=0))
    return ((cs == (j + 1)[:, None]) & bits).to(torch.int64).argmax(1)


def _choose_exact(idx: torch.Tensor, m: int, g, device) -> torch.Tensor:
    """m distinct entries of idx, uniformly."""
    m = min(int(m), int(idx.numel()))
    if m == 0:
        return idx[:0]
    p = torch.randperm(idx.numel(), generator=g, device=device)[:m]
    return idx[p]


# ----------------------------------------------------------------------------------------------
# policies
# ----------------------------------------------------------------------------------------------

def _key_and_digest(g, device):
    k = _rand_u64((3,), g, device).tolist()
    return _u64(k[0]), _u64(k[1]), _u64(k[2])


def _finish_policy(kind_t, sizes_t, window_slots, g, device, k0, k1, dig, disjoint=True) -> Policy:
    """Draw each forward site's targets from the window and lay them out as sorted CSR.

    disjoint=True draws every target of the policy without replacement, so sets of
    different sites never share an address (then any address taken from another site's
    set, or from free_slots, is out of this site's set by construction).
    """
    n_sites = kind_t.numel()
    total = int(sizes_t.sum())
    site_of = torch.repeat_interleave(torch.arange(n_sites, device=device), sizes_t)
    if disjoint:
        assert total <= window_slots
        perm = torch.randperm(window_slots, generator=g, device=device)
        slots = perm[:total]
        free = perm[total:]
        key = (site_of << 32) | slots
        key = torch.sort(key).values
        counts = sizes_t
    else:
        slots = torch.randint(0, window_slots, (total,), generator=g, device=device, dtype=torch.int64)
        key = torch.unique((site_of << 32) | slots)  # sorted, per-site duplicates removed
        counts = torch.bincount(key >> 32, minlength=n_sites)
        fwd = kind_t == PROTECTED_FORWARD
        assert bool((counts[fwd] > 0).all())
        free = None
    tg = CODE_BASE + SLOT_BYTES * (key & 0xFFFFFFFF)
    off = torch.zeros(n_sites + 1, dtype=torch.int64, device=device)
    off[1:] = torch.cumsum(counts, 0)
    return Policy(kind=kind_t.to(torch.uint8).cpu().numpy(),
                  tgt_off=off.cpu().numpy().astype(np.uint32),
                  tgts=tg.cpu().numpy().astype(np.uint64),
                  k0=k0, k1=k1, policy_digest=dig, window_slots=window_slots, free_slots=free)


def _shuffled_kinds(counts: dict, g, device) -> torch.Tensor:
    kinds = torch.cat([torch.full((c,), k, dtype=torch.int64, device=device) for k, c in counts.items()])
    return kinds[torch.randperm(kinds.numel(), generator=g, device=device)]


def _place_sizes(kind_t, fwd_sizes: torch.Tensor, g, device) -> torch.Tensor:
    """Give the forward sites (in a seeded order) the listed set sizes; every other site size 0."""
    sizes = torch.zeros_like(kind_t)
    fwd_idx = torch.nonzero(kind_t == PROTECTED_FORWARD).flatten()
    assert fwd_idx.numel() == fwd_sizes.numel()
    sizes[fwd_idx] = fwd_sizes[torch.randperm(fwd_sizes.numel(), generator=g, device=device)]
    return sizes


# ----------------------------------------------------------------------------------------------
# events
# ----------------------------------------------------------------------------------------------

def _build_events(policy: Policy, site: torch.Tensor, *, mask_mode: str, ret_uniform: float,
                  fwd_uniform: float, g, device, chunk: int = 1 << 20):
    """hdr / val / uniform-flag for the given per-event site ids."""
    n = site.numel()
    kind_t = torch.from_numpy(policy.kind.astype(np.int64)).to(device)
    off_t = torch.from_numpy(policy.tgt_off.astype(np.int64)).to(device)
    tg_t = torch.from_numpy(policy.tgts.view(np.int64)).to(device)
    if tg_t.numel() == 0:
        tg_t = torch.zeros(1, dtype=torch.int64, device=device)
    cnt_t = off_t[1:] - off_t[:-1]
    W = policy.window_slots

    hdr = torch.empty((n, 2), dtype=torch.int64, device=device)
    val = torch.empty((n, 32), dtype=torch.int64, device=device)
    uni = torch.empty(n, dtype=torch.bool, device=device)
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        c = hi - lo
        s = site[lo:hi]
        k = kind_t[s]
        # active masks
        if mask_mode == "p0.9":
            bits = torch.rand((c, 32), generator=g, device=device) < 0.9
        elif mask_mode == "k-uniform":
            kk = torch.randint(1, 33, (c,), generator=g, device=device, dtype=torch.int64)
            bits = _k_of_w_bits(kk, 32, g, device)
        else:
            raise ValueError(mask_mode)
        mask = _pack_bits(bits)
        # context_base = epoch 1 | depth | warp slot, low five bits zero
        depth = torch.randint(0, 8, (c,), generator=g, device=device, dtype=torch.int64)
        slot = torch.randint(0, 1 << 20, (c,), generator=g, device=device, dtype=torch.int64)
        ctx = (1 << 48) | (depth << 37) | (slot << 5)
        hdr[lo:hi, 0] = s | (mask << 32)
        hdr[lo:hi, 1] = ctx
        # lane values: garbage everywhere, then real values in the active lanes of protected events
        v = _rand_u64((c, 32), g, device)
        is_ret = k == PROTECTED_RETURN
        is_fwd = k == PROTECTED_FORWARD
        u = torch.rand(c, generator=g, device=device)
        is_uni = torch.where(is_ret, u < ret_uniform, u < fwd_uniform)
        # returns: 16-byte aligned continuations in the code window
        a_u = torch.randint(0, W, (c, 1), generator=g, device=device, dtype=torch.int64)
        a_d = torch.randint(0, W, (c, 32), generator=g, device=device, dtype=torch.int64)
        addr = CODE_BASE + SLOT_BYTES * torch.where(is_uni[:, None], a_u, a_d)
        v = torch.where(bits & is_ret[:, None], addr, v)
        # forwards: members of the site's own set
        cn = cnt_t[s].clamp(min=1)
        r_u = torch.rand((c, 1), generator=g, device=device, dtype=torch.float64)
        r_d = torch.rand((c, 32), generator=g, device=device, dtype=torch.float64)
        r = torch.where(is_uni[:, None], r_u, r_d)
        pick = off_t[s][:, None] + torch.minimum((r * cn[:, None]).long(), (cn - 1)[:, None])
        pick = torch.where(is_fwd[:, None], pick, torch.zeros_like(pick))
        v = torch.where(bits & is_fwd[:, None], tg_t[pick], v)
        val[lo:hi] = v
        uni[lo:hi] = is_uni & (is_ret | is_fwd)
    return hdr, val, uni


def _plan_return_bitflips(hdr, ret_events, m, g, device, *, max_bits: int = 1, tag_only: bool = False):
    """m return events: one active lane, `tag` or `continuation` (p = 1/2), 1..max_bits distinct bits."""
    ev = _choose_exact(ret_events, m, g, device)
    if ev.numel() == 0:
        return TamperPlan.empty(device)
    mask = (hdr[ev, 0] >> 32) & 0xFFFFFFFF
    ok = mask != 0
    ev, mask = ev[ok], mask[ok]
    lane = _pick_active_lane(mask, g, device)
    nb = torch.randint(1, max_bits + 1, (ev.numel(),), generator=g, device=device, dtype=torch.int64)
    x = _pack_bits(_k_of_w_bits(nb, 64, g, device))
    if tag_only:
        what = torch.full_like(ev, T_TAG_XOR)
    else:
        what = torch.where(torch.rand(ev.numel(), generator=g, device=device) < 0.5, T_TAG_XOR, T_VAL_XOR)
    return TamperPlan(ev, lane, what, x)


def _apply_forward_outofset(policy, hdr, val, uni, fwd_events, m, g, device):
    """m forward events get an address no site allows: the whole warp if uniform, else one lane."""
    ev = _choose_exact(fwd_events, m, g, device)
    if ev.numel() == 0:
        return TamperPlan.empty(device)
    free = policy.free_slots
    assert free is not None and free.numel() > 0
    mask = (hdr[ev, 0] >> 32) & 0xFFFFFFFF
    ok = mask != 0
    ev, mask = ev[ok], mask[ok]
    bad = CODE_BASE + SLOT_BYTES * free[torch.randint(0, free.numel(), (ev.numel(),), generator=g, device=device)]
    lane = _pick_active_lane(mask, g, device)
    u = uni[ev]
    bits = _unpack32(mask)
    rows = val[ev]
    rows = torch.where((bits & u[:, None]) | (~u[:, None] & (torch.arange(32, device=device) == lane[:, None])),
                       bad[:, None], rows)
    val[ev] = rows
    lowest = bits.to(torch.int64).argmax(1)
    return TamperPlan(ev, torch.where(u, lowest, lane), torch.where(u, T_VAL_SET_ALL, T_VAL_SET_LANE), bad)


def _apply_forward_bitflip(hdr, val, fwd_events, m, g, device, *, addr_bits_only: bool = False):
    """m forward events: one active lane's (legal) target XOR one bit."""
    ev = _choose_exact(fwd_events, m, g, device)
    if ev.numel() == 0:
        return TamperPlan.empty(device)
    mask = (hdr[ev, 0] >> 32) & 0xFFFFFFFF
    ok = mask != 0
    ev, mask = ev[ok], mask[ok]
    lane = _pick_active_lane(mask, g, device)
    lo, hi = (4, 28) if addr_bits_only else (0, 64)
    bit = torch.randint(lo, hi, (ev.numel(),), generator=g, device=device, dtype=torch.int64)
    x = torch.ones_like(bit) << bit
    val[ev, lane] ^= x
    return TamperPlan(ev, lane, torch.full_like(ev, T_VAL_XOR), x)


# ----------------------------------------------------------------------------------------------
# the five configs (BASELINE.json "configs")
# ----------------------------------------------------------------------------------------------

# configs 6 and 7 are extra, public-code-SHAPED streams: only the shapes the paper reports —
# a recovered 38-target family at one indirect site and a sealed callback whose wrong-callback run
# records 64 forward-violation checks (Table A10) — no item of any third-party code.
FULL_EVENTS = {1: 65_536, 2: 4_000_000, 3: 16_000_000, 4: 58_000_000, 5: 512_000_000, 6: 50_000, 7: 4_160}
NAMES = {1: "tiny", 2: "backward-only", 3: "forward-only", 4: "mixed-paper-shaped", 5: "stress",
         6: "38-target-family", 7: "wrong-callback-burst"}
DEFAULT_MODE = {1: ENFORCE, 2: ENFORCE, 3: DETECT, 4: ENFORCE, 5: DETECT, 6: ENFORCE, 7: ENFORCE}
BURST_CHECKS = 64
CONFIG5_BATCH = 8_000_000


def make_policy(config: int, device="cpu", *, n_sites: int | None = None, max_set: int = 4096) -> Policy:
    """Policy of config 1..5, seed = config - 1.  n_sites / max_set rescale config 5 only."""
    g = _gen(config - 1, device)
    k0, k1, dig = _key_and_digest(g, device)
    if config == 1:
        kind = _shuffled_kinds({PROTECTED_RETURN: 64, PROTECTED_FORWARD: 8}, g, device)
        sizes = _place_sizes(kind, torch.randint(1, 5, (8,), generator=g, device=device, dtype=torch.int64), g, device)
        return _finish_policy(kind, sizes, 1 << 16, g, device, k0, k1, dig)
    if config == 2:
        kind = torch.full((1343,), PROTECTED_RETURN, dtype=torch.int64, device=device)
        return _finish_policy(kind, torch.zeros_like(kind), 1 << 16, g, device, k0, k1, dig)
    if config == 3:
        kind = torch.full((40,), PROTECTED_FORWARD, dtype=torch.int64, device=device)
        sz = [1] * 40
        picks = torch.rand(114 * 8, generator=g, device=device).tolist()
        it = iter(picks)
        for _ in range(114):  # 40 + 114 = 154 targets, every set 1..16
            open_sites = [i for i in range(40) if sz[i] < 16]
            sz[open_sites[int(next(it) * len(open_sites))]] += 1
        sizes = torch.tensor(sz, dtype=torch.int64, device=device)
        return _finish_policy(kind, sizes, 1 << 16, g, device, k0, k1, dig)
    if config == 4:
        counts = {PROTECTED_RETURN: 1343, PROTECTED_FORWARD: 154, UNSUPPORTED: 15, FALLBACK: 10,
                  PROFILE_EXCLUDED: 99, NO_SURFACE: 5000, FIXED_EDGE: 45000}
        assert sum(counts.values()) == 51621
        kind = _shuffled_kinds(counts, g, device)
        fs = [1] * 109 + [2] * 20 + [3] * 19 + [4, 5, 6, 8, 9, 10]
        sizes = _place_sizes(kind, torch.tensor(fs, dtype=torch.int64, device=device), g, device)
        return _finish_policy(kind, sizes, 1 << 16, g, device, k0, k1, dig)
    if config == 5:
        n_sites = 1_000_000 if n_sites is None else int(n_sites)
        n_fwd = n_sites // 2
        kind = _shuffled_kinds({PROTECTED_RETURN: n_sites - n_fwd, PROTECTED_FORWARD: n_fwd}, g, device)
        u = torch.rand(n_fwd, generator=g, device=device, dtype=torch.float64)
        fs = torch.floor(torch.pow(2.0, u * float(np.log2(max_set)))).long().clamp_(1, max_set)
        sizes = _place_sizes(kind, fs, g, device)
        return _finish_policy(kind, sizes, 1 << 24, g, device, k0, k1, dig, disjoint=False)
    if config == 6:  # one indirect site with a 38-target family, 32 return sites, 8 fixed-edge sites
        kind = _shuffled_kinds({PROTECTED_FORWARD: 1, PROTECTED_RETURN: 32, FIXED_EDGE: 8}, g, device)
        sizes = _place_sizes(kind, torch.tensor([38], dtype=torch.int64, device=device), g, device)
        return _finish_policy(kind, sizes, 1 << 16, g, device, k0, k1, dig)
    if config == 7:  # four sealed callback sites (one legal target each), 8 return sites
        kind = _shuffled_kinds({PROTECTED_FORWARD: 4, PROTECTED_RETURN: 8}, g, device)
        sizes = _place_sizes(kind, torch.ones(4, dtype=torch.int64, device=device), g, device)
        return _finish_policy(kind, sizes, 1 << 16, g, device, k0, k1, dig)
    raise ValueError(f"config {config}")


def make_stream(config: int, device="cpu", *, n_events: int | None = None, policy: Policy | None = None,
                batch_index: int = 0, mode: int | None = None, n_sites: int | None = None,
                max_set: int = 4096, chunk: int = 1 << 20) -> Stream:
    """Config 1..5 stream (n_events rescales it, keeping every proportion).

    For config 5 one call makes ONE batch (default 8 M events) seeded by (4, batch_index);
    even batches are detect, odd batches enforce.
    """
    n = FULL_EVENTS[config] if n_events is None else int(n_events)
    if config == 5 and n_events is None:
        n = CONFIG5_BATCH
    if policy is None:
        policy = make_policy(config, device, n_sites=n_sites, max_set=max_set)
    # batch_index > 0 on configs 1-4 gives the independent streams of the other ranks of a weak-scaling run
    seed = (config - 1) + 1000 + (7919 * (batch_index + 1) if config == 5 else 7919 * batch_index)
    g = _gen(seed, device)
    kind_t = torch.from_numpy(policy.kind.astype(np.int64)).to(device)
    ns = policy.n_sites
    meta: dict = {}

    def zipf_over(kind_sel: torch.Tensor, count: int) -> torch.Tensor:
        ids = torch.nonzero(kind_sel).flatten()
        ids = ids[torch.randperm(ids.numel(), generator=g, device=device)]  # rank -> site
        return ids[_zipf_ranks(count, ids.numel(), 1.1, g, device)]

    if config == 1:
        site = torch.randint(0, ns, (n,), generator=g, device=device, dtype=torch.int64)
        mask_mode, ru, fu = "p0.9", 0.7, 0.9
    elif config == 2:
        site = zipf_over(kind_t == PROTECTED_RETURN, n)
        mask_mode, ru, fu = "p0.9", 0.7, 0.9
    elif config == 3:
        site = torch.randint(0, ns, (n,), generator=g, device=device, dtype=torch.int64)
        mask_mode, ru, fu = "p0.9", 0.7, 0.9
    elif config == 4:
        n_ret = round(n * 38.3 / 58.0)
        n_fwd = round(n * 13.9 / 58.0)
        n_non = n - n_ret - n_fwd
        site = torch.cat([zipf_over(kind_t == PROTECTED_RETURN, n_ret),
                          zipf_over(kind_t == PROTECTED_FORWARD, n_fwd),
                          zipf_over(kind_t >= FIXED_EDGE, n_non)])
        site = site[torch.randperm(n, generator=g, device=device)]  # one interleaved stream
        mask_mode, ru, fu = "p0.9", 0.7, 0.9
        meta.update(n_ret=n_ret, n_fwd=n_fwd, n_non=n_non)
    elif config == 5:
        site = torch.randint(0, ns, (n,), generator=g, device=device, dtype=torch.int64)
        mask_mode, ru, fu = "k-uniform", 0.7, 0.9
    elif config == 6:  # 40 % of the events go through the one gate site
        site = torch.randint(0, ns, (n,), generator=g, device=device, dtype=torch.int64)
        gate = torch.nonzero(kind_t == PROTECTED_FORWARD).flatten()[0]
        site[torch.rand(n, generator=g, device=device) < 0.4] = gate
        mask_mode, ru, fu = "p0.9", 0.7, 0.5
    elif config == 7:  # benign traffic, then one contiguous run of BURST_CHECKS events at one callback site
        site = torch.randint(0, ns, (n,), generator=g, device=device, dtype=torch.int64)
        cb = torch.nonzero(kind_t == PROTECTED_FORWARD).flatten()
        burst_site = cb[int(torch.randint(0, cb.numel(), (1,), generator=g, device=device))]
        b0 = n - BURST_CHECKS - 17
        site[b0:b0 + BURST_CHECKS] = burst_site
        mask_mode, ru, fu = "p0.9", 0.7, 1.0
        meta.update(burst_start=b0, burst_site=int(burst_site))
    else:
        raise ValueError(config)

    hdr, val, uni = _build_events(policy, site, mask_mode=mask_mode, ret_uniform=ru, fwd_uniform=fu,
                                  g=g, device=device, chunk=chunk)
    k_ev = kind_t[site]
    ret_ev = torch.nonzero(k_ev == PROTECTED_RETURN).flatten()
    fwd_ev = torch.nonzero(k_ev == PROTECTED_FORWARD).flatten()

    if config == 1:  # 1 % of events: one bit flipped in the tag or the continuation / target
        rt = _plan_return_bitflips(hdr, ret_ev, round(0.01 * ret_ev.numel()), g, device)
        ft = _apply_forward_bitflip(hdr, val, fwd_ev, round(0.01 * fwd_ev.numel()), g, device)
    elif config == 2:  # 0.1 % single-bit flips in tag or continuation
        rt = _plan_return_bitflips(hdr, ret_ev, round(0.001 * ret_ev.numel()), g, device)
        ft = TamperPlan.empty(device)
    elif config == 3:  # 0.5 % out-of-set targets from the same window
        rt = TamperPlan.empty(device)
        ft = _apply_forward_outofset(policy, hdr, val, uni, fwd_ev, round(0.005 * fwd_ev.numel()), g, device)
    elif config == 4:  # 0.05 % violations on protected events
        rt = _plan_return_bitflips(hdr, ret_ev, round(0.0005 * ret_ev.numel()), g, device)
        ft = _apply_forward_outofset(policy, hdr, val, uni, fwd_ev, round(0.0005 * fwd_ev.numel()), g, device)
    elif config == 6:  # 0.5 % wrong targets at the gate site
        rt = TamperPlan.empty(device)
        ft = _apply_forward_outofset(policy, hdr, val, uni, fwd_ev, round(0.005 * fwd_ev.numel()), g, device)
    elif config == 7:  # every check of the burst carries the wrong callback; nothing else is corrupted
        rt = TamperPlan.empty(device)
        b0 = meta["burst_start"]
        burst = torch.arange(b0, b0 + BURST_CHECKS, device=device)
        burst = burst[(hdr[burst, 0] >> 32) & 0xFFFFFFFF != 0]  # (an empty mask is not a check)
        ft = _apply_forward_outofset(policy, hdr, val, uni, burst, burst.numel(), g, device)
    else:  # config 5: forged tags with 1-8 bit flips; targets one bit away from a legal target
        rt = _plan_return_bitflips(hdr, ret_ev, round(0.01 * ret_ev.numel()), g, device, max_bits=8, tag_only=True)
        ft = _apply_forward_bitflip(hdr, val, fwd_ev, round(0.01 * fwd_ev.numel()), g, device, addr_bits_only=True)

    if mode is None:
        mode = (DETECT if batch_index % 2 == 0 else ENFORCE) if config == 5 else DEFAULT_MODE[config]
    meta.update(config=config, seed=seed, batch_index=batch_index,
                n_return_events=int(ret_ev.numel()), n_forward_events=int(fwd_ev.numel()))
    return Stream(name=NAMES[config], policy=policy, mode=mode, hdr=hdr, val=val, uniform=uni,
                  ret_tamper=rt, fwd_tamper=ft, meta=meta)
