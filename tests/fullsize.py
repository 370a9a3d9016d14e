"""Whole-stream parity at BASELINE.json's full sizes: the oracle judges EVERY event — no
sampling — by running P = os.cpu_count() single-threaded oracle processes over disjoint slices of each chunk of the
stream.  Events are independent given the policy, so the slices' verdicts concatenate and their
counters add (first-violation key: the minimum; each slice keeps the stream's own sequence numbers through
wgo_set_sequence_base).  Test infrastructure: the only thing run in the child processes is `oracle/`.

Children are forked (they inherit the chunk's numpy arrays and the policy without a copy) and never touch CUDA."""
from __future__ import annotations

import multiprocessing as mp
import os

import numpy as np

import oracle

_G = {}  # what the forked workers read: policy, chunk arrays, mode, options


def _work(args):
    lo, hi, seq_lo, op = args
    pol = _G["policy"]
    orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
    if _G.get("binary_search"):
        orc.set_binary_search(True)
    hdr, val = _G["hdr"][lo:hi], _G["val"][lo:hi]
    if op == "sign":
        tags = orc.sign(hdr, val)
        g, _ = orc.read_counters(per_site=False)
        return lo, hi, tags, g, None
    orc.set_sequence_base(seq_lo)
    out = orc.verify(hdr, val, _G["tag"][lo:hi], _G["mode"])
    g, s = orc.read_counters()
    nz = np.nonzero(s.any(axis=1))[0]  # per-site counters travel sparse
    return lo, hi, out, g, (nz, s[nz])


def n_procs() -> int:
    return max(1, min(os.cpu_count() or 1, 32))


def oracle_chunk(policy, op: str, hdr: np.ndarray, val: np.ndarray, tag: np.ndarray | None, mode: int, seq_base: int,
                 binary_search: bool = False):
    """Runs the oracle over one chunk with all cores.  Returns (tags or verdicts [n, ...], summed global counters dict,
    per-site counters [n_sites, 4] or None).  seq_base: sequence number of the chunk's first event."""
    n = hdr.shape[0]
    P = n_procs()
    _G.update(policy=policy, hdr=hdr, val=val, tag=tag, mode=mode, binary_search=binary_search)
    bounds = [n * i // P for i in range(P + 1)]
    jobs = [(bounds[i], bounds[i + 1], seq_base + bounds[i], op) for i in range(P) if bounds[i + 1] > bounds[i]]
    with mp.get_context("fork").Pool(len(jobs)) as pool:
        parts = pool.map(_work, jobs)
    parts.sort(key=lambda t: t[0])
    res = np.concatenate([p[2] for p in parts])
    g = dict(parts[0][3])
    none = (1 << 64) - 1
    for p in parts[1:]:
        for k, v in p[3].items():
            if k == "first_violation_key":
                g[k] = min(g[k], v)
            elif k in ("policy_digest", "last_mode"):
                pass
            else:
                g[k] += v
    site = None
    if op != "sign":
        site = np.zeros((policy.n_sites, 4), dtype=np.uint64)
        for p in parts:
            nz, rows = p[4]
            site[nz] += rows
    assert g["first_violation_key"] <= none
    return res, g, site


def add_counters(total: dict | None, g: dict) -> dict:
    """Counters of consecutive chunks of one call sequence add up (key: minimum)."""
    if total is None:
        return dict(g)
    for k, v in g.items():
        if k == "first_violation_key":
            total[k] = min(total[k], v)
        elif k in ("policy_digest", "last_mode"):
            total[k] = v
        else:
            total[k] += v
    return total
