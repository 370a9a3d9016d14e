"""TEST INFRASTRUCTURE ONLY — ctypes face of the CPU oracle (oracle/wg_oracle.cpp).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product package
``paper_2606_11871_b200`` never does, and this package never imports it.

The oracle is built with plain ``g++ -O2`` (no -march, no intrinsics) into
``oracle/libwg_oracle.so``.  All arrays are numpy, host memory.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "wg_oracle.cpp"
_HDR = _HERE / "wg_oracle.h"
_LIB = _HERE / "libwg_oracle.so"

KIND_PROTECTED_RETURN = 0
KIND_PROTECTED_FORWARD = 1
KIND_FIXED_EDGE = 2
KIND_UNSUPPORTED = 3
KIND_PROFILE_EXCLUDED = 4
KIND_FALLBACK = 5
KIND_NO_SURFACE = 6
KIND_COUNT = 7
MODE_DETECT = 0
MODE_ENFORCE = 1

COUNTER_FIELDS = (
    ["events_total", "events_empty", "events_unknown_site", "events_misrouted"]
    + [f"events_by_kind_{k}" for k in range(7)]
    + ["ret_checks", "fwd_checks", "ret_lanes", "fwd_lanes", "ret_viol", "fwd_viol",
       "ret_viol_events", "fwd_viol_events", "blocked_lanes", "blocked_events",
       "first_violation_key", "signed_lanes", "sign_skipped_events", "policy_digest", "last_mode"]
)
assert len(COUNTER_FIELDS) == 26


def build(force: bool = False) -> Path:
    """Compile the oracle if the library is missing or older than its sources."""
    newest = max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
    if force or not _LIB.exists() or _LIB.stat().st_mtime < newest:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        u64, u32, vp = C.c_uint64, C.c_uint32, C.c_void_p
        L.wgo_siphash24.restype = u64
        L.wgo_siphash24.argtypes = [u64, u64, C.c_char_p, C.c_size_t]
        L.wgo_mac.restype = u64
        L.wgo_mac.argtypes = [u64, u64, u32, u64, u64]
        L.wgo_lane_ctx.restype = u64
        L.wgo_lane_ctx.argtypes = [u64, u32]
        L.wgo_validate_policy.restype = C.c_int
        L.wgo_validate_policy.argtypes = [u32, vp, vp, vp]
        L.wgo_create.restype = vp
        L.wgo_create.argtypes = [u32, vp, vp, vp, u64, u64, u64]
        L.wgo_destroy.restype = None
        L.wgo_destroy.argtypes = [vp]
        L.wgo_reset_counters.restype = None
        L.wgo_reset_counters.argtypes = [vp]
        L.wgo_set_binary_search.restype = None
        L.wgo_set_binary_search.argtypes = [vp, C.c_int]
        L.wgo_sign.restype = None
        L.wgo_sign.argtypes = [vp, vp, vp, vp, u64]
        L.wgo_check.restype = None
        L.wgo_check.argtypes = [vp, vp, vp, vp, vp, u64, C.c_int]
        L.wgo_read_counters.restype = None
        L.wgo_read_counters.argtypes = [vp, vp, vp]
        L.wgo_set_profile.restype = None
        L.wgo_set_profile.argtypes = [vp, u32]
        L.wgo_set_skip_sites.restype = None
        L.wgo_set_skip_sites.argtypes = [vp, vp]
        L.wgo_set_sequence_base.restype = None
        L.wgo_set_sequence_base.argtypes = [vp, C.c_uint64]
        L.wgo_set_ring_capacity.restype = None
        L.wgo_set_ring_capacity.argtypes = [vp, u64]
        L.wgo_read_violations.restype = u64
        L.wgo_read_violations.argtypes = [vp, vp, u64]
        L.wgo_read_first_violation.restype = C.c_int
        L.wgo_read_first_violation.argtypes = [vp, vp]
        L.wgo_read_telemetry.restype = None
        L.wgo_read_telemetry.argtypes = [vp, vp]
        L.wgo_policy_digest.restype = u64
        L.wgo_policy_digest.argtypes = [u32, vp, vp, vp, u64, u64]
        L.wgo_create_bound.restype = vp
        L.wgo_create_bound.argtypes = [u32, vp, vp, vp, u64, u64, u64]
        L.wgo_policy_poke.restype = C.c_int
        L.wgo_policy_poke.argtypes = [vp, C.c_int, u64, u64]
        L.wgo_shadow_configure.restype = C.c_int
        L.wgo_shadow_configure.argtypes = [vp, u32, u32]
        L.wgo_shadow_push.restype = None
        L.wgo_shadow_push.argtypes = [vp, vp, vp, vp, u64, C.c_int]
        L.wgo_shadow_check_ret.restype = None
        L.wgo_shadow_check_ret.argtypes = [vp, vp, vp, vp, u64, C.c_int]
        L.wgo_shadow_read_counters.restype = None
        L.wgo_shadow_read_counters.argtypes = [vp, vp]
        L.wgo_shadow_poke.restype = C.c_int
        L.wgo_shadow_poke.argtypes = [vp, u32, u32, u32, C.c_int, u64]
        L.wgo_shadow_depth.restype = u32
        L.wgo_shadow_depth.argtypes = [vp, u32, u32]
        _lib = L
    return _lib


def siphash24(k0: int, k1: int, msg: bytes) -> int:
    return int(lib().wgo_siphash24(k0, k1, msg, len(msg)))


def mac(k0: int, k1: int, site_id: int, value: int, context_id: int) -> int:
    return int(lib().wgo_mac(k0, k1, site_id, value, context_id))


def lane_ctx(context_base: int, lane: int) -> int:
    return int(lib().wgo_lane_ctx(context_base, lane))


def _ptr(a: np.ndarray | None):
    return None if a is None else a.ctypes.data


def _c(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=dtype)


def validate_policy(kind, tgt_off, tgts) -> int:
    kind = _c(kind, np.uint8)
    tgt_off = _c(tgt_off, np.uint32)
    tgts = _c(tgts, np.uint64)
    assert tgt_off.size == kind.size + 1
    return int(lib().wgo_validate_policy(kind.size, _ptr(kind), _ptr(tgt_off), _ptr(tgts)))


def policy_digest(kind, tgt_off, tgts, k0: int, k1: int) -> int:
    kind, tgt_off, tgts = _c(kind, np.uint8), _c(tgt_off, np.uint32), _c(tgts, np.uint64)
    return int(lib().wgo_policy_digest(kind.size, _ptr(kind), _ptr(tgt_off), _ptr(tgts), k0, k1))


def _hdr_bytes(hdr: np.ndarray) -> np.ndarray:
    """Accept [n,2] (u)int64 rows (site | mask<<32, context_base) and return them as raw rows."""
    h = np.ascontiguousarray(hdr)
    assert h.ndim == 2 and h.shape[1] == 2 and h.dtype.itemsize == 8, (h.shape, h.dtype)
    return h.view(np.uint64)


class Oracle:
    """One loaded policy + key + counters (the oracle's analogue of wg_engine)."""

    def __init__(self, kind, tgt_off, tgts, k0: int, k1: int, policy_digest: int = 0, bound: bool = False):
        """bound=True: wgo_create_bound — the image's digest must equal policy_digest and is folded into the tokens."""
        self.kind = _c(kind, np.uint8)
        self.tgt_off = _c(tgt_off, np.uint32)
        self.tgts = _c(tgts, np.uint64)
        assert self.tgt_off.size == self.kind.size + 1
        self.n_sites = int(self.kind.size)
        create = lib().wgo_create_bound if bound else lib().wgo_create
        self._h = create(self.n_sites, _ptr(self.kind), _ptr(self.tgt_off), _ptr(self.tgts), k0, k1, policy_digest)
        if not self._h:
            raise ValueError("oracle rejected the policy (wgo_validate_policy = %d%s)"
                             % (validate_policy(self.kind, self.tgt_off, self.tgts),
                                ", or its digest is not the expected one" if bound else ""))

    def close(self):
        if getattr(self, "_h", None):
            lib().wgo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # interpreter shutdown
            pass

    def reset_counters(self):
        lib().wgo_reset_counters(self._h)

    def set_binary_search(self, on: bool):
        lib().wgo_set_binary_search(self._h, int(bool(on)))

    def sign(self, hdr: np.ndarray, val: np.ndarray) -> np.ndarray:
        h = _hdr_bytes(hdr)
        n = h.shape[0]
        v = np.ascontiguousarray(val).view(np.uint64).reshape(n, 32)
        tag = np.empty((n, 32), dtype=np.uint64)
        lib().wgo_sign(self._h, _ptr(h), _ptr(v), _ptr(tag), n)
        return tag

    def check(self, hdr: np.ndarray, val: np.ndarray, tag: np.ndarray | None, mode: int) -> np.ndarray:
        """Returns [n,2] uint32: (viol_mask, allow_mask).  tag=None is the forward entry point."""
        h = _hdr_bytes(hdr)
        n = h.shape[0]
        v = np.ascontiguousarray(val).view(np.uint64).reshape(n, 32)
        t = None if tag is None else np.ascontiguousarray(tag).view(np.uint64).reshape(n, 32)
        out = np.empty((n, 2), dtype=np.uint32)
        lib().wgo_check(self._h, _ptr(h), _ptr(v), _ptr(t), _ptr(out), n, int(mode))
        return out

    def verify(self, hdr, val, tag, mode):
        assert tag is not None
        return self.check(hdr, val, tag, mode)

    def check_forward(self, hdr, val, mode):
        return self.check(hdr, val, None, mode)

    def read_counters(self, per_site: bool = True):
        g = np.zeros(26, dtype=np.uint64)
        s = np.zeros((self.n_sites, 4), dtype=np.uint64) if per_site else None
        lib().wgo_read_counters(self._h, _ptr(g), _ptr(s))
        return {k: int(v) for k, v in zip(COUNTER_FIELDS, g)}, s

    # ---- profiles and telemetry (wg_oracle.h; R26-R29) ----
    def set_profile(self, flags: int):
        lib().wgo_set_profile(self._h, int(flags))

    def set_skip_sites(self, skip=None):
        """skip: [n_sites] array, non-zero = left out by the coverage-reduced profile (R40); None clears the set."""
        if skip is None:
            lib().wgo_set_skip_sites(self._h, None)
        else:
            a = np.ascontiguousarray(skip, dtype=np.uint8)
            assert a.size == self.n_sites
            lib().wgo_set_skip_sites(self._h, _ptr(a))

    def set_sequence_base(self, base: int):
        lib().wgo_set_sequence_base(self._h, int(base))

    def set_ring_capacity(self, capacity: int):
        lib().wgo_set_ring_capacity(self._h, int(capacity))

    def read_violations(self, cap: int = 1 << 20) -> np.ndarray:
        out = np.zeros(cap, dtype=VIOLATION_DTYPE)
        n = lib().wgo_read_violations(self._h, _ptr(out), cap)
        return out[:n]

    def read_first_violation(self):
        out = np.zeros(1, dtype=VIOLATION_DTYPE)
        ok = lib().wgo_read_first_violation(self._h, _ptr(out))
        return out[0] if ok else None

    def policy_poke(self, what: int, index: int, xor_value: int):
        if lib().wgo_policy_poke(self._h, int(what), int(index), int(xor_value)) != 0:
            raise ValueError("policy_poke: out of range")

    def read_telemetry(self) -> dict:
        t = np.zeros(len(TELEMETRY_FIELDS), dtype=np.uint64)
        lib().wgo_read_telemetry(self._h, _ptr(t))
        return {k: int(v) for k, v in zip(TELEMETRY_FIELDS, t)}


    # ---- stateful shadow stack (wg_oracle.h; R30-R36) ----
    def shadow_configure(self, n_warp_slots: int, max_depth: int):
        if lib().wgo_shadow_configure(self._h, int(n_warp_slots), int(max_depth)) != 0:
            raise ValueError("max_depth must be in 1..64")

    def _shadow(self, fn, hdr, val, mode):
        hdr = _hdr_bytes(hdr)
        val = _c(val, np.uint64)
        n = hdr.shape[0]
        out = np.zeros((n, 2), dtype=np.uint32)
        fn(self._h, _ptr(hdr), _ptr(val), _ptr(out), n, int(mode))
        return out

    def shadow_push(self, hdr, val, mode):
        return self._shadow(lib().wgo_shadow_push, hdr, val, mode)

    def shadow_check_ret(self, hdr, val, mode):
        return self._shadow(lib().wgo_shadow_check_ret, hdr, val, mode)

    def shadow_read_counters(self) -> dict:
        c = np.zeros(16, dtype=np.uint64)
        lib().wgo_shadow_read_counters(self._h, _ptr(c))
        return {k: int(v) for k, v in zip(SHADOW_FIELDS, c)}

    def shadow_poke(self, warp_slot: int, lane: int, entry_depth: int, field: int, xor_value: int):
        if lib().wgo_shadow_poke(self._h, int(warp_slot), int(lane), int(entry_depth), int(field), int(xor_value)) != 0:
            raise ValueError("shadow_poke: out of range")

    def shadow_depth(self, warp_slot: int, lane: int) -> int:
        return int(lib().wgo_shadow_depth(self._h, int(warp_slot), int(lane)))


PROFILE_SKIP_FORWARD, PROFILE_SKIP_BACKWARD, PROFILE_LOW_TELEMETRY, PROFILE_METADATA_INTEGRITY = 1, 2, 4, 8
PROFILE_COVERAGE_REDUCED = 16
VIOLATION_DTYPE = np.dtype([("seq", "<u8"), ("site_id", "<u4"), ("kind", "<u4"), ("viol_mask", "<u4"),
                            ("active_mask", "<u4"), ("lane", "<u4"), ("mode", "<u4"), ("observed", "<u8"),
                            ("stored", "<u8")])
TELEMETRY_FIELDS = ("skipped_ret_events", "skipped_ret_lanes", "skipped_fwd_events", "skipped_fwd_lanes",
                    "ring_recorded", "ring_dropped", "fwd_meta_fail_events", "skipped_site_events", "skipped_site_lanes")
SHADOW_FIELDS = ("push_events", "push_lanes", "check_events", "check_lanes", "empty_events", "overflow_lanes",
                 "underflow_lanes", "depth_mismatch_lanes", "token_mismatch_lanes", "target_mismatch_lanes",
                 "non_return_events", "slot_overflow_events", "slot_conflict_events", "viol_lanes", "viol_events",
                 "blocked_lanes")
POKE_EXPECTED, POKE_TOKEN, POKE_CALLSITE, POKE_ENTRY_DEPTH, POKE_DEPTH_COUNTER = 0, 1, 2, 3, 4
