"""Thin ctypes face of the C-ABI library ``libwarpguard.so`` (include/warpguard.h), same names.

Argument marshalling only: ``tensor.data_ptr()``, sizes and the current CUDA stream are handed to the
library; every step of the check path (MAC, membership, verdicts, counters) runs in its CUDA kernels.
There is no CPU fallback: a missing library, or a box without a CUDA device, raises.

Tensors follow ``streams.py``: ``hdr`` int64 [n, 2] (the little-endian image of ``wg_event_hdr``),
``val`` / ``tag`` int64 [n, 32], ``out`` int32 [n, 2] = (viol_mask, allow_mask).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libwarpguard.so"

WG_OK, WG_ERR_INVALID_ARG, WG_ERR_BAD_POLICY, WG_ERR_NO_POLICY, WG_ERR_CUDA, WG_ERR_OOM, WG_ERR_INTERNAL = range(7)
WG_ERR_STATIC_LIMIT = 7
WG_STATIC_MAX_SITES, WG_STATIC_MAX_EVENTS = 65536, (1 << 27) - 32  # wg_verify_continuations_static
WG_MODE_DETECT, WG_MODE_ENFORCE = 0, 1

EXPORTS = [
    "wg_load_policy", "wg_sign_continuations", "wg_verify_continuations", "wg_check_forward", "wg_read_counters",
    "wg_reset_counters", "wg_set_sequence_base", "wg_set_skip_sites", "wg_destroy", "wg_strerror", "wg_last_cuda_error",
    "wg_sign_continuations_host", "wg_verify_continuations_host", "wg_check_forward_host",
    "wg_set_profile", "wg_set_ring_capacity", "wg_read_telemetry",
    "wg_shadow_configure", "wg_shadow_push", "wg_shadow_check_ret", "wg_shadow_read_counters", "wg_shadow_poke",
    "wg_shadow_depth", "wg_policy_poke", "wg_get_device_view", "wg_policy_digest",
    "wg_load_policy_bound", "wg_verify_continuations_static",
]


class DeviceView(C.Structure):
    """wg_device_view: pass it by value to a kernel that uses include/warpguard_device.cuh"""
    _fields_ = [("site_recs", C.c_void_p), ("targets", C.c_void_p), ("n_sites", C.c_uint32), ("bind_hi", C.c_uint32),
                ("v_init", C.c_uint64 * 4)]
SHADOW_FIELDS = ("push_events", "push_lanes", "check_events", "check_lanes", "empty_events", "overflow_lanes",
                 "underflow_lanes", "depth_mismatch_lanes", "token_mismatch_lanes", "target_mismatch_lanes",
                 "non_return_events", "slot_overflow_events", "slot_conflict_events", "viol_lanes", "viol_events",
                 "blocked_lanes")

WG_PROFILE_FULL, WG_PROFILE_SKIP_FORWARD, WG_PROFILE_SKIP_BACKWARD, WG_PROFILE_LOW_TELEMETRY = 0, 1, 2, 4
WG_PROFILE_METADATA_INTEGRITY = 8
WG_PROFILE_COVERAGE_REDUCED = 16
VIOLATION_DTYPE = np.dtype([("seq", "<u8"), ("site_id", "<u4"), ("kind", "<u4"), ("viol_mask", "<u4"),
                            ("active_mask", "<u4"), ("lane", "<u4"), ("mode", "<u4"), ("observed", "<u8"),
                            ("stored", "<u8")])  # wg_violation_rec, 48 bytes
TELEMETRY_FIELDS = ("skipped_ret_events", "skipped_ret_lanes", "skipped_fwd_events", "skipped_fwd_lanes",
                    "ring_recorded", "ring_dropped", "fwd_meta_fail_events", "skipped_site_events", "skipped_site_lanes")
# words of wg_telemetry_counters behind TELEMETRY_FIELDS that have no counterpart in the method (engine diagnostics)
TELEMETRY_ENGINE_FIELDS = ("kernel_launches",)

COUNTER_FIELDS = (
    ["events_total", "events_empty", "events_unknown_site", "events_misrouted"]
    + [f"events_by_kind_{k}" for k in range(7)]
    + ["ret_checks", "fwd_checks", "ret_lanes", "fwd_lanes", "ret_viol", "fwd_viol",
       "ret_viol_events", "fwd_viol_events", "blocked_lanes", "blocked_events",
       "first_violation_key", "signed_lanes", "sign_skipped_events", "policy_digest", "last_mode"]
)


class WgError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: wg_status {status} ({strerror(status)})")


class _PolicyDesc(C.Structure):
    _fields_ = [("n_sites", C.c_uint32), ("kind", C.c_void_p), ("tgt_off", C.c_void_p), ("tgts", C.c_void_p),
                ("key", C.c_uint64 * 2), ("policy_digest", C.c_uint64)]


_lib = None


def lib() -> C.CDLL:
    """Loads libwarpguard.so (built in-tree by ``python -m paper_2606_11871_b200.build``).  Fails loudly."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_11871_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, u64, i = C.c_void_p, C.c_uint64, C.c_int
        L.wg_load_policy.argtypes = [C.POINTER(vp), i, C.POINTER(_PolicyDesc)]
        L.wg_load_policy_bound.argtypes = [C.POINTER(vp), i, C.POINTER(_PolicyDesc)]
        L.wg_policy_digest.argtypes = [C.POINTER(_PolicyDesc), C.POINTER(u64)]
        L.wg_sign_continuations.argtypes = [vp, vp, vp, vp, u64, vp]
        L.wg_verify_continuations.argtypes = [vp, vp, vp, vp, vp, u64, i, vp]
        L.wg_check_forward.argtypes = [vp, vp, vp, vp, u64, i, vp]
        L.wg_read_counters.argtypes = [vp, vp, vp, vp]
        L.wg_reset_counters.argtypes = [vp, vp]
        L.wg_set_sequence_base.argtypes = [vp, u64]
        L.wg_set_skip_sites.argtypes = [vp, vp, vp]
        L.wg_destroy.argtypes = [vp]
        L.wg_destroy.restype = None
        L.wg_strerror.argtypes = [i]
        L.wg_strerror.restype = C.c_char_p
        L.wg_last_cuda_error.argtypes = [vp]
        L.wg_sign_continuations_host.argtypes = [vp, vp, vp, vp, u64]
        L.wg_verify_continuations_host.argtypes = [vp, vp, vp, vp, vp, u64, i]
        L.wg_check_forward_host.argtypes = [vp, vp, vp, vp, u64, i]
        L.wg_shadow_configure.argtypes = [vp, C.c_uint32, C.c_uint32, vp]
        L.wg_shadow_push.argtypes = [vp, vp, vp, vp, u64, i, vp]
        L.wg_shadow_check_ret.argtypes = [vp, vp, vp, vp, u64, i, vp]
        L.wg_shadow_read_counters.argtypes = [vp, vp, vp]
        L.wg_shadow_poke.argtypes = [vp, C.c_uint32, C.c_uint32, C.c_uint32, i, u64, vp]
        L.wg_shadow_depth.argtypes = [vp, C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32), vp]
        L.wg_set_profile.argtypes = [vp, C.c_uint32]
        L.wg_policy_poke.argtypes = [vp, i, u64, u64, vp]
        L.wg_get_device_view.argtypes = [vp, C.POINTER(DeviceView)]
        L.wg_set_ring_capacity.argtypes = [vp, u64, vp]
        L.wg_read_telemetry.argtypes = [vp, vp, vp, C.POINTER(C.c_int), vp, u64, C.POINTER(u64), vp]
        L.wg_verify_continuations_static.argtypes = [vp, vp, vp, vp, vp, vp, vp, u64, i, vp]
        for name in EXPORTS:
            if name not in ("wg_destroy", "wg_strerror"):
                getattr(L, name).restype = i
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().wg_strerror(int(status)).decode()


def _chk(status: int, what: str) -> None:
    if status != WG_OK:
        raise WgError(status, what)


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev(t: torch.Tensor, what: str, cols: int, itemsize: int) -> int:
    if not t.is_cuda:
        raise ValueError(f"{what} must be a CUDA tensor (use the *_host calls for host buffers)")
    if not t.is_contiguous() or t.element_size() != itemsize or (t.dim() != 2 or t.shape[1] != cols):
        raise ValueError(f"{what}: expected a contiguous [n, {cols}] tensor of {itemsize}-byte elements, "
                         f"got {tuple(t.shape)} {t.dtype}")
    return t.data_ptr()


def _host(t: torch.Tensor, what: str, cols: int, itemsize: int) -> int:
    if t.is_cuda:
        raise ValueError(f"{what} must be a host tensor")
    if not t.is_contiguous() or t.element_size() != itemsize or (t.dim() != 2 or t.shape[1] != cols):
        raise ValueError(f"{what}: expected a contiguous [n, {cols}] tensor of {itemsize}-byte elements")
    return t.data_ptr()


class Engine:
    """Owner of one ``wg_engine*``.  Method names are the C-ABI's."""

    def __init__(self, device: int | None = None):
        self._h = C.c_void_p(None)
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.n_sites = 0

    # -- wg_load_policy ---------------------------------------------------------------------------
    def wg_load_policy(self, kind, tgt_off, tgts, k0: int, k1: int, policy_digest: int = 0, bound: bool = False) -> None:
        """bound=True calls wg_load_policy_bound: policy_digest must be the image's digest (wg_policy_digest)."""
        kind = np.ascontiguousarray(kind, dtype=np.uint8)
        tgt_off = np.ascontiguousarray(tgt_off, dtype=np.uint32)
        tgts = np.ascontiguousarray(tgts, dtype=np.uint64)
        if tgt_off.size != kind.size + 1:
            raise ValueError("tgt_off must have n_sites + 1 entries")
        d = _PolicyDesc()
        d.n_sites = kind.size
        d.kind = kind.ctypes.data if kind.size else None
        d.tgt_off = tgt_off.ctypes.data
        d.tgts = tgts.ctypes.data if tgts.size else None
        d.key[0] = k0 & (2**64 - 1)
        d.key[1] = k1 & (2**64 - 1)
        d.policy_digest = policy_digest & (2**64 - 1)
        if bound:
            _chk(lib().wg_load_policy_bound(C.byref(self._h), self.device, C.byref(d)), "wg_load_policy_bound")
        else:
            _chk(lib().wg_load_policy(C.byref(self._h), self.device, C.byref(d)), "wg_load_policy")
        self.n_sites = int(kind.size)

    def load(self, policy) -> "Engine":
        self.wg_load_policy(policy.kind, policy.tgt_off, policy.tgts, policy.k0, policy.k1, policy.policy_digest)
        return self

    # -- device-buffer calls ----------------------------------------------------------------------
    def wg_sign_continuations(self, hdr, val, tag=None, stream=None) -> torch.Tensor:
        n = hdr.shape[0]
        if tag is None:
            tag = torch.empty((n, 32), dtype=torch.int64, device=hdr.device)
        _chk(lib().wg_sign_continuations(self._h, _dev(hdr, "hdr", 2, 8), _dev(val, "val", 32, 8),
                                         _dev(tag, "tag", 32, 8), n, _stream_ptr(stream)), "wg_sign_continuations")
        return tag

    def wg_verify_continuations(self, hdr, val, tag, mode: int, out=None, stream=None) -> torch.Tensor:
        n = hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32, device=hdr.device)
        _chk(lib().wg_verify_continuations(self._h, _dev(hdr, "hdr", 2, 8), _dev(val, "val", 32, 8),
                                           _dev(tag, "tag", 32, 8), _dev(out, "out", 2, 4), n, int(mode),
                                           _stream_ptr(stream)), "wg_verify_continuations")
        return out

    def wg_verify_continuations_static(self, hdr, val, tag, mode: int, out=None, counters=None, per_site=None,
                                       stream=None):
        """The allocation-free verify (warpguard.h): scratch in the library's static device array, stateless.
        out [n, 2] int32, counters [26] int64, per_site [n_sites, 4] int64: CUDA tensors the CALLER passes (the library
        allocates nothing; tensors left out are made here, by torch).  Returns (out, counters, per_site); all three are
        valid once `stream` has passed the call's work — counter_dict() synchronises and decodes."""
        n = hdr.shape[0]
        dev = hdr.device
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32, device=dev)
        if counters is None:
            counters = torch.empty(26, dtype=torch.int64, device=dev)
        if per_site is None:
            per_site = torch.empty((self.n_sites, 4), dtype=torch.int64, device=dev)
        if not (counters.is_cuda and counters.is_contiguous() and counters.numel() == 26 and counters.element_size() == 8):
            raise ValueError("counters: expected a contiguous CUDA tensor of 26 8-byte words")
        if not (per_site.is_cuda and per_site.is_contiguous() and tuple(per_site.shape) == (self.n_sites, 4)
                and per_site.element_size() == 8):
            raise ValueError(f"per_site: expected a contiguous CUDA [{self.n_sites}, 4] tensor of 8-byte words")
        _chk(lib().wg_verify_continuations_static(
            self._h, _dev(hdr, "hdr", 2, 8), _dev(val, "val", 32, 8), _dev(tag, "tag", 32, 8), _dev(out, "out", 2, 4),
            C.c_void_p(counters.data_ptr()), C.c_void_p(per_site.data_ptr() if self.n_sites else None), n, int(mode),
            _stream_ptr(stream)), "wg_verify_continuations_static")
        return out, counters, per_site

    @staticmethod
    def counter_dict(counters: torch.Tensor) -> dict:
        """Decodes the 26 words wg_verify_continuations_static wrote (synchronises through the copy to the host)."""
        g = counters.cpu().numpy().view(np.uint64)
        return {k: int(v) for k, v in zip(COUNTER_FIELDS, g)}

    def wg_check_forward(self, hdr, val, mode: int, out=None, stream=None) -> torch.Tensor:
        n = hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32, device=hdr.device)
        _chk(lib().wg_check_forward(self._h, _dev(hdr, "hdr", 2, 8), _dev(val, "val", 32, 8),
                                    _dev(out, "out", 2, 4), n, int(mode), _stream_ptr(stream)), "wg_check_forward")
        return out

    # -- host-buffer calls (end-to-end path) ------------------------------------------------------
    def wg_sign_continuations_host(self, hdr, val, tag=None) -> torch.Tensor:
        n = hdr.shape[0]
        if tag is None:
            tag = torch.empty((n, 32), dtype=torch.int64)
        _chk(lib().wg_sign_continuations_host(self._h, _host(hdr, "hdr", 2, 8), _host(val, "val", 32, 8),
                                              _host(tag, "tag", 32, 8), n), "wg_sign_continuations_host")
        return tag

    def wg_verify_continuations_host(self, hdr, val, tag, mode: int, out=None) -> torch.Tensor:
        n = hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32)
        _chk(lib().wg_verify_continuations_host(self._h, _host(hdr, "hdr", 2, 8), _host(val, "val", 32, 8),
                                                _host(tag, "tag", 32, 8), _host(out, "out", 2, 4), n, int(mode)),
             "wg_verify_continuations_host")
        return out

    def wg_check_forward_host(self, hdr, val, mode: int, out=None) -> torch.Tensor:
        n = hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32)
        _chk(lib().wg_check_forward_host(self._h, _host(hdr, "hdr", 2, 8), _host(val, "val", 32, 8),
                                         _host(out, "out", 2, 4), n, int(mode)), "wg_check_forward_host")
        return out

    # -- counters ---------------------------------------------------------------------------------
    def wg_read_counters(self, per_site: bool = True, stream=None):
        g = np.zeros(26, dtype=np.uint64)
        s = np.zeros((self.n_sites, 4), dtype=np.uint64) if per_site else None
        _chk(lib().wg_read_counters(self._h, g.ctypes.data, None if s is None or s.size == 0 else s.ctypes.data,
                                    _stream_ptr(stream)), "wg_read_counters")
        return {k: int(v) for k, v in zip(COUNTER_FIELDS, g)}, s

    # -- stateful shadow stack (warpguard.h; R30-R36) -------------------------------------
    def wg_shadow_configure(self, n_warp_slots: int, max_depth: int, stream=None) -> None:
        _chk(lib().wg_shadow_configure(self._h, int(n_warp_slots), int(max_depth), _stream_ptr(stream)),
             "wg_shadow_configure")

    def _shadow(self, fn, what, hdr, val, mode, out, stream):
        n = hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32, device=hdr.device)
        _chk(fn(self._h, _dev(hdr, "hdr", 2, 8), _dev(val, "val", 32, 8), _dev(out, "out", 2, 4), n, int(mode),
                _stream_ptr(stream)), what)
        return out

    def wg_shadow_push(self, hdr, val, mode: int, out=None, stream=None) -> torch.Tensor:
        return self._shadow(lib().wg_shadow_push, "wg_shadow_push", hdr, val, mode, out, stream)

    def wg_shadow_check_ret(self, hdr, val, mode: int, out=None, stream=None) -> torch.Tensor:
        return self._shadow(lib().wg_shadow_check_ret, "wg_shadow_check_ret", hdr, val, mode, out, stream)

    def wg_shadow_read_counters(self, stream=None) -> dict:
        c = np.zeros(16, dtype=np.uint64)
        _chk(lib().wg_shadow_read_counters(self._h, c.ctypes.data, _stream_ptr(stream)), "wg_shadow_read_counters")
        return {k: int(v) for k, v in zip(SHADOW_FIELDS, c)}

    def wg_shadow_poke(self, warp_slot: int, lane: int, entry_depth: int, field: int, xor_value: int, stream=None):
        _chk(lib().wg_shadow_poke(self._h, int(warp_slot), int(lane), int(entry_depth), int(field), int(xor_value),
                                  _stream_ptr(stream)), "wg_shadow_poke")

    def wg_shadow_depth(self, warp_slot: int, lane: int, stream=None) -> int:
        d = C.c_uint32(0)
        _chk(lib().wg_shadow_depth(self._h, int(warp_slot), int(lane), C.byref(d), _stream_ptr(stream)),
             "wg_shadow_depth")
        return int(d.value)

    # -- profiles and telemetry (warpguard.h; R26-R29) ----------------------------------
    def wg_set_profile(self, flags: int) -> None:
        _chk(lib().wg_set_profile(self._h, int(flags)), "wg_set_profile")

    def wg_set_skip_sites(self, skip=None, stream=None) -> None:
        """skip: [n_sites] array, non-zero = left out by the coverage-reduced profile; None clears the set."""
        if skip is None:
            _chk(lib().wg_set_skip_sites(self._h, None, _stream_ptr(stream)), "wg_set_skip_sites")
            return
        a = np.ascontiguousarray(skip, dtype=np.uint8)
        if a.size != self.n_sites:
            raise ValueError("skip must have n_sites entries")
        _chk(lib().wg_set_skip_sites(self._h, a.ctypes.data, _stream_ptr(stream)), "wg_set_skip_sites")

    def wg_set_sequence_base(self, base: int) -> None:
        _chk(lib().wg_set_sequence_base(self._h, int(base)), "wg_set_sequence_base")

    def wg_get_device_view(self) -> DeviceView:
        v = DeviceView()
        _chk(lib().wg_get_device_view(self._h, C.byref(v)), "wg_get_device_view")
        return v

    def wg_policy_poke(self, what: int, index: int, xor_value: int, stream=None) -> None:
        _chk(lib().wg_policy_poke(self._h, int(what), int(index), int(xor_value), _stream_ptr(stream)), "wg_policy_poke")

    def wg_set_ring_capacity(self, capacity: int, stream=None) -> None:
        _chk(lib().wg_set_ring_capacity(self._h, int(capacity), _stream_ptr(stream)), "wg_set_ring_capacity")

    def wg_read_telemetry(self, ring_cap: int = 0, stream=None):
        """(telemetry counters dict, first-violation record or None, ring records as a structured array)."""
        t = np.zeros(len(TELEMETRY_FIELDS) + len(TELEMETRY_ENGINE_FIELDS), dtype=np.uint64)
        first = np.zeros(1, dtype=VIOLATION_DTYPE)
        have = C.c_int(0)
        ring = np.zeros(max(int(ring_cap), 1), dtype=VIOLATION_DTYPE)
        n = C.c_uint64(0)
        _chk(lib().wg_read_telemetry(self._h, t.ctypes.data, first.ctypes.data, C.byref(have),
                                     ring.ctypes.data if ring_cap else None, int(ring_cap), C.byref(n),
                                     _stream_ptr(stream)), "wg_read_telemetry")
        self.kernel_launches = int(t[len(TELEMETRY_FIELDS)])
        return ({k: int(v) for k, v in zip(TELEMETRY_FIELDS, t)}, first[0] if have.value else None,
                ring[: n.value] if ring_cap else ring[:0])

    def wg_kernel_launches(self) -> int:
        """wg_telemetry_counters.kernel_launches: CUDA kernels this engine has enqueued since it was created."""
        t = np.zeros(len(TELEMETRY_FIELDS) + len(TELEMETRY_ENGINE_FIELDS), dtype=np.uint64)
        _chk(lib().wg_read_telemetry(self._h, t.ctypes.data, None, None, None, 0, None, _stream_ptr(None)),
             "wg_read_telemetry")
        return int(t[len(TELEMETRY_FIELDS)])

    def wg_reset_counters(self, stream=None) -> None:
        _chk(lib().wg_reset_counters(self._h, _stream_ptr(stream)), "wg_reset_counters")

    def wg_destroy(self) -> None:
        if self._h:
            lib().wg_destroy(self._h)
            self._h = C.c_void_p(None)

    close = wg_destroy

    def __del__(self):
        try:
            self.wg_destroy()
        except Exception:  # interpreter shutdown
            pass


def wg_policy_digest(kind, tgt_off, tgts, k0: int, k1: int) -> int:
    """Digest of a policy image (warpguard.h): host-side, no GPU needed."""
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    tgt_off = np.ascontiguousarray(tgt_off, dtype=np.uint32)
    tgts = np.ascontiguousarray(tgts, dtype=np.uint64)
    d = _PolicyDesc()
    d.n_sites = kind.size
    d.kind = kind.ctypes.data if kind.size else None
    d.tgt_off = tgt_off.ctypes.data
    d.tgts = tgts.ctypes.data if tgts.size else None
    d.key[0] = k0 & (2**64 - 1)
    d.key[1] = k1 & (2**64 - 1)
    out = C.c_uint64(0)
    _chk(lib().wg_policy_digest(C.byref(d), C.byref(out)), "wg_policy_digest")
    return int(out.value)
