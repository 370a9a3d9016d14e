/* warpguard.h — C ABI of the B200-native protected-site CFI check engine (libwarpguard.so).
 *
 * What it computes: the runtime check path of WarpGuard (arxiv/paper_2606_11871), re-cast from an inline
 * helper called by every instrumented SASS CALL / RET / indirect branch into a batched engine over a stream
 * of per-warp check events.  The three helper calls of PAPER.md:228 (§5.3)
 *     push(site, expected_ret, guard)   check_ret(site, observed_ret, guard)   forward check (site, target, guard)
 * become wg_sign_continuations, wg_verify_continuations and wg_check_forward; `guard` is the event's 32-bit
 * active-lane mask ("lanes with P0=false ... must not be checked").
 *
 * Passages: backward token sign / verify PAPER.md:162-168 (§4.4), 242-248 (§5.5), 258 (§5.6); forward
 * membership PAPER.md:172-180 (§4.5), 250-252 (§5.5); lane granularity PAPER.md:190 (§4.7); detect / enforce and
 * fail closed PAPER.md:196-198 (§4.8), 264-266 (§5.7); outcome kinds and the protected denominator
 * PAPER.md:113 (§3), 127 (§4.1), 145-158 (Table 2), 224 (§5.2).  Where the paper is silent or garbled (the MAC
 * formula is lost at PAPER.md:164-166 and 244-246) the readings R1-R25 of DESIGN.md §2 apply: the token is
 * SipHash-2-4 under the 128-bit backend key over the 24-byte message
 *     LE64(zero-extended site_id) || LE64(continuation) || LE64((context_base & ~31) | lane).
 *
 * General rules
 *  - Every call returns a wg_status; nothing throws or aborts.  Data-dependent conditions (unknown site,
 *    tampered tag, out-of-set target) are never errors: they are verdicts and counters.
 *  - `d_*` arguments are caller-owned DEVICE pointers on the engine's device, 16-byte aligned, valid until
 *    `cuda_stream` has executed the call's work; the engine neither frees nor keeps them.  `h_*` / `desc`
 *    arguments are HOST pointers.  `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *  - Policy tables and counters live in engine-owned device memory ("backend-private state", §5.6;
 *    Table A3).  The key, and everything derived from it, is NOT in device global memory at all: the engine keeps it
 *    host-side and hands it to its kernels as launch parameters (constant bank) — "keys are passed to injected helpers
 *    as instrumentation arguments and are not exposed as ordinary target-writable CUDA objects" — so a
 *    device-side read / write primitive (in scope) finds no key material to read through any pointer
 *    this library hands out or keeps.  The policy tables themselves are, as in the paper, ordinary device memory:
 *    the metadata-integrity profile below authenticates them per check.
 *  - Sign / verify / check enqueue work on `cuda_stream` and return without waiting.  Counters accumulate across
 *    calls until wg_reset_counters (synchronous) or the next successful wg_load_policy.  The *_host calls are
 *    synchronous and run on the engine's own streams: they are not ordered after work still pending on a caller
 *    stream, so synchronise that stream first when both forms are mixed.  Calls of one engine may be in flight on
 *    several caller streams at once (each launch takes its own group ticket from a ring of 64): keep fewer than 64
 *    launches of one engine pending across streams; on a single stream there is no limit.
 *  - There is no CPU fallback: without a CUDA device every call that needs one returns WG_ERR_CUDA.
 */
#ifndef WARPGUARD_H
#define WARPGUARD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wg_engine wg_engine; /* opaque; owns device tables, key, counters */

typedef enum {
  WG_OK = 0,
  WG_ERR_INVALID_ARG = 1, /* NULL / misaligned pointer, bad mode, bad device                         */
  WG_ERR_BAD_POLICY = 2,  /* policy rejected at load; nothing was loaded                             */
  WG_ERR_NO_POLICY = 3,   /* engine handle is NULL or holds no policy                                */
  WG_ERR_CUDA = 4,        /* a CUDA runtime call failed (wg_last_cuda_error gives the code)          */
  WG_ERR_OOM = 5,         /* host or device allocation failed                                        */
  WG_ERR_INTERNAL = 6,    /* an engine invariant does not hold (a bug): nothing returned may be trusted      */
  WG_ERR_STATIC_LIMIT = 7 /* wg_verify_continuations_static: more sites or events than its static scratch holds */
} wg_status;

/* Site outcome kinds: PAPER.md:145-154 (Table 2), "protected" split by edge direction. */
typedef enum {
  WG_KIND_PROTECTED_RETURN = 0,
  WG_KIND_PROTECTED_FORWARD = 1,
  WG_KIND_FIXED_EDGE = 2,
  WG_KIND_UNSUPPORTED = 3,
  WG_KIND_PROFILE_EXCLUDED = 4,
  WG_KIND_FALLBACK = 5,
  WG_KIND_NO_SURFACE = 6,
  WG_KIND_COUNT = 7
} wg_kind;

/* PAPER.md:264 (§5.7): detect-only records and continues; enforce blocks the violating transfer. */
typedef enum { WG_MODE_DETECT = 0, WG_MODE_ENFORCE = 1 } wg_mode;

/* Policy description — HOST pointers, copied by wg_load_policy; the caller keeps ownership.
 * Forward record of PAPER.md:250 {site_id, token, target_count, allowed_targets} as CSR. */
typedef struct {
  uint32_t n_sites;        /* site_id in events is a dense index 0 .. n_sites-1 (R5)      */
  const uint8_t* kind;     /* [n_sites] wg_kind                                                      */
  const uint32_t* tgt_off; /* [n_sites + 1] CSR offsets, tgt_off[0] == 0, non-decreasing             */
  const uint64_t* tgts;    /* [tgt_off[n_sites]] per site strictly ascending; may be NULL if empty   */
  uint64_t key[2];         /* k0, k1 = little-endian 64-bit halves of the 128-bit backend key (R20)  */
  uint64_t policy_digest;  /* stored and echoed by wg_read_counters; wg_load_policy does not check it (R25),  */
                           /* wg_load_policy_bound refuses the policy unless it is the image's digest (R39)   */
} wg_policy_desc;

/* One per-warp check event (16 bytes, little-endian).  context_base packs the caller's epoch / depth /
 * warp slot; its low five bits are reserved: the engine binds lane l to (context_base & ~31) | l (R2). */
typedef struct {
  uint32_t site_id;
  uint32_t active_mask;
  uint64_t context_base;
} wg_event_hdr;

/* Per-event result.  viol_mask: active lanes that failed their check.  allow_mask: lanes whose transfer is
 * released — the active mask in detect mode, active & ~viol in enforce mode. */
typedef struct {
  uint32_t viol_mask;
  uint32_t allow_mask;
} wg_verdict;

/* Global outcome counters, all u64 (26 words).  Only non-empty events at protected sites enter
 * ret_checks / fwd_checks (events) and ret_lanes / fwd_lanes (lane verdicts): the protected denominator
 * of PAPER.md:113, 127, 224.  Names follow the paper's ret_viol / fwd_viol counters (Table 3, Table 5). */
typedef struct {
  uint64_t events_total, events_empty, events_unknown_site, events_misrouted;
  uint64_t events_by_kind[7];
  uint64_t ret_checks, fwd_checks;
  uint64_t ret_lanes, fwd_lanes;
  uint64_t ret_viol, fwd_viol; /* violating lanes */
  uint64_t ret_viol_events, fwd_viol_events;
  uint64_t blocked_lanes, blocked_events; /* enforce mode only */
  uint64_t first_violation_key;           /* min((seq << 5) | lane) over violations; UINT64_MAX if none (R12) */
  uint64_t signed_lanes, sign_skipped_events;
  uint64_t policy_digest, last_mode;
} wg_counters;

typedef struct {
  uint64_t events, lanes_checked, lanes_violation, lanes_blocked;
} wg_site_counters;

/* Load (or replace) the policy, PAPER.md:186 (§4.6), 260 (§5.6): validated BEFORE any state is touched; on
 * failure nothing is loaded and an existing engine keeps its previous policy.
 *   eng     in: address of NULL (create) or of an existing handle (replace); out: the handle.
 *   device  CUDA device ordinal.
 * WG_ERR_BAD_POLICY for: kind >= 7; tgt_off[0] != 0 or decreasing; a set not strictly ascending; a
 * protected-forward site with an empty set; a non-forward site owning targets (R16).
 * A successful load zeroes all counters and the event sequence number. */
wg_status wg_load_policy(wg_engine** eng, int device, const wg_policy_desc* desc);

/* Policy-digest binding ("When an enforcement profile requires a policy digest, a
 * mismatch aborts before the policy is used"; R39).
 * wg_policy_digest: SipHash-2-4 under desc->key over LE64(n_sites) || LE64(n_targets) || kind bytes (zero-padded to
 *   8) || tgt_off as LE32 (zero-padded to 8) || tgts as LE64 — computed on the host, at load time only.
 * wg_load_policy_bound: as wg_load_policy, but desc->policy_digest must equal that digest (else WG_ERR_BAD_POLICY,
 *   nothing loaded), and its low 32 bits are folded into the upper half of every backward token's first message word
 *   (LE64(site_id | digest32 << 32)): tokens signed under one policy image do not verify under another.  The
 *   binding holds until the next load. */
wg_status wg_policy_digest(const wg_policy_desc* desc, uint64_t* h_digest);
wg_status wg_load_policy_bound(wg_engine** eng, int device, const wg_policy_desc* desc);

/* Backward push: d_tag[e][l] = token(site, d_val[e][l], lane context) for every active
 * lane of every event whose site is protected-return, 0 for every other lane (R10).
 *   d_hdr [n] wg_event_hdr, d_val [n][32] u64 in, d_tag [n][32] u64 out.  n == 0 is a no-op. */
wg_status wg_sign_continuations(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                uint64_t* d_tag, uint64_t n, void* cuda_stream);

/* Backward check_ret over a stream that may interleave events of ANY site kind: the engine
 * dispatches on the policy's kind (protected-return: recompute the token over the observed continuation and
 * compare with d_tag; protected-forward: membership, tag row ignored; other kinds: counted only, R17).
 *   d_out [n] wg_verdict out.  mode: WG_MODE_DETECT or WG_MODE_ENFORCE. */
wg_status wg_verify_continuations(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                  const uint64_t* d_tag, wg_verdict* d_out, uint64_t n, wg_mode mode,
                                  void* cuda_stream);

/* Forward check: observed target must be a member of the site's set (exact
 * 64-bit equality, R8).  A protected-return event given to this entry point has no tag and fails closed (R14). */
wg_status wg_check_forward(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                           wg_verdict* d_out, uint64_t n, wg_mode mode, void* cuda_stream);

/* Synchronises `cuda_stream`, then copies the counters to HOST memory (diagnostic only,
 * they never feed a verdict).  h_per_site may be NULL, else [n_sites]. */
wg_status wg_read_counters(wg_engine* eng, wg_counters* h_global, wg_site_counters* h_per_site,
                           void* cuda_stream);

/* ---- lifecycle helpers beside the five ---- */
wg_status wg_reset_counters(wg_engine* eng, void* cuda_stream); /* also restarts the event sequence (R12) */
/* The running event index (R12) the next checked event gets; wg_reset_counters and wg_load_policy set it to 0.  A rank
 * that checks the slice [lo, hi) of a sharded stream ("This property is site-local")
 * sets it to lo, so that first_violation_key, the first-violation record and the ring records carry the stream's own
 * sequence numbers.  Takes effect with the next check call; base <= 2^58. */
wg_status wg_set_sequence_base(wg_engine* eng, uint64_t base);
void wg_destroy(wg_engine* eng);                                /* NULL is allowed */
const char* wg_strerror(wg_status s);
int wg_last_cuda_error(const wg_engine* eng); /* cudaError_t of the last WG_ERR_CUDA, 0 if none */

/* ---- profiles and telemetry (readings R26-R29) ----
 * PAPER.md:196 (§4.8): "Fast or attribution profiles that skip kernels, sites, counters, or a CFI direction change
 * the protected set and are reported under separate denominators"; Table A2 names the
 * profiles; PAPER.md:264-266 (§5.7): counters, telemetry buffers and first-violation records are diagnostic —
 * nothing below ever changes a verdict of a site that stays in the protected set.
 *   WG_PROFILE_SKIP_FORWARD   backward-only: non-empty events at protected-forward sites are not judged
 *                             (viol 0, allow = active); they still count in events_total / events_by_kind /
 *                             site.events, and in skipped_fwd_events / skipped_fwd_lanes.
 *   WG_PROFILE_SKIP_BACKWARD  forward-only: the same for protected-return sites, at both check entry points (such
 *                             an event is then neither verified nor "misrouted").  Signing is unaffected.
 *   WG_PROFILE_LOW_TELEMETRY  low-telemetry enforcement: same verdicts, global counters and first-violation
 *                             record; per-site counters and the violation ring are not updated.
 * The flags are engine configuration: they survive wg_reset_counters and wg_load_policy. */
typedef enum {
  WG_PROFILE_FULL = 0,
  WG_PROFILE_SKIP_FORWARD = 1,
  WG_PROFILE_SKIP_BACKWARD = 2,
  WG_PROFILE_LOW_TELEMETRY = 4,
  /* SURVEY.md §8(f-2), "authenticates the record when metadata integrity is enabled ... The forward
   * metadata token is a MAC over site_id, target_count, and allowed_targets", 258; R37-R38: before the
   * membership test of a non-empty event at a protected-forward site the site's record is re-authenticated —
   * SipHash-2-4_key(LE64(site_id) || LE64(target_count) || LE64(t_0) || ...) over the record as it is NOW in the
   * engine's metadata memory must equal the token computed at wg_load_policy; else every active lane violates (a
   * forward check whose lanes all violate) and fwd_meta_fail_events counts the event. */
  WG_PROFILE_METADATA_INTEGRITY = 8,
  /* Coverage-reduced ("profiles that skip kernels, sites, counters, or a CFI direction change the protected
   * set and are reported under separate denominators"; Table A2; R40): the protected sites
   * flagged with wg_set_skip_sites are left out of the protected set.  A non-empty event at such a site is not judged
   * (viol 0, allow = active) at either check entry point (it is never "misrouted"); it counts in events_total /
   * events_by_kind / site.events and in skipped_site_events / skipped_site_lanes, never in ret_* / fwd_*.  A direction
   * skip takes precedence; flags on sites of other kinds mean nothing; signing is unaffected; without this profile
   * flag the skip set is ignored. */
  WG_PROFILE_COVERAGE_REDUCED = 16
} wg_profile_flags;

/* One record per event with viol_mask != 0: lane = lowest violating lane, observed = d_val[event][lane],
 * stored = d_tag[event][lane] when the event was judged as a return check (else 0), kind = 7 for an unknown
 * site, seq = running event index (R12). */
typedef struct {
  uint64_t seq;
  uint32_t site_id, kind, viol_mask, active_mask, lane, mode;
  uint64_t observed, stored;
} wg_violation_rec; /* 48 bytes */

typedef struct {
  uint64_t skipped_ret_events, skipped_ret_lanes, skipped_fwd_events, skipped_fwd_lanes;
  uint64_t ring_recorded, ring_dropped; /* recorded + dropped == events with viol != 0 since the ring was enabled */
  uint64_t fwd_meta_fail_events;        /* forward records that failed their authentication (metadata integrity) */
  uint64_t skipped_site_events, skipped_site_lanes; /* coverage-reduced profile: non-empty events / their active lanes
                                                       at protected sites of the skip set                         */
  uint64_t kernel_launches;             /* CUDA kernels this engine has enqueued since it was created (diagnostic)  */
} wg_telemetry_counters;
/* The attacker's write into the policy metadata, for tests (the paper treats forward records as ordinary writable
 * GPU memory): what = 0: allowed_targets[index] ^= x (index into the CSR array); what = 1: the
 * stored token of site `index` ^= x.  Synchronises cuda_stream. */
wg_status wg_policy_poke(wg_engine* eng, int what, uint64_t index, uint64_t xor_value, void* cuda_stream);

/* WG_ERR_INVALID_ARG for unknown flag bits.  Applies to the calls made after it returns. */
wg_status wg_set_profile(wg_engine* eng, uint32_t flags);
/* The coverage-reduced profile's skip set: h_skip = [n_sites] bytes in HOST memory, non-zero = skipped; NULL clears
 * the set.  Synchronises cuda_stream; belongs to the loaded policy (the next wg_load_policy clears it). */
wg_status wg_set_skip_sites(wg_engine* eng, const uint8_t* h_skip, void* cuda_stream);
/* Bounded violation ring in engine-owned device memory: `capacity` records (0 = off, the default).  Synchronises
 * `cuda_stream`, reallocates, and restarts the ring empty.  When the ring is full further records are dropped and
 * counted; which records a full ring holds is unspecified (any `capacity` of the violating events), their order
 * in the ring is unspecified too.  Capacity survives wg_reset_counters (which empties the ring). */
wg_status wg_set_ring_capacity(wg_engine* eng, uint64_t capacity, void* cuda_stream);
/* Synchronises `cuda_stream`, then copies to HOST memory: the telemetry counters; the first-violation record
 * (*h_have_first = 0 if none since the last reset; it is the record of first_violation_key and is kept even when
 * the ring overflowed or telemetry is low); up to ring_cap ring records (*h_n_ring = how many were copied).
 * h_first / h_ring may be NULL. */
wg_status wg_read_telemetry(wg_engine* eng, wg_telemetry_counters* h_counters, wg_violation_rec* h_first,
                            int* h_have_first, wg_violation_rec* h_ring, uint64_t ring_cap, uint64_t* h_n_ring,
                            void* cuda_stream);

/* ---- stateful shadow stack (readings R30-R36) ----
 * The steps either side of the MAC in the paper's backward mechanism: "one logical shadow stack per CUDA thread
 * slot ... bounded per-thread depth arrays.  Each shadow entry stores expected_return, callsite_id, depth, and
 * token" (§5.5; 162-166 §4.4; 258 §5.6).  thread slot = (warp_slot, lane), warp_slot = bits 36..5 and
 * epoch = bits 63..48 of context_base (its depth field is ignored: the engine owns the depth).  Entry token:
 *     MAC(key, callsite_id, expected_return, epoch << 48 | depth << 37 | warp_slot << 5 | lane).
 * wg_shadow_push: per active lane, depth == max_depth -> overflow: the lane violates, nothing is written; else
 *   the entry {d_val, site, depth, token} is written and the depth incremented.
 * wg_shadow_check_ret: per active lane, depth == 0 -> underflow: violates; else the entry at depth - 1 is read
 *   and the depth decremented whatever the verdict; the lane violates on (first that applies) entry.depth !=
 *   depth - 1; token != MAC over the entry's own fields under the event's epoch; entry.expected_return != d_val or
 *   entry.callsite_id != site.
 * All active lanes violate and no state changes when: the site is unknown or not protected-return; warp_slot >=
 *   n_warp_slots ("if a launch exceeds the configured capacity, the backward check fails closed instead of
 *   wrapping"); the warp_slot occurs more than once in the call (one call = one lock-step step of distinct warps).
 * The shadow arrays are ordinary device memory in the paper's threat model: wg_shadow_poke is the attacker's write
 * (field 0 expected_return, 1 token, 2 callsite_id, 3 entry depth, 4 the slot's depth counter), used by the tests.
 * d_out: verdicts as for the check calls (allow = active & ~viol in enforce mode). */
typedef struct {
  uint64_t push_events, push_lanes, check_events, check_lanes, empty_events;
  uint64_t overflow_lanes, underflow_lanes, depth_mismatch_lanes, token_mismatch_lanes, target_mismatch_lanes;
  uint64_t non_return_events, slot_overflow_events, slot_conflict_events;
  uint64_t viol_lanes, viol_events, blocked_lanes;
} wg_shadow_counters; /* 16 x u64 */
/* (re)allocates and zeroes the shadow state and its counters; max_depth in 1..64; synchronises cuda_stream.
 * Engine-owned device memory: n_warp_slots x (32 x (4 + 32 x max_depth) + 8) bytes — one 32-byte entry per thread
 * slot and depth, a 4-byte depth counter per thread slot, an 8-byte use count per warp slot. */
wg_status wg_shadow_configure(wg_engine* eng, uint32_t n_warp_slots, uint32_t max_depth, void* cuda_stream);
wg_status wg_shadow_push(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val, wg_verdict* d_out,
                         uint64_t n, wg_mode mode, void* cuda_stream);
wg_status wg_shadow_check_ret(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val, wg_verdict* d_out,
                              uint64_t n, wg_mode mode, void* cuda_stream);
wg_status wg_shadow_read_counters(wg_engine* eng, wg_shadow_counters* h_out, void* cuda_stream);
wg_status wg_shadow_poke(wg_engine* eng, uint32_t warp_slot, uint32_t lane, uint32_t entry_depth, int field,
                         uint64_t xor_value, void* cuda_stream);
wg_status wg_shadow_depth(wg_engine* eng, uint32_t warp_slot, uint32_t lane, uint32_t* h_depth, void* cuda_stream);

/* ---- inline device form (include/warpguard_device.cuh) ----
 * What a kernel needs to run the checks at its own sites: the engine's policy tables and the key-derived SipHash
 * initial state.  Pass the view to the kernel BY VALUE — kernel parameter space is where the paper puts the key
 * ("passed to injected helpers as instrumentation arguments"); never copy it into device global memory.
 * It stays valid until the next wg_load_policy or wg_destroy.  site_recs: 16 bytes per site {kind, set offset, set
 * size, flags}; nothing in device memory is key-derived. */
typedef struct {
  const void* site_recs;
  const uint64_t* targets;
  uint32_t n_sites;
  uint32_t bind_hi;    /* low 32 bits of the policy digest when loaded with wg_load_policy_bound (R39), else 0 */
  uint64_t v_init[4];  /* key xor the SipHash constants: key-equivalent, host / parameter space only           */
} wg_device_view;
wg_status wg_get_device_view(wg_engine* eng, wg_device_view* h_view);

/* ---- HOST-buffer entry points (end-to-end path) ----
 * Same semantics as the calls above but every array is in HOST memory (pinned memory gives full PCIe speed,
 * pageable works).  The engine streams the events through its own double-buffered device staging in chunks,
 * runs the same kernels, and returns after the results are back in h_tag / h_out (synchronous). */
wg_status wg_sign_continuations_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                     uint64_t* h_tag, uint64_t n);
wg_status wg_verify_continuations_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                       const uint64_t* h_tag, wg_verdict* h_out, uint64_t n, wg_mode mode);
wg_status wg_check_forward_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                wg_verdict* h_out, uint64_t n, wg_mode mode);

/* ---- allocation-free verify ----
 * For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it):
 * wg_verify_continuations (same dispatch, same verdicts) with the kernel's scratch memory —
 * the launch's group ticket, the counter words it adds into, the first-violation key, the per-site counters — in ONE
 * static device array of the library (2,098,176 bytes, held by every GPU that loads the library until the process
 * exits) instead of the engine's allocations.  The call performs no cudaMalloc / cudaFree and no allocating library
 * call: memsets, one kernel launch and device-to-device copies, all on `cuda_stream`, nothing synchronous.  The first
 * call on a device also resolves the array's address (cudaGetSymbolAddress: no allocation, but make that call outside
 * graph capture).
 *   STATELESS: the engine's cumulative counters, event sequence (R12), violation ring and first-violation record
 *   are neither read nor changed.  The counters of THIS call alone are returned:
 *   d_counters  DEVICE pointer, out (may be NULL): wg_counters of this call; first_violation_key numbers events from
 *               this call's first event (seq = index into d_hdr); policy_digest and last_mode are 0 in this copy.
 *   d_per_site  DEVICE pointer, out (may be NULL): [n_sites] wg_site_counters of this call.
 *   d_hdr / d_val / d_tag / d_out: as wg_verify_continuations (DEVICE, caller-owned).  The engine's profile flags apply.
 *   n == 0 writes zero counters (key UINT64_MAX) and launches nothing.
 * Limits: the loaded policy has at most WG_STATIC_MAX_SITES sites and n <= WG_STATIC_MAX_EVENTS (one launch), else
 * WG_ERR_STATIC_LIMIT and nothing is written.  Other errors as wg_verify_continuations.
 * SHARED: every call, of every engine and every thread, uses the same array on a device, and the array keeps the last
 * call's contents (each call clears what it needs).  Two calls that overlap on the GPU (different streams, or the same
 * graph launched twice concurrently) race on it: order them on one stream.  d_counters / d_per_site are valid once the
 * stream reaches the end of the call's work. */
#define WG_STATIC_MAX_SITES 65536u
#define WG_STATIC_MAX_EVENTS 134217696ull /* 2^27 - 32 */
wg_status wg_verify_continuations_static(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                         const uint64_t* d_tag, wg_verdict* d_out, wg_counters* d_counters,
                                         wg_site_counters* d_per_site, uint64_t n, wg_mode mode, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* WARPGUARD_H */
