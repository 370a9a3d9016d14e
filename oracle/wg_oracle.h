/* wg_oracle.h — TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded CPU oracle for the WarpGuard protected-site CFI
 * check path (arxiv/paper_2606_11871).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * The product (paper_2606_11871_b200/, include/warpguard.h) shares no code,
 * header, table or constant with it; the layouts below are re-declared here on
 * purpose.
 *
 * Everything the oracle computes is an integer function of (policy, key,
 * events, mode, call order), so there is exactly one correct result and the
 * CUDA path must match it bit for bit (SURVEY.md §8(c) "Nature of the result").
 *
 * Passages followed (PAPER.md line numbers):
 *   backward push / check_ret ..... 162-168 (§4.4), 228 (§5.3), 242-248 (§5.5), 258 (§5.6)
 *   forward membership ............ 172-180 (§4.5), 250-252 (§5.5)
 *   lane granularity, guards ...... 190 (§4.7), 230 (§5.3)
 *   detect / enforce .............. 196-198 (§4.8), 264-266 (§5.7)
 *   accounting .................... 113 (§3), 127 (§4.1), 145-158 (Table 2), 224 (§5.2)
 *   MAC primitive ................. the paper's formula is lost in extraction
 *                                   (PAPER.md:164-166, 244-246); reading R1
 *                                   takes SipHash-2-4 as BASELINE.json states.
 *
 * Pins (tests/test_oracle_*.py): SipHash known answers and an OpenSSL
 * EVP_MAC("SIPHASH") cross-check; brute-force Python-set membership; the
 * sign/verify, tamper, replay, guard, mode and accounting invariants.
 * No function in this file is "parity unpinned".
 */
#ifndef WG_ORACLE_H
#define WG_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wgo_engine wgo_engine;

/* Site outcome kinds, PAPER.md:145-154 (Table 2) with "protected" split by edge
 * direction as BASELINE.json's policy table does. */
enum {
  WGO_PROTECTED_RETURN = 0,
  WGO_PROTECTED_FORWARD = 1,
  WGO_FIXED_EDGE = 2,
  WGO_UNSUPPORTED = 3,
  WGO_PROFILE_EXCLUDED = 4,
  WGO_FALLBACK = 5,
  WGO_NO_SURFACE = 6,
  WGO_KIND_COUNT = 7
};
enum { WGO_DETECT = 0, WGO_ENFORCE = 1 };

/* policy validation result */
enum {
  WGO_POLICY_OK = 0,
  WGO_POLICY_BAD_KIND = 1,       /* kind >= 7                                        */
  WGO_POLICY_BAD_OFFSETS = 2,    /* tgt_off[0] != 0 or decreasing                    */
  WGO_POLICY_UNSORTED_SET = 3,   /* a set not strictly ascending                     */
  WGO_POLICY_EMPTY_FORWARD = 4,  /* protected-forward site with no target evidence   */
  WGO_POLICY_STRAY_SET = 5       /* a non-forward site that owns targets             */
};

typedef struct {
  uint32_t site_id;
  uint32_t active_mask;
  uint64_t context_base;
} wgo_event_hdr; /* 16 bytes */

typedef struct {
  uint32_t viol_mask;
  uint32_t allow_mask;
} wgo_verdict; /* 8 bytes */

typedef struct {
  uint64_t events_total, events_empty, events_unknown_site, events_misrouted;
  uint64_t events_by_kind[7];
  uint64_t ret_checks, fwd_checks;
  uint64_t ret_lanes, fwd_lanes;
  uint64_t ret_viol, fwd_viol;
  uint64_t ret_viol_events, fwd_viol_events;
  uint64_t blocked_lanes, blocked_events;
  uint64_t first_violation_key;
  uint64_t signed_lanes, sign_skipped_events;
  uint64_t policy_digest, last_mode;
} wgo_counters; /* 26 x u64 */

typedef struct {
  uint64_t events, lanes_checked, lanes_violation, lanes_blocked;
} wgo_site_counters;

/* SipHash-2-4, 64-bit output, arbitrary length — the plain definition. */
uint64_t wgo_siphash24(uint64_t k0, uint64_t k1, const uint8_t* msg, size_t len);

/* token = SipHash-2-4_key( LE64(site_id) || LE64(value) || LE64(context_id) ) */
uint64_t wgo_mac(uint64_t k0, uint64_t k1, uint32_t site_id, uint64_t value, uint64_t context_id);

/* context id of one lane: low five bits of context_base replaced by the lane */
uint64_t wgo_lane_ctx(uint64_t context_base, uint32_t lane);

int wgo_validate_policy(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off,
                        const uint64_t* tgts);

/* NULL when the policy is rejected (nothing is loaded). Arrays are copied. */
wgo_engine* wgo_create(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off,
                       const uint64_t* tgts, uint64_t k0, uint64_t k1, uint64_t policy_digest);
void wgo_destroy(wgo_engine* e);
void wgo_reset_counters(wgo_engine* e);

/* use_binary_search != 0 switches membership to std::binary_search (config 5
 * timing only; tests prove both agree).  Default is the linear scan. */
void wgo_set_binary_search(wgo_engine* e, int use_binary_search);

void wgo_sign(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val /*[n][32]*/,
              uint64_t* tag /*[n][32] out*/, uint64_t n);

/* tag == NULL is the forward entry point (wg_check_forward); non-NULL is
 * wg_verify_continuations. */
void wgo_check(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, const uint64_t* tag,
               wgo_verdict* out, uint64_t n, int mode);

void wgo_read_counters(const wgo_engine* e, wgo_counters* global,
                       wgo_site_counters* per_site /* [n_sites] or NULL */);

/* ---- profiles and telemetry (§4.8, 264-266 §5.7, Table A2 576-588;
 *      DESIGN.md readings R26-R29) ------------------------------------------------------------------
 * Profile flags change the PROTECTED SET, so what they skip is counted under a separate denominator
 * ("Fast or attribution profiles that skip ... a CFI direction change the protected set and are reported
 * under separate denominators"):
 *   WGO_PROFILE_SKIP_FORWARD   "backward-only: authenticated returns only": a non-empty event at a
 *                              protected-forward site is not judged (viol 0, allow = active); it still counts
 *                              in events_total / events_by_kind / site.events and in skipped_fwd_*.
 *   WGO_PROFILE_SKIP_BACKWARD  "forward-only": the same for protected-return sites (in both entry points:
 *                              such an event is then neither checked nor misrouted).  Signing is not a check
 *                              and is unaffected.
 *   WGO_PROFILE_LOW_TELEMETRY  "same checked transfers with less reporting": verdicts, global counters and
 *                              the first-violation record are unchanged; per-site counters and the violation
 *                              ring are not updated.
 * Violation record: one per event with viol != 0 — "counters, telemetry buffers, and first-violation records
 * are diagnostic": lane = lowest violating lane, observed = val[event][lane], stored =
 * tag[event][lane] when the event was judged as a return check, else 0; kind = 7 for an unknown site. */
/*   WGO_PROFILE_METADATA_INTEGRITY  ("authenticates the record when metadata
 *                              integrity is enabled ... The forward metadata token is a MAC over site_id,
 *                              target_count, and allowed_targets"; 258): before the membership test of a non-empty
 *                              event at a protected-forward site, the site's record is re-authenticated:
 *                                  SipHash-2-4_key( LE64(site_id) || LE64(target_count) || LE64(t_0) || ... )
 *                              over the record AS IT IS NOW in the (writable) metadata memory must equal the token
 *                              computed when the policy was loaded; else every active lane violates (a forward
 *                              check with popc(active) violating lanes) and fwd_meta_fail_events counts it.
 *                              wgo_policy_poke is the attacker's write into that memory. */
/*   WGO_PROFILE_COVERAGE_REDUCED  ("profiles that skip kernels, sites, counters, or a CFI direction
 *                              change the protected set and are reported under separate denominators"; Table A2,
 *                              PAPER.md:586-587 "coverage-reduced"; R40): protected sites flagged by
 *                              wgo_set_skip_sites are left out of the protected set: a non-empty event there is not
 *                              judged (viol 0, allow = active, at either entry point: never "misrouted"); it counts in
 *                              events_total / events_by_kind / site.events and in skipped_site_events / _lanes, never
 *                              in ret_* / fwd_*.  A direction skip (above) takes precedence; flags on sites of other
 *                              kinds mean nothing; signing is unaffected.  Without the profile flag the skip set is
 *                              ignored. */
enum { WGO_PROFILE_SKIP_FORWARD = 1, WGO_PROFILE_SKIP_BACKWARD = 2, WGO_PROFILE_LOW_TELEMETRY = 4,
       WGO_PROFILE_METADATA_INTEGRITY = 8, WGO_PROFILE_COVERAGE_REDUCED = 16 };
typedef struct {
  uint64_t seq;
  uint32_t site_id, kind, viol_mask, active_mask, lane, mode;
  uint64_t observed, stored;
} wgo_violation_rec; /* 48 bytes */
typedef struct {
  uint64_t skipped_ret_events, skipped_ret_lanes, skipped_fwd_events, skipped_fwd_lanes;
  uint64_t ring_recorded, ring_dropped; /* recorded + dropped == events with viol != 0 (ring enabled) */
  uint64_t fwd_meta_fail_events;        /* forward records that failed their authentication */
  uint64_t skipped_site_events, skipped_site_lanes; /* coverage-reduced profile: events / lanes at skipped sites */
} wgo_telemetry_counters;
/* what = 0: allowed_targets[index] ^= x (index into the CSR array); what = 1: the stored token of site `index` ^= x.
 * Returns 0, or -1 when out of range.  The set may become unsorted: membership is the linear scan then. */
int wgo_policy_poke(wgo_engine* e, int what, uint64_t index, uint64_t xor_value);
/* ---- policy-digest binding (second half; R39) ----
 * wgo_policy_digest: SipHash-2-4 under the policy's key over LE64(n_sites) || LE64(n_targets) || kind bytes
 * (zero-padded to 8) || tgt_off as LE32 (zero-padded to 8) || tgts as LE64.
 * wgo_create_bound: NULL unless the image's digest equals expected_digest ("a mismatch aborts before the policy is
 * used"); the engine then folds the digest's low 32 bits into the upper half of every backward token's first
 * message word (LE64(site_id | digest32 << 32)), so tokens do not carry over to another policy image. */
uint64_t wgo_policy_digest(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off, const uint64_t* tgts,
                           uint64_t k0, uint64_t k1);
wgo_engine* wgo_create_bound(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off, const uint64_t* tgts,
                             uint64_t k0, uint64_t k1, uint64_t expected_digest);
void wgo_set_profile(wgo_engine* e, uint32_t flags);
/* skip: [n_sites] bytes, non-zero = the site is in the coverage-reduced profile's skip set; NULL clears the set */
void wgo_set_skip_sites(wgo_engine* e, const uint8_t* skip);
/* The running event index (R12) the NEXT checked event gets.  wgo_reset_counters sets it to 0; a rank that
 * checks the slice [lo, hi) of a sharded stream sets it to lo so that first-violation keys and records carry the
 * stream's own sequence numbers. */
void wgo_set_sequence_base(wgo_engine* e, uint64_t base);
/* capacity 0 (default) disables the ring; the oracle keeps the FIRST `capacity` records in event order
 * (any subset of that size is a valid ring content once it overflows). */
void wgo_set_ring_capacity(wgo_engine* e, uint64_t capacity);
uint64_t wgo_read_violations(const wgo_engine* e, wgo_violation_rec* out, uint64_t cap);
/* returns 1 and fills *out when a violation was seen since the last reset, else 0 */
int wgo_read_first_violation(const wgo_engine* e, wgo_violation_rec* out);
void wgo_read_telemetry(const wgo_engine* e, wgo_telemetry_counters* out);


/* ---- stateful shadow stack (§4.4, 242-248 §5.5, 258 §5.6;
 *      DESIGN.md readings R30-R36) --------------------------------------------------------------------
 * "one logical shadow stack per CUDA thread slot ... bounded per-thread depth arrays.  Each shadow entry stores
 * expected_return, callsite_id, depth, and token".  thread slot = (warp_slot, lane) with
 * warp_slot = bits 36..5 of context_base and epoch = bits 63..48 (the depth field of context_base is ignored:
 * the engine owns the depth).  Token of an entry at depth d:
 *     MAC(key, callsite_id, expected_return, (epoch << 48) | (d << 37) | (warp_slot << 5) | lane).
 * push: per active lane, d = depth: d == max_depth -> overflow, the lane violates and nothing is
 *   written; else the entry {value, site, d, token} is written at d and depth becomes d + 1.
 * check_ret: per active lane, d = depth: d == 0 -> underflow, violates; else the entry at d - 1
 *   is read and the depth becomes d - 1 whatever the verdict (the return consumed the frame); the lane violates
 *   on, in this order: entry.depth != d - 1 (depth mismatch); token != MAC over the ENTRY's own fields under
 *   the event's epoch (token mismatch); entry.expected_return != observed value or entry.callsite_id != site
 *   (target mismatch).  Each violating lane counts under exactly one cause.
 * Event-level failures, all lanes violate, state untouched ("fail closed instead of aliasing"):
 *   unknown site or a site that is not protected-return (non_return); warp_slot >= n_warp_slots (slot
 *   overflow); a warp_slot that occurs more than once in one call (slot conflict: a call is one lock-step step
 *   of distinct warps).  Empty masks are counted and change nothing. */
typedef struct {
  uint64_t push_events, push_lanes, check_events, check_lanes, empty_events;
  uint64_t overflow_lanes, underflow_lanes, depth_mismatch_lanes, token_mismatch_lanes, target_mismatch_lanes;
  uint64_t non_return_events, slot_overflow_events, slot_conflict_events;
  uint64_t viol_lanes, viol_events, blocked_lanes;
} wgo_shadow_counters; /* 16 x u64 */
/* (re)allocates and zeroes the shadow state and its counters; max_depth in 1..64 */
int wgo_shadow_configure(wgo_engine* e, uint32_t n_warp_slots, uint32_t max_depth);
void wgo_shadow_push(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, wgo_verdict* out,
                     uint64_t n, int mode);
void wgo_shadow_check_ret(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, wgo_verdict* out,
                          uint64_t n, int mode);
void wgo_shadow_read_counters(const wgo_engine* e, wgo_shadow_counters* out);
/* the attacker's write into the (ordinary, writable) shadow memory: field 0 expected_return, 1 token,
 * 2 callsite_id, 3 depth of the entry; 4 = the slot's current depth counter (entry_depth ignored) */
int wgo_shadow_poke(wgo_engine* e, uint32_t warp_slot, uint32_t lane, uint32_t entry_depth, int field,
                    uint64_t xor_value);
/* current depth of a thread slot (test read-back) */
uint32_t wgo_shadow_depth(const wgo_engine* e, uint32_t warp_slot, uint32_t lane);

#ifdef __cplusplus
}
#endif
#endif
