// wg_internal.h — what the C-ABI layer (wg_api.cu) and the kernels (wg_kernels.cu) agree on.
// Not installed; the public surface is include/warpguard.h only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wg {

// ---- engine-owned device tables (DESIGN.md §5 "data layout") --------------------------------------
// One 16-byte record per site, gathered once per event.  L2-resident at every config (1 M sites =
// 16 MB).  Nothing key-derived is stored in it — or anywhere else in global memory: the key-derived SipHash initial
// state lives in the kernel parameters only (constant bank), and the per-site part of the MAC is
// recomputed in the kernels' event-parallel phases (2 SipRounds per 32 events).
struct __align__(16) SiteRec {
  uint32_t kind;  // wg_kind
  uint32_t off;   // first element of this site's set in the device copy of `tgts` (u64 index)
  uint32_t cnt;   // number of targets (0 unless protected-forward)
  uint32_t flags; // bit 0: the site is in the coverage-reduced profile's skip set (R40)
};
static_assert(sizeof(SiteRec) == 16, "SiteRec is one 16-byte vector");
enum : uint32_t { SITE_FLAG_SKIP = 1u, SITE_FLAG_HAS_ALLONES = 2u };  // (2: the set contains 0xffff...f, see the hash index)

// Global counter block: the first 26 words have exactly the layout of wg_counters, so a read-out is one
// copy.  Words 24 (policy_digest) and 25 (last_mode) are kept host-side and patched in at read-out.
enum CounterWord {
  C_EVENTS_TOTAL = 0,
  C_EVENTS_EMPTY = 1,
  C_EVENTS_UNKNOWN = 2,
  C_EVENTS_MISROUTED = 3,
  C_BY_KIND = 4,  // 7 words
  C_RET_CHECKS = 11,
  C_FWD_CHECKS = 12,
  C_RET_LANES = 13,
  C_FWD_LANES = 14,
  C_RET_VIOL = 15,
  C_FWD_VIOL = 16,
  C_RET_VIOL_EVENTS = 17,
  C_FWD_VIOL_EVENTS = 18,
  C_BLOCKED_LANES = 19,
  C_BLOCKED_EVENTS = 20,
  C_FIRST_VIOLATION = 21,  // atomicMin, initialised to UINT64_MAX
  C_SIGNED_LANES = 22,
  C_SIGN_SKIPPED = 23,
  C_POLICY_DIGEST = 24,
  C_LAST_MODE = 25,
  // telemetry words behind the 26 words of wg_counters (wg_telemetry_counters; R26-R28)
  C_SKIP_RET_EVENTS = 26,
  C_SKIP_RET_LANES = 27,
  C_SKIP_FWD_EVENTS = 28,
  C_SKIP_FWD_LANES = 29,
  C_RING_TOTAL = 30,  // violation records offered to the ring (recorded = min(total, capacity))
  C_SPARE31 = 31,
  C_META_FAIL = 32,   // forward records that failed their authentication (metadata-integrity profile, R37)
  C_SKIP_SITE_EVENTS = 33,  // non-empty events at protected sites the coverage-reduced profile leaves out (R40)
  C_SKIP_SITE_LANES = 34,
  C_WORDS = 40
};

// Launches of one engine that may be in flight at once on different streams each need their own group ticket: the
// engine hands out the words of a small ring in launch order (wg_api.cu)
constexpr int kSchedSlots = 64;

// Violation record, layout of wg_violation_rec (48 bytes)
struct __align__(8) ViolRec {
  uint64_t seq;
  uint32_t site_id, kind, viol_mask, active_mask, lane, mode;
  uint64_t observed, stored;
};
static_assert(sizeof(ViolRec) == 48, "ViolRec layout");
// First-violation record kept on the device: the record and the key it was written for
struct FirstRec {
  ViolRec rec;
  unsigned long long key;  // UINT64_MAX: none
};
enum : uint32_t { PROFILE_SKIP_FORWARD = 1, PROFILE_SKIP_BACKWARD = 2, PROFILE_LOW_TELEMETRY = 4,
                  PROFILE_METADATA_INTEGRITY = 8, PROFILE_COVERAGE_REDUCED = 16 };

// Per-site counters: 4 x u64 per site, layout of wg_site_counters.
enum SiteWord { S_EVENTS = 0, S_LANES_CHECKED = 1, S_LANES_VIOLATION = 2, S_LANES_BLOCKED = 3 };

// Everything a kernel needs, passed by value (lives in the constant bank: the key never sits in
// caller-addressable memory).
struct Params {
  const uint4* hdr;          // [n] wg_event_hdr as one 16-byte vector
  const uint64_t* val;       // [n][32]
  const uint64_t* tag;       // [n][32] or nullptr (forward entry point)
  uint64_t* tag_out;         // sign only
  uint2* out;                // [n] wg_verdict
  uint64_t n;
  uint64_t seq_base;         // running event index of event 0 of this call (R12)
  const SiteRec* recs;       // [n_sites]
  const uint64_t* tok;       // [n_sites] token of each forward record at load time (metadata-integrity profile, R37)
  const uint64_t* tgts;
  const uint64_t* htab;      // hash index of the target sets (policies too large to stage), or nullptr (wg_check.cu)
  uint64_t n_tgts;           // elements in tgts (v2 stages the whole table in shared memory when it is small)
  unsigned int* sched;       // this launch's group ticket (wg_check.cu): one word of the engine's ring of kSchedSlots
  unsigned long long* glob;  // [C_WORDS]
  unsigned long long* site;  // [n_sites][4]
  uint32_t n_sites;
  uint32_t mode;             // 0 detect, 1 enforce
  uint32_t profile;          // PROFILE_* flags (R26)
  uint32_t pad0;
  uint32_t bind_hi;          // upper half of the token's first message word: low 32 bits of the policy digest when
                             // the policy was loaded with wg_load_policy_bound (R39), else 0
  uint32_t has_ret;          // the policy lists at least one protected-return site (else a verify decides what the forward
                             // entry point decides, and runs its kernel)
  ViolRec* ring;             // violation ring or nullptr
  uint64_t ring_cap;         // its capacity in records
  FirstRec* first;           // first-violation record
  uint64_t v0, v1, v2, v3;   // SipHash initial state: key ^ constants (computed host-side at load)
};

// Shadow-stack state (wg_shadow.cu; R30-R36): structure of arrays, all engine-allocated but, as in the
// paper, treated as attacker-writable: nothing read from it is trusted before its token verifies.
struct ShadowState {
  uint32_t n_slots, max_depth;
  uint32_t* depth_ctr;          // [n_slots][32]
  uint64_t* entry;              // [n_slots][max_depth][32][4]: one 32-byte sector per thread slot and depth,
                                // {expected_return, token, callsite_id | depth << 32, 0}: an active lane writes
                                // its whole sector (two 16-byte stores the L2 merges), so DRAM never has to
                                // read-fill a partially written one; inactive lanes' sectors are not touched
  unsigned long long* uses;     // [n_slots] {stamp of the call that last used the slot << 32 | its occurrences in that call}
  unsigned long long* counters; // [16] wg_shadow_counters
  uint32_t stamp;               // the current call (1, 2, ...): a use count under an older stamp counts as zero, so nothing is cleared
  int per_sm[2];                // resident blocks per SM of the check_ret / push kernel on the engine's device
};
cudaError_t launch_shadow(const Params& p, const ShadowState& sh, bool push, int sm_count, cudaStream_t st,
                          uint64_t* launches);
cudaError_t shadow_occupancy(int* per_sm_push, int* per_sm_check);  // resident blocks per SM on the current device

// launchers (wg_kernels_v2.cu); grid sizing from the SM count of the engine's device.  `launches` (host) counts the
// kernels enqueued, per engine (wg_telemetry_counters.kernel_launches).
cudaError_t launch_sign(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches);
cudaError_t launch_check(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches);
// first-violation record of the events [p.seq_base, p.seq_base + p.n) (one thread; see wg_first_record)
cudaError_t launch_first_record(const Params& p, cudaStream_t st, uint64_t* launches);
// tokens of the forward records as loaded (trusted load time)
cudaError_t launch_build_tokens(uint64_t* tok, const SiteRec* recs, const uint64_t* tgts, uint32_t n_sites,
                                uint64_t v0, uint64_t v1, uint64_t v2, uint64_t v3, cudaStream_t st, uint64_t* launches);
// SiteRec.flags bit 0 <- d_skip[site] != 0 (d_skip == nullptr: cleared), the coverage-reduced profile's skip set (R40)
cudaError_t launch_set_site_flags(SiteRec* recs, const uint8_t* d_skip, uint32_t n_sites, cudaStream_t st, uint64_t* launches);
// hash index of large target sets: htab has 2 * n_tgts + 4 * n_sites slots, pre-filled with all-ones (wg_check.cu)
cudaError_t launch_build_hash(uint64_t* htab, SiteRec* recs, const uint64_t* tgts, uint32_t n_sites, uint64_t n_tgts,
                              cudaStream_t st, uint64_t* launches);
cudaError_t launch_clear_allones_flags(SiteRec* recs, uint32_t n_sites, cudaStream_t st, uint64_t* launches);
uint64_t max_staged_targets();  // larger tables are searched in global memory (and get the hash index)
cudaError_t init_kernels();  // one-time function attributes (dynamic shared memory opt-in) on the current device

}  // namespace wg
