// wg_internal.h — what the C-ABI layer (wg_api.cu) and the kernels (wg_kernels.cu) agree on.
// Not installed; the public surface is include/warpguard.h only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wg {

// ---- engine-owned device tables (DESIGN.md §5 "data layout") --------------------------------------
// One 16-byte row per site, gathered once per event.  L2-resident at every config.
struct __align__(16) SiteRow {
  uint32_t kind;  // wg_kind
  uint32_t off;   // first element of this site's set in the device copy of `tgts` (u64 index)
  uint32_t cnt;   // number of targets (0 unless protected-forward)
  uint32_t pad;
};

// v2 site record: one 64-byte line per site (never straddles a 128-byte cache line), gathered once per event.
//   words 0-3   kind, off, cnt, 0          (same meaning as SiteRow)
//   words 4-11  protected-return sites: SipHash state after absorbing LE64(site_id), with quarter-round A of the
//               next round already applied ("pre-A" mid-state, wg_sip32.cuh), as v0l v0h v1l v1h v2l v2h v3l v3h.
//               Key-derived, so it lives only in engine-owned memory.  Zero for other kinds.
//   words 12-13 protected-forward sites: token of the forward record at load time (SipHash over site_id,
//               target_count, allowed_targets, R37); words 14-15 reserved (0)
struct __align__(16) SiteRec {
  uint32_t kind, off, cnt, pad0;
  uint32_t st[8];
  uint32_t pad1[4];
};
static_assert(sizeof(SiteRec) == 64, "SiteRec is one 64-byte line");

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
  C_WORDS = 40
};

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
                  PROFILE_METADATA_INTEGRITY = 8 };

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
  const SiteRow* rows;       // v1 kernels
  const SiteRec* recs;       // v2 kernels
  const uint64_t* tgts;
  uint64_t n_tgts;           // elements in tgts (v2 stages the whole table in shared memory when it is small)
  unsigned long long* glob;  // [C_WORDS]
  unsigned long long* site;  // [n_sites][4]
  uint32_t n_sites;
  uint32_t mode;             // 0 detect, 1 enforce
  uint32_t profile;          // PROFILE_* flags (R26)
  uint32_t sparse;           // tuning: compacted-lane MAC passes (wg_set_tuning)
  uint32_t bind_hi;          // upper half of the token's first message word: low 32 bits of the policy digest when
                             // the policy was loaded with wg_load_policy_bound (R39), else 0
  uint32_t pad1;
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
};
cudaError_t launch_shadow(const Params& p, const ShadowState& sh, bool push, int sm_count, cudaStream_t st);

// launchers (wg_kernels.cu); grid sizing from the SM count of the engine's device
cudaError_t launch_sign_v1(const Params& p, int sm_count, cudaStream_t st);
cudaError_t launch_check_v1(const Params& p, int sm_count, cudaStream_t st);
// v2 (wg_kernels_v2.cu): tiled, cp.async-staged, mid-state-cached kernels
cudaError_t launch_sign_v2(const Params& p, int sm_count, cudaStream_t st);
cudaError_t launch_check_v2(const Params& p, int sm_count, cudaStream_t st);
cudaError_t launch_build_recs(SiteRec* recs, const SiteRow* rows, const uint64_t* tgts, uint32_t n_sites, uint32_t bind_hi,
                              uint64_t v0, uint64_t v1, uint64_t v2, uint64_t v3, cudaStream_t st);
cudaError_t init_v2();  // one-time function attributes (dynamic shared memory opt-in)
cudaError_t launch_fill_u64(unsigned long long* p, uint64_t n, unsigned long long v, cudaStream_t st);
cudaError_t run_int_pipe_probe(int mix, int sm_count, double* ops_per_s, double* ms);
void count_launch();

}  // namespace wg
