// wg_oracle.cpp — TEST INFRASTRUCTURE ONLY (see wg_oracle.h).
//
// Plain single-threaded C++17.  No intrinsics, no blocking, no fusion, no
// reordering: SipHash-2-4 lane by lane, linear-scan set membership, counters
// updated event by event in stream order.  Written so that a reader can check
// each function against the cited passage by eye.

#include "wg_oracle.h"

#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

namespace {

inline uint64_t rotl64(uint64_t x, unsigned b) { return (x << b) | (x >> (64u - b)); }

// One SipRound (Aumasson & Bernstein, "SipHash: a fast short-input PRF", §2.1
// figure of the ARX network; restated in SURVEY.md §8(c)).
inline void sipround(uint64_t& v0, uint64_t& v1, uint64_t& v2, uint64_t& v3) {
  v0 += v1;
  v1 = rotl64(v1, 13);
  v1 ^= v0;
  v0 = rotl64(v0, 32);
  v2 += v3;
  v3 = rotl64(v3, 16);
  v3 ^= v2;
  v0 += v3;
  v3 = rotl64(v3, 21);
  v3 ^= v0;
  v2 += v1;
  v1 = rotl64(v1, 17);
  v1 ^= v2;
  v2 = rotl64(v2, 32);
}

inline uint64_t load_le64(const uint8_t* p) {
  uint64_t w = 0;
  for (int i = 0; i < 8; ++i) w |= static_cast<uint64_t>(p[i]) << (8 * i);
  return w;
}

inline void store_le64(uint8_t* p, uint64_t w) {
  for (int i = 0; i < 8; ++i) p[i] = static_cast<uint8_t>(w >> (8 * i));
}

inline unsigned popcount32(uint32_t x) {
  unsigned c = 0;
  for (int i = 0; i < 32; ++i) c += (x >> i) & 1u;
  return c;
}

inline unsigned lowest_set_lane(uint32_t x) {  // x != 0
  unsigned i = 0;
  while (((x >> i) & 1u) == 0) ++i;
  return i;
}

}  // namespace

struct wgo_engine {
  uint32_t n_sites = 0;
  std::vector<uint8_t> kind;
  std::vector<uint32_t> tgt_off;
  std::vector<uint64_t> tgts;
  uint64_t k0 = 0, k1 = 0;
  uint64_t seq = 0;  // running event index over check calls (R12)
  int use_binary_search = 0;
  bool poked = false;
  bool bind_digest = false;  // R39: fold the policy digest into the token's first word  // wgo_policy_poke touched the target array: sets may be unsorted
  wgo_counters g;
  std::vector<wgo_site_counters> site;
  // profiles and telemetry (R26-R29)
  uint32_t profile = 0;
  uint64_t ring_capacity = 0;
  std::vector<wgo_violation_rec> ring;
  wgo_telemetry_counters t = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  std::vector<uint8_t> skip_site;  // per site: left out by the coverage-reduced profile (R40); empty = none
  std::vector<uint64_t> fwd_token;  // per site: token of the forward record at load time (R37)
  bool have_first = false;
  wgo_violation_rec first = {};
  // stateful shadow stack (R30-R36): entry (slot, lane, d) lives at ((slot * 32 + lane) * max_depth + d)
  struct ShadowEntry {
    uint64_t expected_return, token;
    uint32_t callsite_id, depth;
  };
  uint32_t sh_slots = 0, sh_max_depth = 0;
  std::vector<ShadowEntry> sh_entry;
  std::vector<uint32_t> sh_depth;  // [slot * 32 + lane]
  wgo_shadow_counters sh = {};
};

extern "C" {

static uint64_t forward_record_token(const wgo_engine* e, uint32_t s);  // defined beside the membership tests


// SipHash-c-d with c = 2 compression rounds and d = 4 finalisation rounds,
// 64-bit output.  Initialisation constants are the ASCII of
// "somepseudorandomlygeneratedbytes"; the last word carries the message
// length mod 256 in its top byte.
uint64_t wgo_siphash24(uint64_t k0, uint64_t k1, const uint8_t* msg, size_t len) {
  uint64_t v0 = k0 ^ 0x736f6d6570736575ULL;
  uint64_t v1 = k1 ^ 0x646f72616e646f6dULL;
  uint64_t v2 = k0 ^ 0x6c7967656e657261ULL;
  uint64_t v3 = k1 ^ 0x7465646279746573ULL;

  const size_t full_words = len / 8;
  for (size_t i = 0; i < full_words; ++i) {
    const uint64_t m = load_le64(msg + 8 * i);
    v3 ^= m;
    sipround(v0, v1, v2, v3);
    sipround(v0, v1, v2, v3);
    v0 ^= m;
  }

  uint64_t last = static_cast<uint64_t>(len & 0xff) << 56;
  const size_t tail = len % 8;
  for (size_t i = 0; i < tail; ++i) last |= static_cast<uint64_t>(msg[8 * full_words + i]) << (8 * i);
  v3 ^= last;
  sipround(v0, v1, v2, v3);
  sipround(v0, v1, v2, v3);
  v0 ^= last;

  v2 ^= 0xff;
  sipround(v0, v1, v2, v3);
  sipround(v0, v1, v2, v3);
  sipround(v0, v1, v2, v3);
  sipround(v0, v1, v2, v3);
  return v0 ^ v1 ^ v2 ^ v3;
}

// Backward token (binds expected return, callsite
// identifier, depth / thread slot / epoch and key material).  DESIGN.md R2-R4:
// message = LE64(zero-extended site_id) || LE64(continuation) || LE64(context_id).
uint64_t wgo_mac(uint64_t k0, uint64_t k1, uint32_t site_id, uint64_t value, uint64_t context_id) {
  uint8_t msg[24];
  store_le64(msg + 0, static_cast<uint64_t>(site_id));
  store_le64(msg + 8, value);
  store_le64(msg + 16, context_id);
  return wgo_siphash24(k0, k1, msg, sizeof msg);
}

// Token as the ENGINE computes it: with digest binding on (R39, "policy binding is checked before
// use") the low 32 bits of the policy digest ride in the upper half of the first message word, so
// a token minted under one policy image does not verify under another.
static uint64_t engine_token(const wgo_engine* e, uint32_t site_id, uint64_t value, uint64_t context_id) {
  uint8_t msg[24];
  const uint64_t w0 = static_cast<uint64_t>(site_id) |
                      (e->bind_digest ? (e->g.policy_digest & 0xffffffffull) << 32 : 0ull);
  store_le64(msg + 0, w0);
  store_le64(msg + 8, value);
  store_le64(msg + 16, context_id);
  return wgo_siphash24(e->k0, e->k1, msg, sizeof msg);
}

// DESIGN.md R2: the caller's context_base has its low five bits reserved for
// the lane, so a lane's token cannot be replayed in another lane (the paper's
// per-thread-slot binding).
uint64_t wgo_lane_ctx(uint64_t context_base, uint32_t lane) {
  return (context_base & ~static_cast<uint64_t>(31)) | static_cast<uint64_t>(lane & 31u);
}

// Load-time policy validation.  "A binding mismatch becomes an abort ... rather
// than a wider allowed target set"; "missing ... target evidence
// receive[s] an unsupported outcome".  DESIGN.md R16.
int wgo_validate_policy(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off,
                        const uint64_t* tgts) {
  for (uint32_t s = 0; s < n_sites; ++s)
    if (kind[s] >= WGO_KIND_COUNT) return WGO_POLICY_BAD_KIND;
  if (tgt_off[0] != 0) return WGO_POLICY_BAD_OFFSETS;
  for (uint32_t s = 0; s < n_sites; ++s)
    if (tgt_off[s + 1] < tgt_off[s]) return WGO_POLICY_BAD_OFFSETS;
  for (uint32_t s = 0; s < n_sites; ++s) {
    const uint32_t lo = tgt_off[s], hi = tgt_off[s + 1];
    if (kind[s] == WGO_PROTECTED_FORWARD) {
      if (hi == lo) return WGO_POLICY_EMPTY_FORWARD;
    } else if (hi != lo) {
      return WGO_POLICY_STRAY_SET;
    }
    for (uint32_t i = lo; i + 1 < hi; ++i)
      if (!(tgts[i] < tgts[i + 1])) return WGO_POLICY_UNSORTED_SET;
  }
  return WGO_POLICY_OK;
}

void wgo_reset_counters(wgo_engine* e) {
  const uint64_t digest = e->g.policy_digest;  // echoed policy binding, not a counter
  std::memset(&e->g, 0, sizeof e->g);
  e->g.policy_digest = digest;
  e->g.first_violation_key = ~static_cast<uint64_t>(0);
  std::fill(e->site.begin(), e->site.end(), wgo_site_counters{0, 0, 0, 0});
  e->seq = 0;
  e->ring.clear();  // profile and ring capacity are configuration and stay
  e->t = wgo_telemetry_counters{};  // every field zero
  e->have_first = false;
}

wgo_engine* wgo_create(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off,
                       const uint64_t* tgts, uint64_t k0, uint64_t k1, uint64_t policy_digest) {
  if (wgo_validate_policy(n_sites, kind, tgt_off, tgts) != WGO_POLICY_OK) return nullptr;
  wgo_engine* e = new (std::nothrow) wgo_engine;
  if (!e) return nullptr;
  e->n_sites = n_sites;
  e->kind.assign(kind, kind + n_sites);
  e->tgt_off.assign(tgt_off, tgt_off + n_sites + 1);
  e->tgts.assign(tgts, tgts + tgt_off[n_sites]);
  e->k0 = k0;
  e->k1 = k1;
  e->site.resize(n_sites);
  e->fwd_token.assign(n_sites, 0);
  for (uint32_t s = 0; s < n_sites; ++s)
    if (kind[s] == WGO_PROTECTED_FORWARD) e->fwd_token[s] = forward_record_token(e, s);
  e->g.policy_digest = policy_digest;
  wgo_reset_counters(e);
  return e;
}

void wgo_destroy(wgo_engine* e) { delete e; }

void wgo_set_binary_search(wgo_engine* e, int use_binary_search) {
  e->use_binary_search = use_binary_search;
}

// Backward push (PAPER.md:228 push(site, expected_ret, guard); 248 "writes the
// authenticated record").  Guard-false lanes are no-ops: tag 0.
void wgo_sign(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, uint64_t* tag,
              uint64_t n) {
  for (uint64_t ev = 0; ev < n; ++ev) {
    const uint32_t s = hdr[ev].site_id;
    const uint32_t a = hdr[ev].active_mask;
    const bool protected_return = s < e->n_sites && e->kind[s] == WGO_PROTECTED_RETURN;
    for (uint32_t lane = 0; lane < 32; ++lane) {
      const bool active = (a >> lane) & 1u;
      uint64_t t = 0;
      if (protected_return && active)
        t = engine_token(e, s, val[ev * 32 + lane], wgo_lane_ctx(hdr[ev].context_base, lane));
      tag[ev * 32 + lane] = t;
    }
    if (protected_return)
      e->g.signed_lanes += popcount32(a);
    else
      e->g.sign_skipped_events += 1;
  }
}

// token of a forward record: SipHash-2-4 over LE64(site_id) || LE64(target_count) || LE64(targets...) as the
// record stands in memory NOW
static uint64_t forward_record_token(const wgo_engine* e, uint32_t s) {
  const uint32_t a = e->tgt_off[s], b = e->tgt_off[s + 1];
  std::vector<uint8_t> msg;
  auto put = [&msg](uint64_t w) {
    for (int i = 0; i < 8; ++i) msg.push_back(static_cast<uint8_t>(w >> (8 * i)));
  };
  put(s);
  put(b - a);
  for (uint32_t i = a; i < b; ++i) put(e->tgts[i]);
  return wgo_siphash24(e->k0, e->k1, msg.data(), msg.size());
}

static bool member_linear(const wgo_engine* e, uint32_t s, uint64_t target) {
  for (uint32_t i = e->tgt_off[s]; i < e->tgt_off[s + 1]; ++i)
    if (e->tgts[i] == target) return true;  // exact 64-bit equality, R8
  return false;
}

static bool member_bsearch(const wgo_engine* e, uint32_t s, uint64_t target) {
  return std::binary_search(e->tgts.begin() + e->tgt_off[s], e->tgts.begin() + e->tgt_off[s + 1],
                            target);
}

// check_ret(site, observed_ret, guard) and the forward check (site, target,
// guard); verdict rules PAPER.md:264; accounting
// PAPER.md:113, 127, 224.  Follows SURVEY.md §8(c) "CHECK" line by line.
void wgo_check(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, const uint64_t* tag,
               wgo_verdict* out, uint64_t n, int mode) {
  for (uint64_t ev = 0; ev < n; ++ev) {
    const uint64_t seq = e->seq++;
    const uint32_t s = hdr[ev].site_id;
    const uint32_t a = hdr[ev].active_mask;
    uint32_t viol = 0;
    bool judged_ret = false;  // the stored tag took part in this event's verdict
    const bool low = (e->profile & WGO_PROFILE_LOW_TELEMETRY) != 0;
    e->g.events_total += 1;

    if (s >= e->n_sites) {
      // unknown site: fail closed, outside every denominator (R13)
      viol = a;
      e->g.events_unknown_site += 1;
    } else {
      const uint8_t k = e->kind[s];
      e->g.events_by_kind[k] += 1;
      if (!low) e->site[s].events += 1;
      if (a == 0) {
        // fully predicated-off instruction: no helper ran (R22)
        e->g.events_empty += 1;
      } else if (k == WGO_PROTECTED_RETURN && (e->profile & WGO_PROFILE_SKIP_BACKWARD)) {
        // forward-only profile: outside the protected set, separate denominator (R26)
        e->t.skipped_ret_events += 1;
        e->t.skipped_ret_lanes += popcount32(a);
      } else if (k == WGO_PROTECTED_FORWARD && (e->profile & WGO_PROFILE_SKIP_FORWARD)) {
        // backward-only profile (R26)
        e->t.skipped_fwd_events += 1;
        e->t.skipped_fwd_lanes += popcount32(a);
      } else if ((k == WGO_PROTECTED_RETURN || k == WGO_PROTECTED_FORWARD) &&
                 (e->profile & WGO_PROFILE_COVERAGE_REDUCED) && !e->skip_site.empty() && e->skip_site[s]) {
        // coverage-reduced profile: this protected site is left out of the protected set; not judged, reported
        // under its own denominator (Table A2 586-587; R40)
        e->t.skipped_site_events += 1;
        e->t.skipped_site_lanes += popcount32(a);
      } else if (k == WGO_PROTECTED_RETURN && tag != nullptr) {
        judged_ret = true;
        for (uint32_t lane = 0; lane < 32; ++lane) {
          if (!((a >> lane) & 1u)) continue;  // inactive lanes are never judged
          const uint64_t expect =
              engine_token(e, s, val[ev * 32 + lane], wgo_lane_ctx(hdr[ev].context_base, lane));
          if (expect != tag[ev * 32 + lane]) viol |= (1u << lane);
        }
        e->g.ret_checks += 1;
        e->g.ret_lanes += popcount32(a);
        e->g.ret_viol += popcount32(viol);
        e->g.ret_viol_events += (viol != 0);
        if (!low) e->site[s].lanes_checked += popcount32(a);
        if (!low) e->site[s].lanes_violation += popcount32(viol);
      } else if (k == WGO_PROTECTED_RETURN) {
        // handed to the forward entry point: no tag, cannot authenticate (R14)
        viol = a;
        e->g.events_misrouted += 1;
      } else if (k == WGO_PROTECTED_FORWARD) {
        bool record_ok = true;
        if (e->profile & WGO_PROFILE_METADATA_INTEGRITY) {  // authenticate the record before use
          record_ok = forward_record_token(e, s) == e->fwd_token[s];
          if (!record_ok) e->t.fwd_meta_fail_events += 1;
        }
        for (uint32_t lane = 0; lane < 32; ++lane) {
          if (!((a >> lane) & 1u)) continue;
          const uint64_t target = val[ev * 32 + lane];
          // an unauthenticated record authorises nothing; a poked set may be unsorted, so scan it
          const bool ok = record_ok && ((e->use_binary_search && !e->poked) ? member_bsearch(e, s, target)
                                                                            : member_linear(e, s, target));
          if (!ok) viol |= (1u << lane);
        }
        e->g.fwd_checks += 1;
        e->g.fwd_lanes += popcount32(a);
        e->g.fwd_viol += popcount32(viol);
        e->g.fwd_viol_events += (viol != 0);
        if (!low) e->site[s].lanes_checked += popcount32(a);
        if (!low) e->site[s].lanes_violation += popcount32(viol);
      } else {
        // fixed-edge / unsupported / profile-excluded / fallback / no-surface:
        // counted above, never judged (R17)
      }
    }

    const uint32_t allow = (mode == WGO_ENFORCE) ? (a & ~viol) : a;
    if (mode == WGO_ENFORCE && viol != 0) {
      e->g.blocked_lanes += popcount32(viol);
      e->g.blocked_events += 1;
      if (s < e->n_sites && !low) e->site[s].lanes_blocked += popcount32(viol);
    }
    if (viol != 0) {
      const uint64_t key = (seq << 5) | lowest_set_lane(viol);
      // the violation record (R27): diagnostic only, it never feeds a verdict
      wgo_violation_rec r;
      r.seq = seq;
      r.site_id = s;
      r.kind = (s < e->n_sites) ? e->kind[s] : 7u;
      r.viol_mask = viol;
      r.active_mask = a;
      r.lane = lowest_set_lane(viol);
      r.mode = static_cast<uint32_t>(mode);
      r.observed = val[ev * 32 + r.lane];
      r.stored = judged_ret ? tag[ev * 32 + r.lane] : 0;
      if (key < e->g.first_violation_key) {  // PAPER.md:266 "records the first violation"
        e->g.first_violation_key = key;
        e->first = r;
        e->have_first = true;
      }
      if (!low && e->ring_capacity != 0) {  // bounded ring (R28)
        if (e->ring.size() < e->ring_capacity) {
          e->ring.push_back(r);
          e->t.ring_recorded += 1;
        } else {
          e->t.ring_dropped += 1;
        }
      }
    }
    out[ev].viol_mask = viol;
    out[ev].allow_mask = allow;
  }
  if (n != 0) e->g.last_mode = static_cast<uint64_t>(mode);
}

// Digest of a policy image (R39): SipHash-2-4 under the policy's key over
//   LE64(n_sites) || LE64(n_targets) || kind[n_sites] (zero-padded to 8 bytes) || tgt_off[n_sites + 1] as LE32
//   (zero-padded to 8 bytes) || tgts as LE64.
uint64_t wgo_policy_digest(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off, const uint64_t* tgts,
                           uint64_t k0, uint64_t k1) {
  std::vector<uint8_t> msg;
  auto put64 = [&msg](uint64_t w) {
    for (int i = 0; i < 8; ++i) msg.push_back(static_cast<uint8_t>(w >> (8 * i)));
  };
  auto pad8 = [&msg]() {
    while (msg.size() % 8) msg.push_back(0);
  };
  const uint64_t nt = tgt_off[n_sites];
  put64(n_sites);
  put64(nt);
  for (uint32_t s = 0; s < n_sites; ++s) msg.push_back(kind[s]);
  pad8();
  for (uint32_t s = 0; s <= n_sites; ++s)
    for (int i = 0; i < 4; ++i) msg.push_back(static_cast<uint8_t>(tgt_off[s] >> (8 * i)));
  pad8();
  for (uint64_t i = 0; i < nt; ++i) put64(tgts[i]);
  return wgo_siphash24(k0, k1, msg.data(), msg.size());
}

// "When an enforcement profile requires a policy digest, a mismatch aborts before the policy is used"
wgo_engine* wgo_create_bound(uint32_t n_sites, const uint8_t* kind, const uint32_t* tgt_off, const uint64_t* tgts,
                             uint64_t k0, uint64_t k1, uint64_t expected_digest) {
  if (wgo_validate_policy(n_sites, kind, tgt_off, tgts) != WGO_POLICY_OK) return nullptr;
  if (wgo_policy_digest(n_sites, kind, tgt_off, tgts, k0, k1) != expected_digest) return nullptr;
  wgo_engine* e = wgo_create(n_sites, kind, tgt_off, tgts, k0, k1, expected_digest);
  if (e) e->bind_digest = true;
  return e;
}

void wgo_set_profile(wgo_engine* e, uint32_t flags) { e->profile = flags; }

void wgo_set_skip_sites(wgo_engine* e, const uint8_t* skip) {
  e->skip_site.clear();
  if (skip) e->skip_site.assign(skip, skip + e->n_sites);
}

// the sequence number the next checked event gets (R12; sharded streams: a rank's events keep their global numbers)
void wgo_set_sequence_base(wgo_engine* e, uint64_t base) { e->seq = base; }

int wgo_policy_poke(wgo_engine* e, int what, uint64_t index, uint64_t xor_value) {
  if (what == 0 && index < e->tgts.size()) {
    e->tgts[index] ^= xor_value;
    e->poked = true;
    return 0;
  }
  if (what == 1 && index < e->n_sites) {
    e->fwd_token[index] ^= xor_value;
    return 0;
  }
  return -1;
}

void wgo_set_ring_capacity(wgo_engine* e, uint64_t capacity) {
  e->ring_capacity = capacity;
  if (e->ring.size() > capacity) {  // shrinking drops the tail, and says so
    e->t.ring_dropped += e->ring.size() - capacity;
    e->t.ring_recorded = capacity;
    e->ring.resize(capacity);
  }
}

uint64_t wgo_read_violations(const wgo_engine* e, wgo_violation_rec* out, uint64_t cap) {
  const uint64_t n = e->ring.size() < cap ? e->ring.size() : cap;
  for (uint64_t i = 0; i < n; ++i) out[i] = e->ring[i];
  return n;
}

int wgo_read_first_violation(const wgo_engine* e, wgo_violation_rec* out) {
  if (!e->have_first) return 0;
  *out = e->first;
  return 1;
}

void wgo_read_telemetry(const wgo_engine* e, wgo_telemetry_counters* out) { *out = e->t; }

void wgo_read_counters(const wgo_engine* e, wgo_counters* global, wgo_site_counters* per_site) {
  if (global) *global = e->g;
  if (per_site)
    for (uint32_t s = 0; s < e->n_sites; ++s) per_site[s] = e->site[s];
}

// ---------------------------------------------------------------------------------------------------
// stateful shadow stack, PAPER.md:162-166, 242-248, 258 (wg_oracle.h; R30-R36)
// ---------------------------------------------------------------------------------------------------
int wgo_shadow_configure(wgo_engine* e, uint32_t n_warp_slots, uint32_t max_depth) {
  if (max_depth == 0 || max_depth > 64) return -1;
  e->sh_slots = n_warp_slots;
  e->sh_max_depth = max_depth;
  e->sh_entry.assign(static_cast<size_t>(n_warp_slots) * 32 * max_depth, wgo_engine::ShadowEntry{0, 0, 0, 0});
  e->sh_depth.assign(static_cast<size_t>(n_warp_slots) * 32, 0u);
  e->sh = wgo_shadow_counters{};
  return 0;
}

static uint64_t shadow_ctx(uint64_t context_base, uint32_t depth, uint32_t lane) {
  const uint64_t epoch = context_base >> 48;
  const uint64_t slot = (context_base >> 5) & 0xffffffffull;
  return (epoch << 48) | (static_cast<uint64_t>(depth) << 37) | (slot << 5) | lane;
}

// 0: process per lane; else every active lane violates and the state is untouched
static int shadow_event_failure(wgo_engine* e, const std::vector<uint32_t>& uses, const wgo_event_hdr& h) {
  const uint32_t s = h.site_id;
  const uint64_t slot = (h.context_base >> 5) & 0xffffffffull;
  if (s >= e->n_sites || e->kind[s] != WGO_PROTECTED_RETURN) return 1;  // not a return site of the policy
  if (slot >= e->sh_slots) return 2;                                     // thread-slot overflow
  if (uses[slot] > 1) return 3;                                          // one call = one step of distinct warps
  return 0;
}

static void shadow_run(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, wgo_verdict* out,
                       uint64_t n, int mode, bool push) {
  // how often each warp slot occurs in this call (non-empty or not: the header alone decides)
  std::vector<uint32_t> uses(e->sh_slots, 0u);
  for (uint64_t ev = 0; ev < n; ++ev) {
    const uint64_t slot = (hdr[ev].context_base >> 5) & 0xffffffffull;
    if (slot < e->sh_slots) uses[slot] += 1;
  }
  for (uint64_t ev = 0; ev < n; ++ev) {
    const wgo_event_hdr& h = hdr[ev];
    const uint32_t a = h.active_mask;
    uint32_t viol = 0;
    if (a == 0) {
      e->sh.empty_events += 1;
    } else {
      (push ? e->sh.push_events : e->sh.check_events) += 1;
      (push ? e->sh.push_lanes : e->sh.check_lanes) += popcount32(a);
      const int fail = shadow_event_failure(e, uses, h);
      if (fail) {
        viol = a;
        if (fail == 1) e->sh.non_return_events += 1;
        if (fail == 2) e->sh.slot_overflow_events += 1;
        if (fail == 3) e->sh.slot_conflict_events += 1;
      } else {
        const uint64_t slot = (h.context_base >> 5) & 0xffffffffull;
        for (uint32_t lane = 0; lane < 32; ++lane) {
          if (!((a >> lane) & 1u)) continue;  // guard-false lanes made no call / return
          uint32_t& d = e->sh_depth[slot * 32 + lane];
          wgo_engine::ShadowEntry* st = &e->sh_entry[(slot * 32 + lane) * e->sh_max_depth];
          if (push) {
            if (d >= e->sh_max_depth) {  // overflow fails closed instead of wrapping
              viol |= 1u << lane;
              e->sh.overflow_lanes += 1;
              continue;
            }
            st[d].expected_return = val[ev * 32 + lane];
            st[d].callsite_id = h.site_id;
            st[d].depth = d;
            st[d].token = engine_token(e, h.site_id, val[ev * 32 + lane], shadow_ctx(h.context_base, d, lane));
            d += 1;
          } else {
            if (d == 0) {  // underflow
              viol |= 1u << lane;
              e->sh.underflow_lanes += 1;
              continue;
            }
            d -= 1;  // the return consumes the frame whatever the verdict (R33)
            if (d >= e->sh_max_depth) {  // a corrupted counter points past the bounded array: no such entry
              viol |= 1u << lane;
              e->sh.depth_mismatch_lanes += 1;
              continue;
            }
            const wgo_engine::ShadowEntry& r = st[d];
            if (r.depth != d) {
              viol |= 1u << lane;
              e->sh.depth_mismatch_lanes += 1;
            } else if (r.token != engine_token(e, r.callsite_id, r.expected_return,
                                          shadow_ctx(h.context_base, r.depth, lane))) {
              viol |= 1u << lane;
              e->sh.token_mismatch_lanes += 1;
            } else if (r.expected_return != val[ev * 32 + lane] || r.callsite_id != h.site_id) {
              viol |= 1u << lane;
              e->sh.target_mismatch_lanes += 1;
            }
          }
        }
      }
    }
    if (viol) {
      e->sh.viol_lanes += popcount32(viol);
      e->sh.viol_events += 1;
      if (mode == WGO_ENFORCE) e->sh.blocked_lanes += popcount32(viol);
    }
    out[ev].viol_mask = viol;
    out[ev].allow_mask = (mode == WGO_ENFORCE) ? (a & ~viol) : a;
  }
}

void wgo_shadow_push(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, wgo_verdict* out,
                     uint64_t n, int mode) {
  shadow_run(e, hdr, val, out, n, mode, true);
}

void wgo_shadow_check_ret(wgo_engine* e, const wgo_event_hdr* hdr, const uint64_t* val, wgo_verdict* out,
                          uint64_t n, int mode) {
  shadow_run(e, hdr, val, out, n, mode, false);
}

void wgo_shadow_read_counters(const wgo_engine* e, wgo_shadow_counters* out) { *out = e->sh; }

int wgo_shadow_poke(wgo_engine* e, uint32_t warp_slot, uint32_t lane, uint32_t entry_depth, int field,
                    uint64_t xor_value) {
  if (warp_slot >= e->sh_slots || lane >= 32) return -1;
  if (field == 4) {
    e->sh_depth[static_cast<size_t>(warp_slot) * 32 + lane] ^= static_cast<uint32_t>(xor_value);
    return 0;
  }
  if (entry_depth >= e->sh_max_depth) return -1;
  wgo_engine::ShadowEntry& r = e->sh_entry[(static_cast<size_t>(warp_slot) * 32 + lane) * e->sh_max_depth + entry_depth];
  switch (field) {
    case 0: r.expected_return ^= xor_value; return 0;
    case 1: r.token ^= xor_value; return 0;
    case 2: r.callsite_id ^= static_cast<uint32_t>(xor_value); return 0;
    case 3: r.depth ^= static_cast<uint32_t>(xor_value); return 0;
  }
  return -1;
}

uint32_t wgo_shadow_depth(const wgo_engine* e, uint32_t warp_slot, uint32_t lane) {
  return e->sh_depth[static_cast<size_t>(warp_slot) * 32 + lane];
}

}  // extern "C"
