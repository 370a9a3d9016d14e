// wg_check.cu — the check path on sm_100a: wg_sign_continuations, wg_verify_continuations, wg_check_forward.
//
// Steps: a1 event fetch + guard, a2 policy lookup, a3 MAC sign, a4 MAC verify + compare,
// a5 forward membership, a6 verdicts, a7 counters, a8 first-violation record.  Paper passages: backward token
// PAPER.md:162, 248; forward membership PAPER.md:174-178, 250-252; guards PAPER.md:190, 230; detect / enforce
// PAPER.md:264; accounting PAPER.md:113, 127, 224.  Readings: DESIGN.md §2.  Kernel design: DESIGN.md §6.
//
// What bounds it (measured, profiles/): a SipRound is 20 ALU-pipe instructions (4 IADD3 with carry-out, 8 LOP3,
// 8 SHF) + 4 IMAD.X on the FMA pipe, and every ALU-pipe instruction costs 2 issue cycles per warp on sm_100a, so a
// round is 40 cycles per warp per SM sub-partition whatever the occupancy or ILP.  VOTE, ISETP, SEL, PRMT and LEA are
// ALU-pipe instructions too; IMAD (FMA pipe), POPC / FLO / BREV (XU), SHFL / LDS / LDG (LSU), branches (CBU) and the
// uniform datapath are not.  The kernel is therefore built to (1) run fewer rounds, (2) never run a round on an
// inactive lane, and (3) spend as few ALU-pipe instructions as possible on anything else.
//
// Mapping.  A persistent warp walks over GROUPS of 32 consecutive events.  Per group it runs
//   "event-parallel" phases (lane i <-> event i): header, site record (16 bytes, L2), classification, counters that
//       need no verdict; the part of the MAC that is the same for every lane of an event — the site word always, the
//       continuation word too when it is warp-uniform — from the key-derived initial state in the kernel parameters
//       (nothing key-derived is ever read from memory); the membership search of warp-uniform forward targets;
//   a "producer" loop (lane l <-> lane l, one trip per protected event): the event's value row straight from global
//       memory (one coalesced 256-byte load, no shared-memory staging), the warp-uniformity test, and for return events
//       the ACTIVE lanes appended, compacted, to one of two work queues in shared memory (warp-uniform /
//       lane-divergent continuation); lane-divergent forward targets are searched here;
//   "consumer" passes (lane j <-> queue item j): 32 queued (event, lane) items per pass, whatever events they
//       belong to — the per-lane tail of the MAC (8 of the 12 SipRounds for a warp-uniform continuation, 10
//       otherwise) and the compare, tags gathered from global memory.  Only FULL passes run; what is left over (< 32
//       items per queue) is carried into the next group, so no SipRound is ever spent on an inactive lane;
//   the event-parallel epilogue of the PREVIOUS group (its last items were consumed by this group's first passes):
//       verdict store, violation counters, first violation.
// Rows are pulled into L2 by `prefetch.global.L2` shortly before they are read (value rows of the next group behind this
// group's passes, tag rows at the head of the group's own passes); when the policy's whole target table is small it is
// staged in shared memory once per CTA by one TMA bulk copy.
#include "wg_internal.h"
#include "../../include/warpguard_sip32.cuh"

namespace wg {

namespace {

enum : int { MODE_VERIFY = 0, MODE_FORWARD = 1, MODE_SIGN = 2 };
enum : uint32_t { K_RET = 0, K_FWD = 1 };
// what the kernel does with an event
enum : uint32_t { CLS_NONE = 0, CLS_COUNT = 1, CLS_RET = 2, CLS_FWD = 3, CLS_FAIL = 4, CLS_SKIP_DIR = 5, CLS_SKIP_SITE = 6 };

#ifndef WG_WARPS
#define WG_WARPS 20
#endif
constexpr int kWarps = WG_WARPS;       // warps per CTA, one CTA per SM (sign / verify: the 96-register pass code)
constexpr int kThreads = kWarps * 32;
// The forward entry point (and a verify over a policy without return sites: the same decisions) has no MAC pass: its
// warps wait on shared-memory and shuffle latencies with nothing else to issue, so it wants more of them — 64
// registers, no work queue in shared memory.
#ifndef WG_WARPS_FWD
#define WG_WARPS_FWD 32
#endif
constexpr int kWarpsFwd = WG_WARPS_FWD;
constexpr uint32_t kSmemMax = 232448;  // 227 KB opt-in shared memory per CTA on sm_100a
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kMaxCacheSlots = 2048;  // slots of the per-site counter cache in shared memory (12 bytes each)

// ---- shared-memory carve-up ----------------------------------------------------------------------
// CTA part: [tgts staged: stage_bytes][per-site counter cache: site_bytes][cnt64: 40 x u64][bykind: 12 x u32][mbar, pad]
//           [violation counts: 8 x u32][smallest first-violation key: u64, pad]
// warp part: event records [2 groups][33] x 80 B (record 32 of a group is a dummy that absorbs the padding trips of
// the producer loop), the work queue (u16 items = record slot * 32 + lane; warp-uniform items from the front, lane-divergent
// items from the back), and the producer's list of the group's protected events (16 B each)
//   record: +0  SipHash state the event's consumer passes start from (8 words); a forward event parks its set range
//               {offset, count} at +16 instead
//           +32 ctx lo (context_base & ~31), +36 ctx hi, +40 (8 B) pointer to the event's tag row (sign: the row to
//               write) minus 8 * 32 * slot, so that pointer + 8 * (queue item's low half = slot * 32 + lane) is the
//               lane's element: one IMAD.WIDE on the FMA pipe, no 64-bit add on the ALU pipe
//           +48 active mask, +52 queue mask (the active mask of a return check, else 0), +56 violation mask,
//           +60 lanes whose value differs from the first active lane's (0: warp-uniform)
//           +64 meta = cls | kind << 4, +68 site id, +72 (8 B) pointer to the event's value row, biased the same way
//   (80 bytes: every 16-byte field stays 16-byte aligned)
constexpr uint32_t kRecBytes = 80;
constexpr uint32_t kGroupRecs = 33;
constexpr uint32_t kRecArea = 2 * kGroupRecs * kRecBytes;  // 5,280 B
#ifndef WG_QUEUE
#define WG_QUEUE (1024 + 128)
#endif
constexpr uint32_t kQueueItems = WG_QUEUE;       // one group adds at most 1,024 items; each queue carries < 64
#ifndef WG_BATCH
#define WG_BATCH 4
#endif
constexpr uint32_t kBatch = WG_BATCH;              // row loads in flight per lane in the producer loop
constexpr uint32_t kListBytes = 40 * 16;           // up to 32 protected events, padded to a multiple of kBatch
constexpr uint32_t kWarpBytes = kRecArea + kQueueItems * 2 + kListBytes;
constexpr uint32_t kWarpBytesFwd = kRecArea + kListBytes;  // the forward kernels queue nothing
// kernels that look forward targets up in the hash index (verify / forward, table not staged) add a queue of lookups
constexpr uint32_t kFwdQueueItems = 512;            // drained when more than 256 wait: 8 trips add at most 256
constexpr uint32_t kFwdQueueBytes = kFwdQueueItems * 2;
constexpr uint32_t kCtaFixedBytes = C_WORDS * 8 + 16 * 4 + 16 + 48;  // cnt64, bykind + rare-event counts (u32), mbar, violation counts (8 x u32), first-violation key
constexpr uint32_t kLeft = kSmemMax - kCtaFixedBytes - kWarps * kWarpBytes;
constexpr uint32_t kMaxStageTgts = (kLeft / 16 * 2) < 2048 ? (kLeft / 16 * 2) : 2048;
static_assert(kWarps * (kWarpBytes + kFwdQueueBytes) + kCtaFixedBytes + 4096 <= kSmemMax, "too many warps for the shared memory");
static_assert(kWarpsFwd * (kWarpBytesFwd + kFwdQueueBytes) + kCtaFixedBytes + 4096 <= kSmemMax, "too many forward warps for the shared memory");
static_assert(kWarpsFwd * kWarpBytesFwd + kCtaFixedBytes + 2048 * 8 + 64 * 12 <= kSmemMax, "the staged table must fit beside the forward warps");

// ---- PTX helpers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ uint4 ldg_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
// value rows are read twice by a lane-divergent event (uniformity test, then the consumer's gather): keep them in L1
__device__ __forceinline__ uint2 ldg_v2_keep(const void* p) {
  uint2 r;
  asm volatile("ld.global.ca.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
  return r;
}
// tags are read once
__device__ __forceinline__ uint2 ldg_v2_stream(const void* p) {
  uint2 r;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream_v2(void* p, uint32_t a, uint32_t b) {
  asm volatile("st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ uint4 lds_v4(uint32_t a) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a));
  return r;
}
__device__ __forceinline__ uint2 lds_v2(uint32_t a) {
  uint2 r;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(a));
  return r;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
  uint32_t r;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(a));
  return r;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t a) {
  uint32_t r;
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(r) : "r"(a));
  return r;
}
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t x) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"(static_cast<unsigned short>(x)) : "memory");
}
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t x) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(x) : "memory");
}
__device__ __forceinline__ void sts_v4(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void sts_v2(uint32_t a, uint32_t x, uint32_t y) {
  asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(a), "r"(x), "r"(y) : "memory");
}
// one 256-byte row -> L2.  A prefetch pulls 64 bytes (measured: 2 sectors per request), so a row takes four (one
// `cp.async.bulk.prefetch.L2` of 256 bytes and two prefetches 128 bytes apart were measured: slower / rows half fetched).
__device__ __forceinline__ void prefetch_row_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];\n\tprefetch.global.L2 [%0+64];\n\tprefetch.global.L2 [%0+128];\n\tprefetch.global.L2 [%0+192];" ::"l"(p) : "memory");
}
// L2 policy "evict last" for what every batch of a stream comes back to: site records and per-site counters
__device__ __forceinline__ uint64_t l2_keep_policy() {
  uint64_t pol;
  asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint4 ldg_v4_l2keep(const void* p, uint64_t pol) {
  uint4 r;
  asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p), "l"(pol));
  return r;
}
// {kind, off, cnt} of a site record, without the flags word: a kernel that never reads the flags would leave the fourth
// destination register of a 16-byte load dead, ptxas reuses it at once, and the write-after-write hazard then waits for
// the load right where it was issued (measured on config 3: 8.7 % of the stall samples at the head of every group)
__device__ __forceinline__ uint4 ldg_rec3_l2keep(const void* p, uint64_t pol) {
  uint4 r;
  asm volatile("ld.global.nc.L2::cache_hint.v2.u32 {%0,%1}, [%2], %3;" : "=r"(r.x), "=r"(r.y) : "l"(p), "l"(pol));
  asm volatile("ld.global.nc.L2::cache_hint.u32 %0, [%1+8], %2;" : "=r"(r.z) : "l"(p), "l"(pol));
  r.w = 0u;
  return r;
}
__device__ __forceinline__ void red_add_u64_l2keep(unsigned long long* p, unsigned long long v, uint64_t pol) {
  asm volatile("red.global.add.L2::cache_hint.u64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void atoms_or(uint32_t a, uint32_t x) {
  asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(a), "r"(x) : "memory");
}
// a * b + c on the FMA pipe (address arithmetic inside the ALU-bound loops)
__device__ __forceinline__ uint32_t mad32(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
// base + 8 * element (ptxas turns it into a shift pair on the FMA pipe and a 64-bit add on the ALU pipe; passing the
// multiplier in a register, so that it has to stay an IMAD.WIDE, was measured: the array base lives in uniform registers,
// which IMAD.WIDE cannot take as its addend, so the 64-bit add stays and the kernel gets slower, 13.37 -> 13.72 ms)
__device__ __forceinline__ const uint64_t* elem_ptr(const uint64_t* base, uint32_t elem) {
  uint64_t r;
  asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(r) : "r"(elem), "l"(reinterpret_cast<uint64_t>(base)));
  return reinterpret_cast<const uint64_t*>(r);
}
// d = a & b and t = (d != 0) ? 1 : 0 ... as ONE LOP3 that writes the value and a predicate (ptxas emits two otherwise)
__device__ __forceinline__ void and_test(uint32_t a, uint32_t b, uint32_t& d, uint32_t& t) {
  asm("{ .reg .pred p, q;\n\t"
      "setp.ne.u32 q, 0, 0;\n\t"
      "lop3.or.b32 %0|p, %2, %3, 0, 0xc0, q;\n\t"
      "selp.u32 %1, 1, 0, p; }"
      : "=r"(d), "=r"(t)
      : "r"(a), "r"(b));
}
// biased row pointer (two 32-bit halves from a record) + 8 * queue item: the address of the item's element
__device__ __forceinline__ const uint64_t* item_ptr(uint32_t lo, uint32_t hi, uint32_t item) {
  uint64_t r;
  asm("{ .reg .b64 b; mov.b64 b, {%2, %3}; mad.wide.u32 %0, %1, 8, b; }" : "=l"(r) : "r"(item), "r"(lo), "r"(hi));
  return reinterpret_cast<const uint64_t*>(r);
}
// base + byte offset
__device__ __forceinline__ const char* byte_ptr(const char* base, uint32_t off) {
  uint64_t r;
  asm("mad.wide.u32 %0, %1, 1, %2;" : "=l"(r) : "r"(off), "l"(reinterpret_cast<uint64_t>(base)));
  return reinterpret_cast<const char*>(r);
}

// TMA: 1-D bulk copy global -> shared with completion on an mbarrier (whole-table staging of the target sets)
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n"
      "WG_MBAR_WAIT:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra WG_MBAR_DONE;\n\t"
      "bra WG_MBAR_WAIT;\n"
      "WG_MBAR_DONE:\n\t}" ::"r"(mbar),
      "r"(parity)
      : "memory");
}

// exact-equality membership in a strictly ascending set: branch-free lower-bound walk, then one compare
// (R8).  cnt >= 1 for every protected-forward site (validated at load).
template <bool STAGED>
__device__ __forceinline__ bool member(const Params& p, uint32_t tg_s, uint32_t off, uint32_t cnt, uint32_t vl,
                                       uint32_t vh) {
  const uint64_t v = (static_cast<uint64_t>(vh) << 32) | vl;
  uint32_t lo = 0, len = cnt;
  if constexpr (STAGED) {
    const uint32_t base = tg_s + off * 8;
    while (len > 1) {
      const uint32_t half = len >> 1;
      const uint2 m = lds_v2(base + (lo + half) * 8);
      const uint64_t mid = (static_cast<uint64_t>(m.y) << 32) | m.x;
      lo = (mid <= v) ? lo + half : lo;
      len -= half;
    }
    const uint2 m = lds_v2(base + lo * 8);
    return m.x == vl && m.y == vh;
  } else {
    const uint64_t* set = p.tgts + off;
    // large sets live in L2 / HBM and every probe is a dependent load: quaternary steps issue three independent
    // probes at once and halve the number of dependent rounds (config 5: sets up to 4,096 entries)
    while (len > 8) {
      const uint32_t q = len >> 2;
      const uint64_t m1 = __ldg(set + lo + q), m2 = __ldg(set + lo + 2 * q), m3 = __ldg(set + lo + 3 * q);
      if (m3 <= v) {
        lo += 3 * q;
        len -= 3 * q;
      } else {
        lo += (m2 <= v) ? 2 * q : (m1 <= v) ? q : 0u;
        len = q;
      }
    }
    while (len > 1) {
      const uint32_t half = len >> 1;
      const uint64_t mid = __ldg(set + lo + half);
      lo = (mid <= v) ? lo + half : lo;
      len -= half;
    }
    return __ldg(set + lo) == v;
  }
}

// ---- hash index of the large target sets (policies whose table is not staged in shared memory) --------------------
// A binary search over a set in L2 / HBM is up to 12 DEPENDENT loads (7 with quaternary steps): on config 5 (sets up to
// 4,096 entries) the check kernel spent most of its time waiting on them (ALU pipe 48 % busy).  At load time the engine
// therefore builds, per forward site, an open-addressing hash table of the site's targets in its own memory:
//   slots of site s: htab[(2 * off(s) + 4 * s + 2) & ~3 ...), 4 * nb(s) of them, nb(s) = ceil(cnt(s) / 2) buckets of 4
//   slots: load factor <= 1/2, tables derived from the site record alone, no extra field; the rounding makes every
//   bucket ONE aligned 32-byte sector (without it the buckets of a site with an odd offset straddled two sectors, often
//   in two DRAM bursts: measured 105 bytes of DRAM traffic per lookup on config 5) and still fits the 2 T + 4 S slots;
//   a target goes to the first free slot of bucket b = mulhi(hash(v), nb), b + 1, ... (linear probing by bucket).
// Membership is then ONE 32-byte load in the common case: found if a slot equals v, absent if the bucket has a free
// slot, else the next bucket.  Exactly the set's membership (R8): the table holds the set's
// elements and nothing else.  The all-ones word marks a free slot; a set that contains it carries SITE_FLAG_HAS_ALLONES.
// The metadata-integrity profile authenticates the SORTED record, so it searches that, not the index; wg_policy_poke
// rebuilds the index from the rewritten array.
constexpr uint64_t kFree = ~0ull;
__host__ __device__ __forceinline__ uint64_t hash_base(uint32_t site, uint32_t off) {
  return (2ull * off + 4ull * site + 2ull) & ~3ull;
}
__host__ __device__ __forceinline__ uint32_t hash_target(uint32_t lo, uint32_t hi) {
  uint32_t h = lo * 0x9e3779b1u ^ (hi + 0x7f4a7c15u) * 0x85ebca6bu;
  h ^= h >> 15;
  h *= 0x2c1b3c6du;
  h ^= h >> 13;
  return h;
}
// the same lookup in two halves, so that a pass can have the first bucket of several lookups in flight at once
struct HashProbe {
  const ulonglong2* tab;
  uint32_t nb, b;
};
__device__ __forceinline__ HashProbe hash_probe(const Params& p, uint32_t site, uint32_t off, uint32_t cnt, uint32_t vl,
                                                uint32_t vh) {
  HashProbe h;
  h.nb = (cnt + 1u) >> 1;
  h.tab = reinterpret_cast<const ulonglong2*>(p.htab + hash_base(site, off));
  h.b = __umulhi(hash_target(vl, vh), h.nb);
  return h;
}
__device__ __forceinline__ bool hash_resolve(HashProbe h, uint32_t flags, uint32_t vl, uint32_t vh, ulonglong2 x, ulonglong2 y) {
  if ((vl & vh) == 0xffffffffu) return (flags & SITE_FLAG_HAS_ALLONES) != 0u;
  const uint64_t v = (static_cast<uint64_t>(vh) << 32) | vl;
  for (uint32_t i = 1;; ++i) {
    if (x.x == v || x.y == v || y.x == v || y.y == v) return true;
    if (x.x == kFree || x.y == kFree || y.x == kFree || y.y == kFree || i >= h.nb) return false;
    h.b = h.b + 1u == h.nb ? 0u : h.b + 1u;  // (rare: a full bucket without the value)
    x = __ldg(h.tab + 2u * h.b);
    y = __ldg(h.tab + 2u * h.b + 1u);
  }
}

__device__ __forceinline__ Sip32 init_state(const Params& p) {
  return Sip32{static_cast<uint32_t>(p.v0), static_cast<uint32_t>(p.v0 >> 32), static_cast<uint32_t>(p.v1),
               static_cast<uint32_t>(p.v1 >> 32), static_cast<uint32_t>(p.v2), static_cast<uint32_t>(p.v2 >> 32),
               static_cast<uint32_t>(p.v3), static_cast<uint32_t>(p.v3 >> 32)};
}

// token of a forward record ("a MAC over site_id, target_count, and allowed_targets"; R37):
// SipHash-2-4 over LE64(site_id) || LE64(cnt) || LE64(t_0) ... LE64(t_cnt-1), read through `load(i)`
template <typename LoadTarget>
__device__ __forceinline__ uint2 record_token(Sip32 s, uint32_t site, uint32_t cnt, LoadTarget load) {
  sip_absorb(s, site, 0u);
  sip_absorb(s, cnt, 0u);
  for (uint32_t i = 0; i < cnt; ++i) {
    const uint2 t = load(i);
    sip_absorb(s, t.x, t.y);
  }
  uint2 out;
  sip_finish_len(s, ((8u * (cnt + 2u)) & 0xffu) << 24, 0u, 0u, out.x, out.y);
  return out;
}

__device__ __forceinline__ Sip32 lds_state(uint32_t a) {
  const uint4 x = lds_v4(a), y = lds_v4(a + 16);
  return Sip32{x.x, x.y, x.z, x.w, y.x, y.y, y.z, y.w};
}

// warp-uniform running counters of one warp (flushed once at the end)
struct WarpCtr {
  uint32_t ret_checks, fwd_checks, ret_lanes, fwd_lanes;  // sign: ret_lanes = signed lanes, fwd_checks = skipped events
};

// ---------------------------------------------------------------------------------------------------
// MODE_VERIFY = wg_verify_continuations, MODE_FORWARD = wg_check_forward, MODE_SIGN = wg_sign_continuations.
// STAGED: the whole target table sits in shared memory.  TEL: a profile flag is set or the violation ring is on
// (compiled out of the ordinary launch).
// ---------------------------------------------------------------------------------------------------
template <int MODE, bool STAGED, bool TEL>
__global__ void __launch_bounds__(((MODE == MODE_FORWARD && STAGED) ? kWarpsFwd : kWarps) * 32, 1)
    wg_check_kernel(const Params p, const uint32_t stage_bytes, const uint32_t site_bytes) {
  // warps of this CTA.  (The forward kernel that looks targets up in the hash index keeps the 20-warp shape: at 64
  // registers it spills, and its lookups wait on DRAM, not on the shared-memory unit — measured on config 5's forward
  // entry: 0.80 ms with 20 warps, 0.90 ms with 32.)
  constexpr uint32_t kW = (MODE == MODE_FORWARD && STAGED) ? kWarpsFwd : kWarps;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint32_t lane, lanebit;
  asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));
  asm volatile("shl.b32 %0, 1, %1;" : "=r"(lanebit) : "r"(lane));
  const uint32_t ltmask = lanebit - 1u;
  // the shuffle tells the compiler that the warp index (and what derives from it) is warp-uniform
  const uint32_t warp = __shfl_sync(kFull, threadIdx.x >> 5, 0);
  const uint32_t smem0 = smem_u32(smem_raw);
  const uint32_t tg_s = smem0;
  // Per-site counter cache (site_bytes = 12 bytes x a power-of-two number of slots, or 0): a direct-mapped table in
  // shared memory, two candidate slots per site, {owner site, events, lanes checked}.  A slot is claimed by the first site that
  // asks for it (one compare-and-swap) and keeps it for the whole launch; that site's per-event counts are shared-memory
  // atomics from then on, flushed once per CTA.  Sites that find their slot taken use one reduction per event
  // straight to L2, as every site did before.  Why: under Zipf(1.1) one site takes 17 % of the events, and 13 M
  // same-address L2 reductions per launch serialise behind one another — measured 13.3 to 21 ms per verify launch from
  // run to run, against 12.9 ms without per-site counters.  A policy with no more sites than slots has every site cached
  // (config 3: 40 sites, whose global counters span a handful of L2 lines).
  uint32_t* site_s = reinterpret_cast<uint32_t*>(smem_raw + stage_bytes);
  const uint32_t cta_off = stage_bytes + site_bytes;
  unsigned long long* cnt64 = reinterpret_cast<unsigned long long*>(smem_raw + cta_off);
  uint32_t* bykind = reinterpret_cast<uint32_t*>(smem_raw + cta_off + C_WORDS * 8);
  const uint32_t mbar_cta = smem0 + cta_off + C_WORDS * 8 + 64;
  // violation counts of this CTA (ret lanes, fwd lanes, ret events, fwd events, blocked lanes, blocked events) and its
  // smallest first-violation key: a stream with 1 % violating events (config 5) sent 7 same-address reductions per
  // violating group to L2, where they queue behind one another (10 % of the launch, measured); once per CTA instead
  uint32_t* viol_s = reinterpret_cast<uint32_t*>(smem_raw + cta_off + C_WORDS * 8 + 80);
  unsigned long long* key_s = reinterpret_cast<unsigned long long*>(smem_raw + cta_off + C_WORDS * 8 + 112);
  constexpr bool FQ = MODE != MODE_SIGN && !STAGED;  // forward lookups go through the hash index and its queue
  constexpr uint32_t kQBytes = MODE == MODE_FORWARD ? 0u : kQueueItems * 2u;  // (the forward kernels have no work queue)
  const uint32_t rec_s = smem0 + cta_off + kCtaFixedBytes + warp * (kRecArea + kQBytes + kListBytes + (FQ ? kFwdQueueBytes : 0u));
  const uint32_t q_s = rec_s + kRecArea;                    // uniform items: q_s + 2 * k
  const uint32_t q_top = q_s + (kQueueItems - 1) * 2;        // divergent items: q_top - 2 * k
  const uint32_t list_s = q_s + kQBytes;
  const uint32_t fq_s = list_s + kListBytes;                // forward lookups (FQ): fq_s + 2 * k
  if (lane < 2) {  // the two dummy records: no active lane, nothing to queue
    sts_v4(rec_s + (lane * kGroupRecs + 32u) * kRecBytes + 32, 0u, 0u, 0u, 0u);
    sts_v4(rec_s + (lane * kGroupRecs + 32u) * kRecBytes + 48, 0u, 0u, 0u, 0u);
  }

  if (threadIdx.x < C_WORDS) cnt64[threadIdx.x] = 0ull;
  const uint32_t tbl_slots = site_bytes / 12u, tbl_mask = tbl_slots - 1u;  // site_s: [slots] owner, [slots][2] counts
  for (uint32_t i = threadIdx.x; i < site_bytes / 4; i += blockDim.x) site_s[i] = i < tbl_slots ? 0xffffffffu : 0u;
  if (threadIdx.x < 12) bykind[threadIdx.x] = 0u;  // 7 by-kind counts, then unknown / empty / misrouted events
  if (threadIdx.x < 8) viol_s[threadIdx.x] = 0u;
  if (threadIdx.x == 0) *key_s = ~0ull;
  if (threadIdx.x == 0) mbar_init(mbar_cta, 1);
  __syncthreads();
  if constexpr (STAGED) {
    if (threadIdx.x == 0) {
      mbar_expect_tx(mbar_cta, stage_bytes);
      tma_bulk_g2s(tg_s, p.tgts, stage_bytes, mbar_cta);
    }
    mbar_wait(mbar_cta, 0);
  }

  // a launch covers at most 2^27 events (wg_api.cu), so event and element indices (event * 32 + lane) fit 32 bits
  const uint32_t n_ev = static_cast<uint32_t>(p.n);
  const uint32_t n_groups = (n_ev + 31u) / 32u;
  // Groups are handed out dynamically, to the whole grid, from one ticket counter in global memory (one of a ring of
  // counters the engine owns, zeroed by the launcher): a warp takes four consecutive groups per ticket (one 64-bit-free atomic per 128 events; the claim is made
  // three groups before the group is needed, so its latency is never waited for), single groups near the end of the
  // stream so that the launch ends evenly.  A warp that waits longer on memory simply takes fewer groups; no SM, and no
  // sub-partition with one warp more than its neighbours, holds the launch back.
  // (A short stream — fewer than 16 groups per warp — is dealt out statically, group = warp + k * warps: the tickets of
  // 3,000 warps that all start at once would queue on the one counter for longer than such a launch lasts.)
  const bool dyn = n_groups >= 16u * gridDim.x * kW;
  uint32_t wnext = warp * gridDim.x + blockIdx.x, wleft = 0;  // (static dealing: consecutive groups go to different SMs)
  const uint32_t tail_from = n_groups > 8u * gridDim.x * kW ? n_groups - 8u * gridDim.x * kW : 0u;
  unsigned int* const sched = p.sched;
  auto claim = [&]() __attribute__((always_inline)) -> uint32_t {
    if (!dyn) {
      const uint32_t g = wnext;
      wnext += gridDim.x * kW;
      return g;
    }
    if (wleft == 0u) {
      const uint32_t sz = wnext < tail_from ? 4u : 1u;
      uint32_t t = 0;
      if (lane == 0) t = atomicAdd(sched, sz);
      wnext = __shfl_sync(kFull, t, 0);
      wleft = sz;
    }
    --wleft;
    return wnext++;
  };
  uint32_t gi = claim();
  uint32_t g_nxt = claim();
  const bool enforce = p.mode != 0;
  // large sets: the hash index, unless the metadata-integrity profile wants the authenticated sorted record searched
  const bool use_hash = FQ && !(TEL && (p.profile & PROFILE_METADATA_INTEGRITY));
  const Sip32 s_init = init_state(p);
  WarpCtr c = {0, 0, 0, 0};
  uint32_t par = 0;          // which half of the record area this group uses
  uint32_t nu = 0, nd = 0;   // items in the uniform / divergent queue (carried items first)
  bool have_prev = false;    // a previous group still waits for its epilogue
  uint32_t prev_e0 = 0;

  // ---- consumer passes ------------------------------------------------------------------------------
  // One pass = 64 queue items, two per lane (items k0 + lane and k0 + 32 + lane of the uniform or of the divergent
  // queue): twice the instruction-level parallelism of the dependent SipRound chains for the same instruction count.
  // ONE copy of this code serves both queues and the partial passes that flush them (on_a / on_b; a lane with on_b
  // false works on item a twice and drops the second result): with the producer and the event-parallel phases it has
  // to fit the 32 KB instruction cache — a version with one specialised copy per case ran at half speed on
  // no_instruction stalls.
  auto pass2 = [&](bool div, uint32_t k0, bool on_a, bool on_b) __attribute__((always_inline)) {
    if (!on_a) return;
    const uint32_t kb = on_b ? k0 + 32u : k0;
    const uint32_t qa = div ? mad32(k0 + lane, 0xfffffffeu, q_top) : mad32(k0 + lane, 2u, q_s);
    const uint32_t qb = div ? mad32(kb + lane, 0xfffffffeu, q_top) : mad32(kb + lane, 2u, q_s);
    const uint32_t ia = lds_u16(qa), ib = lds_u16(qb);            // slot * 32 + lane of the event
    const uint32_t ra = mad32(ia >> 5, kRecBytes, rec_s), rb = mad32(ib >> 5, kRecBytes, rec_s);  // the events' records
    const uint4 ca = lds_v4(ra + 32), cb = lds_v4(rb + 32);        // ctx lo, ctx hi, biased tag row pointer
    Sip32 sa = lds_state(ra), sb = lds_state(rb);
    const uint64_t* pa = item_ptr(ca.z, ca.w, ia);
    const uint64_t* pb = item_ptr(cb.z, cb.w, ib);
    uint2 ta = make_uint2(0u, 0u), tb = make_uint2(0u, 0u);
    if constexpr (MODE != MODE_SIGN) {
      ta = ldg_v2_stream(pa);
      tb = ldg_v2_stream(pb);
    }
    if (div) {
      // lane-divergent continuation: the states are the sites' pre-A states; absorb each item's own value, then bring
      // the states to where a warp-uniform event's state starts (B folded into v3, quarter A of the next round done)
      const uint2 wa = lds_v2(ra + 72), wb = lds_v2(rb + 72);  // biased value row pointers
      const uint2 va = ldg_v2_keep(item_ptr(wa.x, wa.y, ia)), vb = ldg_v2_keep(item_ptr(wb.x, wb.y, ib));
      sip_absorb_preA2(sa, sb, va.x, va.y, vb.x, vb.y);
      sip_qA(sa);
      sip_qA(sb);
      sa.v3l ^= ca.x; sa.v3h ^= ca.y;
      sb.v3l ^= cb.x; sb.v3h ^= cb.y;
    }
    const uint32_t la = ia & 31u, lb = ib & 31u;
    uint32_t al, ah, bl, bh;
    sa.v3l ^= la;
    sb.v3l ^= lb;
    sip_tail_ctxlane2(sa, sb, ca.x ^ la, ca.y, cb.x ^ lb, cb.y, ta.x, ta.y, tb.x, tb.y, al, ah, bl, bh);
    if constexpr (MODE == MODE_SIGN) {
      st_stream_v2(const_cast<uint64_t*>(pa), al, ah);
      if (on_b) st_stream_v2(const_cast<uint64_t*>(pb), bl, bh);
    } else {
      if ((al | ah | bl | bh) != 0u) {  // rare: a lane's token does not match
        if ((al | ah) != 0u) atoms_or(ra + 56, 1u << la);
        if ((bl | bh) != 0u) atoms_or(rb + 56, 1u << lb);  // (with on_b false this repeats item a's bit: harmless)
      }
    }
  };
  // run every full pass of both queues, then move what is left (< 64 items each) to the queue heads.
  // flush: also run a partial pass, leaving the queue empty.
  auto drain = [&](bool flush_u, bool flush_d) __attribute__((always_inline)) {
#pragma unroll 1
    for (uint32_t cl = 0; cl < 2u; ++cl) {
      const bool div = cl != 0u;
      const uint32_t n = div ? nd : nu;
      const bool flush = div ? flush_d : flush_u;
      const uint32_t kend = (flush ? n + 63u : n) & ~63u;  // where the passes stop (beyond n: a partial last pass)
      uint32_t k = 0;
#pragma unroll 1
      for (; k < kend; k += 64u) pass2(div, k, k + lane < n, k + 32u + lane < n);
      k = k < n ? k : n;
      const uint32_t r = n - k;  // < 64 items stay: two per lane
      uint32_t c0 = 0, c1 = 0;
      if (lane < r) c0 = lds_u16(div ? q_top - (k + lane) * 2u : q_s + (k + lane) * 2u);
      if (lane + 32u < r) c1 = lds_u16(div ? q_top - (k + 32u + lane) * 2u : q_s + (k + 32u + lane) * 2u);
      __syncwarp();
      if (lane < r) sts_u16(div ? q_top - lane * 2u : q_s + lane * 2u, c0);
      if (lane + 32u < r) sts_u16(div ? q_top - (32u + lane) * 2u : q_s + (32u + lane) * 2u, c1);
      if (div) nd = r; else nu = r;
    }
    __syncwarp();
  };

  // ---- forward lookups in the hash index (FQ): 64 queue items, two per lane, so that a lane has the buckets of two
  //      lookups in flight and the warp waits once per 64 lookups — not once per lane-divergent event plus once for the
  //      group's warp-uniform targets (config 5: 2.6 waits on DRAM per group, 25 % of the launch).  A target outside its
  //      set sets the lane's bit in the record's violation word; the event's own lane widens that to the whole active
  //      mask for a warp-uniform target afterwards. ----
  auto fpass = [&](uint32_t k0, uint32_t n) __attribute__((always_inline)) {
    if constexpr (FQ) {
      const uint32_t ka = k0 + lane < n ? k0 + lane : k0, kb = k0 + 32u + lane < n ? k0 + 32u + lane : k0;
      const uint32_t ia = lds_u16(fq_s + ka * 2u), ib = lds_u16(fq_s + kb * 2u);  // (past the end: item k0 once more)
      const uint32_t ra = mad32(ia >> 5, kRecBytes, rec_s), rb = mad32(ib >> 5, kRecBytes, rec_s);
      const uint2 wa = lds_v2(ra + 72), wb = lds_v2(rb + 72);  // biased value row pointers
      const uint2 va = ldg_v2_keep(item_ptr(wa.x, wa.y, ia)), vb = ldg_v2_keep(item_ptr(wb.x, wb.y, ib));
      const uint4 fa = lds_v4(ra), fb = lds_v4(rb);            // offset, count, flags of the events' sets
      const HashProbe ha = hash_probe(p, lds_u32(ra + 68), fa.x, fa.y, va.x, va.y);
      const HashProbe hb = hash_probe(p, lds_u32(rb + 68), fb.x, fb.y, vb.x, vb.y);
      const ulonglong2 xa = __ldg(ha.tab + 2u * ha.b), ya = __ldg(ha.tab + 2u * ha.b + 1u);
      const ulonglong2 xb = __ldg(hb.tab + 2u * hb.b), yb = __ldg(hb.tab + 2u * hb.b + 1u);
      if (!hash_resolve(ha, fa.z, va.x, va.y, xa, ya)) atoms_or(ra + 56, 1u << (ia & 31u));
      if (!hash_resolve(hb, fb.z, vb.x, vb.y, xb, yb)) atoms_or(rb + 56, 1u << (ib & 31u));
    }
  };

  // ---- event-parallel epilogue of a finished group: verdicts (a6), violation counters (a7), first violation (a8) ----
  auto epilogue = [&](uint32_t rpar, uint32_t e0) __attribute__((always_inline)) {
    if constexpr (MODE != MODE_SIGN) {
      const uint32_t ra = rec_s + (rpar * kGroupRecs + lane) * kRecBytes;
      const uint4 m = lds_v4(ra + 48);   // active, queue mask, viol, -
      const uint2 ms = lds_v2(ra + 64);  // meta, site
      const uint32_t active = m.x, cls = ms.x & 15u, kind = (ms.x >> 4) & 15u, viol = m.z, site = ms.y;
      const bool valid = cls != CLS_NONE;
      if (valid) st_stream_v2(p.out + (e0 + lane), viol, enforce ? (active & ~viol) : active);
      // violations are rare (0.05 % of events in the paper-shaped stream): one warp-uniform branch per group
      if (__ballot_sync(kFull, viol != 0u)) {
        const uint32_t pv = __popc(viol);
        const bool judged = cls == CLS_RET || cls == CLS_FWD;
        const bool known = valid && kind < 7u;
        const uint32_t rv = __reduce_add_sync(kFull, cls == CLS_RET ? pv : 0u);
        const uint32_t fv = __reduce_add_sync(kFull, cls == CLS_FWD ? pv : 0u);
        const uint32_t av = __reduce_add_sync(kFull, pv);
        const uint32_t rve = __popc(__ballot_sync(kFull, cls == CLS_RET && viol != 0u));
        const uint32_t fve = __popc(__ballot_sync(kFull, cls == CLS_FWD && viol != 0u));
        const uint32_t ave = __popc(__ballot_sync(kFull, viol != 0u));
        // first violation: smallest (seq << 5 | lane); seq = running event index (R12)
        unsigned long long key = ~0ull;
        if (viol) key = ((p.seq_base + (e0 + lane)) << 5) | static_cast<uint32_t>(__ffs(viol) - 1);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
          const unsigned long long o = __shfl_xor_sync(kFull, key, d);
          key = o < key ? o : key;
        }
        if (lane == 0) {  // (32-bit shared-memory atomics; a launch has fewer than 2^27 events, so no count wraps)
          if (rv) atomicAdd(&viol_s[0], rv);
          if (fv) atomicAdd(&viol_s[1], fv);
          if (rve) atomicAdd(&viol_s[2], rve);
          if (fve) atomicAdd(&viol_s[3], fve);
          if (enforce) {
            atomicAdd(&viol_s[4], av);
            atomicAdd(&viol_s[5], ave);
          }
          if (key < *reinterpret_cast<volatile unsigned long long*>(key_s)) atomicMin(key_s, key);  // (settles quickly)
        }
        if (TEL && viol && !(p.profile & PROFILE_LOW_TELEMETRY) && p.ring_cap != 0) {
          // violation ring (R27, R28): diagnostic, bounded; a full ring drops and counts
          const unsigned long long slot = atomicAdd(p.glob + C_RING_TOTAL, 1ull);
          if (slot < p.ring_cap) {
            const uint32_t fl = static_cast<uint32_t>(__ffs(viol) - 1);
            ViolRec r;
            r.seq = p.seq_base + (e0 + lane);
            r.site_id = site;
            r.kind = kind;
            r.viol_mask = viol;
            r.active_mask = active;
            r.lane = fl;
            r.mode = p.mode;
            r.observed = p.val[(e0 + lane) * 32u + fl];
            r.stored = (MODE == MODE_VERIFY && cls == CLS_RET) ? p.tag[(e0 + lane) * 32u + fl] : 0ull;
            p.ring[slot] = r;
          }
        }
        if (viol && known && !(TEL && (p.profile & PROFILE_LOW_TELEMETRY))) {
          unsigned long long* sc = p.site + static_cast<uint64_t>(site) * 4;  // (rare: straight to L2)
          if (judged) atomicAdd(sc + S_LANES_VIOLATION, static_cast<unsigned long long>(pv));
          if (enforce) atomicAdd(sc + S_LANES_BLOCKED, static_cast<unsigned long long>(pv));
        }
      }
    }
  };

  // ---- software pipeline of the event-parallel loads: the header two groups ahead, the site record one group ahead,
  //      so that the rows of the NEXT group can be pulled into L2 while this group is computed ----
  auto load_hdr = [&](uint32_t g) __attribute__((always_inline)) -> uint4 {  // (tickets run a few groups past the end: no 32-bit wrap)
    const uint32_t e = g * 32u + lane;
    return (g < n_groups && e < n_ev) ? ldg_v4(p.hdr + e) : make_uint4(0xffffffffu, 0u, 0u, 0u);
  };
  auto load_rec = [&](const uint4& h) __attribute__((always_inline)) -> uint4 {
    if (!FQ && !TEL)  // (the flags: hash index and coverage-reduced profile only)
      return h.x < p.n_sites ? ldg_rec3_l2keep(p.recs + h.x, l2_keep_policy()) : make_uint4(7u, 0u, 0u, 0u);
    return h.x < p.n_sites ? ldg_v4_l2keep(p.recs + h.x, l2_keep_policy()) : make_uint4(7u, 0u, 0u, 0u);
  };
  uint4 h_cur = load_hdr(gi);
  uint4 h_nxt = load_hdr(g_nxt);
  uint4 r_cur = load_rec(h_cur);

  // One trip per group of this warp, plus one last trip over an empty group (no valid event) that flushes the queues and
  // runs the last real group's epilogue: the drain / epilogue code exists once (the kernel must stay small enough for
  // the instruction cache: a version that inlined it twice ran at half speed on no_instruction stalls).
  bool last = gi >= n_groups;
  if (!last) do {
    last = gi >= n_groups;
    const uint32_t gn = g_nxt;
    const uint32_t e0 = gi * 32u;
    g_nxt = claim();
    const uint4 r_nxt = load_rec(h_nxt);
    const uint4 h_nn = load_hdr(g_nxt);
    const uint32_t rbase = rec_s + par * (kGroupRecs * kRecBytes);
    const uint32_t ra_me = rbase + lane * kRecBytes;
    const uint32_t slot_me = par * kGroupRecs + lane;
    const uint32_t cu = nu, cd = nd;  // items carried over from the previous group

    // ---- event-parallel: classify (a1, a2) ----
    const bool valid = e0 + lane < n_ev;
    const uint32_t site = h_cur.x;
    const uint32_t active = valid ? h_cur.y : 0u;
    const bool known = valid && site < p.n_sites;
    const uint32_t kind = known ? r_cur.x : 7u;
    const uint32_t off = r_cur.y, cnt = r_cur.z;
    uint32_t cls = CLS_NONE;
    if (valid) {
      if (known) {
        if constexpr (MODE == MODE_SIGN) {
          cls = (kind == K_RET && active != 0u) ? CLS_RET : CLS_COUNT;
        } else {
          if (active == 0u)
            cls = CLS_COUNT;  // fully predicated off: counted, not a check (R22)
          else if (TEL && ((kind == K_RET && (p.profile & PROFILE_SKIP_BACKWARD)) ||
                           (kind == K_FWD && (p.profile & PROFILE_SKIP_FORWARD))))
            cls = CLS_SKIP_DIR;   // outside this profile's protected set: separate denominator (R26)
          else if (TEL && (kind == K_RET || kind == K_FWD) && (p.profile & PROFILE_COVERAGE_REDUCED) &&
                   (r_cur.w & SITE_FLAG_SKIP))
            cls = CLS_SKIP_SITE;  // a site the coverage-reduced profile leaves out: separate denominator (R40)
          else if (kind == K_RET)
            cls = (MODE == MODE_VERIFY) ? CLS_RET : CLS_FAIL;  // no tag at the forward entry point (R14)
          else if (kind == K_FWD)
            cls = CLS_FWD;
          else
            cls = CLS_COUNT;  // non-protected kinds are only counted (R17)
        }
      } else {
        cls = (MODE == MODE_SIGN) ? CLS_COUNT : CLS_FAIL;  // unknown site: fail closed (R13)
      }
    }
    const uint32_t na = __popc(active);
    const uint32_t first = active ? static_cast<uint32_t>(__ffs(active) - 1) : 0u;
    const uint32_t m_ret = __ballot_sync(kFull, cls == CLS_RET);
    const uint32_t m_fwd = (MODE == MODE_SIGN) ? 0u : __ballot_sync(kFull, cls == CLS_FWD);
    uint32_t viol = (cls == CLS_FAIL) ? active : 0u;  // fail closed (R13, R14)
    {
      const uint64_t tp = reinterpret_cast<uint64_t>(MODE == MODE_SIGN ? p.tag_out : p.tag) + static_cast<uint64_t>(e0 + lane) * 256u -
                          static_cast<uint64_t>(slot_me) * 256u;
      const uint64_t vp = reinterpret_cast<uint64_t>(p.val) + static_cast<uint64_t>(e0 + lane) * 256u - static_cast<uint64_t>(slot_me) * 256u;
      // (the forward kernels run no MAC pass: nobody reads the context or the tag row there, and only the hash-index
      // lookups read the value-row pointer; their warps queue on the shared-memory unit, so what is not read is not written)
      if constexpr (MODE != MODE_FORWARD)
        sts_v4(ra_me + 32, h_cur.z & ~31u, h_cur.w, static_cast<uint32_t>(tp), static_cast<uint32_t>(tp >> 32));
      if constexpr (MODE != MODE_FORWARD || FQ)
        sts_v2(ra_me + 72, static_cast<uint32_t>(vp), static_cast<uint32_t>(vp >> 32));
    }
    sts_v4(ra_me + 48, active, cls == CLS_RET ? active : 0u, viol, 0u);
    sts_v2(ra_me + 64, cls | (kind << 4), site);
    if (FQ && cls == CLS_FWD) sts_v4(ra_me, off, cnt, r_cur.w, 0u);  // the set a queued lookup searches

    // ---- the producer's list of the group's protected events (event-parallel), padded to a multiple of kBatch with
    //      trips on the group's dummy record (no active lane: nothing is queued, nothing counted), so that a batch is
    //      straight-line code and every sync operation in it sees the whole warp ----
    const uint32_t need = (MODE == MODE_SIGN) ? m_ret : (m_ret | m_fwd);
    const uint32_t n_need = __popc(need);
    if (need != 0u) {
      const uint32_t row0 = static_cast<uint32_t>(__ffs(need) - 1) * 256u;  // a row that is read anyway (padding trips)
      // (bit 5 of the last word: a forward event; the shuffle that takes this word as its source lane reads bits 0-4)
      if (need & lanebit)
        // (third word: the queue item base; a forward kernel without the hash index queues nothing and carries the
        // event's active mask there instead, which saves the producer one shared-memory load per event)
        sts_v4(list_s + __popc(need & ltmask) * 16u, ra_me, lane * 256u, (MODE == MODE_FORWARD && !FQ) ? active : slot_me * 32u,
               first | ((FQ && cls == CLS_FWD) ? 32u : 0u));
      if (lane < ((kBatch - n_need) & (kBatch - 1u)))
        sts_v4(list_s + (n_need + lane) * 16u, rbase + 32u * kRecBytes, row0, (MODE == MODE_FORWARD && !FQ) ? 0u : (slot_me - lane + 32u) * 32u, 0u);
    }
    __syncwarp();  // the records and the list are visible to every lane
    // value rows, straight from global memory: one coalesced 256-byte load per event, kBatch in flight per lane; the
    // first batch is issued now and lands while the counters below are updated
    const char* vrow = reinterpret_cast<const char*>(elem_ptr(p.val, e0 * 32u + lane));
    uint2 va[kBatch], vb[kBatch];
    auto load_batch = [&](uint2 (&v)[kBatch], uint32_t b0) {
#pragma unroll
      for (int j = 0; j < static_cast<int>(kBatch); ++j) v[j] = ldg_v2_keep(byte_ptr(vrow, lds_u32(list_s + (b0 + j) * 16u + 4u)));
    };
    if (need != 0u) load_batch(va, 0u);

    // ---- counters that need no verdict (a7) ----
    const uint32_t judged_na = (cls == CLS_RET || cls == CLS_FWD) ? na : 0u;
    if constexpr (MODE == MODE_SIGN) {
      const bool is_ret = known && kind == K_RET;
      c.ret_lanes += __reduce_add_sync(kFull, is_ret ? na : 0u);           // signed lanes
      c.fwd_checks += __popc(__ballot_sync(kFull, valid && !is_ret));      // events that sign nothing
    } else {
      if (__ballot_sync(kFull, valid && (!known || active == 0u || cls == CLS_FAIL))) {  // uncommon events
        const uint32_t u = __popc(__ballot_sync(kFull, valid && !known));
        const uint32_t em = __popc(__ballot_sync(kFull, known && active == 0u));
        const uint32_t mr = __popc(__ballot_sync(kFull, known && cls == CLS_FAIL));
        if (lane == 0) {  // (32-bit shared-memory atomics: a 64-bit one is a compare-and-swap loop)
          if (u) atomicAdd(&bykind[8 + 0], u);
          if (em) atomicAdd(&bykind[8 + 1], em);
          if (mr) atomicAdd(&bykind[8 + 2], mr);
        }
      }
      c.ret_checks += __popc(m_ret);
      c.fwd_checks += __popc(m_fwd);
      c.ret_lanes += __reduce_add_sync(kFull, cls == CLS_RET ? na : 0u);
      c.fwd_lanes += __reduce_add_sync(kFull, cls == CLS_FWD ? na : 0u);
      if (known) atomicAdd(&bykind[kind], 1u);
      if constexpr (TEL) {
        if (p.profile & (PROFILE_SKIP_FORWARD | PROFILE_SKIP_BACKWARD | PROFILE_COVERAGE_REDUCED)) {
          const bool sd = cls == CLS_SKIP_DIR, ss = cls == CLS_SKIP_SITE;
          const uint32_t sr = __ballot_sync(kFull, sd && kind == K_RET);
          const uint32_t sf = __ballot_sync(kFull, sd && kind == K_FWD);
          const uint32_t sse = __ballot_sync(kFull, ss);
          const uint32_t srl = __reduce_add_sync(kFull, (sd && kind == K_RET) ? na : 0u);
          const uint32_t sfl = __reduce_add_sync(kFull, (sd && kind == K_FWD) ? na : 0u);
          const uint32_t ssl = __reduce_add_sync(kFull, ss ? na : 0u);
          if (lane == 0) {
            if (sr) atomicAdd(cnt64 + C_SKIP_RET_EVENTS, static_cast<unsigned long long>(__popc(sr)));
            if (srl) atomicAdd(cnt64 + C_SKIP_RET_LANES, static_cast<unsigned long long>(srl));
            if (sf) atomicAdd(cnt64 + C_SKIP_FWD_EVENTS, static_cast<unsigned long long>(__popc(sf)));
            if (sfl) atomicAdd(cnt64 + C_SKIP_FWD_LANES, static_cast<unsigned long long>(sfl));
            if (sse) atomicAdd(cnt64 + C_SKIP_SITE_EVENTS, static_cast<unsigned long long>(__popc(sse)));
            if (ssl) atomicAdd(cnt64 + C_SKIP_SITE_LANES, static_cast<unsigned long long>(ssl));
          }
        }
      }
      if (TEL && (p.profile & PROFILE_LOW_TELEMETRY)) {
        // "same checked transfers with less reporting" (PAPER.md Table A2): no per-site counters
      } else if (known) {
        bool cached = false;
        if (site_bytes) {
          // two candidate slots per site: a hot site that finds its first slot taken by an earlier (cold) site still
          // gets cached nearly always
          uint32_t slot = site & tbl_mask;
          uint32_t owner = site_s[slot];
          if (owner == 0xffffffffu) owner = atomicCAS(&site_s[slot], 0xffffffffu, site);  // claim a free slot
          if (owner != site && owner != 0xffffffffu) {
            slot = ((site * 0x9e3779b1u) >> 16) & tbl_mask;
            owner = site_s[slot];
            if (owner == 0xffffffffu) owner = atomicCAS(&site_s[slot], 0xffffffffu, site);
          }
          cached = owner == site || owner == 0xffffffffu;
          if (cached) {
            atomicAdd(&site_s[tbl_slots + 2u * slot], 1u);
            if (judged_na) atomicAdd(&site_s[tbl_slots + 2u * slot + 1u], judged_na);
          }
        }
        if (!cached) {  // one reduction per event straight to L2
          unsigned long long* sc = p.site + static_cast<uint64_t>(site) * 4;
          red_add_u64_l2keep(sc + S_EVENTS, 1ull, l2_keep_policy());
          if (judged_na) red_add_u64_l2keep(sc + S_LANES_CHECKED, static_cast<unsigned long long>(judged_na), l2_keep_policy());
        }
      }
    }

    // ---- producer loop (lane-parallel), one trip per protected event: warp-uniformity of the row just loaded, and
    //      for a return check the active lanes appended, compacted, to the queue of its class.  Double-buffered: the
    //      next batch's rows are requested before this batch is looked at. ----
    uint32_t divbits = 0;  // forward kernels: bit e = event e of the group has lane-divergent targets (warp-uniform word)
    if (need != 0u) {
      uint32_t qu = q_s + nu * 2u, qd = q_top - nd * 2u;  // where the next uniform / divergent item goes
      uint32_t qf = fq_s;                                  // ... and the next forward lookup
      auto consume_batch = [&](const uint2 (&v)[kBatch], uint32_t b0) {
#pragma unroll
        for (int j = 0; j < static_cast<int>(kBatch); ++j) {
          const uint4 le = lds_v4(list_s + (b0 + j) * 16u);  // record, row byte offset, queue item base, first active lane
          uint2 am;                                          // active, queue mask
          if constexpr (MODE == MODE_FORWARD && !FQ)
            am = make_uint2(le.z, 0u);
          else
            am = lds_v2(le.x + 48);
          const uint32_t rx = __shfl_sync(kFull, v[j].x, le.w), ry = __shfl_sync(kFull, v[j].y, le.w);
          uint32_t diff, div_;
          and_test(__ballot_sync(kFull, v[j].x != rx || v[j].y != ry), am.x, diff, div_);
          if constexpr (MODE == MODE_FORWARD)
            divbits |= div_ << ((le.y >> 8) & 31u);  // (kept in a register: one shared-memory store less per event)
          else
            sts_u32(le.x + 60, diff);  // (every lane stores the same word)
          if (FQ && use_hash && (le.w & 32u)) {
            // a forward event: one lookup for a warp-uniform target (the first active lane's), else one per active lane
            const uint32_t fm = div_ != 0u ? am.x : (1u << (le.w & 31u));
            if (fm & lanebit) sts_u16(mad32(__popc(fm & ltmask), 2u, qf), le.z + lane);
            qf = mad32(__popc(fm), 2u, qf);
            continue;
          }
          if (MODE == MODE_FORWARD || m_ret == 0u) continue;  // a group without return checks has nothing to queue
          const uint32_t rank = __popc(am.y & ltmask), nae = __popc(am.y);
          const bool div = div_ != 0u, act = (am.y & lanebit) != 0u;
          const uint32_t addr = div ? mad32(rank, 0xfffffffeu, qd) : mad32(rank, 2u, qu);
          if (act) sts_u16(addr, le.z + lane);
          qd = div ? mad32(nae, 0xfffffffeu, qd) : qd;
          qu = div ? qu : mad32(nae, 2u, qu);
          if (MODE == MODE_SIGN && !act && am.x != 0u)  // inactive lanes sign nothing (R10)
            st_stream_v2(const_cast<char*>(byte_ptr(reinterpret_cast<const char*>(elem_ptr(p.tag_out, e0 * 32u + lane)), le.y)), 0u, 0u);
        }
      };
#pragma unroll 1
      for (uint32_t b0 = 0;; b0 += 2u * kBatch) {
        const bool done = b0 >= n_need;
        if (FQ && use_hash) {
          // the queued forward lookups: all of them once the group's events are through, or when the next two batches
          // might not fit (one copy of this code: it sits at the loop head, which the last, empty trip also reaches)
          const uint32_t nf = (qf - fq_s) >> 1;
          if (nf != 0u && (done || nf > kFwdQueueItems - 2u * kBatch * 32u)) {
            __syncwarp();
#pragma unroll 1
            for (uint32_t k = 0; k < nf; k += 64u) fpass(k, nf);
            qf = fq_s;
            __syncwarp();
          }
        }
        if (done) break;
        const bool more = b0 + kBatch < n_need;
        if (more) load_batch(vb, b0 + kBatch);
        consume_batch(va, b0);
        if (more) {
          if (b0 + 2u * kBatch < n_need) load_batch(va, b0 + 2u * kBatch);
          consume_batch(vb, b0 + kBatch);
        }
      }
      nu = (qu - q_s) >> 1;
      nd = (q_top - qd) >> 1;
    }
    if constexpr (MODE == MODE_SIGN) {
      // every event that is not a return check gets a zero row (R10): non-return sites, empty masks; written as
      // 16-byte stores: a half-warp covers one 256-byte row, one instruction covers two events
      const uint32_t zmask = __ballot_sync(kFull, valid && cls != CLS_RET);
      if (zmask) {
        const uint32_t half = lane >> 4, chunk = lane & 15u;
#pragma unroll 4
        for (int j = 0; j < 16; ++j) {
          const uint32_t e = 2u * j + half;
          if ((zmask >> e) & 1u)
            asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%1,%1,%1};" ::"l"(elem_ptr(p.tag_out, (e0 + e) * 32u + chunk * 2u)), "r"(0u) : "memory");
        }
      }
    }
    __syncwarp();

    // ---- event-parallel: per-event part of the MAC; search of warp-uniform forward targets ----
    {
      const bool judged = cls == CLS_RET || cls == CLS_FWD;
      const bool is_uni = judged && (MODE == MODE_FORWARD ? ((divbits >> lane) & 1u) == 0u : lds_u32(ra_me + 60) == 0u);
      uint32_t ul = 0, uh = 0;
      if (is_uni && !(use_hash && cls == CLS_FWD)) {
        const uint2 r = ldg_v2_keep(elem_ptr(p.val, (e0 + lane) * 32u + first));  // the event's one value (an L1 hit)
        ul = r.x;
        uh = r.y;
      }
      if (MODE != MODE_FORWARD && m_ret != 0u) {
        // the site word of the MAC, once per event; the key-derived initial state exists in the kernel parameters only
        // (constant bank).  Leaves the "pre-A" state the lane-divergent tails start from.
        Sip32 st = s_init;
        sip_absorb(st, site, p.bind_hi);  // LE64(site_id | digest32 << 32): zero-extended site id unless bound (R3, R5, R39)
        sip_qA(st);
        if (is_uni) {
          sip_absorb_preA(st, ul, uh);  // the continuation word, once per event
          sip_qA(st);                   // quarter A of the context word's first round
          st.v3l ^= h_cur.z & ~31u;     // and the lane-independent bits of the context word
          st.v3h ^= h_cur.w;
        }
        if (cls == CLS_RET) {
          sts_v4(ra_me, st.v0l, st.v0h, st.v1l, st.v1h);
          sts_v4(ra_me + 16, st.v2l, st.v2h, st.v3l, st.v3h);
        }
      }
      if constexpr (MODE != MODE_SIGN) {
        bool bad_rec = false;
        if constexpr (TEL) {
          // metadata integrity: the forward record is re-authenticated before it is used, once per
          // event; a record that fails authorises nothing: every active lane violates
          if (p.profile & PROFILE_METADATA_INTEGRITY) {
            if (cls == CLS_FWD) {
              const uint2 tok = __ldg(reinterpret_cast<const uint2*>(p.tok) + site);
              uint2 tk;
              if constexpr (STAGED) {
                const uint32_t base = tg_s + off * 8;
                tk = record_token(s_init, site, cnt, [&](uint32_t i) { return lds_v2(base + i * 8); });
              } else {
                const uint2* set = reinterpret_cast<const uint2*>(p.tgts + off);
                tk = record_token(s_init, site, cnt, [&](uint32_t i) { return __ldcg(set + i); });
              }
              bad_rec = tk.x != tok.x || tk.y != tok.y;
            }
            const uint32_t m_bad = __ballot_sync(kFull, bad_rec);
            if (m_bad && lane == 0)
              atomicAdd(p.glob + C_META_FAIL, static_cast<unsigned long long>(__popc(m_bad)));
          }
        }
        // lane-divergent forward targets are searched per lane, one event at a time (per-warp checking
        // only after proving uniformity); a warp-uniform target is searched once, by the event's lane
        uint32_t fviol = 0;
        if (use_hash) {
          // the lookups went through the queue; a warp-uniform target outside the set fails every active lane
          if (cls == CLS_FWD) {
            const uint32_t v = lds_u32(ra_me + 56);
            sts_u32(ra_me + 56, is_uni ? (v != 0u ? active : 0u) : v);
          }
        } else {
          for (uint32_t m = __ballot_sync(kFull, cls == CLS_FWD && !is_uni && !bad_rec); m; m &= m - 1) {
            const uint32_t e = __ffs(m) - 1;
            const uint32_t a = __shfl_sync(kFull, active, e);
            const uint32_t o2 = __shfl_sync(kFull, off, e), c2 = __shfl_sync(kFull, cnt, e);
            const uint2 v = ldg_v2_keep(elem_ptr(p.val, (e0 + e) * 32u + lane));
            const bool in = member<STAGED>(p, tg_s, o2, c2, v.x, v.y);
            const uint32_t vb = __ballot_sync(kFull, (a & lanebit) && !in);
            if (lane == e) fviol = vb;
          }
          if (cls == CLS_FWD) {
            if (bad_rec)
              fviol = active;
            else if (is_uni)
              fviol = member<STAGED>(p, tg_s, off, cnt, ul, uh) ? 0u : active;
            sts_u32(ra_me + 56, fviol);
          }
        }
      }
    }
    // ---- tag rows -> L2: lane i pulls the tag row of event i of THIS group if it is a return check; the passes that
    //      gather from it start below (their first items are carried ones, whose rows came in a group ago).  Rows that
    //      were fetched a whole group ahead sat in L2 for up to two groups: with 2,960 warps that footprint (up to
    //      97 MB of rows) did not fit beside a large policy's tables, and rows were fetched from DRAM twice (measured:
    //      config 5 read 5.72 GB per batch, 4.95 GB now; config 4 26.8 -> 24.7 GB per launch, its algorithmic bytes) ----
    if (MODE == MODE_VERIFY && cls == CLS_RET)
      prefetch_row_l2(reinterpret_cast<const char*>(elem_ptr(p.tag, (e0 + lane) * 32u)));
    __syncwarp();

    // ---- consumer passes: every full pass; carried items of the previous group go first.  If a queue still holds
    //      items of the previous group and cannot fill a pass, it is flushed with a partial pass (rare). ----
    // (carried items are the oldest: any full pass consumes them; fewer than 64 are carried per queue)
    drain(last || (cu != 0u && nu < 64u), last || (cd != 0u && nd < 64u));
    // ---- the next group's value rows -> L2, as late as possible (see above): lane i pulls row i of the next group if
    //      that event will need it (its site record has arrived by now); rows nobody will read are not fetched ----
    if (gn < n_groups) {
      const bool v_nxt = gn * 32u + lane < n_ev && h_nxt.y != 0u;
      const bool ret_nxt = v_nxt && r_nxt.x == K_RET, fwd_nxt = v_nxt && r_nxt.x == K_FWD;
      if (MODE == MODE_FORWARD ? fwd_nxt : (MODE == MODE_SIGN ? ret_nxt : (ret_nxt || fwd_nxt)))
        prefetch_row_l2(reinterpret_cast<const char*>(elem_ptr(p.val, (gn * 32u + lane) * 32u)));
    }
    if (have_prev) epilogue(par ^ 1u, prev_e0);
    have_prev = true;
    prev_e0 = e0;
    par ^= 1u;
    gi = gn;
    h_cur = h_nxt;
    r_cur = r_nxt;
    h_nxt = h_nn;
    __syncwarp();
  } while (!last);

  // ---- flush: warp registers -> CTA shared memory -> one global atomic per counter per CTA ----
  if (lane == 0) {
    if constexpr (MODE == MODE_SIGN) {
      if (c.ret_lanes) atomicAdd(cnt64 + C_SIGNED_LANES, static_cast<unsigned long long>(c.ret_lanes));
      if (c.fwd_checks) atomicAdd(cnt64 + C_SIGN_SKIPPED, static_cast<unsigned long long>(c.fwd_checks));
    } else {
      if (c.ret_checks) atomicAdd(cnt64 + C_RET_CHECKS, static_cast<unsigned long long>(c.ret_checks));
      if (c.fwd_checks) atomicAdd(cnt64 + C_FWD_CHECKS, static_cast<unsigned long long>(c.fwd_checks));
      if (c.ret_lanes) atomicAdd(cnt64 + C_RET_LANES, static_cast<unsigned long long>(c.ret_lanes));
      if (c.fwd_lanes) atomicAdd(cnt64 + C_FWD_LANES, static_cast<unsigned long long>(c.fwd_lanes));
    }
  }
  // every event of the launch is counted once (the kernel walks all of them)
  if (MODE != MODE_SIGN && blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(cnt64 + C_EVENTS_TOTAL, static_cast<unsigned long long>(p.n));
  __syncthreads();
  if (threadIdx.x < C_WORDS) {  // (words updated in global memory directly, and the host-side words, stay 0 here)
    unsigned long long v = cnt64[threadIdx.x];
    if (threadIdx.x >= C_BY_KIND && threadIdx.x < C_BY_KIND + 7) v = bykind[threadIdx.x - C_BY_KIND];
    if (threadIdx.x == C_EVENTS_UNKNOWN) v = bykind[8 + 0];
    if (threadIdx.x == C_EVENTS_EMPTY) v = bykind[8 + 1];
    if (threadIdx.x == C_EVENTS_MISROUTED) v = bykind[8 + 2];
    if (threadIdx.x == C_RET_VIOL) v = viol_s[0];
    if (threadIdx.x == C_FWD_VIOL) v = viol_s[1];
    if (threadIdx.x == C_RET_VIOL_EVENTS) v = viol_s[2];
    if (threadIdx.x == C_FWD_VIOL_EVENTS) v = viol_s[3];
    if (threadIdx.x == C_BLOCKED_LANES) v = viol_s[4];
    if (threadIdx.x == C_BLOCKED_EVENTS) v = viol_s[5];
    if (v) atomicAdd(p.glob + threadIdx.x, v);
  }
  if (MODE != MODE_SIGN && threadIdx.x == 0 && *key_s != ~0ull) atomicMin(p.glob + C_FIRST_VIOLATION, *key_s);
  for (uint32_t i = threadIdx.x; i < tbl_slots; i += blockDim.x) {  // the cached sites' counts, once per CTA
    const uint32_t owner = site_s[i];
    if (owner != 0xffffffffu) {
      const uint32_t ev = site_s[tbl_slots + 2u * i], ln = site_s[tbl_slots + 2u * i + 1u];
      unsigned long long* sc = p.site + static_cast<uint64_t>(owner) * 4;
      if (ev) atomicAdd(sc + S_EVENTS, static_cast<unsigned long long>(ev));
      if (ln) atomicAdd(sc + S_LANES_CHECKED, static_cast<unsigned long long>(ln));
    }
  }
}

// first-violation record (R29), one thread, enqueued behind every check launch: the launch is over, so
// the key is final for it; if the key moved into that launch's event range the full record of that event is written.
// Deterministic, and nothing on the hot path: violations only did the atomicMin they always did.
__global__ void wg_first_record(const Params p, const int has_tag) {
  const unsigned long long key = p.glob[C_FIRST_VIOLATION];
  const unsigned long long seq = key >> 5;
  if (key == ~0ull || key == p.first->key || seq < p.seq_base || seq - p.seq_base >= p.n) return;
  const uint64_t i = seq - p.seq_base;
  const uint32_t fl = static_cast<uint32_t>(key & 31u);
  const uint4 hh = p.hdr[i];
  const uint2 o = p.out[i];
  ViolRec r;
  r.seq = seq;
  r.site_id = hh.x;
  r.kind = hh.x < p.n_sites ? p.recs[hh.x].kind : 7u;
  r.viol_mask = o.x;
  r.active_mask = hh.y;
  r.lane = fl;
  r.mode = p.mode;
  r.observed = p.val[i * 32 + fl];
  const bool skipped = (r.kind == K_RET && (p.profile & PROFILE_SKIP_BACKWARD)) ||
                       (hh.x < p.n_sites && (p.profile & PROFILE_COVERAGE_REDUCED) && (p.recs[hh.x].flags & SITE_FLAG_SKIP));
  const bool judged_ret = has_tag && r.kind == K_RET && !skipped;
  r.stored = judged_ret ? p.tag[i * 32 + fl] : 0ull;
  p.first->rec = r;
  p.first->key = key;
}

// tokens of the forward records as loaded (trusted load time; R37), one thread per site
__global__ void wg_build_tokens(uint64_t* tok, const SiteRec* recs, const uint64_t* tgts, uint32_t n_sites, uint64_t v0,
                                uint64_t v1, uint64_t v2, uint64_t v3) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_sites) return;
  const SiteRec r = recs[s];
  uint64_t t = 0;
  if (r.kind == K_FWD) {
    const uint2* set = reinterpret_cast<const uint2*>(tgts + r.off);
    const Sip32 s0{static_cast<uint32_t>(v0), static_cast<uint32_t>(v0 >> 32), static_cast<uint32_t>(v1),
                   static_cast<uint32_t>(v1 >> 32), static_cast<uint32_t>(v2), static_cast<uint32_t>(v2 >> 32),
                   static_cast<uint32_t>(v3), static_cast<uint32_t>(v3 >> 32)};
    const uint2 tk = record_token(s0, s, r.cnt, [&](uint32_t i) { return set[i]; });
    t = (static_cast<uint64_t>(tk.y) << 32) | tk.x;
  }
  tok[s] = t;
}

// hash index build (load time): one thread per target finds its site (binary search over the records' offsets) and
// claims the first free slot of its probe sequence
__global__ void wg_build_hash(uint64_t* htab, SiteRec* recs, const uint64_t* tgts, uint32_t n_sites, uint64_t n_tgts) {
  const uint64_t i = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n_tgts) return;
  uint32_t lo = 0, len = n_sites;  // last site with off <= i that owns targets: sites without targets share offsets
  while (len > 1) {
    const uint32_t half = len >> 1;
    if (recs[lo + half].off <= i) lo += half;
    len -= half;
  }
  while (recs[lo].cnt == 0u || recs[lo].off + recs[lo].cnt <= i) --lo;  // (step back over empty sites at the same offset)
  const SiteRec r = recs[lo];
  const uint64_t v = tgts[i];
  if (v == kFree) {  // the free-slot marker cannot be stored: the site's record carries a flag instead
    atomicOr(&recs[lo].flags, SITE_FLAG_HAS_ALLONES);
    return;
  }
  const uint32_t nb = (r.cnt + 1u) >> 1;
  unsigned long long* tab = reinterpret_cast<unsigned long long*>(htab + hash_base(lo, r.off));
  uint32_t b = __umulhi(hash_target(static_cast<uint32_t>(v), static_cast<uint32_t>(v >> 32)), nb);
  for (;;) {
    for (uint32_t k = 0; k < 4u; ++k)
      if (atomicCAS(tab + 4u * b + k, kFree, v) == kFree) return;
    b = b + 1u == nb ? 0u : b + 1u;
  }
}

__global__ void wg_set_site_flags(SiteRec* recs, const uint8_t* skip, uint32_t n_sites) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n_sites) recs[s].flags = (recs[s].flags & ~SITE_FLAG_SKIP) | ((skip && skip[s]) ? SITE_FLAG_SKIP : 0u);
}

__global__ void wg_clear_allones_flags(SiteRec* recs, uint32_t n_sites) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n_sites) recs[s].flags &= ~SITE_FLAG_HAS_ALLONES;
}

template <int MODE>
cudaError_t launch_mode(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches) {
  const uint64_t n_groups = (p.n + 31) / 32;
  const uint64_t want = n_groups;  // a short stream is spread over all SMs, a few warps each, not packed into a few full CTAs
  const int grid = static_cast<int>(want < static_cast<uint64_t>(sm_count) ? want : sm_count);
  const bool staged = MODE != MODE_SIGN && p.n_tgts > 0 && p.n_tgts <= kMaxStageTgts;
  const uint32_t W = (MODE == MODE_FORWARD && staged) ? kWarpsFwd : kWarps;  // (the kernel's kW)
  const uint32_t stage_bytes = staged ? static_cast<uint32_t>((p.n_tgts * 8 + 15) & ~15ull) : 0u;
  // the per-site counter cache: the largest power-of-two slot count <= kMaxCacheSlots that fits beside the staged
  // targets (and no more than twice the policy needs); sign keeps no per-site counters
  const uint32_t warp_bytes = (MODE == MODE_FORWARD ? kWarpBytesFwd : kWarpBytes) +
                              ((MODE != MODE_SIGN && !staged) ? kFwdQueueBytes : 0u);  // (the kernel's FQ)
  uint32_t site_bytes = 0;
  if (MODE != MODE_SIGN && p.n_sites > 0) {
    const uint32_t left = kSmemMax - kCtaFixedBytes - W * warp_bytes;
    uint32_t slots = kMaxCacheSlots;
    while (slots >= 64u && (stage_bytes + slots * 12u > left || slots / 2u >= p.n_sites)) slots /= 2u;
    if (slots >= 64u) site_bytes = slots * 12u;
  }
  const uint32_t smem = stage_bytes + site_bytes + kCtaFixedBytes + W * warp_bytes;
  const bool tel = MODE != MODE_SIGN && (p.profile != 0 || p.ring_cap != 0);
  {  // the launch's group ticket starts at 0
    const cudaError_t e = cudaMemsetAsync(p.sched, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
  }
  if (tel) {
    if constexpr (MODE != MODE_SIGN) {
      if (staged)
        wg_check_kernel<MODE, true, true><<<grid, W * 32, smem, st>>>(p, stage_bytes, site_bytes);
      else
        wg_check_kernel<MODE, false, true><<<grid, W * 32, smem, st>>>(p, stage_bytes, site_bytes);
    }
  } else if (staged) {
    wg_check_kernel<MODE, true, false><<<grid, W * 32, smem, st>>>(p, stage_bytes, site_bytes);
  } else {
    wg_check_kernel<MODE, false, false><<<grid, W * 32, smem, st>>>(p, stage_bytes, site_bytes);
  }
  ++*launches;
  return cudaGetLastError();
}

template <int MODE, bool STAGED>
cudaError_t opt_in() {
  if constexpr (MODE != MODE_SIGN) {
    const cudaError_t e = cudaFuncSetAttribute(wg_check_kernel<MODE, STAGED, true>,
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(kSmemMax));
    if (e != cudaSuccess) return e;
  }
  return cudaFuncSetAttribute(wg_check_kernel<MODE, STAGED, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              static_cast<int>(kSmemMax));
}

}  // namespace

cudaError_t init_kernels() {
  cudaError_t e;
  if ((e = opt_in<MODE_VERIFY, true>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_VERIFY, false>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_FORWARD, true>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_FORWARD, false>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_SIGN, false>()) != cudaSuccess) return e;
  return cudaSuccess;
}

cudaError_t launch_sign(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches) {
  return launch_mode<MODE_SIGN>(p, sm_count, st, launches);
}

cudaError_t launch_check(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches) {
  // without a return site in the policy no event can be a return check: the verify decides exactly what the forward entry
  // point decides (unknown sites fail closed in both) and runs its leaner, wider kernel
  return (p.tag && p.has_ret) ? launch_mode<MODE_VERIFY>(p, sm_count, st, launches) : launch_mode<MODE_FORWARD>(p, sm_count, st, launches);
}

cudaError_t launch_first_record(const Params& p, cudaStream_t st, uint64_t* launches) {
  wg_first_record<<<1, 1, 0, st>>>(p, p.tag != nullptr);
  ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_clear_allones_flags(SiteRec* recs, uint32_t n_sites, cudaStream_t st, uint64_t* launches) {
  if (n_sites == 0) return cudaSuccess;
  wg_clear_allones_flags<<<(n_sites + 255) / 256, 256, 0, st>>>(recs, n_sites);
  ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_build_hash(uint64_t* htab, SiteRec* recs, const uint64_t* tgts, uint32_t n_sites, uint64_t n_tgts,
                              cudaStream_t st, uint64_t* launches) {
  if (n_tgts == 0) return cudaSuccess;
  wg_build_hash<<<static_cast<unsigned>((n_tgts + 255) / 256), 256, 0, st>>>(htab, recs, tgts, n_sites, n_tgts);
  ++*launches;
  return cudaGetLastError();
}

uint64_t max_staged_targets() { return kMaxStageTgts; }

cudaError_t launch_set_site_flags(SiteRec* recs, const uint8_t* d_skip, uint32_t n_sites, cudaStream_t st, uint64_t* launches) {
  if (n_sites == 0) return cudaSuccess;
  wg_set_site_flags<<<(n_sites + 255) / 256, 256, 0, st>>>(recs, d_skip, n_sites);
  ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_build_tokens(uint64_t* tok, const SiteRec* recs, const uint64_t* tgts, uint32_t n_sites, uint64_t v0,
                                uint64_t v1, uint64_t v2, uint64_t v3, cudaStream_t st, uint64_t* launches) {
  if (n_sites == 0) return cudaSuccess;
  wg_build_tokens<<<(n_sites + 255) / 256, 256, 0, st>>>(tok, recs, tgts, n_sites, v0, v1, v2, v3);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace wg
