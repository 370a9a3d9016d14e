// wg_kernels_v2.cu — the check path on sm_100a, second mapping: a warp owns a TILE of 16 consecutive events.
//
// Steps: a1 event fetch + guard, a2 policy lookup, a3 MAC sign, a4 MAC verify + compare,
// a5 forward membership, a6 verdicts, a7 counters, a8 first-violation record.  Paper passages: backward token
// PAPER.md:162, 248; forward membership PAPER.md:174-178, 250-252; guards PAPER.md:190, 230; detect / enforce
// PAPER.md:264; accounting PAPER.md:113, 127, 224.  Readings: DESIGN.md §2.  Kernel design: DESIGN.md §6.
//
// What bounds it (measured, profiles/): the SipRound is 20 ALU-pipe instructions (4 IADD3 with carry-out,
// 8 LOP3, 8 SHF) + 4 IMAD.X on the FMA pipe, and every ALU-pipe instruction costs 2 issue cycles per warp on
// sm_100a, so a round is 40 cycles per warp per SM sub-partition whatever the occupancy or ILP.  The kernel is
// therefore built to (1) run fewer rounds and (2) spend as few ALU-pipe instructions as possible on anything else.
//
// Per tile the warp runs two kinds of phases:
//   "event-parallel" (lane i <-> event i of the tile): header decode, policy gather (one 64-byte SiteRec),
//       classification, the part of the MAC that is the same for every lane of an event — the per-site
//       mid-state comes from the SiteRec, and when the event's continuation is warp-uniform the continuation
//       word is absorbed here too, ONCE per event instead of once per lane — the membership search of
//       warp-uniform forward targets (each unique target is searched once per warp), verdict / counter epilogue;
//   "lane-parallel" (lane l <-> lane l of one event): the per-lane tail of the MAC (8 of the 12 SipRounds for
//       a warp-uniform continuation, 10 otherwise) and the compare; per-lane searches of lane-divergent targets.
// Event rows reach shared memory by TMA bulk copies (cp.async.bulk, one copy per run of consecutive needed rows,
// only the rows the tile needs) that complete on the warp's own mbarrier; 20 warps per SM keep the ALU pipe fed while
// other warps wait for their rows.  When the policy's whole target table is small (<= kMaxStageTgts entries)
// every CTA stages it in shared memory once with one more bulk copy.
// Counters: warp-uniform registers + shared-memory atomics, flushed once per CTA; per-site counters live in shared
// memory for small policies, else one L2 reduction per event and counter.
#include "wg_internal.h"
#include "../../include/warpguard_sip32.cuh"

namespace wg {

namespace {

enum : int { MODE_VERIFY = 0, MODE_FORWARD = 1, MODE_SIGN = 2 };
enum : uint32_t { K_RET = 0, K_FWD = 1 };
// what the tile does with an event
enum : uint32_t { CLS_NONE = 0, CLS_COUNT = 1, CLS_RET = 2, CLS_FWD = 3, CLS_FAIL = 4, CLS_SKIP = 5 };

#ifndef WG_TILE
#define WG_TILE 16
#endif
#ifndef WG_WARPS_CHECK
#define WG_WARPS_CHECK 20
#endif
#ifndef WG_WARPS_SIGN
#define WG_WARPS_SIGN 20
#endif
constexpr int kT = WG_TILE;            // events per tile (<= 32: one lane per event in the event-parallel phases)
static_assert(kT == 8 || kT == 16 || kT == 32, "tile size");
constexpr uint32_t kSmemMax = 232448;  // 227 KB opt-in shared memory per CTA on sm_100a
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kMaxSmemSites = 1024;  // policies up to this size keep their per-site counters in shared memory

// ---- shared-memory carve-up ----------------------------------------------------------------------
// CTA part: [tgts staged: stage_bytes][per-site counters: site_bytes][cnt64: 32 x u64][bykind: 8 x u32][mbar: u64, pad]
// warp part: raw headers [2][T] x 16 B (this tile, next tile), decoded headers [T] x 16 B
//            {8 * first active lane, active mask, context_base & ~31 (lo), context_base (hi)},
//            per-event SipHash states [T] x 32 B, the warp's mbarrier, value rows [T][32] u64,
//            (verify only) tag rows [T][32] u64
template <int MODE>
struct WarpLayout {
  static constexpr uint32_t kRaw = 0;
  static constexpr uint32_t kDec = kRaw + 2 * kT * 16;
  static constexpr uint32_t kSt = kDec + kT * 16;
  static constexpr uint32_t kBar = kSt + kT * 32;
  static constexpr uint32_t kViol = kBar + 16;  // [T] u32 violation masks of the tile
  static constexpr uint32_t kList = kViol + kT * 4;  // [T * 32] u16 work items (event * 32 + lane) of the sparse path
  static constexpr uint32_t kVal = kList + (MODE == MODE_FORWARD ? 0 : kT * 64);
  static constexpr uint32_t kTag = kVal + kT * 256;
  static constexpr uint32_t kBytes = kTag + (MODE == MODE_VERIFY ? kT * 256 : 0);
};
constexpr uint32_t kCtaFixedBytes = 32 * 8 + 8 * 4 + 16 + 16;  // cnt64, bykind, mbar (+pad to 16)

// warps per CTA (one CTA per SM) and the largest target table that still fits beside the warps' buffers
template <int MODE>
struct Cfg {
  static constexpr int kWarps = (MODE == MODE_SIGN) ? WG_WARPS_SIGN : WG_WARPS_CHECK;
  static constexpr int kThreads = kWarps * 32;
  static constexpr uint32_t kLeft = kSmemMax - kCtaFixedBytes - kWarps * WarpLayout<MODE>::kBytes;
  static constexpr uint32_t kMaxStageTgts = (kLeft / 16 * 2) < 2048 ? (kLeft / 16 * 2) : 2048;
};

// ---- PTX helpers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ uint4 ldg_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream_v2(void* p, uint32_t a, uint32_t b) {
  asm volatile("st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}
// tag row store of the sign kernels: the token for an active lane, zero for an inactive one (R10), as two
// predicated stores (one ALU-pipe instruction for the predicate instead of two selects)
__device__ __forceinline__ void st_tag_or_zero(void* p, uint32_t on, uint32_t lo, uint32_t hi) {
  asm volatile(
      "{\n\t.reg .pred q;\n\t"
      "setp.ne.u32 q, %3, 0;\n\t"
      "@q st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};\n\t"
      "@!q st.global.L1::no_allocate.v2.u32 [%0], {%4,%4};\n\t}" ::"l"(p),
      "r"(lo), "r"(hi), "r"(on), "r"(0u)
      : "memory");
}
__device__ __forceinline__ void st_stream_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d)
               : "memory");
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
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "r"(x) : "memory");
}
__device__ __forceinline__ void atoms_or(uint32_t a, uint32_t x) {
  asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(a), "r"(x) : "memory");
}
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t x) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(x) : "memory");
}
// a * b + c on the FMA pipe (address arithmetic inside the ALU-bound loops)
__device__ __forceinline__ uint32_t mad32(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ void sts_v4(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

// TMA 1-D bulk copy global -> shared, completion on an mbarrier (whole-table staging of the target sets)
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
__device__ __forceinline__ void tma_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
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
    // large sets live in L2 / HBM and every probe is a dependent ~1 us load: quaternary steps issue three
    // independent probes at once and halve the number of dependent rounds (config 5: sets up to 4,096 entries;
    // measured 2.55 -> 2.38 ms per batch; 8-ary steps were slower again, 2.49 ms: more traffic than latency saved)
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
// token of a forward record ("a MAC over site_id, target_count, and allowed_targets"; R37):
// SipHash-2-4 over LE64(site_id) || LE64(cnt) || LE64(t_0) ... LE64(t_cnt-1), read through `load(i)`
template <typename LoadTarget>
__device__ __forceinline__ uint2 record_token(uint64_t v0, uint64_t v1, uint64_t v2, uint64_t v3, uint32_t site,
                                              uint32_t cnt, LoadTarget load) {
  Sip32 s{static_cast<uint32_t>(v0), static_cast<uint32_t>(v0 >> 32), static_cast<uint32_t>(v1),
          static_cast<uint32_t>(v1 >> 32), static_cast<uint32_t>(v2), static_cast<uint32_t>(v2 >> 32),
          static_cast<uint32_t>(v3), static_cast<uint32_t>(v3 >> 32)};
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

// what lane i knows about event i of the tile
struct TileEv {
  uint32_t site, active, cls, kind;
  uint32_t off, cnt;  // protected-forward: the site's set
  uint32_t tokl, tokh;  // protected-forward: the record's token at load time (metadata-integrity profile)
  Sip32 st;           // protected-return: the site's pre-A mid-state
};

// warp-uniform running counters of one warp (flushed once at the end)
struct WarpCtr {
  uint32_t total, empty, unknown, misrouted, ret_checks, fwd_checks, ret_lanes, fwd_lanes, signed_lanes, skipped;
};

// event-parallel: decode header i, gather the SiteRec, classify (a1, a2); leaves the decoded header
// {8 * first active lane, active, context_base & ~31 (lo), context_base (hi)} in shared memory for the
// lane-parallel phases
template <int MODE, bool TEL>
__device__ __forceinline__ TileEv classify(const Params& p, uint32_t raw_s, uint32_t dec_s, uint64_t tile,
                                           uint32_t lane) {
  TileEv ev;
  ev.site = 0;
  ev.active = 0;
  ev.cls = CLS_NONE;
  ev.kind = 7;
  ev.off = 0;
  ev.cnt = 0;
  ev.tokl = 0;
  ev.tokh = 0;
  ev.st = Sip32{0, 0, 0, 0, 0, 0, 0, 0};
  const uint64_t e = tile * kT + lane;
  const bool valid = lane < kT && e < p.n;
  if (lane < kT && !valid) sts_v4(dec_s + lane * 16, 0u, 0u, 0u, 0u);  // ragged tail: a harmless record
  if (valid) {
    const uint4 h = lds_v4(raw_s + lane * 16);
    ev.site = h.x;
    ev.active = h.y;
    sts_v4(dec_s + lane * 16, h.y ? static_cast<uint32_t>(__ffs(h.y) - 1) * 8u : 0u, h.y, h.z & ~31u, h.w);
    if (h.x < p.n_sites) {
      const uint4 a = ldg_v4(p.recs + h.x);
      ev.kind = a.x;
      ev.off = a.y;
      ev.cnt = a.z;
      if (TEL && a.x == K_FWD && (p.profile & PROFILE_METADATA_INTEGRITY)) {
        const uint2 d = __ldg(reinterpret_cast<const uint2*>(p.tok) + h.x);
        ev.tokl = d.x;
        ev.tokh = d.y;
      }
      if constexpr (MODE == MODE_SIGN) {
        ev.cls = (a.x == K_RET && h.y != 0) ? CLS_RET : CLS_COUNT;
      } else {
        if (h.y == 0)
          ev.cls = CLS_COUNT;  // fully predicated off: counted, not a check (R22)
        else if (TEL && ((a.x == K_RET && (p.profile & PROFILE_SKIP_BACKWARD)) ||
                         (a.x == K_FWD && (p.profile & PROFILE_SKIP_FORWARD))))
          ev.cls = CLS_SKIP;   // outside this profile's protected set: separate denominator (R26)
        else if (a.x == K_RET)
          ev.cls = (MODE == MODE_VERIFY) ? CLS_RET : CLS_FAIL;  // no tag at the forward entry point (R14)
        else if (a.x == K_FWD)
          ev.cls = CLS_FWD;
        else
          ev.cls = CLS_COUNT;  // non-protected kinds are only counted (R17)
      }
    } else {
      ev.cls = (MODE == MODE_SIGN) ? CLS_COUNT : CLS_FAIL;  // unknown site: fail closed (R13)
    }
  }
  return ev;
}

__device__ __forceinline__ Sip32 lds_state(uint32_t a) {
  const uint4 x = lds_v4(a), y = lds_v4(a + 16);
  return Sip32{x.x, x.y, x.z, x.w, y.x, y.y, y.z, y.w};
}

// ---------------------------------------------------------------------------------------------------
// the tile kernel: MODE_VERIFY = wg_verify_continuations, MODE_FORWARD = wg_check_forward, MODE_SIGN =
// wg_sign_continuations.  STAGED: the whole target table sits in shared memory.
// ---------------------------------------------------------------------------------------------------
// TEL: a profile flag is set or the violation ring is on (compiled out of the ordinary launch).
// SPARSE: the lane-parallel MAC passes run over a compacted list of ACTIVE (event, lane) items instead of one pass
// per event — for streams whose active masks are far from full (config 5: 1-32 lanes, half of a pass would idle).
template <int MODE, bool STAGED, bool TEL, bool SPARSE>
__global__ void __launch_bounds__(Cfg<MODE>::kThreads, 1) wg_tile_kernel(const Params p, const uint32_t stage_bytes,
                                                                                const uint32_t site_bytes) {
  using L = WarpLayout<MODE>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t lanebit = 1u << lane;
  // the shuffle tells the compiler that the warp index (and what derives from it) is warp-uniform
  const uint32_t warp = __shfl_sync(kFull, threadIdx.x >> 5, 0);
  const uint32_t smem0 = smem_u32(smem_raw);
  const uint32_t tg_s = smem0;
  // small policies (site_bytes != 0): per-site counters are accumulated in shared memory as 4 x u32 per site and
  // flushed once per CTA.  With few sites the global counter array spans only a few L2 slices and the reductions
  // of 148 SMs would queue on them (config 3: 40 sites, 7.6 ms -> see DESIGN.md §9).
  uint32_t* site_s = reinterpret_cast<uint32_t*>(smem_raw + stage_bytes);
  const uint32_t cta_off = stage_bytes + site_bytes;
  unsigned long long* cnt64 = reinterpret_cast<unsigned long long*>(smem_raw + cta_off);
  uint32_t* bykind = reinterpret_cast<uint32_t*>(smem_raw + cta_off + 256);
  const uint32_t mbar_cta = smem0 + cta_off + 256 + 32;
  const uint32_t warp_s = smem0 + cta_off + kCtaFixedBytes + warp * L::kBytes;
  const uint32_t dec_s = warp_s + L::kDec;
  const uint32_t st_s = warp_s + L::kSt;
  const uint32_t mbar = warp_s + L::kBar;
  const uint32_t viol_s = warp_s + L::kViol;
  const uint32_t list_s = warp_s + L::kList;
  const uint32_t val_s = warp_s + L::kVal;
  const uint32_t tag_s = warp_s + L::kTag;
  const uint32_t val_lane_s = val_s + lane * 8, tag_lane_s = tag_s + lane * 8;  // this lane's column of the rows

  if (threadIdx.x < 32) cnt64[threadIdx.x] = 0ull;
  for (uint32_t i = threadIdx.x; i < site_bytes / 4; i += blockDim.x) site_s[i] = 0u;
  if (threadIdx.x < 8) bykind[threadIdx.x] = 0u;
  if (threadIdx.x == 0) mbar_init(mbar_cta, 1);
  if (lane == 0) mbar_init(mbar, 1);
  __syncthreads();
  if constexpr (STAGED) {
    if (threadIdx.x == 0) {
      mbar_expect_tx(mbar_cta, stage_bytes);
      tma_bulk_g2s(tg_s, p.tgts, stage_bytes, mbar_cta);
    }
    mbar_wait(mbar_cta, 0);
  }

  const uint64_t n_tiles = (p.n + kT - 1) / kT;
  constexpr int kWarps = Cfg<MODE>::kWarps;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * kWarps;
  uint64_t t = static_cast<uint64_t>(blockIdx.x) * kWarps + warp;
  const bool enforce = p.mode != 0;
  WarpCtr c = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  uint32_t phase = 0, rb = 0;  // mbarrier phase parity; which raw-header buffer holds this tile

  // prologue: raw headers of the first tile
  if (t < n_tiles) {
    if (lane == 0) {
      const uint64_t left = p.n - t * kT;
      const uint32_t bytes = static_cast<uint32_t>(left < kT ? left : kT) * 16u;
      mbar_expect_tx(mbar, bytes);
      tma_bulk_g2s(warp_s + L::kRaw, p.hdr + t * kT, bytes, mbar);
    }
    mbar_wait(mbar, phase);
    phase ^= 1u;
  }

  while (t < n_tiles) {
    const uint64_t tn = t + stride;
    const uint64_t e0 = t * kT;
    uint64_t* const tag_out_lane = (MODE == MODE_SIGN) ? p.tag_out + (e0 * 32 + lane) : nullptr;  // this lane's column
    // ---- event-parallel: decode, gather, classify (a1, a2) ----
    TileEv ev = classify<MODE, TEL>(p, warp_s + L::kRaw + rb * kT * 16, dec_s, t, lane);
    const uint32_t m_ret = __ballot_sync(kFull, ev.cls == CLS_RET);
    if (MODE != MODE_FORWARD && m_ret != 0u) {
      // the site word of the MAC, once per event: the key-derived initial state exists in the kernel parameters only
      // (constant bank), never in global memory; leaves the "pre-A" state the tails start from
      ev.st = Sip32{static_cast<uint32_t>(p.v0), static_cast<uint32_t>(p.v0 >> 32), static_cast<uint32_t>(p.v1),
                    static_cast<uint32_t>(p.v1 >> 32), static_cast<uint32_t>(p.v2), static_cast<uint32_t>(p.v2 >> 32),
                    static_cast<uint32_t>(p.v3), static_cast<uint32_t>(p.v3 >> 32)};
      sip_absorb(ev.st, ev.site, p.bind_hi);  // LE64(site_id | digest32 << 32): zero-extended site id unless bound (R3, R5, R39)
      sip_qA(ev.st);
    }
    const uint32_t m_fwd = __ballot_sync(kFull, ev.cls == CLS_FWD);

    // ---- rows of this tile and raw headers of the next: TMA bulk copies onto the warp's mbarrier ----
    {
      uint32_t hdr_bytes = 0;
      if (tn < n_tiles) {
        const uint64_t left = p.n - tn * kT;
        hdr_bytes = static_cast<uint32_t>(left < kT ? left : kT) * 16u;
      }
      const uint32_t rows = __popc(m_ret | m_fwd) + (MODE == MODE_VERIFY ? __popc(m_ret) : 0);
      if (lane == 0) mbar_expect_tx(mbar, rows * 256u + hdr_bytes);
      __syncwarp();
      // one bulk copy per RUN of consecutive needed rows (a bulk copy is issued by one elected lane at a time, so
      // fewer, longer copies cost fewer issue slots): the first lane of a run copies the whole run
      {
        const uint32_t need = m_ret | m_fwd;
        const uint32_t here = need >> lane;
        if ((here & 1u) && (lane == 0u || !((need >> (lane - 1u)) & 1u))) {
          const uint32_t len = static_cast<uint32_t>(__ffs(~here)) - 1u;
          tma_bulk_g2s(val_s + lane * 256, p.val + (e0 + lane) * 32, len * 256u, mbar);
        }
        if constexpr (MODE == MODE_VERIFY) {
          const uint32_t here_t = m_ret >> lane;
          if ((here_t & 1u) && (lane == 0u || !((m_ret >> (lane - 1u)) & 1u))) {
            const uint32_t len = static_cast<uint32_t>(__ffs(~here_t)) - 1u;
            tma_bulk_g2s(tag_s + lane * 256, p.tag + (e0 + lane) * 32, len * 256u, mbar);
          }
        }
      }
      if (lane == 0 && hdr_bytes) {
        tma_bulk_g2s(warp_s + L::kRaw + (rb ^ 1u) * kT * 16, p.hdr + tn * kT, hdr_bytes, mbar);
        // a tile without return events is HBM-bound work (280 B / event, a few instructions): pull the next
        // tile's value rows into L2 now, so that its row copies find them there (one more tile of bytes in flight)
        if (MODE != MODE_SIGN && m_ret == 0u) tma_prefetch_l2(p.val + tn * kT * 32, hdr_bytes * 16u);
      }
    }

    // ---- while the rows fly: everything of the epilogue that does not depend on a verdict (a7) ----
    const bool valid = ev.cls != CLS_NONE;
    const bool known = valid && ev.kind < 7u;
    const uint32_t na = __popc(ev.active);
    const uint32_t judged_na = (ev.cls == CLS_RET || ev.cls == CLS_FWD) ? na : 0u;
    unsigned long long* sc = p.site + static_cast<uint64_t>(ev.site) * 4;
    uint32_t tile_ret_lanes = 0;  // active lanes over the tile's return events
    if constexpr (MODE == MODE_SIGN) {
      const bool is_ret = known && ev.kind == K_RET;
      tile_ret_lanes = __reduce_add_sync(kFull, is_ret ? na : 0u);
      c.signed_lanes += tile_ret_lanes;
      c.skipped += __popc(__ballot_sync(kFull, valid && !is_ret));
    } else {
      c.total += __popc(__ballot_sync(kFull, valid));
      if (__ballot_sync(kFull, valid && (!known || ev.active == 0u || ev.cls == CLS_FAIL))) {  // uncommon events
        c.unknown += __popc(__ballot_sync(kFull, valid && !known));
        c.empty += __popc(__ballot_sync(kFull, known && ev.active == 0u));
        c.misrouted += __popc(__ballot_sync(kFull, known && ev.cls == CLS_FAIL));
      }
      c.ret_checks += __popc(m_ret);
      c.fwd_checks += __popc(m_fwd);
      tile_ret_lanes = __reduce_add_sync(kFull, ev.cls == CLS_RET ? na : 0u);
      c.ret_lanes += tile_ret_lanes;
      c.fwd_lanes += __reduce_add_sync(kFull, ev.cls == CLS_FWD ? na : 0u);
      if (known) atomicAdd(&bykind[ev.kind], 1u);
      if (TEL && (p.profile & (PROFILE_SKIP_FORWARD | PROFILE_SKIP_BACKWARD))) {
        const uint32_t sr = __ballot_sync(kFull, ev.cls == CLS_SKIP && ev.kind == K_RET);
        const uint32_t sf = __ballot_sync(kFull, ev.cls == CLS_SKIP && ev.kind == K_FWD);
        const uint32_t srl = __reduce_add_sync(kFull, (ev.cls == CLS_SKIP && ev.kind == K_RET) ? na : 0u);
        const uint32_t sfl = __reduce_add_sync(kFull, (ev.cls == CLS_SKIP && ev.kind == K_FWD) ? na : 0u);
        if (lane == 0) {
          if (sr) atomicAdd(cnt64 + C_SKIP_RET_EVENTS, static_cast<unsigned long long>(__popc(sr)));
          if (srl) atomicAdd(cnt64 + C_SKIP_RET_LANES, static_cast<unsigned long long>(srl));
          if (sf) atomicAdd(cnt64 + C_SKIP_FWD_EVENTS, static_cast<unsigned long long>(__popc(sf)));
          if (sfl) atomicAdd(cnt64 + C_SKIP_FWD_LANES, static_cast<unsigned long long>(sfl));
        }
      }
      if (TEL && (p.profile & PROFILE_LOW_TELEMETRY)) {
        // "same checked transfers with less reporting" (PAPER.md Table A2): no per-site counters
      } else if (site_bytes) {
        // per-site counters in shared memory (small policies)
        if (known) {
          atomicAdd(&site_s[ev.site * 4 + S_EVENTS], 1u);
          if (judged_na) atomicAdd(&site_s[ev.site * 4 + S_LANES_CHECKED], judged_na);
        }
      } else {
        // per-site counters in global memory, one reduction per event straight to L2: measured faster than merging equal sites of the tile first
        // (__match_any_sync + shuffles cost more ALU-pipe slots than the hot site's reductions cost in L2:
        // config 4 verify 14.90 -> 14.64 ms, config 2 1.457 -> 1.449 ms)
        if (known) {
          atomicAdd(sc + S_EVENTS, 1ull);
          if (judged_na) atomicAdd(sc + S_LANES_CHECKED, static_cast<unsigned long long>(judged_na));
        }
      }
    }

    mbar_wait(mbar, phase);  // rows (and the next raw headers) have landed
    phase ^= 1u;

    // ---- which events carry one warp-uniform value?  (a5 dedupe)  Unrolled over the tile:
    //      three independent shared-memory loads and ~6 ALU instructions per event, one REDUX per tile ----
    uint32_t uni = 0;
    if (MODE != MODE_SIGN || m_ret != 0u) {  // (a sign tile without return events has nothing to detect)
      uint32_t mism = 0;
#pragma unroll
      for (int e = 0; e < kT; ++e) {
        const uint2 d = lds_v2(dec_s + e * 16);  // {8 * first active lane, active}
        const uint2 v = lds_v2(val_s + e * 256 + lane * 8);
        const uint2 r = lds_v2(val_s + e * 256 + d.x);
        if ((((v.x ^ r.x) | (v.y ^ r.y)) != 0u) && (d.y & lanebit)) mism |= 1u << e;
      }
      uni = ~__reduce_or_sync(kFull, mism) & (m_ret | m_fwd);
    }

    // ---- event-parallel: per-event part of the MAC; batched search of warp-uniform forward targets ----
    uint32_t viol = 0;
    uint32_t m_bad_rec = 0;  // events whose forward record failed its authentication
    {
      const bool is_uni = (uni >> lane) & 1u;
      uint32_t ul = 0, uh = 0;
      if (is_uni) {
        const uint2 d = lds_v2(dec_s + lane * 16);
        const uint2 r = lds_v2(val_s + lane * 256 + d.x);  // the event's one value
        ul = r.x;
        uh = r.y;
      }
      if (ev.cls == CLS_RET) {
        Sip32 s = ev.st;  // pre-A state after the site word
        if (is_uni) {
          const uint4 d = lds_v4(dec_s + lane * 16);
          sip_absorb_preA(s, ul, uh);  // the continuation word, once per event
          sip_qA(s);                   // quarter A of the context word's first round
          s.v3l ^= d.z;                // and the lane-independent bits of the context word
          s.v3h ^= d.w;
        }
        sts_v4(st_s + lane * 32, s.v0l, s.v0h, s.v1l, s.v1h);
        sts_v4(st_s + lane * 32 + 16, s.v2l, s.v2h, s.v3l, s.v3h);
      }
      if constexpr (MODE != MODE_SIGN) {
        if constexpr (TEL) {
          // metadata integrity: the forward record is re-authenticated before it is used, once per
          // event; a record that fails authorises nothing: every active lane violates
          if (p.profile & PROFILE_METADATA_INTEGRITY) {
            bool bad_rec = false;
            if (ev.cls == CLS_FWD) {
              uint2 tk;
              if constexpr (STAGED) {
                const uint32_t base = tg_s + ev.off * 8;
                tk = record_token(p.v0, p.v1, p.v2, p.v3, ev.site, ev.cnt, [&](uint32_t i) { return lds_v2(base + i * 8); });
              } else {
                const uint2* set = reinterpret_cast<const uint2*>(p.tgts + ev.off);
                tk = record_token(p.v0, p.v1, p.v2, p.v3, ev.site, ev.cnt, [&](uint32_t i) { return __ldcg(set + i); });
              }
              bad_rec = tk.x != ev.tokl || tk.y != ev.tokh;
            }
            m_bad_rec = __ballot_sync(kFull, bad_rec);
            if (m_bad_rec && lane == 0)
              atomicAdd(p.glob + C_META_FAIL, static_cast<unsigned long long>(__popc(m_bad_rec)));
            if (bad_rec) viol = ev.active;
          }
        }
        if (ev.cls == CLS_FWD && is_uni && !((m_bad_rec >> lane) & 1u))
          viol = member<STAGED>(p, tg_s, ev.off, ev.cnt, ul, uh) ? 0u : ev.active;
        if (ev.cls == CLS_FAIL) viol = ev.active;  // fail closed (R13, R14)
        if (lane < kT) sts_u32(viol_s + lane * 4, viol);  // the lane-parallel loops below overwrite their events
      }
    }
    __syncwarp();

    // the sparse instantiation decides per tile: compaction pays when at least a quarter of the lanes of the
    // tile's return events are idle (the list costs ~8 instructions per event, a saved pass ~200)
    if (SPARSE && MODE != MODE_FORWARD && tile_ret_lanes * 4u <= 96u * static_cast<uint32_t>(__popc(m_ret))) {
      // ---- sparse path: work items = the ACTIVE lanes of the tile's return events, uniform events from the front
      //      of the list, divergent ones from the back; 32 items per pass whatever event they belong to ----
      uint32_t n_u = 0, n_d = 0;
      for (uint32_t m = m_ret; m; m &= m - 1) {
        const uint32_t e = __ffs(m) - 1;
        const uint32_t a = lds_u32(dec_s + e * 16 + 4);
        const bool is_u = (uni >> e) & 1u;
        const uint32_t pos = __popc(a & (lanebit - 1u));
        if (a & lanebit) {
          sts_u16(list_s + 2u * (is_u ? n_u + pos : (kT * 32u - 1u) - (n_d + pos)), e * 32u + lane);
        } else if (MODE == MODE_SIGN) {
          st_stream_v2(p.tag_out + ((e0 + e) * 32 + lane), 0u, 0u);  // inactive lanes sign nothing (R10)
        }
        const uint32_t na_e = __popc(a);
        if (is_u) n_u += na_e; else n_d += na_e;
      }
      __syncwarp();
      for (uint32_t k0 = 0; k0 < n_u; k0 += 32) {
        const bool on = k0 + lane < n_u;
        const uint32_t item = lds_u16(list_s + 2u * (on ? k0 + lane : 0u));
        const uint32_t e = item >> 5, l = item & 31u;
        const uint4 h = lds_v4(dec_s + e * 16);
        const Sip32 st = lds_state(st_s + e * 32);
        uint32_t dl, dh;
        if constexpr (MODE == MODE_SIGN) {
          sip_tail_lane(st, l, h.z, h.w, 0u, 0u, dl, dh);
          if (on) st_stream_v2(p.tag_out + (e0 * 32 + item), dl, dh);
        } else {
          const uint2 tg = lds_v2(tag_s + item * 8);
          sip_tail_lane(st, l, h.z, h.w, tg.x, tg.y, dl, dh);
          if (on && (dl | dh) != 0u) atoms_or(viol_s + e * 4, 1u << l);
        }
      }
      for (uint32_t k0 = 0; k0 < n_d; k0 += 32) {
        const bool on = k0 + lane < n_d;
        const uint32_t item = lds_u16(list_s + 2u * ((kT * 32u - 1u) - (on ? k0 + lane : 0u)));
        const uint32_t e = item >> 5, l = item & 31u;
        const uint4 h = lds_v4(dec_s + e * 16);
        const Sip32 st = lds_state(st_s + e * 32);
        const uint2 v = lds_v2(val_s + item * 8);
        uint32_t dl, dh;
        if constexpr (MODE == MODE_SIGN) {
          sip_tail_val_lane(st, v.x, v.y, l, h.z, h.w, 0u, 0u, dl, dh);
          if (on) st_stream_v2(p.tag_out + (e0 * 32 + item), dl, dh);
        } else {
          const uint2 tg = lds_v2(tag_s + item * 8);
          sip_tail_val_lane(st, v.x, v.y, l, h.z, h.w, tg.x, tg.y, dl, dh);
          if (on && (dl | dh) != 0u) atoms_or(viol_s + e * 4, 1u << l);
        }
      }
    } else {
    // ---- lane-parallel: protected-return events with a warp-uniform continuation (8 rounds per lane) ----
    for (uint32_t m = m_ret & uni; m; m &= m - 1) {
      const uint32_t e = __ffs(m) - 1;
      const uint4 h = lds_v4(mad32(e, 16u, dec_s));
      const Sip32 s = lds_state(mad32(e, 32u, st_s));
      uint32_t dl, dh;
      if constexpr (MODE == MODE_SIGN) {
        sip_tail_lane(s, lane, h.z, h.w, 0u, 0u, dl, dh);
        st_tag_or_zero(tag_out_lane + e * 32, h.y & lanebit, dl, dh);
      } else {
        const uint2 tg = lds_v2(mad32(e, 256u, tag_lane_s));
        sip_tail_lane(s, lane, h.z, h.w, tg.x, tg.y, dl, dh);
        // inactive lanes computed on garbage: masked out after the vote (R10)
        const uint32_t vb = __ballot_sync(kFull, (dl | dh) != 0u) & h.y;
        if (lane == 0) sts_u32(mad32(e, 4u, viol_s), vb);
      }
    }
    // ---- lane-parallel: protected-return events with lane-divergent continuations (10 rounds per lane) ----
    for (uint32_t m = m_ret & ~uni; m; m &= m - 1) {
      const uint32_t e = __ffs(m) - 1;
      const uint4 h = lds_v4(mad32(e, 16u, dec_s));
      const Sip32 s = lds_state(mad32(e, 32u, st_s));
      const uint2 v = lds_v2(mad32(e, 256u, val_lane_s));
      uint32_t dl, dh;
      if constexpr (MODE == MODE_SIGN) {
        sip_tail_val_lane(s, v.x, v.y, lane, h.z, h.w, 0u, 0u, dl, dh);
        st_tag_or_zero(tag_out_lane + e * 32, h.y & lanebit, dl, dh);
      } else {
        const uint2 tg = lds_v2(mad32(e, 256u, tag_lane_s));
        sip_tail_val_lane(s, v.x, v.y, lane, h.z, h.w, tg.x, tg.y, dl, dh);
        const uint32_t vb = __ballot_sync(kFull, (dl | dh) != 0u) & h.y;
        if (lane == 0) sts_u32(mad32(e, 4u, viol_s), vb);
      }
    }
    }  // dense path
    // ---- lane-parallel: protected-forward events with lane-divergent targets ----
    if constexpr (MODE != MODE_SIGN) {
      for (uint32_t m = m_fwd & ~uni & ~m_bad_rec; m; m &= m - 1) {
        const uint32_t e = __ffs(m) - 1;
        const uint32_t a = lds_u32(dec_s + e * 16 + 4);
        const uint32_t off = __shfl_sync(kFull, ev.off, e), cnt = __shfl_sync(kFull, ev.cnt, e);
        const uint2 v = lds_v2(val_s + e * 256 + lane * 8);
        const bool bad = (a & lanebit) && !member<STAGED>(p, tg_s, off, cnt, v.x, v.y);
        const uint32_t vb = __ballot_sync(kFull, bad);
        if (lane == 0) sts_u32(viol_s + e * 4, vb);
      }
      __syncwarp();
      if (lane < kT) viol = lds_u32(viol_s + lane * 4);  // event-parallel again: lane i <-> event i
    }

    // ---- event-parallel epilogue: verdicts (a6), violation counters (a7), first violation (a8) ----
    if constexpr (MODE == MODE_SIGN) {
      // every row the loops above did not write is a zero row (R10): non-return sites, empty masks
      // written as 16-byte stores: a half-warp covers one 256-byte row, one instruction covers two events
      const uint32_t zmask = __ballot_sync(kFull, valid && ev.cls != CLS_RET);
      if (zmask) {
        const uint32_t half = lane >> 4, chunk = lane & 15u;
#pragma unroll
        for (int j = 0; j < kT / 2; ++j) {
          const uint32_t e = 2u * j + half;
          if ((zmask >> e) & 1u) st_stream_v4(p.tag_out + ((e0 + e) * 32 + chunk * 2), 0u, 0u, 0u, 0u);
        }
      }
    } else {
      if (valid) st_stream_v2(p.out + (e0 + lane), viol, enforce ? (ev.active & ~viol) : ev.active);
      // violations are rare (0.05 % of events in the paper-shaped stream): one warp-uniform branch per tile
      if (__ballot_sync(kFull, viol != 0u)) {
        const uint32_t pv = __popc(viol);
        const uint32_t rv = __reduce_add_sync(kFull, ev.cls == CLS_RET ? pv : 0u);
        const uint32_t fv = __reduce_add_sync(kFull, ev.cls == CLS_FWD ? pv : 0u);
        const uint32_t av = __reduce_add_sync(kFull, pv);
        const uint32_t rve = __popc(__ballot_sync(kFull, ev.cls == CLS_RET && viol != 0u));
        const uint32_t fve = __popc(__ballot_sync(kFull, ev.cls == CLS_FWD && viol != 0u));
        const uint32_t ave = __popc(__ballot_sync(kFull, viol != 0u));
        // first violation: smallest (seq << 5 | lane); seq = running event index (R12)
        unsigned long long key = ~0ull;
        if (viol) key = ((p.seq_base + e0 + lane) << 5) | static_cast<uint32_t>(__ffs(viol) - 1);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
          const unsigned long long o = __shfl_xor_sync(kFull, key, d);
          key = o < key ? o : key;
        }
        if (lane == 0) {
          if (rv) atomicAdd(p.glob + C_RET_VIOL, static_cast<unsigned long long>(rv));
          if (fv) atomicAdd(p.glob + C_FWD_VIOL, static_cast<unsigned long long>(fv));
          if (rve) atomicAdd(p.glob + C_RET_VIOL_EVENTS, static_cast<unsigned long long>(rve));
          if (fve) atomicAdd(p.glob + C_FWD_VIOL_EVENTS, static_cast<unsigned long long>(fve));
          if (enforce) {
            atomicAdd(p.glob + C_BLOCKED_LANES, static_cast<unsigned long long>(av));
            atomicAdd(p.glob + C_BLOCKED_EVENTS, static_cast<unsigned long long>(ave));
          }
          atomicMin(p.glob + C_FIRST_VIOLATION, key);
        }
        if (TEL && viol && !(p.profile & PROFILE_LOW_TELEMETRY) && p.ring_cap != 0) {
          // violation ring (R27, R28): diagnostic, bounded; a full ring drops and counts
          const unsigned long long slot = atomicAdd(p.glob + C_RING_TOTAL, 1ull);
          if (slot < p.ring_cap) {
            const uint32_t fl = static_cast<uint32_t>(__ffs(viol) - 1);
            ViolRec r;
            r.seq = p.seq_base + e0 + lane;
            r.site_id = ev.site;
            r.kind = ev.kind;
            r.viol_mask = viol;
            r.active_mask = ev.active;
            r.lane = fl;
            r.mode = p.mode;
            r.observed = p.val[(e0 + lane) * 32 + fl];
            r.stored = (MODE == MODE_VERIFY && ev.cls == CLS_RET) ? p.tag[(e0 + lane) * 32 + fl] : 0ull;
            p.ring[slot] = r;
          }
        }
        if (viol && known && !(TEL && (p.profile & PROFILE_LOW_TELEMETRY))) {
          if (site_bytes) {
            if (judged_na) atomicAdd(&site_s[ev.site * 4 + S_LANES_VIOLATION], pv);
            if (enforce) atomicAdd(&site_s[ev.site * 4 + S_LANES_BLOCKED], pv);
          } else {
            if (judged_na) atomicAdd(sc + S_LANES_VIOLATION, static_cast<unsigned long long>(pv));
            if (enforce) atomicAdd(sc + S_LANES_BLOCKED, static_cast<unsigned long long>(pv));
          }
        }
      }
    }
    __syncwarp();  // every lane is done with this tile's shared memory before the next tile's copies land
    t = tn;
    rb ^= 1u;
  }

  // ---- flush: warp registers -> CTA shared memory -> one global atomic per counter per CTA ----
  if (lane == 0) {
    if constexpr (MODE == MODE_SIGN) {
      if (c.signed_lanes) atomicAdd(cnt64 + C_SIGNED_LANES, static_cast<unsigned long long>(c.signed_lanes));
      if (c.skipped) atomicAdd(cnt64 + C_SIGN_SKIPPED, static_cast<unsigned long long>(c.skipped));
    } else {
      if (c.total) atomicAdd(cnt64 + C_EVENTS_TOTAL, static_cast<unsigned long long>(c.total));
      if (c.empty) atomicAdd(cnt64 + C_EVENTS_EMPTY, static_cast<unsigned long long>(c.empty));
      if (c.unknown) atomicAdd(cnt64 + C_EVENTS_UNKNOWN, static_cast<unsigned long long>(c.unknown));
      if (c.misrouted) atomicAdd(cnt64 + C_EVENTS_MISROUTED, static_cast<unsigned long long>(c.misrouted));
      if (c.ret_checks) atomicAdd(cnt64 + C_RET_CHECKS, static_cast<unsigned long long>(c.ret_checks));
      if (c.fwd_checks) atomicAdd(cnt64 + C_FWD_CHECKS, static_cast<unsigned long long>(c.fwd_checks));
      if (c.ret_lanes) atomicAdd(cnt64 + C_RET_LANES, static_cast<unsigned long long>(c.ret_lanes));
      if (c.fwd_lanes) atomicAdd(cnt64 + C_FWD_LANES, static_cast<unsigned long long>(c.fwd_lanes));
    }
  }
  __syncthreads();
  if (threadIdx.x < C_RING_TOTAL) {  // words 24, 25 (digest, last mode) are host-side: their slots stay 0 here
    unsigned long long v = cnt64[threadIdx.x];
    if (threadIdx.x >= C_BY_KIND && threadIdx.x < C_BY_KIND + 7) v = bykind[threadIdx.x - C_BY_KIND];
    if (v) atomicAdd(p.glob + threadIdx.x, v);
  }
  for (uint32_t i = threadIdx.x; i < site_bytes / 4; i += blockDim.x) {
    const uint32_t v = site_s[i];
    if (v) atomicAdd(p.site + i, static_cast<unsigned long long>(v));
  }
}

// first-violation record (R29), one thread, enqueued behind every check launch: the launch is over, so
// the key is final for it; if the key moved into that launch's event range the full record of that event is written.
// Deterministic, and nothing on the hot path: violations only did the atomicMin they always did.  (An earlier version
// let the last CTA of the tile kernel do this behind a ticket counter; it cost config 3 five per cent.)
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
  const bool judged_ret = has_tag && r.kind == K_RET && !(p.profile & PROFILE_SKIP_BACKWARD);
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
    const uint2 tk = record_token(v0, v1, v2, v3, s, r.cnt, [&](uint32_t i) { return set[i]; });
    t = (static_cast<uint64_t>(tk.y) << 32) | tk.x;
  }
  tok[s] = t;
}

template <int MODE>
uint32_t smem_bytes(uint32_t stage_bytes) {  // stage_bytes: staged targets + shared-memory site counters
  return stage_bytes + kCtaFixedBytes + Cfg<MODE>::kWarps * WarpLayout<MODE>::kBytes;
}

template <int MODE>
cudaError_t launch_tile(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches) {
  const uint64_t n_tiles = (p.n + kT - 1) / kT;
  constexpr int kWarps = Cfg<MODE>::kWarps;
  constexpr int kThreads = Cfg<MODE>::kThreads;
  const uint64_t want = (n_tiles + kWarps - 1) / kWarps;
  const int grid = static_cast<int>(want < static_cast<uint64_t>(sm_count) ? want : sm_count);
  const bool staged = MODE != MODE_SIGN && p.n_tgts > 0 && p.n_tgts <= Cfg<MODE>::kMaxStageTgts;
  const uint32_t stage_bytes = staged ? static_cast<uint32_t>((p.n_tgts * 8 + 15) & ~15ull) : 0u;
  // per-site counters in shared memory when the policy is small and they fit beside the staged targets
  uint32_t site_bytes = 0;
  if (MODE != MODE_SIGN && p.n_sites > 0 && p.n_sites <= kMaxSmemSites &&
      stage_bytes + p.n_sites * 16u <= Cfg<MODE>::kLeft)
    site_bytes = p.n_sites * 16u;
  const uint32_t smem = smem_bytes<MODE>(stage_bytes + site_bytes);
  const bool tel = MODE != MODE_SIGN && (p.profile != 0 || p.ring_cap != 0);
  if (tel) {
    if constexpr (MODE != MODE_SIGN) {
      if (staged)
        wg_tile_kernel<MODE, true, true, false><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
      else
        wg_tile_kernel<MODE, false, true, false><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
    }
  } else if (MODE != MODE_FORWARD && p.sparse) {
    if constexpr (MODE != MODE_FORWARD) {
      if (staged)
        wg_tile_kernel<MODE, true, false, true><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
      else
        wg_tile_kernel<MODE, false, false, true><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
    }
  } else if (staged) {
    wg_tile_kernel<MODE, true, false, false><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
  } else {
    wg_tile_kernel<MODE, false, false, false><<<grid, kThreads, smem, st>>>(p, stage_bytes, site_bytes);
  }
  ++*launches;
  return cudaGetLastError();
}

template <int MODE, bool STAGED>
cudaError_t opt_in() {
  if constexpr (MODE != MODE_SIGN) {
    const cudaError_t e = cudaFuncSetAttribute(wg_tile_kernel<MODE, STAGED, true, false>,
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(kSmemMax));
    if (e != cudaSuccess) return e;
  }
  if constexpr (MODE != MODE_FORWARD) {
    const cudaError_t e = cudaFuncSetAttribute(wg_tile_kernel<MODE, STAGED, false, true>,
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(kSmemMax));
    if (e != cudaSuccess) return e;
  }
  return cudaFuncSetAttribute(wg_tile_kernel<MODE, STAGED, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
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
  return launch_tile<MODE_SIGN>(p, sm_count, st, launches);
}

cudaError_t launch_check(const Params& p, int sm_count, cudaStream_t st, uint64_t* launches) {
  return p.tag ? launch_tile<MODE_VERIFY>(p, sm_count, st, launches) : launch_tile<MODE_FORWARD>(p, sm_count, st, launches);
}

cudaError_t launch_first_record(const Params& p, cudaStream_t st, uint64_t* launches) {
  wg_first_record<<<1, 1, 0, st>>>(p, p.tag != nullptr);
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
