// wg_kernels_v2.cu — the check path on sm_100a, second mapping: a warp owns a TILE of T consecutive events.
//
// Steps: a1 event fetch + guard, a2 policy lookup, a3 MAC sign, a4 MAC verify + compare,
// a5 forward membership, a6 verdicts, a7 counters, a8 first-violation record.  Paper passages: backward token
// PAPER.md:162, 248; forward membership PAPER.md:174-178, 250-252; guards PAPER.md:190, 230; detect / enforce
// PAPER.md:264; accounting PAPER.md:113, 127, 224.  Readings: DESIGN.md §2.  Kernel design: DESIGN.md §6.
//
// Per tile the warp runs two kinds of phases:
//   "event-parallel" (lane i <-> event i of the tile): header decode, policy gather (one 64-byte SiteRec),
//       classification, the part of the MAC that is the same for every lane of an event — the per-site
//       mid-state comes from the SiteRec, and when the event's continuation is warp-uniform the continuation
//       word is absorbed here too, ONCE per event instead of once per lane — the membership search of
//       warp-uniform forward targets (each unique target is searched once per warp), verdict / counter epilogue;
//   "lane-parallel" (lane l <-> lane l of one event): the per-lane tail of the MAC (8 of the 12 SipRounds for
//       a warp-uniform continuation, 10 otherwise) and the compare; per-lane searches of lane-divergent targets.
// Event rows reach shared memory by cp.async (16-byte chunks, only the rows a tile needs), double-buffered:
// the rows of tile k+1 are in flight while tile k is computed.  When the policy's whole target table is small
// (<= kMaxStageTgts entries) every CTA stages it in shared memory once with one TMA bulk copy.
// Counters: warp-uniform registers + shared-memory atomics, flushed once per CTA; per-site counters are
// aggregated over equal sites of a tile (__match_any_sync) before the global reduction.
#include "wg_internal.h"
#include "wg_sip32.cuh"

namespace wg {

namespace {

enum : int { MODE_VERIFY = 0, MODE_FORWARD = 1, MODE_SIGN = 2 };
enum : uint32_t { K_RET = 0, K_FWD = 1 };
// what the tile does with an event
enum : uint32_t { CLS_NONE = 0, CLS_COUNT = 1, CLS_RET = 2, CLS_FWD = 3, CLS_FAIL = 4 };

constexpr int kT = 16;                 // events per tile
constexpr int kWarps = 12;             // warps per CTA, one CTA per SM
constexpr int kThreads = kWarps * 32;
constexpr uint32_t kMaxStageTgts = 2048;  // 16 KB of shared memory for the target table
constexpr uint32_t kFull = 0xffffffffu;

// ---- shared-memory carve-up ----------------------------------------------------------------------
// CTA part: [tgts staged: stage_bytes][cnt64: 32 x u64][bykind: 8 x u32][mbar: u64, pad]
// warp part: hdr[3][T] uint4, st[T][8] u32, val[2][T][32] u64, (verify only) tag[2][T][32] u64
template <int MODE>
struct WarpLayout {
  static constexpr uint32_t kHdr = 0;
  static constexpr uint32_t kSt = kHdr + 3 * kT * 16;
  static constexpr uint32_t kVal = kSt + kT * 32;
  static constexpr uint32_t kTag = kVal + 2 * kT * 256;
  static constexpr uint32_t kBytes = kTag + (MODE == MODE_VERIFY ? 2 * kT * 256 : 0);
};
constexpr uint32_t kCtaFixedBytes = 32 * 8 + 8 * 4 + 16 + 16;  // cnt64, bykind, mbar (+pad to 16)

// ---- PTX helpers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ uint4 ldg_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
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
    while (len > 1) {
      const uint32_t half = len >> 1;
      const uint64_t mid = __ldg(set + lo + half);
      lo = (mid <= v) ? lo + half : lo;
      len -= half;
    }
    return __ldg(set + lo) == v;
  }
}

// what lane i knows about event i of a tile
struct TileEv {
  uint32_t site, active, cls, kind;
  uint32_t off, cnt;  // protected-forward: the site's set
  Sip32 st;           // protected-return: the site's pre-A mid-state
};

// warp-uniform running counters of one warp (flushed once at the end)
struct WarpCtr {
  uint32_t total, empty, unknown, misrouted, ret_checks, fwd_checks, ret_lanes, fwd_lanes, signed_lanes, skipped;
};

template <int MODE>
__device__ __forceinline__ void issue_hdr(const Params& p, uint32_t hdr_s, uint64_t tile, uint32_t buf,
                                          uint32_t lane) {
  const uint64_t e = tile * kT + lane;
  if (lane < kT && e < p.n) cp_async16(hdr_s + (buf * kT + lane) * 16, p.hdr + e);
}

// rows of the tile: one cp.async instruction moves 16 B per lane = two 256-byte rows per warp instruction
template <int MODE>
__device__ __forceinline__ void issue_rows(const Params& p, uint32_t warp_s, uint64_t tile, uint32_t buf,
                                           uint32_t need_val, uint32_t need_tag, uint32_t lane) {
  using L = WarpLayout<MODE>;
  const uint32_t half = lane >> 4, chunk = lane & 15;
  const uint64_t e0 = tile * kT;
#pragma unroll
  for (int j = 0; j < kT / 2; ++j) {
    const uint32_t e = 2 * j + half;
    const uint64_t g = (e0 + e) * 32 + chunk * 2;
    const uint32_t s = ((buf * kT + e) * 32 + chunk * 2) * 8;
    if ((need_val >> e) & 1u) cp_async16(warp_s + L::kVal + s, p.val + g);
    if constexpr (MODE == MODE_VERIFY) {
      if ((need_tag >> e) & 1u) cp_async16(warp_s + L::kTag + s, p.tag + g);
    }
  }
}

// event-parallel: decode header i, gather the SiteRec, classify (a1, a2)
template <int MODE>
__device__ __forceinline__ TileEv classify(const Params& p, uint32_t hdr_s, uint64_t tile, uint32_t buf,
                                           uint32_t lane) {
  TileEv ev;
  ev.site = 0;
  ev.active = 0;
  ev.cls = CLS_NONE;
  ev.kind = 7;
  ev.off = 0;
  ev.cnt = 0;
  ev.st = Sip32{0, 0, 0, 0, 0, 0, 0, 0};
  const uint64_t e = tile * kT + lane;
  if (lane < kT && e < p.n) {
    const uint4 h = lds_v4(hdr_s + (buf * kT + lane) * 16);
    ev.site = h.x;
    ev.active = h.y;
    if (h.x < p.n_sites) {
      const SiteRec* r = p.recs + h.x;
      const uint4 a = ldg_v4(r);
      ev.kind = a.x;
      ev.off = a.y;
      ev.cnt = a.z;
      if (a.x == K_RET && MODE != MODE_FORWARD) {
        const uint4 b = ldg_v4(reinterpret_cast<const char*>(r) + 16);
        const uint4 c = ldg_v4(reinterpret_cast<const char*>(r) + 32);
        ev.st = Sip32{b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
      }
      if constexpr (MODE == MODE_SIGN) {
        ev.cls = (a.x == K_RET && h.y != 0) ? CLS_RET : CLS_COUNT;
      } else {
        if (h.y == 0)
          ev.cls = CLS_COUNT;  // fully predicated off: counted, not a check (R22)
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
template <int MODE, bool STAGED>
__global__ void __launch_bounds__(kThreads, 1) wg_tile_kernel(const Params p, const uint32_t stage_bytes) {
  using L = WarpLayout<MODE>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t smem0 = smem_u32(smem_raw);
  const uint32_t tg_s = smem0;
  unsigned long long* cnt64 = reinterpret_cast<unsigned long long*>(smem_raw + stage_bytes);
  uint32_t* bykind = reinterpret_cast<uint32_t*>(smem_raw + stage_bytes + 256);
  const uint32_t mbar = smem0 + stage_bytes + 256 + 32;
  const uint32_t warp_s = smem0 + stage_bytes + kCtaFixedBytes + warp * L::kBytes;
  const uint32_t hdr_s = warp_s + L::kHdr;
  const uint32_t st_s = warp_s + L::kSt;

  if (threadIdx.x < 32) cnt64[threadIdx.x] = 0ull;
  if (threadIdx.x < 8) bykind[threadIdx.x] = 0u;
  if constexpr (STAGED) {
    if (threadIdx.x == 0) mbar_init(mbar, 1);
  }
  __syncthreads();
  if constexpr (STAGED) {
    if (threadIdx.x == 0) {
      mbar_expect_tx(mbar, stage_bytes);
      tma_bulk_g2s(tg_s, p.tgts, stage_bytes, mbar);
    }
    mbar_wait(mbar, 0);
  }

  const uint64_t n_tiles = (p.n + kT - 1) / kT;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * kWarps;
  uint64_t t = static_cast<uint64_t>(blockIdx.x) * kWarps + warp;
  const bool enforce = p.mode != 0;
  WarpCtr c = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};

  // ---- prologue: header of the first tile, its classification, its rows + the header of the second ----
  TileEv nx = classify<MODE>(p, hdr_s, n_tiles, 0, lane);  // an all-NONE tile (tile index past the end)
  uint32_t hb = 0, hb1 = 1, hb2 = 2, rb = 0;
  if (t < n_tiles) {
    issue_hdr<MODE>(p, hdr_s, t, hb, lane);
    cp_async_commit();
    cp_async_wait_all();
    __syncwarp();
    nx = classify<MODE>(p, hdr_s, t, hb, lane);
    const uint32_t nr = __ballot_sync(kFull, nx.cls == CLS_RET);
    const uint32_t nf = __ballot_sync(kFull, nx.cls == CLS_FWD);
    issue_rows<MODE>(p, warp_s, t, rb, nr | nf, nr, lane);
    if (t + stride < n_tiles) issue_hdr<MODE>(p, hdr_s, t + stride, hb1, lane);
    cp_async_commit();
  }

  while (t < n_tiles) {
    const TileEv ev = nx;
    const uint64_t tn = t + stride;
    cp_async_wait_all();  // rows of this tile and the header of the next have landed
    __syncwarp();
    const uint32_t m_ret = __ballot_sync(kFull, ev.cls == CLS_RET);
    const uint32_t m_fwd = __ballot_sync(kFull, ev.cls == CLS_FWD);
    const uint32_t hdr_t = hdr_s + hb * kT * 16;                 // this tile's headers
    const uint32_t val_t = warp_s + L::kVal + rb * kT * 256;     // this tile's value rows
    const uint32_t tag_t = warp_s + L::kTag + rb * kT * 256;     // this tile's tag rows (verify)

    // next tile: header decode + SiteRec gather now, so the gather latency hides behind the next phase
    if (tn < n_tiles) nx = classify<MODE>(p, hdr_s, tn, hb1, lane);

    // ---- which events carry one warp-uniform value?  (a5 dedupe) ----
    uint32_t uni = 0, ul = 0, uh = 0;
    for (uint32_t m = m_ret | m_fwd; m; m &= m - 1) {
      const uint32_t e = __ffs(m) - 1;
      const uint32_t a = lds_u32(hdr_t + e * 16 + 4);
      const uint2 v = lds_v2(val_t + e * 256 + lane * 8);
      const uint2 r = lds_v2(val_t + e * 256 + (__ffs(a) - 1) * 8);  // first active lane's value
      const bool same = ((v.x == r.x) && (v.y == r.y)) || !((a >> lane) & 1u);
      if (__all_sync(kFull, same)) {
        uni |= 1u << e;
        if (lane == e) {
          ul = r.x;
          uh = r.y;
        }
      }
    }

    // ---- rows of the next tile + header of the one after go in flight now ----
    if (tn < n_tiles) {
      const uint32_t nr = __ballot_sync(kFull, nx.cls == CLS_RET);
      const uint32_t nf = __ballot_sync(kFull, nx.cls == CLS_FWD);
      issue_rows<MODE>(p, warp_s, tn, rb ^ 1u, nr | nf, nr, lane);
      if (tn + stride < n_tiles) issue_hdr<MODE>(p, hdr_s, tn + stride, hb2, lane);
    }
    cp_async_commit();

    // ---- event-parallel: per-event part of the MAC; batched search of warp-uniform forward targets ----
    uint32_t viol = 0;
    if (ev.cls == CLS_RET) {
      Sip32 s = ev.st;  // pre-A state after the site word
      if ((uni >> lane) & 1u) {
        sip_absorb_preA(s, ul, uh);  // the continuation word, once per event
        sip_qA(s);                   // and quarter A of the context word's first round
      }
      sts_v4(st_s + lane * 32, s.v0l, s.v0h, s.v1l, s.v1h);
      sts_v4(st_s + lane * 32 + 16, s.v2l, s.v2h, s.v3l, s.v3h);
    }
    if constexpr (MODE != MODE_SIGN) {
      if (ev.cls == CLS_FWD && ((uni >> lane) & 1u))
        viol = member<STAGED>(p, tg_s, ev.off, ev.cnt, ul, uh) ? 0u : ev.active;
      if (ev.cls == CLS_FAIL) viol = ev.active;  // fail closed (R13, R14)
    }
    __syncwarp();

    // ---- lane-parallel: protected-return events with a warp-uniform continuation (8 rounds per lane) ----
    for (uint32_t m = m_ret & uni; m; m &= m - 1) {
      const uint32_t e = __ffs(m) - 1;
      const uint4 h = lds_v4(hdr_t + e * 16);
      const Sip32 s = lds_state(st_s + e * 32);
      const bool on = (h.y >> lane) & 1u;
      uint32_t dl, dh;
      if constexpr (MODE == MODE_SIGN) {
        sip_tail_ctx(s, (h.z & ~31u) | lane, h.w, 0u, 0u, dl, dh);
        st_stream_v2(p.tag_out + ((t * kT + e) * 32 + lane), on ? dl : 0u, on ? dh : 0u);
      } else {
        const uint2 tg = lds_v2(tag_t + e * 256 + lane * 8);
        sip_tail_ctx(s, (h.z & ~31u) | lane, h.w, tg.x, tg.y, dl, dh);
        const uint32_t vb = __ballot_sync(kFull, on && ((dl | dh) != 0u));
        if (lane == e) viol = vb;
      }
    }
    // ---- lane-parallel: protected-return events with lane-divergent continuations (10 rounds per lane) ----
    for (uint32_t m = m_ret & ~uni; m; m &= m - 1) {
      const uint32_t e = __ffs(m) - 1;
      const uint4 h = lds_v4(hdr_t + e * 16);
      const Sip32 s = lds_state(st_s + e * 32);
      const uint2 v = lds_v2(val_t + e * 256 + lane * 8);
      const bool on = (h.y >> lane) & 1u;
      uint32_t dl, dh;
      if constexpr (MODE == MODE_SIGN) {
        sip_tail_val_ctx(s, v.x, v.y, (h.z & ~31u) | lane, h.w, 0u, 0u, dl, dh);
        st_stream_v2(p.tag_out + ((t * kT + e) * 32 + lane), on ? dl : 0u, on ? dh : 0u);
      } else {
        const uint2 tg = lds_v2(tag_t + e * 256 + lane * 8);
        sip_tail_val_ctx(s, v.x, v.y, (h.z & ~31u) | lane, h.w, tg.x, tg.y, dl, dh);
        const uint32_t vb = __ballot_sync(kFull, on && ((dl | dh) != 0u));
        if (lane == e) viol = vb;
      }
    }
    // ---- lane-parallel: protected-forward events with lane-divergent targets ----
    if constexpr (MODE != MODE_SIGN) {
      for (uint32_t m = m_fwd & ~uni; m; m &= m - 1) {
        const uint32_t e = __ffs(m) - 1;
        const uint32_t a = lds_u32(hdr_t + e * 16 + 4);
        const uint32_t off = __shfl_sync(kFull, ev.off, e), cnt = __shfl_sync(kFull, ev.cnt, e);
        const uint2 v = lds_v2(val_t + e * 256 + lane * 8);
        const bool bad = ((a >> lane) & 1u) && !member<STAGED>(p, tg_s, off, cnt, v.x, v.y);
        const uint32_t vb = __ballot_sync(kFull, bad);
        if (lane == e) viol = vb;
      }
    }

    // ---- event-parallel epilogue: verdicts (a6), counters (a7), first violation (a8) ----
    const bool valid = ev.cls != CLS_NONE;
    const bool known = valid && ev.kind < 7u;
    const uint32_t na = __popc(ev.active);
    if constexpr (MODE == MODE_SIGN) {
      // every row the loops above did not write is a zero row (R10): non-return sites, empty masks
      for (uint32_t m = __ballot_sync(kFull, valid && ev.cls != CLS_RET); m; m &= m - 1) {
        const uint32_t e = __ffs(m) - 1;
        st_stream_v2(p.tag_out + ((t * kT + e) * 32 + lane), 0u, 0u);
      }
      const bool is_ret = known && ev.kind == K_RET;
      c.signed_lanes += __reduce_add_sync(kFull, is_ret ? na : 0u);
      c.skipped += __popc(__ballot_sync(kFull, valid && !is_ret));
    } else {
      if (valid) st_stream_v2(p.out + (t * kT + lane), viol, enforce ? (ev.active & ~viol) : ev.active);
      c.total += __popc(__ballot_sync(kFull, valid));
      c.unknown += __popc(__ballot_sync(kFull, valid && !known));
      c.empty += __popc(__ballot_sync(kFull, known && ev.active == 0u));
      c.misrouted += __popc(__ballot_sync(kFull, known && ev.cls == CLS_FAIL));
      c.ret_checks += __popc(m_ret);
      c.fwd_checks += __popc(m_fwd);
      const uint32_t judged_na = (ev.cls == CLS_RET || ev.cls == CLS_FWD) ? na : 0u;
      c.ret_lanes += __reduce_add_sync(kFull, ev.cls == CLS_RET ? na : 0u);
      c.fwd_lanes += __reduce_add_sync(kFull, ev.cls == CLS_FWD ? na : 0u);
      if (known) atomicAdd(&bykind[ev.kind], 1u);

      // per-site counters: equal sites of the tile are merged first (Zipf: the hottest site is ~1/6 of all events)
      const uint32_t m_known = __ballot_sync(kFull, known);
      uint32_t grp = 0;
      if (known) grp = __match_any_sync(m_known, ev.site);
      uint32_t sum = judged_na;
      for (uint32_t m = __ballot_sync(kFull, __popc(grp) > 1); m; m &= m - 1) {
        const uint32_t j = __ffs(m) - 1;
        const uint32_t x = __shfl_sync(kFull, judged_na, j);
        if (((grp >> j) & 1u) && j != lane) sum += x;
      }
      unsigned long long* sc = p.site + static_cast<uint64_t>(ev.site) * 4;
      if (known && lane == static_cast<uint32_t>(__ffs(grp) - 1)) {
        atomicAdd(sc + S_EVENTS, static_cast<unsigned long long>(__popc(grp)));
        if (sum) atomicAdd(sc + S_LANES_CHECKED, static_cast<unsigned long long>(sum));
      }

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
        if (viol) key = ((p.seq_base + t * kT + lane) << 5) | static_cast<uint32_t>(__ffs(viol) - 1);
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
        if (viol && known) {
          if (judged_na) atomicAdd(sc + S_LANES_VIOLATION, static_cast<unsigned long long>(pv));
          if (enforce) atomicAdd(sc + S_LANES_BLOCKED, static_cast<unsigned long long>(pv));
        }
      }
    }

    t = tn;
    rb ^= 1u;
    const uint32_t h0 = hb;
    hb = hb1;
    hb1 = hb2;
    hb2 = h0;
  }
  cp_async_wait_all();

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
  if (threadIdx.x < 24) {
    unsigned long long v = cnt64[threadIdx.x];
    if (threadIdx.x >= C_BY_KIND && threadIdx.x < C_BY_KIND + 7) v = bykind[threadIdx.x - C_BY_KIND];
    if (v) atomicAdd(p.glob + threadIdx.x, v);
  }
}

// SiteRec table from the v1 rows: the pre-A mid-state of every protected-return site (runs once per policy load)
__global__ void wg_build_recs(SiteRec* recs, const SiteRow* rows, uint32_t n_sites, uint64_t v0, uint64_t v1,
                              uint64_t v2, uint64_t v3) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_sites) return;
  const SiteRow r = rows[s];
  SiteRec o;
  o.kind = r.kind;
  o.off = r.off;
  o.cnt = r.cnt;
  o.pad0 = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) o.st[i] = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) o.pad1[i] = 0;
  if (r.kind == K_RET) {
    Sip32 st{static_cast<uint32_t>(v0), static_cast<uint32_t>(v0 >> 32), static_cast<uint32_t>(v1),
             static_cast<uint32_t>(v1 >> 32), static_cast<uint32_t>(v2), static_cast<uint32_t>(v2 >> 32),
             static_cast<uint32_t>(v3), static_cast<uint32_t>(v3 >> 32)};
    sip_absorb(st, s, 0u);  // LE64(zero-extended site_id) (R3, R5)
    sip_qA(st);             // quarter A of the continuation word's first round
    o.st[0] = st.v0l; o.st[1] = st.v0h; o.st[2] = st.v1l; o.st[3] = st.v1h;
    o.st[4] = st.v2l; o.st[5] = st.v2h; o.st[6] = st.v3l; o.st[7] = st.v3h;
  }
  recs[s] = o;
}

template <int MODE>
uint32_t smem_bytes(uint32_t stage_bytes) {
  return stage_bytes + kCtaFixedBytes + kWarps * WarpLayout<MODE>::kBytes;
}

template <int MODE>
cudaError_t launch_tile(const Params& p, int sm_count, cudaStream_t st) {
  const uint64_t n_tiles = (p.n + kT - 1) / kT;
  const uint64_t want = (n_tiles + kWarps - 1) / kWarps;
  const int grid = static_cast<int>(want < static_cast<uint64_t>(sm_count) ? want : sm_count);
  const bool staged = MODE != MODE_SIGN && p.n_tgts > 0 && p.n_tgts <= kMaxStageTgts;
  const uint32_t stage_bytes = staged ? static_cast<uint32_t>((p.n_tgts * 8 + 15) & ~15ull) : 0u;
  const uint32_t smem = smem_bytes<MODE>(stage_bytes);
  if (staged)
    wg_tile_kernel<MODE, true><<<grid, kThreads, smem, st>>>(p, stage_bytes);
  else
    wg_tile_kernel<MODE, false><<<grid, kThreads, smem, st>>>(p, stage_bytes);
  count_launch();
  return cudaGetLastError();
}

template <int MODE, bool STAGED>
cudaError_t opt_in() {
  return cudaFuncSetAttribute(wg_tile_kernel<MODE, STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              static_cast<int>(smem_bytes<MODE>(STAGED ? kMaxStageTgts * 8 : 0)));
}

}  // namespace

cudaError_t init_v2() {
  cudaError_t e;
  if ((e = opt_in<MODE_VERIFY, true>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_VERIFY, false>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_FORWARD, true>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_FORWARD, false>()) != cudaSuccess) return e;
  if ((e = opt_in<MODE_SIGN, false>()) != cudaSuccess) return e;
  return cudaSuccess;
}

cudaError_t launch_sign_v2(const Params& p, int sm_count, cudaStream_t st) {
  return launch_tile<MODE_SIGN>(p, sm_count, st);
}

cudaError_t launch_check_v2(const Params& p, int sm_count, cudaStream_t st) {
  return p.tag ? launch_tile<MODE_VERIFY>(p, sm_count, st) : launch_tile<MODE_FORWARD>(p, sm_count, st);
}

cudaError_t launch_build_recs(SiteRec* recs, const SiteRow* rows, uint32_t n_sites, uint64_t v0, uint64_t v1,
                              uint64_t v2, uint64_t v3, cudaStream_t st) {
  if (n_sites == 0) return cudaSuccess;
  wg_build_recs<<<(n_sites + 255) / 256, 256, 0, st>>>(recs, rows, n_sites, v0, v1, v2, v3);
  count_launch();
  return cudaGetLastError();
}

}  // namespace wg
