// wg_shadow.cu — the stateful backward mechanism around the MAC: one bounded shadow stack per CUDA thread slot
// (§4.4, 242-250 §5.5, 258 §5.6; readings R30-R36).
//
// "Each shadow entry stores expected_return, callsite_id, depth, and token for the current slot".
// thread slot = (warp_slot, lane); warp_slot = bits 36..5 and epoch = bits 63..48 of the event's context_base.
// Token of the entry at depth d:  MAC(key, callsite_id, expected_return, epoch<<48 | d<<37 | warp_slot<<5 | lane).
// The shadow memory is ordinary (attacker-writable) device memory — wg_shadow_poke is that write — so nothing
// read from it is trusted before the token verifies.
//
// Layout (structure of arrays, so that the 32 lanes of a warp touch 256 contiguous bytes per field):
//   depth_ctr[slot][32] u32;  entry[slot][d][32][4] u64 = {expected, token, callsite | depth << 32, 0}: one 32-byte
//   sector per thread slot and depth, written whole by its (active) lane.
// Mapping: a warp owns a tile of 32 events; header decode and classification run with lane i <-> event i, the per
// thread-slot part (depth counter, entry, MAC, compare) lane-parallel, one pass per event (each lane owns its own stack).
// A call is one lock-step step of DISTINCT warps: a counting pass marks warp slots that occur twice in the call
// and those events fail closed; the marks carry the call's stamp, so no clearing pass is needed.
#include "wg_internal.h"
#include "../../include/warpguard_sip32.cuh"

namespace wg {

namespace {

constexpr uint32_t kFull = 0xffffffffu;
enum : uint32_t { K_RET = 0 };

__device__ __forceinline__ uint32_t slot_of(uint32_t ctx_lo, uint32_t ctx_hi) {
  return (ctx_lo >> 5) | (ctx_hi << 27);  // bits 36..5 of context_base
}

// counting pass: {stamp << 32 | occurrences} per warp slot.  The max installs this call's stamp with a zero count
// over whatever an earlier call left (older stamps are smaller), the add counts; nothing has to be cleared afterwards.
__global__ void wg_shadow_mark(const uint4* __restrict__ hdr, uint64_t n, unsigned long long* uses, uint32_t n_slots,
                               uint32_t stamp) {
  uint64_t i = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * blockDim.x;
  for (; i < n; i += stride) {
    const uint4 h = hdr[i];
    const uint32_t slot = slot_of(h.z, h.w);
    if (slot < n_slots) {
      atomicMax(uses + slot, static_cast<unsigned long long>(stamp) << 32);
      atomicAdd(uses + slot, 1ull);
    }
  }
}

// full 12-round token from the key-derived initial state (entries whose callsite is not the event's site)
__device__ __forceinline__ void mac_full(const Params& p, uint32_t site, uint32_t vl, uint32_t vh, uint32_t cl,
                                         uint32_t ch, uint32_t& outl, uint32_t& outh) {
  Sip32 s{static_cast<uint32_t>(p.v0), static_cast<uint32_t>(p.v0 >> 32), static_cast<uint32_t>(p.v1),
          static_cast<uint32_t>(p.v1 >> 32), static_cast<uint32_t>(p.v2), static_cast<uint32_t>(p.v2 >> 32),
          static_cast<uint32_t>(p.v3), static_cast<uint32_t>(p.v3 >> 32)};
  sip_absorb(s, site, p.bind_hi);
  sip_absorb(s, vl, vh);
  sip_absorb(s, cl, ch);
  sip_finish(s, 0u, 0u, outl, outh);
}

enum ShWord {  // wg_shadow_counters
  SH_PUSH_EVENTS = 0, SH_PUSH_LANES, SH_CHECK_EVENTS, SH_CHECK_LANES, SH_EMPTY_EVENTS,
  SH_OVERFLOW, SH_UNDERFLOW, SH_DEPTH_MISMATCH, SH_TOKEN_MISMATCH, SH_TARGET_MISMATCH,
  SH_NON_RETURN, SH_SLOT_OVERFLOW, SH_SLOT_CONFLICT, SH_VIOL_LANES, SH_VIOL_EVENTS, SH_BLOCKED_LANES, SH_WORDS
};

struct StageE {
  uint32_t exl, exh, tkl, tkh, callsite, depth;
};

// ---------------------------------------------------------------------------------------------------
// Tile mapping: a warp owns 32 consecutive events.  What a warp-per-event kernel (the first version of this file, see
// git history) does once per EVENT with all 32 lanes doing the same thing — header decode, SiteRec gather, use count,
// the fail-closed classification, the event counters, the verdict store — is done here once per TILE with lane i <-> event i
// ("event-parallel", as in wg_kernels_v2.cu); only the part that really is per thread slot (depth counter, value,
// entry, MAC, compare) runs lane-parallel, one pass per ordinary event, fed from shared memory.  The per-lane loads
// of a pass are dependent round trips (depth counter -> entry), so they are issued two passes (counter, value) and
// one pass (entry) ahead; only those 9 registers rotate.
// ---------------------------------------------------------------------------------------------------
// Tile size / block size sweep on B200 (1 Mi warps, depth 4; push / check_ret ms per call): 8 x 256 threads 0.55 / 0.60,
// 16 x 128 0.55 / 0.58, 16 x 256 0.55 / 0.58, 32 x 128 0.58 / 0.58, 32 x 256 0.55 / 0.57, 32 x 512 0.54 / 0.55.
// Again on the final kernels (whole-sector entries, warp-uniform prefix): 16 x 512 0.474 / 0.526, 32 x 256 0.490 / 0.562,
// 32 x 384 0.480 / 0.537, 32 x 512 0.467 / 0.517 — 32 resident warps at 64 registers beat 24 at 71 - 73.
#ifndef WG_SH_THREADS
#define WG_SH_THREADS 512
#endif
#ifndef WG_SH_TILE
#define WG_SH_TILE 32
#endif
constexpr int kST = WG_SH_TILE;  // events per tile (<= 32: one lane per event in the event-parallel phase)
static_assert(kST == 8 || kST == 16 || kST == 32, "tile size");
constexpr int kTileThreads = WG_SH_THREADS;
constexpr int kTileWarps = kTileThreads / 32;
enum : uint32_t { ST_NONE = 0, ST_EMPTY, ST_NON_RETURN, ST_SLOT_OVERFLOW, ST_SLOT_CONFLICT, ST_NORMAL };

struct TileSmem {
  uint4 rec[kST];        // {active, slot, site, context hi without the depth: epoch<<16 | slot>>27}
  uint4 st[kST][2];      // the site's pre-A mid-state
  uint4 ust[kST][2];     // the state after the site word AND the value of the event's first active lane (+ quarter A)
  uint2 vf[kST];         // that value
};

__device__ __forceinline__ uint32_t sm_addr(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ uint4 lds4(uint32_t a) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a));
  return r;
}

__device__ __forceinline__ uint2 lds2(uint32_t a) {
  uint2 r;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(a));
  return r;
}

template <bool PUSH>
__global__ void __launch_bounds__(kTileThreads, 1024 / kTileThreads) wg_shadow_tile_kernel(const Params p, const ShadowState sh) {
  __shared__ unsigned long long sm[SH_WORDS];
  __shared__ __align__(16) TileSmem tiles[kTileWarps];
  // (volatile: ptxas otherwise re-derives the lane from SR_TID at every guard, an S2R round trip each time)
  uint32_t lane, lanebit;
  asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));
  asm volatile("shl.b32 %0, 1, %1;" : "=r"(lanebit) : "r"(lane));
  const uint32_t warp = __shfl_sync(kFull, threadIdx.x >> 5, 0);
  TileSmem& ts = tiles[warp];
  const uint32_t rec_s = sm_addr(ts.rec), st_s = sm_addr(ts.st), ust_s = sm_addr(ts.ust), vf_s = sm_addr(ts.vf);
  const uint64_t n_tiles = (p.n + kST - 1) / kST;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * kTileWarps;
  // the warp-uniform-value prefix (8 of 12 rounds per lane): check_ret 0.544 -> 0.514 ms, push 0.500 -> 0.474 ms.
  // (While the entry fields lived in three separate rows, push waited on DRAM read-filling its partially written
  // sectors and the prefix made it slower, 0.539 -> 0.559 ms; the switch is kept for such measurements.)
  constexpr bool kFast = true;
  const bool enforce = p.mode != 0;
  const uint32_t max_depth = sh.max_depth;
  uint32_t c[SH_WORDS];
#pragma unroll
  for (int i = 0; i < SH_WORDS; ++i) c[i] = 0;

  // lane-parallel loads of one pass.  S1: the lane's depth counter and value; S2 (check): the entry under the counter.
  struct S1 { uint32_t d, vl, vh; };
  auto load1 = [&](uint32_t i, uint64_t e0) -> S1 {
    S1 r{0u, 0u, 0u};
    if (i < static_cast<uint32_t>(kST)) {
      const uint4 a = lds4(rec_s + i * 16);
      if (a.x & lanebit) {
        r.d = sh.depth_ctr[static_cast<uint64_t>(a.y) * 32 + lane];
        const uint2 v = *reinterpret_cast<const uint2*>(p.val + (e0 + i) * 32 + lane);
        r.vl = v.x;
        r.vh = v.y;
      }
    }
    return r;
  };
  auto load2 = [&](uint32_t i, const S1& b) -> StageE {
    StageE x{0u, 0u, 0u, 0u, 0u, 0u};
    if constexpr (!PUSH) {
      if (i < static_cast<uint32_t>(kST)) {
        const uint4 a = lds4(rec_s + i * 16);
        if ((a.x & lanebit) && b.d != 0u && b.d - 1u < max_depth) {
          const uint4* en = reinterpret_cast<const uint4*>(sh.entry) + ((static_cast<uint64_t>(a.y) * max_depth + (b.d - 1u)) * 32 + lane) * 2;
          const uint4 et = en[0], m = en[1];
          x = StageE{et.x, et.y, et.z, et.w, m.x, m.y};
        }
      }
    }
    return x;
  };
  // index of the lowest set bit of m, or kST ("no pass") when m is empty
  auto first = [](uint32_t m) -> uint32_t { return m ? static_cast<uint32_t>(__ffs(m)) - 1u : static_cast<uint32_t>(kST); };

  // event-parallel loads of a tile, in the order they can be asked for: the header; then what it addresses (site
  // record, use count of the warp slot).  Two tiles ahead / one tile ahead, so a tile starts with both in registers.
  struct TB { uint32_t kind, uses, vfl, vfh; };
  auto load_th = [&](uint64_t t) -> uint4 {
    const uint64_t e = t * kST + lane;
    return (t < n_tiles && lane < static_cast<uint32_t>(kST) && e < p.n) ? __ldg(reinterpret_cast<const uint4*>(p.hdr) + e)
                                                                         : make_uint4(0u, 0u, 0u, 0u);
  };
  auto load_tb = [&](const uint4& h, uint64_t t) -> TB {
    TB b;
    b.kind = 7u;
    b.uses = b.vfl = b.vfh = 0u;
    if (h.y != 0u) {  // (a lane without an event holds a zero header)
      // the value of the event's first active lane: when every active lane carries it (a warp-uniform return
      // address) its two SipRounds are done once per event, 32 events at a time, instead of once per lane
      if constexpr (kFast) {
        const uint2 vf = *reinterpret_cast<const uint2*>(p.val + (t * kST + lane) * 32 + (__ffs(h.y) - 1));
        b.vfl = vf.x;
        b.vfh = vf.y;
      }
      if (h.x < p.n_sites) b.kind = __ldg(reinterpret_cast<const uint32_t*>(p.recs + h.x));
      const uint32_t slot = slot_of(h.z, h.w);
      if (slot < sh.n_slots) b.uses = static_cast<uint32_t>(sh.uses[slot]);  // (the slot carries this call's stamp)
    }
    return b;
  };
  const uint64_t t_first = static_cast<uint64_t>(blockIdx.x) * kTileWarps + warp;
  uint4 h_cur = load_th(t_first), h_nxt = load_th(t_first + stride);
  TB b_cur = load_tb(h_cur, t_first);

  for (uint64_t t = t_first; t < n_tiles; t += stride) {
    const uint64_t e0 = t * kST;
    const uint4 h_nn = load_th(t + 2 * stride);
    const TB b_nxt = load_tb(h_nxt, t + stride);
    // ---- event-parallel: header, site record, use count, classification, event counters ----
    const uint64_t e = e0 + lane;
    const bool valid = lane < static_cast<uint32_t>(kST) && e < p.n;
    const uint4 h = h_cur;
    const uint32_t a = h.y, slot = slot_of(h.z, h.w);
    uint32_t status = ST_NONE;
    if (valid) {
      status = ST_EMPTY;  // no lane executed the call / return
      if (a != 0u) {
        if (b_cur.kind != K_RET) {
          status = ST_NON_RETURN;  // unknown site, or not a return site of the policy: fail closed, state untouched
        } else if (slot >= sh.n_slots) {
          status = ST_SLOT_OVERFLOW;  // thread-slot overflow fails closed instead of wrapping
        } else if (b_cur.uses > 1u) {
          status = ST_SLOT_CONFLICT;  // the same warp twice in one lock-step call
        } else {
          status = ST_NORMAL;
          ts.rec[lane] = make_uint4(a, slot, h.x, (slot >> 27) | (h.w & 0xffff0000u));
          if constexpr (kFast) ts.vf[lane] = make_uint2(b_cur.vfl, b_cur.vfh);
        }
      }
    }
    // the site word of the MAC, once per event, 32 events at a time: the key-derived initial state exists in the kernel
    // parameters only (constant bank), never in global memory; leaves the "pre-A" state the tails start from
    Sip32 u{static_cast<uint32_t>(p.v0), static_cast<uint32_t>(p.v0 >> 32), static_cast<uint32_t>(p.v1),
            static_cast<uint32_t>(p.v1 >> 32), static_cast<uint32_t>(p.v2), static_cast<uint32_t>(p.v2 >> 32),
            static_cast<uint32_t>(p.v3), static_cast<uint32_t>(p.v3 >> 32)};
    sip_absorb(u, h.x, p.bind_hi);
    sip_qA(u);
    if (status == ST_NORMAL) {
      ts.st[lane][0] = make_uint4(u.v0l, u.v0h, u.v1l, u.v1h);
      ts.st[lane][1] = make_uint4(u.v2l, u.v2h, u.v3l, u.v3h);
    }
    if constexpr (kFast) {  // the MAC prefix of a warp-uniform value, for all events of the tile at once (used by the passes that find
       // every MAC-computing lane on that value; harmless garbage for the others)
      sip_absorb_preA(u, b_cur.vfl, b_cur.vfh);
      sip_qA(u);
      if (status == ST_NORMAL) {
        ts.ust[lane][0] = make_uint4(u.v0l, u.v0h, u.v1l, u.v1h);
        ts.ust[lane][1] = make_uint4(u.v2l, u.v2h, u.v3l, u.v3h);
      }
    }
    uint32_t viol = (status >= ST_NON_RETURN && status <= ST_SLOT_CONFLICT) ? a : 0u;
    const uint32_t m_norm = __ballot_sync(kFull, status == ST_NORMAL);
    {
      const uint32_t m_live = __ballot_sync(kFull, status >= ST_NON_RETURN);
      c[PUSH ? SH_PUSH_EVENTS : SH_CHECK_EVENTS] += __popc(m_live);
      c[PUSH ? SH_PUSH_LANES : SH_CHECK_LANES] += __reduce_add_sync(kFull, status >= ST_NON_RETURN ? __popc(a) : 0u);
      if (__ballot_sync(kFull, status != ST_NORMAL && status != ST_NONE)) {  // uncommon events
        c[SH_EMPTY_EVENTS] += __popc(__ballot_sync(kFull, status == ST_EMPTY));
        c[SH_NON_RETURN] += __popc(__ballot_sync(kFull, status == ST_NON_RETURN));
        c[SH_SLOT_OVERFLOW] += __popc(__ballot_sync(kFull, status == ST_SLOT_OVERFLOW));
        c[SH_SLOT_CONFLICT] += __popc(__ballot_sync(kFull, status == ST_SLOT_CONFLICT));
      }
    }
    __syncwarp();

    // ---- lane-parallel: one pass per ordinary event (distinct warp slots, so the passes touch disjoint state) ----
    // (Unrolling this loop three times over three named register sets, so that no loaded register is ever copied
    // before its pass, was measured with the earlier three-row entry layout: push 0.56 ms, check_ret 0.56 ms — no
    // gain for push and a loss for check_ret through its register count.)
    uint32_t m = m_norm;
    uint32_t i0 = first(m);
    m &= m - 1u;
    uint32_t i1 = first(m);
    m = m ? (m & (m - 1u)) : 0u;
    S1 b0 = load1(i0, e0), b1 = load1(i1, e0);
    StageE x0 = load2(i0, b0);
    while (i0 < static_cast<uint32_t>(kST)) {
      const uint32_t i2 = first(m);
      m = m ? (m & (m - 1u)) : 0u;
      const S1 b2 = load1(i2, e0);
      const StageE x1 = load2(i1, b1);

      const uint4 ra = lds4(rec_s + i0 * 16);
      uint2 vf = make_uint2(0u, 0u);
      if constexpr (kFast) vf = lds2(vf_s + i0 * 8);
      const uint32_t act = ra.x, sl = ra.y, site = ra.z;
      const bool on = (act & lanebit) != 0u;
      const uint32_t vl = b0.vl, vh = b0.vh;
      uint32_t d = b0.d;
      uint32_t cause = 0;  // 0 ok, else SH_* word of the lane's one cause
      // which lanes reach the MAC, and over which (callsite, value)
      bool mac = false;
      uint32_t ml = vl, mh = vh, msite = site;
      uint32_t* dctr = sh.depth_ctr + static_cast<uint64_t>(sl) * 32 + lane;
      if (on) {
        if (PUSH) {
          if (d >= max_depth)
            cause = SH_OVERFLOW;
          else
            mac = true;
        } else {
          if (d == 0) {
            cause = SH_UNDERFLOW;
          } else {
            d -= 1;
            *dctr = d;  // the return consumes the frame whatever the verdict (R33)
            // a corrupted counter may point past the arrays' depth: such an entry does not exist -> depth mismatch
            if (d >= max_depth || x0.depth != d) {
              cause = SH_DEPTH_MISMATCH;
            } else {
              mac = true;  // the token is verified over the ENTRY's own fields under the event's epoch
              ml = x0.exl;
              mh = x0.exh;
              msite = x0.callsite;
            }
          }
        }
      }
      // context: epoch<<48 | d<<37 | slot<<5 | lane
      const uint32_t bl = sl << 5, bh = ra.w | (d << 5);
      uint32_t tl = 0, th = 0;
      if (kFast && __all_sync(kFull, !mac || (ml == vf.x && mh == vf.y && msite == site))) {
        // the ordinary case: one return address for the whole warp — 8 of the 12 rounds per lane
        if (mac) {
          const uint4 s0 = lds4(ust_s + i0 * 32), s1 = lds4(ust_s + i0 * 32 + 16);
          sip_tail_ctx(Sip32{s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w}, bl | lane, bh, 0u, 0u, tl, th);
        }
      } else if (mac) {
        if (msite == site) {  // the site's cached mid-state saves the first word's rounds
          const uint4 s0 = lds4(st_s + i0 * 32), s1 = lds4(st_s + i0 * 32 + 16);
          sip_tail_val_lane(Sip32{s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w}, ml, mh, lane, bl, bh, 0u, 0u, tl, th);
        } else {
          mac_full(p, msite, ml, mh, bl | lane, bh, tl, th);
        }
      }
      if (mac) {
        if (PUSH) {
          uint4* en = reinterpret_cast<uint4*>(sh.entry) + ((static_cast<uint64_t>(sl) * max_depth + d) * 32 + lane) * 2;
          en[0] = make_uint4(vl, vh, tl, th);
          en[1] = make_uint4(site, d, 0u, 0u);
          *dctr = d + 1;
        } else {
          if (tl != x0.tkl || th != x0.tkh)
            cause = SH_TOKEN_MISMATCH;
          else if (x0.exl != vl || x0.exh != vh || x0.callsite != site)
            cause = SH_TARGET_MISMATCH;
        }
      }
      const uint32_t vb = __ballot_sync(kFull, cause != 0);
      if (vb) {  // rare: one cause per violating lane
#pragma unroll
        for (int k = SH_OVERFLOW; k <= SH_TARGET_MISMATCH; ++k) c[k] += __popc(__ballot_sync(kFull, cause == k));
      }
      if (lane == i0) viol = vb;  // event-parallel again below: lane i <-> event i

      i0 = i1;
      i1 = i2;
      b0 = b1;
      b1 = b2;
      x0 = x1;
    }

    // ---- event-parallel: verdicts and violation counters ----
    if (valid) p.out[e] = make_uint2(viol, enforce ? (a & ~viol) : a);
    const uint32_t m_viol = __ballot_sync(kFull, viol != 0u);
    if (m_viol) {
      const uint32_t lanes = __reduce_add_sync(kFull, __popc(viol));
      c[SH_VIOL_LANES] += lanes;
      c[SH_VIOL_EVENTS] += __popc(m_viol);
      if (enforce) c[SH_BLOCKED_LANES] += lanes;
    }
    __syncwarp();  // every lane is done with this tile's records before the next tile overwrites them
    h_cur = h_nxt;
    h_nxt = h_nn;
    b_cur = b_nxt;
  }

  if (threadIdx.x < SH_WORDS) sm[threadIdx.x] = 0ull;
  __syncthreads();
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < SH_WORDS; ++i)
      if (c[i]) atomicAdd(sm + i, static_cast<unsigned long long>(c[i]));
  }
  __syncthreads();
  if (threadIdx.x < SH_WORDS && sm[threadIdx.x]) atomicAdd(sh.counters + threadIdx.x, sm[threadIdx.x]);
}

}  // namespace

cudaError_t shadow_occupancy(int* per_sm_push, int* per_sm_check) {
  cudaError_t err;
  if ((err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm_push, wg_shadow_tile_kernel<true>, kTileThreads, 0)) != cudaSuccess)
    return err;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm_check, wg_shadow_tile_kernel<false>, kTileThreads, 0);
}

cudaError_t launch_shadow(const Params& p, const ShadowState& sh, bool push, int sm_count, cudaStream_t st,
                          uint64_t* launches) {
  const uint64_t want_m = (p.n + 255) / 256;
  const int grid_m = static_cast<int>(want_m < static_cast<uint64_t>(sm_count) * 8 ? want_m : sm_count * 8);
  wg_shadow_mark<<<grid_m, 256, 0, st>>>(p.hdr, p.n, sh.uses, sh.n_slots, sh.stamp);
  ++*launches;
  // persistent warps: exactly the blocks that are resident at once (occupancy resolved per engine at configure time)
  const int per_sm = sh.per_sm[push] > 0 ? sh.per_sm[push] : 1;
  const uint64_t units = (p.n + kST - 1) / kST;  // a warp's unit of work: a tile
  const uint64_t want = (units + kTileWarps - 1) / kTileWarps;
  const uint64_t resident = static_cast<uint64_t>(sm_count) * per_sm;
  const int grid = static_cast<int>(want < resident ? want : resident);
  if (push)
    wg_shadow_tile_kernel<true><<<grid, kTileThreads, 0, st>>>(p, sh);
  else
    wg_shadow_tile_kernel<false><<<grid, kTileThreads, 0, st>>>(p, sh);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace wg
