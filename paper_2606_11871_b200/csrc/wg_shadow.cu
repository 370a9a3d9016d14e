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
//   depth_ctr[slot][32] u32;  expected[slot][d][32] u64;  token[slot][d][32] u64;  meta[slot][d][32] {callsite, depth}.
// Mapping: one warp per event (the state access is a gather by warp slot; each lane owns its own stack).
// A call is one lock-step step of DISTINCT warps: a counting pass marks warp slots that occur twice in the call
// and those events fail closed; a clearing pass resets the marks.
#include "wg_internal.h"
#include "../../include/warpguard_sip32.cuh"

namespace wg {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr uint32_t kFull = 0xffffffffu;
enum : uint32_t { K_RET = 0 };

__device__ __forceinline__ uint32_t slot_of(uint32_t ctx_lo, uint32_t ctx_hi) {
  return (ctx_lo >> 5) | (ctx_hi << 27);  // bits 36..5 of context_base
}

__global__ void wg_shadow_mark(const uint4* __restrict__ hdr, uint64_t n, uint32_t* uses, uint32_t n_slots, int clear) {
  uint64_t i = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * blockDim.x;
  for (; i < n; i += stride) {
    const uint4 h = hdr[i];
    const uint32_t slot = slot_of(h.z, h.w);
    if (slot < n_slots) {
      if (clear)
        uses[slot] = 0u;
      else
        atomicAdd(uses + slot, 1u);
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

// what an event needs from memory, in the order it can be asked for: the header; then what the header addresses
// (site record, use count of the warp slot, the lane's value and depth counter); then (check) the entry the depth
// counter addresses.  Every load is a dependent HBM / L2 round trip, so the kernel keeps three events in flight per
// warp: while event k is computed, the entry of k+1, the header-addressed words of k+2 and the header of k+3 fly.
struct StageB {
  uint4 rec0, sb, sc;  // SiteRec: {kind, off, cnt, -}; pre-A mid-state after the site word
  uint32_t uses, d, vl, vh;
};
struct StageE {
  uint32_t exl, exh, tkl, tkh, callsite, depth;
};

template <bool PUSH>
__global__ void __launch_bounds__(kThreads) wg_shadow_kernel(const Params p, const ShadowState sh) {
  __shared__ unsigned long long sm[SH_WORDS];
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t warp0 = (static_cast<uint64_t>(blockIdx.x) * kThreads + threadIdx.x) >> 5;
  const uint64_t nwarps = static_cast<uint64_t>(gridDim.x) * kWarps;
  const bool enforce = p.mode != 0;
  uint32_t c[SH_WORDS];
#pragma unroll
  for (int i = 0; i < SH_WORDS; ++i) c[i] = 0;

  auto load_h = [&](uint64_t e) -> uint4 { return e < p.n ? __ldg(reinterpret_cast<const uint4*>(p.hdr) + e) : make_uint4(0u, 0u, 0u, 0u); };
  auto load_b = [&](const uint4& h, uint64_t e) -> StageB {
    StageB b;
    b.rec0 = make_uint4(7u, 0u, 0u, 0u);
    b.sb = b.sc = make_uint4(0u, 0u, 0u, 0u);
    b.uses = b.d = b.vl = b.vh = 0u;
    if (e < p.n && h.y != 0u) {
      const uint32_t slot = slot_of(h.z, h.w);
      const bool on = (h.y >> lane) & 1u;
      if (h.x < p.n_sites) {
        const uint4* r = reinterpret_cast<const uint4*>(p.recs + h.x);
        b.rec0 = __ldg(r);
        b.sb = __ldg(r + 1);
        b.sc = __ldg(r + 2);
      }
      if (slot < sh.n_slots) {
        b.uses = sh.uses[slot];
        if (on) b.d = sh.depth_ctr[static_cast<uint64_t>(slot) * 32 + lane];
      }
      if (on) {
        const uint2 v = *reinterpret_cast<const uint2*>(p.val + e * 32 + lane);
        b.vl = v.x;
        b.vh = v.y;
      }
    }
    return b;
  };
  auto load_e = [&](const uint4& h, const StageB& b) -> StageE {
    StageE x{0u, 0u, 0u, 0u, 0u, 0u};
    if constexpr (!PUSH) {
      const uint32_t slot = slot_of(h.z, h.w);
      if (((h.y >> lane) & 1u) && slot < sh.n_slots && b.d != 0u && b.d - 1u < sh.max_depth) {
        const uint64_t idx = (static_cast<uint64_t>(slot) * sh.max_depth + (b.d - 1u)) * 32 + lane;
        const uint2 ex = *reinterpret_cast<const uint2*>(sh.expected + idx);
        const uint2 tk = *reinterpret_cast<const uint2*>(sh.token + idx);
        const uint2 m = sh.meta[idx];
        x = StageE{ex.x, ex.y, tk.x, tk.y, m.x, m.y};
      }
    }
    return x;
  };

  // prologue: fill the pipeline
  uint4 h0 = load_h(warp0), h1 = load_h(warp0 + nwarps), h2 = load_h(warp0 + 2 * nwarps);
  StageB b0 = load_b(h0, warp0), b1 = load_b(h1, warp0 + nwarps);
  StageE x0 = load_e(h0, b0);

  for (uint64_t e = warp0; e < p.n; e += nwarps) {
    // loads of the events behind this one
    const uint4 h3 = load_h(e + 3 * nwarps);
    const StageB b2 = load_b(h2, e + 2 * nwarps);
    const StageE x1 = load_e(h1, b1);

    const uint4 h = h0;
    const uint32_t site = h.x, a = h.y;
    const uint32_t slot = slot_of(h.z, h.w);
    uint32_t viol = 0;
    if (a == 0) {
      c[SH_EMPTY_EVENTS] += 1;  // no lane executed the call / return
    } else {
      c[PUSH ? SH_PUSH_EVENTS : SH_CHECK_EVENTS] += 1;
      c[PUSH ? SH_PUSH_LANES : SH_CHECK_LANES] += __popc(a);
      if (b0.rec0.x != K_RET) {  // unknown site, or not a return site of the policy: fail closed, state untouched
        viol = a;
        c[SH_NON_RETURN] += 1;
      } else if (slot >= sh.n_slots) {  // thread-slot overflow fails closed instead of wrapping
        viol = a;
        c[SH_SLOT_OVERFLOW] += 1;
      } else if (b0.uses > 1u) {  // the same warp twice in one lock-step call
        viol = a;
        c[SH_SLOT_CONFLICT] += 1;
      } else {
        const bool on = (a >> lane) & 1u;
        const uint32_t vl = b0.vl, vh = b0.vh;
        uint32_t* dctr = sh.depth_ctr + static_cast<uint64_t>(slot) * 32 + lane;
        uint32_t d = b0.d;
        uint32_t cause = 0;  // 0 ok, else SH_* word of the lane's one cause
        const Sip32 s_site{b0.sb.x, b0.sb.y, b0.sb.z, b0.sb.w, b0.sc.x, b0.sc.y, b0.sc.z, b0.sc.w};  // pre-A state after the site word
        if (on) {
          if (PUSH) {
            if (d >= sh.max_depth) {
              cause = SH_OVERFLOW;
            } else {
              // context: epoch<<48 | d<<37 | slot<<5 | lane (lane is injected by the tail)
              const uint32_t bl = slot << 5, bh = (slot >> 27) | (d << 5) | (h.w & 0xffff0000u);
              uint32_t tl, th;
              sip_tail_val_lane(s_site, vl, vh, lane, bl, bh, 0u, 0u, tl, th);
              const uint64_t idx = (static_cast<uint64_t>(slot) * sh.max_depth + d) * 32 + lane;
              *reinterpret_cast<uint2*>(sh.expected + idx) = make_uint2(vl, vh);
              *reinterpret_cast<uint2*>(sh.token + idx) = make_uint2(tl, th);
              sh.meta[idx] = make_uint2(site, d);
              *dctr = d + 1;
            }
          } else {
            if (d == 0) {
              cause = SH_UNDERFLOW;
            } else {
              d -= 1;
              *dctr = d;  // the return consumes the frame whatever the verdict (R33)
              // a corrupted counter may point past the arrays' depth: such an entry does not exist -> depth mismatch
              if (d >= sh.max_depth) {
                cause = SH_DEPTH_MISMATCH;
              } else if (x0.depth != d) {
                cause = SH_DEPTH_MISMATCH;
              } else {
                // the token is verified over the ENTRY's own fields under the event's epoch
                const uint32_t bl = slot << 5, bh = (slot >> 27) | (d << 5) | (h.w & 0xffff0000u);
                uint32_t tl, th;
                if (x0.callsite == site) {  // the ordinary case: the site's cached mid-state saves the first word's rounds
                  sip_tail_val_lane(s_site, x0.exl, x0.exh, lane, bl, bh, 0u, 0u, tl, th);
                } else {
                  mac_full(p, x0.callsite, x0.exl, x0.exh, bl | lane, bh, tl, th);
                }
                if (tl != x0.tkl || th != x0.tkh)
                  cause = SH_TOKEN_MISMATCH;
                else if (x0.exl != vl || x0.exh != vh || x0.callsite != site)
                  cause = SH_TARGET_MISMATCH;
              }
            }
          }
        }
        viol = __ballot_sync(kFull, cause != 0);
        if (viol) {  // rare: one cause per violating lane
#pragma unroll
          for (int k = SH_OVERFLOW; k <= SH_TARGET_MISMATCH; ++k) c[k] += __popc(__ballot_sync(kFull, cause == k));
        }
      }
    }
    if (viol) {
      c[SH_VIOL_LANES] += __popc(viol);
      c[SH_VIOL_EVENTS] += 1;
      if (enforce) c[SH_BLOCKED_LANES] += __popc(viol);
    }
    if (lane == 0) p.out[e] = make_uint2(viol, enforce ? (a & ~viol) : a);

    h0 = h1;
    h1 = h2;
    h2 = h3;
    b0 = b1;
    b1 = b2;
    x0 = x1;
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

cudaError_t launch_shadow(const Params& p, const ShadowState& sh, bool push, int sm_count, cudaStream_t st) {
  const uint64_t want_m = (p.n + 255) / 256;
  const int grid_m = static_cast<int>(want_m < static_cast<uint64_t>(sm_count) * 8 ? want_m : sm_count * 8);
  wg_shadow_mark<<<grid_m, 256, 0, st>>>(p.hdr, p.n, sh.uses, sh.n_slots, 0);
  count_launch();
  // persistent warps, three events in flight each: exactly the blocks that are resident at once
  static int per_sm[2] = {0, 0};
  if (per_sm[push] == 0) {
    int nb = 0;
    const cudaError_t err = push ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, wg_shadow_kernel<true>, kThreads, 0)
                                 : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, wg_shadow_kernel<false>, kThreads, 0);
    if (err != cudaSuccess) return err;
    per_sm[push] = nb > 0 ? nb : 1;
  }
  const uint64_t want = (p.n + kWarps - 1) / kWarps;
  const uint64_t resident = static_cast<uint64_t>(sm_count) * per_sm[push];
  const int grid = static_cast<int>(want < resident ? want : resident);
  if (push)
    wg_shadow_kernel<true><<<grid, kThreads, 0, st>>>(p, sh);
  else
    wg_shadow_kernel<false><<<grid, kThreads, 0, st>>>(p, sh);
  count_launch();
  wg_shadow_mark<<<grid_m, 256, 0, st>>>(p.hdr, p.n, sh.uses, sh.n_slots, 1);
  count_launch();
  return cudaGetLastError();
}

}  // namespace wg
