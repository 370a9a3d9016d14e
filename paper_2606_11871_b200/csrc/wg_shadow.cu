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

  for (uint64_t e = warp0; e < p.n; e += nwarps) {
    const uint4 h = p.hdr[e];
    const uint32_t site = h.x, a = h.y;
    const uint32_t slot = slot_of(h.z, h.w);
    uint32_t viol = 0;
    if (a == 0) {
      c[SH_EMPTY_EVENTS] += 1;  // no lane executed the call / return
    } else {
      c[PUSH ? SH_PUSH_EVENTS : SH_CHECK_EVENTS] += 1;
      c[PUSH ? SH_PUSH_LANES : SH_CHECK_LANES] += __popc(a);
      uint4 rec0 = make_uint4(7u, 0u, 0u, 0u);
      if (site < p.n_sites) rec0 = __ldg(reinterpret_cast<const uint4*>(p.recs + site));
      if (rec0.x != K_RET) {  // unknown site, or not a return site of the policy: fail closed, state untouched
        viol = a;
        c[SH_NON_RETURN] += 1;
      } else if (slot >= sh.n_slots) {  // thread-slot overflow fails closed instead of wrapping
        viol = a;
        c[SH_SLOT_OVERFLOW] += 1;
      } else if (sh.uses[slot] > 1u) {  // the same warp twice in one lock-step call
        viol = a;
        c[SH_SLOT_CONFLICT] += 1;
      } else {
        const bool on = (a >> lane) & 1u;
        const uint64_t v = on ? p.val[e * 32 + lane] : 0ull;
        const uint32_t vl = static_cast<uint32_t>(v), vh = static_cast<uint32_t>(v >> 32);
        uint32_t* dctr = sh.depth_ctr + static_cast<uint64_t>(slot) * 32 + lane;
        uint32_t d = on ? *dctr : 0u;
        uint32_t cause = 0;  // 0 ok, else SH_* word of the lane's one cause
        if (on) {
          if (PUSH) {
            if (d >= sh.max_depth) {
              cause = SH_OVERFLOW;
            } else {
              const uint4 b = __ldg(reinterpret_cast<const uint4*>(p.recs + site) + 1);
              const uint4 cc = __ldg(reinterpret_cast<const uint4*>(p.recs + site) + 2);
              const Sip32 s{b.x, b.y, b.z, b.w, cc.x, cc.y, cc.z, cc.w};  // pre-A state after the site word
              // context: epoch<<48 | d<<37 | slot<<5 | lane (lane is injected by the tail)
              const uint32_t bl = slot << 5, bh = (slot >> 27) | (d << 5) | (h.w & 0xffff0000u);
              uint32_t tl, th;
              sip_tail_val_lane(s, vl, vh, lane, bl, bh, 0u, 0u, tl, th);
              const uint64_t idx = (static_cast<uint64_t>(slot) * sh.max_depth + d) * 32 + lane;
              sh.expected[idx] = v;
              sh.token[idx] = (static_cast<uint64_t>(th) << 32) | tl;
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
              } else {
                const uint64_t idx = (static_cast<uint64_t>(slot) * sh.max_depth + d) * 32 + lane;
                const uint64_t ex = sh.expected[idx], tk = sh.token[idx];
                const uint2 m = sh.meta[idx];
                if (m.y != d) {
                  cause = SH_DEPTH_MISMATCH;
                } else {
                  // the token is verified over the ENTRY's own fields under the event's epoch
                  const uint32_t bl = slot << 5, bh = (slot >> 27) | (d << 5) | (h.w & 0xffff0000u);
                  uint32_t tl, th;
                  if (m.x == site) {  // the ordinary case: the site's cached mid-state saves the first word's rounds
                    const uint4 b = __ldg(reinterpret_cast<const uint4*>(p.recs + site) + 1);
                    const uint4 cc = __ldg(reinterpret_cast<const uint4*>(p.recs + site) + 2);
                    const Sip32 s{b.x, b.y, b.z, b.w, cc.x, cc.y, cc.z, cc.w};
                    sip_tail_val_lane(s, static_cast<uint32_t>(ex), static_cast<uint32_t>(ex >> 32), lane, bl, bh, 0u,
                                      0u, tl, th);
                  } else {
                    mac_full(p, m.x, static_cast<uint32_t>(ex), static_cast<uint32_t>(ex >> 32), bl | lane, bh, tl, th);
                  }
                  if (((static_cast<uint64_t>(th) << 32) | tl) != tk)
                    cause = SH_TOKEN_MISMATCH;
                  else if (ex != v || m.x != site)
                    cause = SH_TARGET_MISMATCH;
                }
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
  const uint64_t want = (p.n + kWarps - 1) / kWarps;
  const int grid = static_cast<int>(want < static_cast<uint64_t>(sm_count) * 8 ? want : sm_count * 8);
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
