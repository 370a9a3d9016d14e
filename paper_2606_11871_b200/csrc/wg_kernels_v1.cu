// wg_kernels_v1.cu — the FIRST (baseline) mapping of the check path on sm_100a, kept selectable (WG_IMPL=v1) so
// that the v2 kernels of wg_kernels_v2.cu can be measured against it (profiles/):  sign (a3), verify (a4), forward membership (a5), verdicts (a6),
// aggregated counters (a7) and the first-violation record (a8) of SURVEY.md §8(a).
//
// Mapping (v1, "warp per event"): one warp owns one event at a time, thread l owns lane l of it.  The 16-byte
// header is one broadcast load, the value / tag rows are one fully coalesced 256-byte load each
// (ld.global.nc, no L1 allocation: every byte is read once), the verdict is one 8-byte store by lane 0.
// Counters are warp-uniform registers flushed once per warp through shared memory, then one global atomic
// per counter per CTA; per-site counters are one red.global per event by two lanes.
//
// Paper passages: backward token PAPER.md:162, 248; forward membership PAPER.md:174-178, 250-252; guards
// PAPER.md:190, 230; detect / enforce PAPER.md:264; accounting PAPER.md:113, 127, 224.  Readings: DESIGN.md §2.
#include "wg_internal.h"
#include "wg_siphash.cuh"

namespace wg {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

enum : uint32_t { K_RET = 0, K_FWD = 1 };

__device__ __forceinline__ uint4 ld_stream_v4(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ uint64_t ld_stream_u64(const uint64_t* p) {
  uint64_t r;
  asm volatile("ld.global.nc.L1::no_allocate.u64 %0, [%1];" : "=l"(r) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.global.L1::no_allocate.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_stream_v2(uint2* p, uint32_t a, uint32_t b) {
  asm volatile("st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}

__device__ __forceinline__ Sip init_state(const Params& p) { return Sip{p.v0, p.v1, p.v2, p.v3}; }

// full token of one lane: absorb site, continuation, lane context, length word; finalise (R1-R4)
__device__ __forceinline__ uint64_t token(const Params& p, uint32_t site, uint64_t value, uint64_t ctx) {
  Sip s = init_state(p);
  absorb(s, static_cast<uint64_t>(site));
  return mac_tail_from_w1(s, value, ctx);
}

// exact-equality membership in a strictly ascending set, branch-free lower-bound walk (R8)
__device__ __forceinline__ bool member(const uint64_t* __restrict__ set, uint32_t cnt, uint64_t v) {
  uint32_t lo = 0, len = cnt;  // cnt >= 1 for every protected-forward site (validated at load)
  while (len > 1) {
    const uint32_t half = len >> 1;
    const uint64_t mid = __ldg(set + lo + half);
    lo = (mid <= v) ? lo + half : lo;
    len -= half;
  }
  return __ldg(set + lo) == v;
}

// warp-uniform counters of one warp, flushed at the end
struct WarpCounters {
  uint32_t w[24];
  uint64_t first;
};

__device__ __forceinline__ void flush_counters(const WarpCounters& c, unsigned long long* glob,
                                               unsigned long long* sm) {
  const int lane = threadIdx.x & 31;
  if (threadIdx.x < C_WORDS) sm[threadIdx.x] = (threadIdx.x == C_FIRST_VIOLATION) ? ~0ull : 0ull;
  __syncthreads();
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < 24; ++i)
      if (i != C_FIRST_VIOLATION && c.w[i]) atomicAdd(sm + i, static_cast<unsigned long long>(c.w[i]));
    if (c.first != ~0ull) atomicMin(sm + C_FIRST_VIOLATION, static_cast<unsigned long long>(c.first));
  }
  __syncthreads();
  if (threadIdx.x < 24) {
    const unsigned long long v = sm[threadIdx.x];
    if (threadIdx.x == C_FIRST_VIOLATION) {
      if (v != ~0ull) atomicMin(glob + C_FIRST_VIOLATION, v);
    } else if (v) {
      atomicAdd(glob + threadIdx.x, v);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// sign: backward push
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) wg_sign_v1(const Params p) {
  __shared__ unsigned long long sm[C_WORDS];
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t warp0 = (static_cast<uint64_t>(blockIdx.x) * kThreads + threadIdx.x) >> 5;
  const uint64_t nwarps = static_cast<uint64_t>(gridDim.x) * kWarps;
  WarpCounters c;
#pragma unroll
  for (int i = 0; i < 24; ++i) c.w[i] = 0;
  c.first = ~0ull;

  for (uint64_t e = warp0; e < p.n; e += nwarps) {
    const uint4 h = ld_stream_v4(p.hdr + e);
    const uint32_t site = h.x, active = h.y;
    bool prot = false;
    if (site < p.n_sites) prot = __ldg(reinterpret_cast<const uint32_t*>(p.rows + site)) == K_RET;
    uint64_t t = 0;
    if (prot) {
      c.w[C_SIGNED_LANES] += __popc(active);
      if ((active >> lane) & 1u) {
        const uint64_t v = ld_stream_u64(p.val + e * 32 + lane);
        const uint64_t ctx = (pack64(h.z, h.w) & ~31ull) | lane;
        t = token(p, site, v, ctx);
      }
    } else {
      c.w[C_SIGN_SKIPPED] += 1;
    }
    st_stream_u64(p.tag_out + e * 32 + lane, t);
  }
  flush_counters(c, p.glob, sm);
}

// ---------------------------------------------------------------------------------------------------
// check: backward check_ret + forward check over a stream of any site kinds
// ---------------------------------------------------------------------------------------------------
template <bool HAS_TAG>
__global__ void __launch_bounds__(kThreads) wg_check_v1(const Params p) {
  __shared__ unsigned long long sm[C_WORDS];
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t warp0 = (static_cast<uint64_t>(blockIdx.x) * kThreads + threadIdx.x) >> 5;
  const uint64_t nwarps = static_cast<uint64_t>(gridDim.x) * kWarps;
  const bool enforce = p.mode != 0;
  WarpCounters c;
#pragma unroll
  for (int i = 0; i < 24; ++i) c.w[i] = 0;
  c.first = ~0ull;

  for (uint64_t e = warp0; e < p.n; e += nwarps) {
    const uint4 h = ld_stream_v4(p.hdr + e);
    const uint32_t site = h.x, active = h.y;
    const uint32_t na = __popc(active);
    uint32_t viol = 0;
    c.w[C_EVENTS_TOTAL] += 1;
    if (site >= p.n_sites) {  // unknown site: fail closed, outside every denominator (R13)
      viol = active;
      c.w[C_EVENTS_UNKNOWN] += 1;
    } else {
      const uint4 row = __ldg(reinterpret_cast<const uint4*>(p.rows + site));
      const uint32_t kind = row.x;
      unsigned long long* sc = p.site + static_cast<uint64_t>(site) * 4;
      bool judged = false;
      // events_by_kind: kind is warp-uniform, a 7-way select keeps the counters in registers
#pragma unroll
      for (int k = 0; k < 7; ++k) c.w[C_BY_KIND + k] += (kind == static_cast<uint32_t>(k));
      if (active == 0) {
        c.w[C_EVENTS_EMPTY] += 1;  // fully predicated off: not a check (R22)
      } else if (kind == K_RET) {
        if (HAS_TAG) {
          bool bad = false;
          if ((active >> lane) & 1u) {  // inactive lanes are never read nor judged
            const uint64_t v = ld_stream_u64(p.val + e * 32 + lane);
            const uint64_t t = ld_stream_u64(p.tag + e * 32 + lane);
            const uint64_t ctx = (pack64(h.z, h.w) & ~31ull) | lane;
            bad = token(p, site, v, ctx) != t;
          }
          viol = __ballot_sync(0xffffffffu, bad);
          c.w[C_RET_CHECKS] += 1;
          c.w[C_RET_LANES] += na;
          c.w[C_RET_VIOL] += __popc(viol);
          c.w[C_RET_VIOL_EVENTS] += (viol != 0);
          judged = true;
        } else {  // no tag at the forward entry point: cannot authenticate, fail closed (R14)
          viol = active;
          c.w[C_EVENTS_MISROUTED] += 1;
        }
      } else if (kind == K_FWD) {
        bool bad = false;
        if ((active >> lane) & 1u) {
          const uint64_t v = ld_stream_u64(p.val + e * 32 + lane);
          bad = !member(p.tgts + row.y, row.z, v);
        }
        viol = __ballot_sync(0xffffffffu, bad);
        c.w[C_FWD_CHECKS] += 1;
        c.w[C_FWD_LANES] += na;
        c.w[C_FWD_VIOL] += __popc(viol);
        c.w[C_FWD_VIOL_EVENTS] += (viol != 0);
        judged = true;
      }
      // per-site counters (diagnostic only): lane 0 events, lane 1 lanes_checked, ...
      if (lane == 0) atomicAdd(sc + S_EVENTS, 1ull);
      if (judged) {
        if (lane == 1) atomicAdd(sc + S_LANES_CHECKED, static_cast<unsigned long long>(na));
        if (viol) {
          if (lane == 2) atomicAdd(sc + S_LANES_VIOLATION, static_cast<unsigned long long>(__popc(viol)));
        }
      }
      if (enforce && viol && lane == 3) atomicAdd(sc + S_LANES_BLOCKED, static_cast<unsigned long long>(__popc(viol)));
    }
    const uint32_t allow = enforce ? (active & ~viol) : active;
    if (viol) {
      if (enforce) {
        c.w[C_BLOCKED_LANES] += __popc(viol);
        c.w[C_BLOCKED_EVENTS] += 1;
      }
      const uint64_t key = ((p.seq_base + e) << 5) | static_cast<uint32_t>(__ffs(viol) - 1);
      c.first = key < c.first ? key : c.first;
    }
    if (lane == 0) st_stream_v2(p.out + e, viol, allow);
  }
  flush_counters(c, p.glob, sm);
}

__global__ void wg_fill_u64(unsigned long long* p, uint64_t n, unsigned long long v) {
  uint64_t i = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * blockDim.x;
  for (; i < n; i += stride) p[i] = v;
}

int grid_for(uint64_t n_events, int sm_count, int ctas_per_sm) {
  const uint64_t want = (n_events + kWarps - 1) / kWarps;
  const uint64_t cap = static_cast<uint64_t>(sm_count) * ctas_per_sm;
  return static_cast<int>(want < cap ? (want ? want : 1) : cap);
}

}  // namespace

cudaError_t launch_sign_v1(const Params& p, int sm_count, cudaStream_t st) {
  wg_sign_v1<<<grid_for(p.n, sm_count, 8), kThreads, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_check_v1(const Params& p, int sm_count, cudaStream_t st) {
  const int grid = grid_for(p.n, sm_count, 8);
  if (p.tag)
    wg_check_v1<true><<<grid, kThreads, 0, st>>>(p);
  else
    wg_check_v1<false><<<grid, kThreads, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_fill_u64(unsigned long long* p, uint64_t n, unsigned long long v, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  uint64_t blocks = (n + 255) / 256;
  if (blocks > 1184) blocks = 1184;
  wg_fill_u64<<<static_cast<int>(blocks), 256, 0, st>>>(p, n, v);
  count_launch();
  return cudaGetLastError();
}

}  // namespace wg
