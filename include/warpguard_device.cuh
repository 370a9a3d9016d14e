// warpguard_device.cuh — the check as an INLINE device helper: a kernel calls it at its own call / return /
// indirect-branch sites, one call per thread, the consumption-time form the paper deploys (§5.1,
// 228-230 §5.3 "push(site, expected_ret, guard), check_ret(site, observed_ret, guard), forward check (site, target,
// guard)"; WG-PC's callback-free checks).
//
// Same arithmetic as the batched engine (R1-R8): token = SipHash-2-4 over LE64(site_id) ||
// LE64(continuation) || LE64(context_id); forward check = exact membership in the site's sorted set.  The view is
// obtained from the engine with wg_get_device_view() and passed to the kernel BY VALUE (kernel parameter space), the
// analogue of "keys are passed to injected helpers as instrumentation arguments and are not exposed as ordinary
// target-writable CUDA objects".  The caller applies the guard: a predicated-off lane simply does
// not call.  These helpers keep no counters: what to do with a false verdict (trap, record) is the
// calling kernel's profile.
#pragma once
#include <stdint.h>

#include "warpguard.h"
#include "warpguard_sip32.cuh"

// sign / verify: `context_id` is the full 64-bit context word of THIS thread (the batched API's
// (context_base & ~31) | lane).  Unknown or non-return sites: sign returns 0, verify returns false (fail closed).
// The key-derived SipHash initial state comes from the view, i.e. from kernel parameter space; nothing key-derived
// is read from device memory.
__device__ __forceinline__ uint64_t wg_dev_sign(const wg_device_view& v, uint32_t site_id, uint64_t continuation,
                                                uint64_t context_id) {
  if (site_id >= v.n_sites) return 0;
  const uint4 a = __ldg(reinterpret_cast<const uint4*>(v.site_recs) + site_id);
  if (a.x != WG_KIND_PROTECTED_RETURN) return 0;
  wg::Sip32 s{static_cast<uint32_t>(v.v_init[0]), static_cast<uint32_t>(v.v_init[0] >> 32),
              static_cast<uint32_t>(v.v_init[1]), static_cast<uint32_t>(v.v_init[1] >> 32),
              static_cast<uint32_t>(v.v_init[2]), static_cast<uint32_t>(v.v_init[2] >> 32),
              static_cast<uint32_t>(v.v_init[3]), static_cast<uint32_t>(v.v_init[3] >> 32)};
  uint32_t tl, th;
  wg::sip_absorb(s, site_id, v.bind_hi);  // LE64(site_id | digest32 << 32) (R3, R39)
  wg::sip_absorb(s, static_cast<uint32_t>(continuation), static_cast<uint32_t>(continuation >> 32));
  wg::sip_absorb(s, static_cast<uint32_t>(context_id), static_cast<uint32_t>(context_id >> 32));
  wg::sip_finish(s, 0u, 0u, tl, th);
  return (static_cast<uint64_t>(th) << 32) | tl;
}

__device__ __forceinline__ bool wg_dev_verify(const wg_device_view& v, uint32_t site_id, uint64_t observed,
                                              uint64_t context_id, uint64_t stored_tag) {
  if (site_id >= v.n_sites) return false;
  if (__ldg(reinterpret_cast<const uint4*>(v.site_recs) + site_id).x != WG_KIND_PROTECTED_RETURN) return false;
  return wg_dev_sign(v, site_id, observed, context_id) == stored_tag;
}

// forward check: true iff `target` is a member of the site's set (branch-free lower-bound walk)
__device__ __forceinline__ bool wg_dev_check_forward(const wg_device_view& v, uint32_t site_id, uint64_t target) {
  if (site_id >= v.n_sites) return false;
  const uint4 a = __ldg(reinterpret_cast<const uint4*>(v.site_recs) + site_id);
  if (a.x != WG_KIND_PROTECTED_FORWARD) return false;
  const uint64_t* set = v.targets + a.y;
  uint32_t lo = 0, len = a.z;
  while (len > 1) {
    const uint32_t half = len >> 1;
    lo = (__ldg(set + lo + half) <= target) ? lo + half : lo;
    len -= half;
  }
  return __ldg(set + lo) == target;
}
