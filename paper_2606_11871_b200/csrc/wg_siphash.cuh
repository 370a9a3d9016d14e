// wg_siphash.cuh — the backward token on the sm_100a integer pipes.
//
// token = SipHash-2-4_key( LE64(site_id) || LE64(continuation) || LE64(context_id) ), 64-bit output
// (R1-R4; the paper's own formula is lost at PAPER.md:164-166 / 244-246, "keyed token" over the
// return state PAPER.md:162, 258).  The 24-byte message is exactly three 64-bit words, so the MAC is
//     absorb(w0) absorb(w1) absorb(w2) absorb(0x18 << 56) finalise
// with absorb(m) = { v3 ^= m; SipRound; SipRound; v0 ^= m } — 12 SipRounds in all.  The engine splits it at
// word boundaries: the state after w0 (site) — and after w1 when the warp's continuation is uniform — is
// computed once per EVENT, the rest once per active LANE.
//
// Instruction selection (checked with cuobjdump -sass): all arithmetic is on 32-bit halves.
// A 64-bit add is IADD3 + IADD3.X / IMAD.X, a rotate is two funnel shifts (SHF.L.W), rotate-by-32 is a register
// rename, xor is LOP3.  Nothing touches memory; the key-derived initial state arrives in kernel parameters.
#pragma once
#include <cstdint>

namespace wg {

struct Sip {
  uint64_t v0, v1, v2, v3;
};

__device__ __forceinline__ uint64_t pack64(uint32_t lo, uint32_t hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
  return r;
}
__device__ __forceinline__ void unpack64(uint64_t x, uint32_t& lo, uint32_t& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(x));
}

// rotate left by a compile-time amount 0 < B < 64, B != 32: two funnel shifts
template <int B>
__device__ __forceinline__ uint64_t rotl(uint64_t x) {
  uint32_t lo, hi;
  unpack64(x, lo, hi);
  if constexpr (B == 32) {
    return pack64(hi, lo);
  } else if constexpr (B < 32) {
    return pack64(__funnelshift_l(hi, lo, B), __funnelshift_l(lo, hi, B));
  } else {
    return pack64(__funnelshift_l(lo, hi, B - 32), __funnelshift_l(hi, lo, B - 32));
  }
}

__device__ __forceinline__ void sipround(Sip& s) {
  s.v0 += s.v1;
  s.v1 = rotl<13>(s.v1);
  s.v1 ^= s.v0;
  s.v0 = rotl<32>(s.v0);
  s.v2 += s.v3;
  s.v3 = rotl<16>(s.v3);
  s.v3 ^= s.v2;
  s.v0 += s.v3;
  s.v3 = rotl<21>(s.v3);
  s.v3 ^= s.v0;
  s.v2 += s.v1;
  s.v1 = rotl<17>(s.v1);
  s.v1 ^= s.v2;
  s.v2 = rotl<32>(s.v2);
}

// one 8-byte message word: c = 2 compression rounds
__device__ __forceinline__ void absorb(Sip& s, uint64_t m) {
  s.v3 ^= m;
  sipround(s);
  sipround(s);
  s.v0 ^= m;
}

// d = 4 finalisation rounds
__device__ __forceinline__ uint64_t finalise(Sip& s) {
  s.v2 ^= 0xffull;
  sipround(s);
  sipround(s);
  sipround(s);
  sipround(s);
  return s.v0 ^ s.v1 ^ s.v2 ^ s.v3;
}

// length word of a 24-byte message: no tail bytes, length in the top byte
constexpr uint64_t kLenWord = 0x18ull << 56;

// remaining work of one lane once the per-event prefix state is known
__device__ __forceinline__ uint64_t mac_tail_from_w1(Sip s, uint64_t value, uint64_t context_id) {
  absorb(s, value);
  absorb(s, context_id);
  absorb(s, kLenWord);
  return finalise(s);
}
__device__ __forceinline__ uint64_t mac_tail_from_w2(Sip s, uint64_t context_id) {
  absorb(s, context_id);
  absorb(s, kLenWord);
  return finalise(s);
}

}  // namespace wg
