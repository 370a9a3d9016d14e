// warpguard_sip32.cuh — SipHash-2-4 on 32-bit register halves: the device-side MAC of the engine kernels
// (paper_2606_11871_b200/csrc) and of the inline device API (warpguard_device.cuh).
//
// token = SipHash-2-4_key( LE64(site_id) || LE64(continuation) || LE64(context_id) ), 64-bit output
// (R1-R4; formula lost at PAPER.md:164-166 / 244-246, "keyed token" over the return state
// PAPER.md:162, 258).  Three message words + the length word 0x18<<56, c = 2, d = 4: 12 SipRounds.
//
// Why halves: sm_100a has no 64-bit integer ALU.  Written on explicit lo/hi registers the round is exactly
//     4 x (IADD3 + carry IADD3.X / IMAD.X)   8 x LOP3   8 x SHF.L.W   rotate-by-32 = register rename
// = 24 instructions and no MOV / pack traffic (the 64-bit formulation of v1 cost ~40 per round).  Measured
// issue costs on B200 (wg_probe_int_pipe): every ALU-pipe instruction (IADD3, LOP3, SHF) holds the pipe
// for 2 cycles per warp, so the round is 40 cycles per warp per sub-partition: 76.8 int32 ops / SM / clk.
//
// The round is split in its four quarter-steps so that work which does not depend on the next message word
// can be hoisted: a word m enters through v3 only, and quarter A touches (v0, v1) only, so A of the first
// round after an injection can run BEFORE the word is known ("pre-A" states).
#pragma once
#include <cstdint>

namespace wg {

struct Sip32 {
  uint32_t v0l, v0h, v1l, v1h, v2l, v2h, v3l, v3h;
};

// a += b (64-bit) on halves; ptxas picks IADD3 + IADD3.X or IMAD.X for the carry half
__device__ __forceinline__ void add64(uint32_t& al, uint32_t& ah, uint32_t bl, uint32_t bh) {
  asm("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, %3;" : "+r"(al), "+r"(ah) : "r"(bl), "r"(bh));
}

// (l, h) = rotl64((l, h), B), 0 < B < 64, B != 32: two funnel shifts
template <int B>
__device__ __forceinline__ void rotl64(uint32_t& l, uint32_t& h) {
  static_assert(B > 0 && B < 64 && B != 32, "rotate amount");
  const uint32_t ol = l, oh = h;
  if constexpr (B < 32) {
    h = __funnelshift_l(ol, oh, B);  // (oh << B) | (ol >> (32 - B))
    l = __funnelshift_l(oh, ol, B);
  } else {
    h = __funnelshift_l(oh, ol, B - 32);
    l = __funnelshift_l(ol, oh, B - 32);
  }
}

__device__ __forceinline__ void swap32(uint32_t& l, uint32_t& h) {
  const uint32_t t = l;
  l = h;
  h = t;
}

// quarter A: v0 += v1; v1 = rotl(v1,13); v1 ^= v0; v0 = rotl(v0,32)
__device__ __forceinline__ void sip_qA(Sip32& s) {
  add64(s.v0l, s.v0h, s.v1l, s.v1h);
  rotl64<13>(s.v1l, s.v1h);
  s.v1l ^= s.v0l;
  s.v1h ^= s.v0h;
  swap32(s.v0l, s.v0h);
}
// quarter B: v2 += v3; v3 = rotl(v3,16); v3 ^= v2
__device__ __forceinline__ void sip_qB(Sip32& s) {
  add64(s.v2l, s.v2h, s.v3l, s.v3h);
  rotl64<16>(s.v3l, s.v3h);
  s.v3l ^= s.v2l;
  s.v3h ^= s.v2h;
}
// quarter C: v0 += v3; v3 = rotl(v3,21); v3 ^= v0
__device__ __forceinline__ void sip_qC(Sip32& s) {
  add64(s.v0l, s.v0h, s.v3l, s.v3h);
  rotl64<21>(s.v3l, s.v3h);
  s.v3l ^= s.v0l;
  s.v3h ^= s.v0h;
}
// quarter D: v2 += v1; v1 = rotl(v1,17); v1 ^= v2; v2 = rotl(v2,32)
__device__ __forceinline__ void sip_qD(Sip32& s) {
  add64(s.v2l, s.v2h, s.v1l, s.v1h);
  rotl64<17>(s.v1l, s.v1h);
  s.v1l ^= s.v2l;
  s.v1h ^= s.v2h;
  swap32(s.v2l, s.v2h);
}

__device__ __forceinline__ void sip_round(Sip32& s) {
  sip_qA(s);
  sip_qB(s);
  sip_qC(s);
  sip_qD(s);
}

// one message word, c = 2 rounds
__device__ __forceinline__ void sip_absorb(Sip32& s, uint32_t ml, uint32_t mh) {
  s.v3l ^= ml;
  s.v3h ^= mh;
  sip_round(s);
  sip_round(s);
  s.v0l ^= ml;
  s.v0h ^= mh;
}
// the same when quarter A of the first round was already applied to s (a "pre-A" state)
__device__ __forceinline__ void sip_absorb_preA(Sip32& s, uint32_t ml, uint32_t mh) {
  s.v3l ^= ml;
  s.v3h ^= mh;
  sip_qB(s);
  sip_qC(s);
  sip_qD(s);
  sip_round(s);
  s.v0l ^= ml;
  s.v0h ^= mh;
}

// length word of the 24-byte message: 0x18 << 56, i.e. lo = 0, hi = 0x18000000
constexpr uint32_t kLenHi = 0x18000000u;

// absorb the length word, then d = 4 finalisation rounds; the 64-bit output is returned XORed with
// (xl, xh) — pass the stored tag to get 0 exactly when the token matches, or 0 to get the token itself.
// (len_hi: the last message word of a message of whole 8-byte words is its byte length mod 256 in the top byte)
__device__ __forceinline__ void sip_finish_len(Sip32& s, uint32_t len_hi, uint32_t xl, uint32_t xh, uint32_t& outl,
                                               uint32_t& outh);
__device__ __forceinline__ void sip_finish(Sip32& s, uint32_t xl, uint32_t xh, uint32_t& outl, uint32_t& outh) {
  sip_finish_len(s, kLenHi, xl, xh, outl, outh);
}
__device__ __forceinline__ void sip_finish_len(Sip32& s, uint32_t len_hi, uint32_t xl, uint32_t xh, uint32_t& outl,
                                               uint32_t& outh) {
  s.v3h ^= len_hi;
  sip_round(s);
  sip_round(s);
  s.v0h ^= len_hi;
  s.v2l ^= 0xffu;
  sip_round(s);
  sip_round(s);
  sip_round(s);
  sip_round(s);
  outl = s.v0l ^ s.v1l ^ s.v2l ^ s.v3l ^ xl;
  outh = s.v0h ^ s.v1h ^ s.v2h ^ s.v3h ^ xh;
}

// The context word of lane l is (B | l) with B = context_base & ~31 (R2), and B | l == B ^ l.
// per-lane tail when the event's state already covers site and continuation (warp-uniform continuation), has
// quarter A of the next round applied, AND has B already folded into v3 (done once per event): the lane only
// injects its own five bits.
__device__ __forceinline__ void sip_tail_lane(Sip32 s, uint32_t lane, uint32_t bl, uint32_t bh, uint32_t xl,
                                              uint32_t xh, uint32_t& outl, uint32_t& outh) {
  s.v3l ^= lane;
  sip_qB(s);
  sip_qC(s);
  sip_qD(s);
  sip_round(s);
  s.v0l ^= bl ^ lane;
  s.v0h ^= bh;
  sip_finish(s, xl, xh, outl, outh);
}
// per-lane tail from the site's pre-A state (lane-divergent continuation)
__device__ __forceinline__ void sip_tail_val_lane(Sip32 s, uint32_t vl, uint32_t vh, uint32_t lane, uint32_t bl,
                                                  uint32_t bh, uint32_t xl, uint32_t xh, uint32_t& outl,
                                                  uint32_t& outh) {
  sip_absorb_preA(s, vl, vh);
  s.v3l ^= bl ^ lane;
  s.v3h ^= bh;
  sip_round(s);
  sip_round(s);
  s.v0l ^= bl ^ lane;
  s.v0h ^= bh;
  sip_finish(s, xl, xh, outl, outh);
}

// The two tails of the compacted consumer passes (csrc/wg_check.cu): the lane index comes from a work item, so the
// caller hands in the whole context word (cl, ch) = (B ^ lane, B >> 32).
// (1) warp-uniform continuation: s covers site and continuation, has quarter A of the next round applied and B folded
//     into v3, and the caller has XORed the lane's five bits into s.v3l.
__device__ __forceinline__ void sip_tail_ctxlane(Sip32 s, uint32_t cl, uint32_t ch, uint32_t xl, uint32_t xh,
                                                 uint32_t& outl, uint32_t& outh) {
  sip_qB(s);
  sip_qC(s);
  sip_qD(s);
  sip_round(s);
  s.v0l ^= cl;
  s.v0h ^= ch;
  sip_finish(s, xl, xh, outl, outh);
}
// (2) lane-divergent continuation: s is the site's pre-A state.
__device__ __forceinline__ void sip_tail_val_ctx(Sip32 s, uint32_t vl, uint32_t vh, uint32_t cl, uint32_t ch,
                                                 uint32_t xl, uint32_t xh, uint32_t& outl, uint32_t& outh) {
  sip_absorb_preA(s, vl, vh);
  s.v3l ^= cl;
  s.v3h ^= ch;
  sip_round(s);
  sip_round(s);
  s.v0l ^= cl;
  s.v0h ^= ch;
  sip_finish(s, xl, xh, outl, outh);
}

// The same two tails for TWO independent items per thread, interleaved quarter by quarter so that the instruction
// stream offers the scheduler two dependent chains instead of one.
__device__ __forceinline__ void sip_round2(Sip32& a, Sip32& b) {
  sip_qA(a); sip_qA(b);
  sip_qB(a); sip_qB(b);
  sip_qC(a); sip_qC(b);
  sip_qD(a); sip_qD(b);
}
// one message word into two pre-A states (quarter A of the first round already applied)
__device__ __forceinline__ void sip_absorb_preA2(Sip32& a, Sip32& b, uint32_t mal, uint32_t mah, uint32_t mbl, uint32_t mbh) {
  a.v3l ^= mal; a.v3h ^= mah; b.v3l ^= mbl; b.v3h ^= mbh;
  sip_qB(a); sip_qB(b);
  sip_qC(a); sip_qC(b);
  sip_qD(a); sip_qD(b);
  sip_round2(a, b);
  a.v0l ^= mal; a.v0h ^= mah; b.v0l ^= mbl; b.v0h ^= mbh;
}
__device__ __forceinline__ void sip_finish2(Sip32& a, Sip32& b, uint32_t xal, uint32_t xah, uint32_t xbl, uint32_t xbh,
                                            uint32_t& oal, uint32_t& oah, uint32_t& obl, uint32_t& obh) {
  a.v3h ^= kLenHi; b.v3h ^= kLenHi;
  sip_round2(a, b);
  sip_round2(a, b);
  a.v0h ^= kLenHi; b.v0h ^= kLenHi;
  a.v2l ^= 0xffu; b.v2l ^= 0xffu;
  sip_round2(a, b);
  sip_round2(a, b);
  sip_round2(a, b);
  sip_round2(a, b);
  oal = a.v0l ^ a.v1l ^ a.v2l ^ a.v3l ^ xal;
  oah = a.v0h ^ a.v1h ^ a.v2h ^ a.v3h ^ xah;
  obl = b.v0l ^ b.v1l ^ b.v2l ^ b.v3l ^ xbl;
  obh = b.v0h ^ b.v1h ^ b.v2h ^ b.v3h ^ xbh;
}
__device__ __forceinline__ void sip_tail_ctxlane2(Sip32 a, Sip32 b, uint32_t cal, uint32_t cah, uint32_t cbl, uint32_t cbh,
                                                  uint32_t xal, uint32_t xah, uint32_t xbl, uint32_t xbh,
                                                  uint32_t& oal, uint32_t& oah, uint32_t& obl, uint32_t& obh) {
  sip_qB(a); sip_qB(b);
  sip_qC(a); sip_qC(b);
  sip_qD(a); sip_qD(b);
  sip_round2(a, b);
  a.v0l ^= cal; a.v0h ^= cah;
  b.v0l ^= cbl; b.v0h ^= cbh;
  sip_finish2(a, b, xal, xah, xbl, xbh, oal, oah, obl, obh);
}
__device__ __forceinline__ void sip_tail_val_ctx2(Sip32 a, Sip32 b, uint32_t val, uint32_t vah, uint32_t vbl, uint32_t vbh,
                                                  uint32_t cal, uint32_t cah, uint32_t cbl, uint32_t cbh,
                                                  uint32_t xal, uint32_t xah, uint32_t xbl, uint32_t xbh,
                                                  uint32_t& oal, uint32_t& oah, uint32_t& obl, uint32_t& obh) {
  a.v3l ^= val; a.v3h ^= vah; b.v3l ^= vbl; b.v3h ^= vbh;
  sip_qB(a); sip_qB(b);
  sip_qC(a); sip_qC(b);
  sip_qD(a); sip_qD(b);
  sip_round2(a, b);
  a.v0l ^= val; a.v0h ^= vah; b.v0l ^= vbl; b.v0h ^= vbh;
  a.v3l ^= cal; a.v3h ^= cah; b.v3l ^= cbl; b.v3h ^= cbh;
  sip_round2(a, b);
  sip_round2(a, b);
  a.v0l ^= cal; a.v0h ^= cah; b.v0l ^= cbl; b.v0h ^= cbh;
  sip_finish2(a, b, xal, xah, xbl, xbh, oal, oah, obl, obh);
}

// per-lane tail when the event's state already covers site and continuation and has quarter A of the next round
// applied, but the context word (cl, ch) is the lane's own in every bit (shadow stack: the depth is part of it)
__device__ __forceinline__ void sip_tail_ctx(Sip32 s, uint32_t cl, uint32_t ch, uint32_t xl, uint32_t xh,
                                             uint32_t& outl, uint32_t& outh) {
  sip_absorb_preA(s, cl, ch);
  sip_finish(s, xl, xh, outl, outh);
}

}  // namespace wg
