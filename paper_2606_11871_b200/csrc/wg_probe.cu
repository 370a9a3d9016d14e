// wg_probe.cu — register-only integer micro-benchmark.  NOT part of libwarpguard.so: it is built into its own
// libwg_probe.so, which only bench.py loads (measurement helper, no part of the check path).  One C entry point:
//   int wg_probe_int_pipe(int device, int mix, double* ops_per_s, double* ms);   returns a cudaError_t (0 = ok)
//   mix: 0 = IADD3 only, 1 = LOP3 only, 2 = SHF only, 3 = IMAD only, 4 = IMAD.WIDE.U32 only, 5 = ALU:FMA 1:1 (LOP3 +
//        IMAD), 6 = SipRound-shaped ALU mix (IADD3 / LOP3 / SHF, 8:8:8), 7 = IMAD.HI.U32 only, 8 = ALU:FMA 2:1,
//        9 = ALU:FMA 1:1 (SHF + IMAD.HI.U32), 10 = 64-bit-add pairs (counts PAIRS), 11 = the SipRound itself (two
//        independent states per thread, 24 int32 operations per round): the ceiling of any SipHash kernel on this GPU.
// It answers "what can the sm_100a integer pipes issue?" so that the ALU roofline of the MAC kernel has a
// measured denominator beside the one derived from unit counts.  Every chain is a dependent
// sequence of one instruction kind; 8 independent chains per thread and 16 resident warps per SMSP keep the
// pipes full.  `asm volatile` pins the instruction selection (checked with cuobjdump -sass).
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/warpguard_sip32.cuh"

namespace wg {
namespace {

constexpr int kChains = 8;
constexpr int kInner = 64;    // unrolled steps per chain per loop trip
constexpr int kTrips = 512;   // loop trips
constexpr int kThreads = 256;

#define STEP_IADD(x, y) asm volatile("add.u32 %0, %0, %1;" : "+r"(x) : "r"(y))
#define STEP_LOP(x, y) asm volatile("xor.b32 %0, %0, %1;" : "+r"(x) : "r"(y))
#define STEP_SHF(x, y) asm volatile("shf.l.wrap.b32 %0, %0, %1, 13;" : "+r"(x) : "r"(y))
#define STEP_IMAD(x, y) asm volatile("mad.lo.u32 %0, %0, %1, %1;" : "+r"(x) : "r"(y))
#define STEP_IMADHI(x, y) asm volatile("mad.hi.u32 %0, %0, %1, %1;" : "+r"(x) : "r"(y))
#define STEP_IMADX(x, y) asm volatile("{ .reg .b32 t; add.cc.u32 t, %0, %1; madc.lo.u32 %0, %0, 1, %1; }" : "+r"(x) : "r"(y))
#define STEP_WIDE(x64, y) asm volatile("{ .reg .b32 lo, hi; mov.b64 {lo, hi}, %0; mad.wide.u32 %0, lo, %1, %0; }" : "+l"(x64) : "r"(y))

template <int MIX>
__global__ void __launch_bounds__(kThreads) wg_int_probe(uint32_t* sink, uint32_t y) {
  uint32_t x[kChains];
  uint64_t w[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) {
    x[i] = threadIdx.x * 2654435761u + i;
    w[i] = (static_cast<uint64_t>(x[i]) << 32) | blockIdx.x;
  }
  for (int t = 0; t < kTrips; ++t) {
#pragma unroll
    for (int s = 0; s < kInner; ++s) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        // the second operand is the NEIGHBOUR chain's current value: no step can be folded algebraically
        // (x ^ y ^ y, x + y + y -> one IADD3) and every step still has kChains independent instructions in flight
        uint32_t& o = x[(i + 1) % kChains];
        if (MIX == 0) STEP_IADD(x[i], o);
        if (MIX == 1) STEP_LOP(x[i], o);
        if (MIX == 2) STEP_SHF(x[i], o);
        if (MIX == 3) STEP_IMAD(x[i], o);
        if (MIX == 4) STEP_WIDE(w[i], static_cast<uint32_t>(w[(i + 1) % kChains]));
        if (MIX == 5) {  // ALU : FMA = 1 : 1
          if (i & 1) STEP_LOP(x[i], o); else STEP_IMAD(x[i], o);
        }
        if (MIX == 6) {  // SipRound-shaped ALU mix 1 : 1 : 1
          if ((s + i) % 3 == 0) STEP_IADD(x[i], o);
          if ((s + i) % 3 == 1) STEP_LOP(x[i], o);
          if ((s + i) % 3 == 2) STEP_SHF(x[i], o);
        }
        if (MIX == 7) STEP_IMADHI(x[i], o);
        if (MIX == 8) {  // ALU : FMA = 2 : 1
          if ((s + i) % 3 == 0) STEP_IMAD(x[i], o);
          if ((s + i) % 3 == 1) STEP_LOP(x[i], o);
          if ((s + i) % 3 == 2) STEP_SHF(x[i], o);
        }
        if (MIX == 9) {  // ALU : FMA = 1 : 1 with IMAD.HI on the FMA side
          if (i & 1) STEP_SHF(x[i], o); else STEP_IMADHI(x[i], o);
        }
        if (MIX == 10) STEP_IMADX(x[i], o);
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) acc ^= x[i] ^ static_cast<uint32_t>(w[i]) ^ static_cast<uint32_t>(w[i] >> 32);
  if (acc == 0x12345678u) sink[0] = acc;  // practically never; keeps the chains live
}

// mix 11: the SipRound itself (wg_sip32.cuh), two independent states per thread, 16 rounds per loop trip.
// Reported as 24 int32 lane-operations per round (8 add halves, 8 xor halves, 8 funnel shifts): the ceiling
// any SipHash kernel on this GPU can reach, whatever its occupancy.
constexpr int kSipRoundsPerTrip = 16;
constexpr int kSipTrips = 1024;
__global__ void __launch_bounds__(kThreads) wg_sip_probe(uint32_t* sink, uint32_t y) {
  Sip32 s[2];
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const uint32_t x = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + y + i * 977u;
    s[i] = Sip32{x, x ^ 0x1234567u, x * 3u, x * 5u, x * 7u, x * 11u, x * 13u, x * 17u};
  }
  for (int t = 0; t < kSipTrips; ++t) {
#pragma unroll
    for (int r = 0; r < kSipRoundsPerTrip; ++r) {
      sip_round(s[0]);
      sip_round(s[1]);
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int i = 0; i < 2; ++i)
    acc ^= s[i].v0l ^ s[i].v0h ^ s[i].v1l ^ s[i].v1h ^ s[i].v2l ^ s[i].v2h ^ s[i].v3l ^ s[i].v3h;
  if (acc == 0x12345678u) sink[0] = acc;
}

cudaError_t run_sip(int sm_count, uint32_t* sink, double* ops_per_s, double* ms_out) {
  const int grid = sm_count * 4;  // 4 CTAs x 8 warps = 8 warps per sub-partition
  cudaEvent_t a, b;
  cudaError_t err;
  if ((err = cudaEventCreate(&a)) != cudaSuccess) return err;
  if ((err = cudaEventCreate(&b)) != cudaSuccess) return err;
  float best = 1e30f;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(a, nullptr);
    wg_sip_probe<<<grid, kThreads>>>(sink, 0x9e3779b9u + rep);
    cudaEventRecord(b, nullptr);
    if ((err = cudaEventSynchronize(b)) != cudaSuccess) return err;
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  const double rounds = static_cast<double>(grid) * kThreads * 2.0 * kSipRoundsPerTrip * kSipTrips;
  *ops_per_s = rounds * 24.0 / (best * 1e-3);
  *ms_out = best;
  return cudaGetLastError();
}

template <int MIX>
cudaError_t run(int sm_count, uint32_t* sink, double* ops_per_s, double* ms_out) {
  const int grid = sm_count * 8;  // 8 CTAs x 8 warps = 64 warps per SM
  cudaEvent_t a, b;
  cudaError_t err;
  if ((err = cudaEventCreate(&a)) != cudaSuccess) return err;
  if ((err = cudaEventCreate(&b)) != cudaSuccess) return err;
  float best = 1e30f;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(a, nullptr);
    wg_int_probe<MIX><<<grid, kThreads>>>(sink, 0x9e3779b9u + rep);
    cudaEventRecord(b, nullptr);
    if ((err = cudaEventSynchronize(b)) != cudaSuccess) return err;
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  const double ops = static_cast<double>(grid) * kThreads * kChains * kInner * static_cast<double>(kTrips);
  *ops_per_s = ops / (best * 1e-3);
  *ms_out = best;
  return cudaGetLastError();
}

}  // namespace

cudaError_t run_int_pipe_probe(int mix, int sm_count, double* ops_per_s, double* ms) {
  uint32_t* sink = nullptr;
  cudaError_t err = cudaMalloc(&sink, 256);
  if (err != cudaSuccess) return err;
  switch (mix) {
    case 0: err = run<0>(sm_count, sink, ops_per_s, ms); break;
    case 1: err = run<1>(sm_count, sink, ops_per_s, ms); break;
    case 2: err = run<2>(sm_count, sink, ops_per_s, ms); break;
    case 3: err = run<3>(sm_count, sink, ops_per_s, ms); break;
    case 4: err = run<4>(sm_count, sink, ops_per_s, ms); break;
    case 5: err = run<5>(sm_count, sink, ops_per_s, ms); break;
    case 6: err = run<6>(sm_count, sink, ops_per_s, ms); break;
    case 7: err = run<7>(sm_count, sink, ops_per_s, ms); break;
    case 8: err = run<8>(sm_count, sink, ops_per_s, ms); break;
    case 9: err = run<9>(sm_count, sink, ops_per_s, ms); break;
    case 10: err = run<10>(sm_count, sink, ops_per_s, ms); break;
    case 11: err = run_sip(sm_count, sink, ops_per_s, ms); break;
    default: err = cudaErrorInvalidValue;
  }
  cudaFree(sink);
  return err;
}

}  // namespace wg

extern "C" int wg_probe_int_pipe(int device, int mix, double* ops_per_s, double* ms) {
  if (!ops_per_s || !ms || mix < 0 || mix > 11) return static_cast<int>(cudaErrorInvalidValue);
  int prev = 0, sms = 0;
  cudaError_t err;
  if ((err = cudaGetDevice(&prev)) != cudaSuccess) return static_cast<int>(err);
  if ((err = cudaSetDevice(device)) != cudaSuccess) return static_cast<int>(err);
  if ((err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) == cudaSuccess)
    err = wg::run_int_pipe_probe(mix, sms, ops_per_s, ms);
  cudaSetDevice(prev);
  return static_cast<int>(err);
}
