// wg_api.cu — the C-ABI of include/warpguard.h: argument checks, policy validation (a bad
// policy loads nothing), engine-owned device tables, launches, counter read-out, and the HOST-buffer entry
// points that stream events through a double-buffered device staging area.  No verdict, MAC or membership
// arithmetic happens on the host: every step of the path runs in the kernels of wg_check.cu and wg_shadow.cu.
#include <cstring>
#include <new>
#include <vector>

#include "../../include/warpguard.h"
#include "wg_internal.h"

struct wg_engine {
  int device = 0;
  int sm_count = 0;
  bool loaded = false;
  uint32_t n_sites = 0;
  uint64_t n_tgts = 0;
  wg::SiteRec* d_recs = nullptr;  // site records {kind, set range, flags}, 16 B each; nothing key-derived
  uint64_t* d_tok = nullptr;       // [n_sites] forward-record tokens at load time (metadata-integrity profile, R37)
  unsigned int* d_sched = nullptr; // ring of group tickets, one per launch in flight (wg_check.cu)
  uint32_t sched_next = 0;
  uint64_t* d_htab = nullptr;      // hash index of the target sets when the table is too large to stage (wg_check.cu)
  uint32_t bind_hi = 0;            // digest32 folded into the tokens (wg_load_policy_bound), else 0
  bool has_ret = false;            // the policy lists a protected-return site
  uint32_t profile = 0;            // WG_PROFILE_* flags (configuration: survives resets and policy loads)
  uint64_t ring_cap = 0;           // violation ring capacity in records (0 = off)
  wg::ViolRec* d_ring = nullptr;
  wg::FirstRec* d_first = nullptr;  // first-violation record + the key it belongs to
  wg::ShadowState sh = {0, 0, nullptr, nullptr, nullptr, nullptr, 0, {0, 0}};  // stateful shadow stack
  uint64_t launches = 0;          // kernels this engine has enqueued (wg_telemetry_counters.kernel_launches)
  uint64_t* d_tgts = nullptr;
  unsigned long long* d_glob = nullptr;  // [C_WORDS]
  unsigned long long* d_site = nullptr;  // [n_sites][4]
  uint64_t v_init[4] = {0, 0, 0, 0};     // key ^ SipHash constants
  uint64_t digest = 0;
  uint64_t seq = 0;        // running event index over check calls (R12), assigned at call time
  uint64_t last_mode = 0;  // mode of the last non-empty check call
  int last_cuda_error = 0;
  // staging for the *_host entry points (allocated on first use)
  uint64_t stage_cap = 0;  // events per buffer
  void* d_stage[2] = {nullptr, nullptr};
  cudaStream_t st[2] = {nullptr, nullptr};
  cudaEvent_t ev_done[2] = {nullptr, nullptr};
  cudaEvent_t ev_rec = nullptr;  // orders the first-violation-record kernels of consecutive chunks across the two streams
};

namespace {

struct DeviceGuard {
  int prev = -1;
  bool ok = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) return;
    ok = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

wg_status cuda_fail(wg_engine* e, cudaError_t err) {
  if (e) e->last_cuda_error = static_cast<int>(err);
  cudaGetLastError();  // clear the sticky-free error state
  return err == cudaErrorMemoryAllocation ? WG_ERR_OOM : WG_ERR_CUDA;
}

#define WG_CUDA(e, call)                                  \
  do {                                                    \
    cudaError_t err__ = (call);                           \
    if (err__ != cudaSuccess) return cuda_fail(e, err__); \
  } while (0)

bool aligned(const void* p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

// R16: everything that would widen or blur an allowed set is rejected before any state is touched.
bool policy_ok(const wg_policy_desc* d) {
  const uint32_t n = d->n_sites;
  if (d->tgt_off[0] != 0) return false;
  for (uint32_t s = 0; s < n; ++s) {
    if (d->kind[s] >= WG_KIND_COUNT) return false;
    const uint32_t a = d->tgt_off[s], b = d->tgt_off[s + 1];
    if (b < a) return false;
    const bool fwd = d->kind[s] == WG_KIND_PROTECTED_FORWARD;
    if (fwd && a == b) return false;   // no target evidence: must have been labelled unsupported
    if (!fwd && a != b) return false;  // a set nobody may consult
    if (a != b && d->tgts == nullptr) return false;
    for (uint32_t i = a + 1; i < b; ++i)
      if (!(d->tgts[i - 1] < d->tgts[i])) return false;  // strictly ascending: sorted, no duplicates
  }
  return true;
}

void free_tables(wg_engine* e) {
  cudaFree(e->d_recs);
  e->d_recs = nullptr;
  cudaFree(e->d_tok);
  e->d_tok = nullptr;
  cudaFree(e->d_htab);
  e->d_htab = nullptr;
  cudaFree(e->d_sched);
  e->d_sched = nullptr;
  cudaFree(e->d_tgts);
  cudaFree(e->d_glob);
  cudaFree(e->d_site);
  e->d_tgts = nullptr;
  e->d_glob = nullptr;
  e->d_site = nullptr;
  e->loaded = false;
}

void free_shadow(wg_engine* e) {
  cudaFree(e->sh.depth_ctr);
  cudaFree(e->sh.entry);
  cudaFree(e->sh.uses);
  cudaFree(e->sh.counters);
  e->sh = wg::ShadowState{0, 0, nullptr, nullptr, nullptr, nullptr, 0, {0, 0}};
}

void free_staging(wg_engine* e) {
  for (int i = 0; i < 2; ++i) {
    if (e->d_stage[i]) cudaFree(e->d_stage[i]);
    if (e->st[i]) cudaStreamDestroy(e->st[i]);
    if (e->ev_done[i]) cudaEventDestroy(e->ev_done[i]);
    e->d_stage[i] = nullptr;
    e->st[i] = nullptr;
    e->ev_done[i] = nullptr;
  }
  if (e->ev_rec) cudaEventDestroy(e->ev_rec);
  e->ev_rec = nullptr;
  e->stage_cap = 0;
}

wg_status zero_counters(wg_engine* e, cudaStream_t st) {
  WG_CUDA(e, cudaMemsetAsync(e->d_glob, 0, sizeof(unsigned long long) * wg::C_WORDS, st));
  WG_CUDA(e, cudaMemsetAsync(e->d_glob + wg::C_FIRST_VIOLATION, 0xff, sizeof(unsigned long long), st));
  if (e->n_sites)
    WG_CUDA(e, cudaMemsetAsync(e->d_site, 0, sizeof(unsigned long long) * 4 * e->n_sites, st));
  if (e->d_first) {
    WG_CUDA(e, cudaMemsetAsync(e->d_first, 0, sizeof(wg::FirstRec), st));
    WG_CUDA(e, cudaMemsetAsync(&e->d_first->key, 0xff, sizeof(unsigned long long), st));
  }
  e->seq = 0;
  e->last_mode = 0;
  return WG_OK;
}

wg::Params base_params(const wg_engine* e) {
  wg::Params p;
  std::memset(&p, 0, sizeof(p));
  p.recs = e->d_recs;
  p.tok = e->d_tok;
  p.htab = e->d_htab;
  p.sched = e->d_sched;  // (the check / sign launch sites pick the ring slot)
  p.n_tgts = e->n_tgts;
  p.profile = e->profile;
  p.bind_hi = e->bind_hi;
  p.has_ret = e->has_ret ? 1u : 0u;
  p.ring = e->d_ring;
  p.ring_cap = e->d_ring ? e->ring_cap : 0;
  p.first = e->d_first;
  p.tgts = e->d_tgts;
  p.glob = e->d_glob;
  p.site = e->d_site;
  p.n_sites = e->n_sites;
  p.v0 = e->v_init[0];
  p.v1 = e->v_init[1];
  p.v2 = e->v_init[2];
  p.v3 = e->v_init[3];
  return p;
}

// element indices event * 32 + lane stay below 2^32 inside a launch, and so does every 32-bit lane count a warp or a CTA
// keeps (at most 32 lanes per event): strictly fewer than 2^27 events
constexpr uint64_t kMaxLaunchEvents = (1ull << 27) - 32;

// rec_after: an event the first-violation-record kernel waits for (host path: the record kernel of the previous chunk,
// which ran on the other staging stream), or nullptr
wg_status check_common(wg_engine* e, const wg_event_hdr* d_hdr, const uint64_t* d_val, const uint64_t* d_tag,
                       bool has_tag, wg_verdict* d_out, uint64_t n, wg_mode mode, cudaStream_t st,
                       cudaEvent_t rec_after = nullptr) {
  if (!e || !e->loaded) return WG_ERR_NO_POLICY;
  if (mode != WG_MODE_DETECT && mode != WG_MODE_ENFORCE) return WG_ERR_INVALID_ARG;
  if (n == 0) return WG_OK;  // R24: nothing changes
  if (!d_hdr || !d_val || !d_out || (has_tag && !d_tag)) return WG_ERR_INVALID_ARG;
  if (!aligned(d_hdr, 16) || !aligned(d_val, 16) || !aligned(d_out, 8) || (has_tag && !aligned(d_tag, 16)))
    return WG_ERR_INVALID_ARG;
  if (n > (1ull << 58)) return WG_ERR_INVALID_ARG;  // (seq << 5) must not wrap
  DeviceGuard g(e->device);
  if (!g.ok) return cuda_fail(e, cudaErrorInvalidDevice);
  // one launch covers at most kMaxLaunchEvents events: the kernels keep per-warp counters in 32-bit registers
  for (uint64_t lo = 0; lo < n; lo += kMaxLaunchEvents) {
    const uint64_t m = (n - lo < kMaxLaunchEvents) ? (n - lo) : kMaxLaunchEvents;
    wg::Params p = base_params(e);
    p.hdr = reinterpret_cast<const uint4*>(d_hdr + lo);
    p.val = d_val + lo * 32;
    p.tag = has_tag ? d_tag + lo * 32 : nullptr;
    p.out = reinterpret_cast<uint2*>(d_out + lo);
    p.n = m;
    p.seq_base = e->seq;
    p.mode = static_cast<uint32_t>(mode);
    p.sched = e->d_sched + (e->sched_next++ % wg::kSchedSlots) * 16;  // (64 bytes apart)
    WG_CUDA(e, wg::launch_check(p, e->sm_count, st, &e->launches));
    // first-violation record (R29): one thread behind the check launch; the launch is over, so the key is final for it
    if (rec_after) WG_CUDA(e, cudaStreamWaitEvent(st, rec_after, 0));
    WG_CUDA(e, wg::launch_first_record(p, st, &e->launches));
    e->seq += m;
  }
  e->last_mode = static_cast<uint64_t>(mode);
  return WG_OK;
}

wg_status sign_common(wg_engine* e, const wg_event_hdr* d_hdr, const uint64_t* d_val, uint64_t* d_tag,
                      uint64_t n, cudaStream_t st) {
  if (!e || !e->loaded) return WG_ERR_NO_POLICY;
  if (n == 0) return WG_OK;
  if (!d_hdr || !d_val || !d_tag) return WG_ERR_INVALID_ARG;
  if (!aligned(d_hdr, 16) || !aligned(d_val, 16) || !aligned(d_tag, 16)) return WG_ERR_INVALID_ARG;
  DeviceGuard g(e->device);
  if (!g.ok) return cuda_fail(e, cudaErrorInvalidDevice);
  for (uint64_t lo = 0; lo < n; lo += kMaxLaunchEvents) {
    const uint64_t m = (n - lo < kMaxLaunchEvents) ? (n - lo) : kMaxLaunchEvents;
    wg::Params p = base_params(e);
    p.hdr = reinterpret_cast<const uint4*>(d_hdr + lo);
    p.val = d_val + lo * 32;
    p.tag_out = d_tag + lo * 32;
    p.n = m;
    p.sched = e->d_sched + (e->sched_next++ % wg::kSchedSlots) * 16;
    WG_CUDA(e, wg::launch_sign(p, e->sm_count, st, &e->launches));
  }
  return WG_OK;
}

// ---- host-buffer streaming -------------------------------------------------------------------------
constexpr uint64_t kStageEvents = 1ull << 18;  // 256 Ki events per buffer: 4 MiB hdr + 64 MiB val + 64 MiB tag + 2 MiB out
constexpr uint64_t kBytesPerStagedEvent = 16 + 256 + 256 + 8;

wg_status ensure_staging(wg_engine* e) {
  if (e->stage_cap) return WG_OK;
  cudaError_t err = cudaSuccess;
  for (int i = 0; i < 2 && err == cudaSuccess; ++i) {
    if ((err = cudaMalloc(&e->d_stage[i], kStageEvents * kBytesPerStagedEvent)) != cudaSuccess) break;
    if ((err = cudaStreamCreateWithFlags(&e->st[i], cudaStreamNonBlocking)) != cudaSuccess) break;
    err = cudaEventCreateWithFlags(&e->ev_done[i], cudaEventDisableTiming);
  }
  if (err == cudaSuccess) err = cudaEventCreateWithFlags(&e->ev_rec, cudaEventDisableTiming);
  if (err != cudaSuccess) {
    free_staging(e);  // all or nothing: a half-built staging area is not kept (the next call starts over)
    return cuda_fail(e, err);
  }
  e->stage_cap = kStageEvents;
  return WG_OK;
}

struct StageView {
  wg_event_hdr* hdr;
  uint64_t* val;
  uint64_t* tag;
  wg_verdict* out;
};
StageView stage_view(void* base) {
  char* b = static_cast<char*>(base);
  StageView v;
  v.hdr = reinterpret_cast<wg_event_hdr*>(b);
  v.val = reinterpret_cast<uint64_t*>(b + kStageEvents * 16);
  v.tag = reinterpret_cast<uint64_t*>(b + kStageEvents * (16 + 256));
  v.out = reinterpret_cast<wg_verdict*>(b + kStageEvents * (16 + 256 + 256));
  return v;
}

enum HostOp { OP_SIGN, OP_VERIFY, OP_FORWARD };

wg_status host_common(wg_engine* e, HostOp op, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                      const uint64_t* h_tag_in, uint64_t* h_tag_out, wg_verdict* h_out, uint64_t n, wg_mode mode) {
  if (!e || !e->loaded) return WG_ERR_NO_POLICY;
  if (op != OP_SIGN && mode != WG_MODE_DETECT && mode != WG_MODE_ENFORCE) return WG_ERR_INVALID_ARG;
  if (n == 0) return WG_OK;
  if (!h_hdr || !h_val) return WG_ERR_INVALID_ARG;
  if (op == OP_SIGN && !h_tag_out) return WG_ERR_INVALID_ARG;
  if (op == OP_VERIFY && !h_tag_in) return WG_ERR_INVALID_ARG;
  if (op != OP_SIGN && !h_out) return WG_ERR_INVALID_ARG;
  DeviceGuard g(e->device);
  if (!g.ok) return cuda_fail(e, cudaErrorInvalidDevice);
  wg_status s = ensure_staging(e);
  if (s != WG_OK) return s;

  // The chunks alternate between two staging streams, so two check kernels may overlap.  Their first-violation-record
  // kernels must not: each one waits (ev_rec) for the record kernel of the chunk before it, so the records are written
  // in chunk order by one kernel at a time, and the last writer is the chunk that holds the final minimum key.
  int buf = 0;
  bool rec_pending = false;
  auto chunk = [&](uint64_t lo, cudaStream_t st, const StageView& v) -> wg_status {
    const uint64_t m = (n - lo < kStageEvents) ? (n - lo) : kStageEvents;
    // the previous use of this buffer (two chunks ago) finished when its stream's D2H did: same stream, in order
    WG_CUDA(e, cudaMemcpyAsync(v.hdr, h_hdr + lo, m * 16, cudaMemcpyHostToDevice, st));
    WG_CUDA(e, cudaMemcpyAsync(v.val, h_val + lo * 32, m * 256, cudaMemcpyHostToDevice, st));
    if (op == OP_VERIFY)
      WG_CUDA(e, cudaMemcpyAsync(v.tag, h_tag_in + lo * 32, m * 256, cudaMemcpyHostToDevice, st));
    if (op == OP_SIGN) {
      const wg_status s2 = sign_common(e, v.hdr, v.val, v.tag, m, st);
      if (s2 != WG_OK) return s2;
      WG_CUDA(e, cudaMemcpyAsync(h_tag_out + lo * 32, v.tag, m * 256, cudaMemcpyDeviceToHost, st));
    } else {
      const wg_status s2 = check_common(e, v.hdr, v.val, v.tag, op == OP_VERIFY, v.out, m, mode, st, rec_pending ? e->ev_rec : nullptr);
      if (s2 != WG_OK) return s2;
      WG_CUDA(e, cudaEventRecord(e->ev_rec, st));
      rec_pending = true;
      WG_CUDA(e, cudaMemcpyAsync(h_out + lo, v.out, m * 8, cudaMemcpyDeviceToHost, st));
    }
    return WG_OK;
  };
  for (uint64_t lo = 0; lo < n && s == WG_OK; lo += kStageEvents, buf ^= 1) s = chunk(lo, e->st[buf], stage_view(e->d_stage[buf]));
  // whatever happened, nothing of this call may still be copying from or into the caller's host buffers on return
  const cudaError_t e0 = cudaStreamSynchronize(e->st[0]), e1 = cudaStreamSynchronize(e->st[1]);
  if (s != WG_OK) return s;
  if (e0 != cudaSuccess) return cuda_fail(e, e0);
  if (e1 != cudaSuccess) return cuda_fail(e, e1);
  return WG_OK;
}

}  // namespace

extern "C" {

// SipHash-2-4 on the host, for the load-time digest of a policy image only (no check runs on the host)
static uint64_t host_siphash24(uint64_t k0, uint64_t k1, const std::vector<uint8_t>& m) {
  auto rotl = [](uint64_t x, int b) { return (x << b) | (x >> (64 - b)); };
  uint64_t v0 = k0 ^ 0x736f6d6570736575ull, v1 = k1 ^ 0x646f72616e646f6dull;
  uint64_t v2 = k0 ^ 0x6c7967656e657261ull, v3 = k1 ^ 0x7465646279746573ull;
  auto round = [&]() {
    v0 += v1; v1 = rotl(v1, 13); v1 ^= v0; v0 = rotl(v0, 32);
    v2 += v3; v3 = rotl(v3, 16); v3 ^= v2;
    v0 += v3; v3 = rotl(v3, 21); v3 ^= v0;
    v2 += v1; v1 = rotl(v1, 17); v1 ^= v2; v2 = rotl(v2, 32);
  };
  const size_t n = m.size(), full = n / 8;
  for (size_t i = 0; i < full; ++i) {
    uint64_t w = 0;
    for (int j = 0; j < 8; ++j) w |= static_cast<uint64_t>(m[8 * i + j]) << (8 * j);
    v3 ^= w; round(); round(); v0 ^= w;
  }
  uint64_t last = static_cast<uint64_t>(n & 0xff) << 56;
  for (size_t j = 0; j < n % 8; ++j) last |= static_cast<uint64_t>(m[8 * full + j]) << (8 * j);
  v3 ^= last; round(); round(); v0 ^= last;
  v2 ^= 0xff; round(); round(); round(); round();
  return v0 ^ v1 ^ v2 ^ v3;
}

static wg_status load_common(wg_engine** eng, int device, const wg_policy_desc* desc, uint32_t bind_hi);

wg_status wg_policy_digest(const wg_policy_desc* desc, uint64_t* h_digest) {
  if (!desc || !h_digest || !desc->tgt_off || (desc->n_sites && !desc->kind)) return WG_ERR_INVALID_ARG;
  if (!policy_ok(desc)) return WG_ERR_BAD_POLICY;
  const uint32_t n = desc->n_sites;
  const uint64_t nt = desc->tgt_off[n];
  std::vector<uint8_t> m;
  try {
    m.reserve(16 + n + 8 + 4 * (static_cast<size_t>(n) + 1) + 8 + 8 * nt);
  } catch (const std::bad_alloc&) {
    return WG_ERR_OOM;
  }
  auto put64 = [&m](uint64_t w) {
    for (int i = 0; i < 8; ++i) m.push_back(static_cast<uint8_t>(w >> (8 * i)));
  };
  put64(n);
  put64(nt);
  for (uint32_t s = 0; s < n; ++s) m.push_back(desc->kind[s]);
  while (m.size() % 8) m.push_back(0);
  for (uint32_t s = 0; s <= n; ++s)
    for (int i = 0; i < 4; ++i) m.push_back(static_cast<uint8_t>(desc->tgt_off[s] >> (8 * i)));
  while (m.size() % 8) m.push_back(0);
  for (uint64_t i = 0; i < nt; ++i) put64(desc->tgts[i]);
  *h_digest = host_siphash24(desc->key[0], desc->key[1], m);
  return WG_OK;
}

wg_status wg_load_policy(wg_engine** eng, int device, const wg_policy_desc* desc) {
  return load_common(eng, device, desc, 0u);
}

wg_status wg_load_policy_bound(wg_engine** eng, int device, const wg_policy_desc* desc) {
  uint64_t d = 0;
  const wg_status s = wg_policy_digest(desc, &d);
  if (s != WG_OK) return s;
  if (d != desc->policy_digest) return WG_ERR_BAD_POLICY;  // "a mismatch aborts before the policy is used"
  return load_common(eng, device, desc, static_cast<uint32_t>(d));
}

static wg_status load_common(wg_engine** eng, int device, const wg_policy_desc* desc, uint32_t bind_hi) {
  if (!eng || !desc) return WG_ERR_INVALID_ARG;
  if (desc->n_sites && (!desc->kind || !desc->tgt_off)) return WG_ERR_INVALID_ARG;
  if (!desc->tgt_off) return WG_ERR_INVALID_ARG;
  if (!policy_ok(desc)) return WG_ERR_BAD_POLICY;  // before any state is touched

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return WG_ERR_CUDA;  // no CPU fallback
  }
  if (device < 0 || device >= ndev) return WG_ERR_INVALID_ARG;
  DeviceGuard g(device);
  if (!g.ok) return WG_ERR_CUDA;

  const uint32_t n = desc->n_sites;
  const uint64_t nt = desc->tgt_off[n];
  // build the new tables completely (in `tmp`, on the new device) before anything of an existing engine is replaced:
  // whatever fails below leaves *eng exactly as it was, and leaks nothing
  std::vector<wg::SiteRec> recs;
  try {
    recs.resize(n);
  } catch (const std::bad_alloc&) {
    return WG_ERR_OOM;
  }
  for (uint32_t s = 0; s < n; ++s) {
    recs[s].kind = desc->kind[s];
    recs[s].off = desc->tgt_off[s];
    recs[s].cnt = desc->tgt_off[s + 1] - desc->tgt_off[s];
    recs[s].flags = 0;
    for (uint32_t i = desc->tgt_off[s]; i < desc->tgt_off[s + 1]; ++i)
      if (desc->tgts[i] == ~0ull) recs[s].flags |= wg::SITE_FLAG_HAS_ALLONES;
  }
  wg_engine tmp;
  tmp.device = device;
  tmp.n_sites = n;
  tmp.n_tgts = nt;
  // SipHash initialisation: key xor the constant "somepseudorandomlygeneratedbytes" (R1, R20).  Kept host-side and
  // handed to the kernels as parameters (constant bank): the key never sits in device global memory.
  tmp.v_init[0] = desc->key[0] ^ 0x736f6d6570736575ull;
  tmp.v_init[1] = desc->key[1] ^ 0x646f72616e646f6dull;
  tmp.v_init[2] = desc->key[0] ^ 0x6c7967656e657261ull;
  tmp.v_init[3] = desc->key[1] ^ 0x7465646279746573ull;
  wg::FirstRec* new_first = nullptr;
  cudaError_t err = cudaSuccess;
  auto fail = [&](cudaError_t e2) {
    free_tables(&tmp);
    cudaFree(new_first);
    return cuda_fail(*eng, e2);  // (records the code in an existing engine; a first load has nowhere to record it)
  };
  if ((err = cudaDeviceGetAttribute(&tmp.sm_count, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess)
    return fail(err);
  // the target table is padded to an even element count so that the TMA bulk copy that stages it moves whole
  // 16-byte units; the pad element is never addressed by a search
  const uint64_t nt_pad = (nt + 1) & ~1ull;
  if ((err = cudaMalloc(&tmp.d_tgts, sizeof(uint64_t) * (nt_pad ? nt_pad : 2))) != cudaSuccess) return fail(err);
  if ((err = cudaMemset(tmp.d_tgts, 0, sizeof(uint64_t) * (nt_pad ? nt_pad : 2))) != cudaSuccess) return fail(err);
  if ((err = cudaMalloc(&tmp.d_recs, sizeof(wg::SiteRec) * (n ? n : 1))) != cudaSuccess) return fail(err);
  if ((err = cudaMalloc(&tmp.d_tok, sizeof(uint64_t) * (n ? n : 1))) != cudaSuccess) return fail(err);
  if ((err = cudaMalloc(&tmp.d_sched, wg::kSchedSlots * 64)) != cudaSuccess) return fail(err);
  if ((err = wg::init_kernels()) != cudaSuccess) return fail(err);
  if ((err = cudaMalloc(&tmp.d_glob, sizeof(unsigned long long) * wg::C_WORDS)) != cudaSuccess) return fail(err);
  if ((err = cudaMalloc(&tmp.d_site, sizeof(unsigned long long) * 4 * (n ? n : 1))) != cudaSuccess) return fail(err);
  if (n && (err = cudaMemcpy(tmp.d_recs, recs.data(), sizeof(wg::SiteRec) * n, cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(err);
  if (nt && (err = cudaMemcpy(tmp.d_tgts, desc->tgts, sizeof(uint64_t) * nt, cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(err);
  // large policies: the hash index of the target sets (one 32-byte load per membership test instead of a binary search)
  if (nt > wg::max_staged_targets()) {
    const size_t slots = 2 * static_cast<size_t>(nt) + 4 * static_cast<size_t>(n);
    if ((err = cudaMalloc(&tmp.d_htab, slots * 8)) != cudaSuccess) return fail(err);
    if ((err = cudaMemset(tmp.d_htab, 0xff, slots * 8)) != cudaSuccess) return fail(err);
    if ((err = wg::launch_build_hash(tmp.d_htab, tmp.d_recs, tmp.d_tgts, n, nt, nullptr, &tmp.launches)) != cudaSuccess)
      return fail(err);
  }
  // tokens of the forward records, computed on the device at (trusted) load time (R37)
  if ((err = wg::launch_build_tokens(tmp.d_tok, tmp.d_recs, tmp.d_tgts, n, tmp.v_init[0], tmp.v_init[1], tmp.v_init[2],
                                     tmp.v_init[3], nullptr, &tmp.launches)) != cudaSuccess)
    return fail(err);
  if ((err = cudaStreamSynchronize(nullptr)) != cudaSuccess) return fail(err);
  wg_engine* e = *eng;
  const bool moved = e && e->device != device;
  if (!e || moved || !e->d_first) {
    if ((err = cudaMalloc(&new_first, sizeof(wg::FirstRec))) != cudaSuccess) return fail(err);
  }
  if (!e) {
    e = new (std::nothrow) wg_engine();
    if (!e) {
      free_tables(&tmp);
      cudaFree(new_first);
      return WG_ERR_OOM;
    }
  } else {
    DeviceGuard g2(e->device);
    cudaDeviceSynchronize();  // nothing may still be reading the tables we are about to drop
    free_tables(e);
    if (moved) {
      // everything else the engine owns lives on the OLD device: staging, first-violation record, ring (its capacity is
      // configuration and is re-created empty on the new device below), shadow state (dropped: wg_shadow_configure again)
      free_staging(e);
      cudaFree(e->d_first);
      e->d_first = nullptr;
      cudaFree(e->d_ring);
      e->d_ring = nullptr;
      free_shadow(e);
    }
  }
  e->device = device;
  e->sm_count = tmp.sm_count;
  e->n_sites = n;
  e->n_tgts = nt;
  e->d_recs = tmp.d_recs;
  e->d_tok = tmp.d_tok;
  e->d_htab = tmp.d_htab;
  e->d_sched = tmp.d_sched;
  e->d_tgts = tmp.d_tgts;
  e->d_glob = tmp.d_glob;
  e->d_site = tmp.d_site;
  e->launches += tmp.launches;
  for (int i = 0; i < 4; ++i) e->v_init[i] = tmp.v_init[i];
  e->digest = desc->policy_digest;
  e->bind_hi = bind_hi;
  e->has_ret = false;
  for (uint32_t s2 = 0; s2 < n; ++s2) e->has_ret = e->has_ret || desc->kind[s2] == WG_KIND_PROTECTED_RETURN;
  if (new_first) e->d_first = new_first;
  e->loaded = true;
  *eng = e;
  if (moved && e->ring_cap) {
    cudaError_t e5 = cudaMalloc(&e->d_ring, sizeof(wg::ViolRec) * e->ring_cap);
    if (e5 != cudaSuccess) {
      e->ring_cap = 0;  // the ring is diagnostic: the policy is loaded, the ring is off
      e->d_ring = nullptr;
      cuda_fail(e, e5);
    }
  }
  wg_status s = zero_counters(e, nullptr);
  if (s != WG_OK) return s;
  WG_CUDA(e, cudaStreamSynchronize(nullptr));
  return WG_OK;
}

wg_status wg_sign_continuations(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                uint64_t* d_tag, uint64_t n, void* cuda_stream) {
  return sign_common(eng, d_hdr, d_val, d_tag, n, static_cast<cudaStream_t>(cuda_stream));
}

wg_status wg_verify_continuations(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                  const uint64_t* d_tag, wg_verdict* d_out, uint64_t n, wg_mode mode,
                                  void* cuda_stream) {
  return check_common(eng, d_hdr, d_val, d_tag, true, d_out, n, mode, static_cast<cudaStream_t>(cuda_stream));
}

wg_status wg_check_forward(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val, wg_verdict* d_out,
                           uint64_t n, wg_mode mode, void* cuda_stream) {
  return check_common(eng, d_hdr, d_val, nullptr, false, d_out, n, mode, static_cast<cudaStream_t>(cuda_stream));
}

wg_status wg_read_counters(wg_engine* eng, wg_counters* h_global, wg_site_counters* h_per_site,
                           void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (!h_global) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WG_CUDA(eng, cudaStreamSynchronize(st));
  static_assert(sizeof(wg_counters) == 26 * 8, "wg_counters layout");
  WG_CUDA(eng, cudaMemcpy(h_global, eng->d_glob, sizeof(wg_counters), cudaMemcpyDeviceToHost));
  h_global->policy_digest = eng->digest;
  h_global->last_mode = eng->last_mode;
  if (h_per_site && eng->n_sites)
    WG_CUDA(eng, cudaMemcpy(h_per_site, eng->d_site, sizeof(wg_site_counters) * eng->n_sites,
                            cudaMemcpyDeviceToHost));
  return WG_OK;
}

wg_status wg_reset_counters(wg_engine* eng, void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  // synchronous: the *_host calls run on the engine's own staging streams, which are not ordered after work the
  // caller enqueued on `cuda_stream`; when this returns the counters are zero for every later call, whatever its stream
  const wg_status s = zero_counters(eng, static_cast<cudaStream_t>(cuda_stream));
  if (s != WG_OK) return s;
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  return WG_OK;
}

void wg_destroy(wg_engine* eng) {
  if (!eng) return;
  {
    DeviceGuard g(eng->device);
    if (g.ok) {
      cudaDeviceSynchronize();
      free_staging(eng);
      free_tables(eng);
      cudaFree(eng->d_ring);
      cudaFree(eng->d_first);
      free_shadow(eng);
    }
  }
  delete eng;
}

const char* wg_strerror(wg_status s) {
  switch (s) {
    case WG_OK: return "ok";
    case WG_ERR_INVALID_ARG: return "invalid argument";
    case WG_ERR_BAD_POLICY: return "policy rejected; nothing loaded";
    case WG_ERR_NO_POLICY: return "no policy loaded";
    case WG_ERR_CUDA: return "CUDA runtime error (no device or call failed)";
    case WG_ERR_OOM: return "out of memory";
    case WG_ERR_INTERNAL: return "engine invariant violated";
    case WG_ERR_STATIC_LIMIT: return "beyond the limits of the allocation-free entry point (WG_STATIC_MAX_SITES / WG_STATIC_MAX_EVENTS)";
  }
  return "unknown status";
}

int wg_last_cuda_error(const wg_engine* eng) { return eng ? eng->last_cuda_error : 0; }

// ---- stateful shadow stack (wg_shadow.cu) ----------------------------------------------------------
wg_status wg_shadow_configure(wg_engine* eng, uint32_t n_warp_slots, uint32_t max_depth, void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (max_depth == 0 || max_depth > 64) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WG_CUDA(eng, cudaStreamSynchronize(st));
  free_shadow(eng);
  wg::ShadowState sh = {n_warp_slots, max_depth, nullptr, nullptr, nullptr, nullptr, 0, {0, 0}};
  WG_CUDA(eng, wg::shadow_occupancy(&sh.per_sm[1], &sh.per_sm[0]));  // resolved once per configuration, on this device
  const size_t lanes = static_cast<size_t>(n_warp_slots ? n_warp_slots : 1) * 32;
  const size_t entries = lanes * max_depth;
  cudaError_t err;
  if ((err = cudaMalloc(&sh.depth_ctr, lanes * 4)) != cudaSuccess || (err = cudaMalloc(&sh.entry, entries * 32)) != cudaSuccess ||
      (err = cudaMalloc(&sh.uses, lanes / 32 * 8)) != cudaSuccess || (err = cudaMalloc(&sh.counters, 16 * 8)) != cudaSuccess) {
    eng->sh = sh;
    free_shadow(eng);
    return cuda_fail(eng, err);
  }
  eng->sh = sh;
  WG_CUDA(eng, cudaMemsetAsync(sh.depth_ctr, 0, lanes * 4, st));
  WG_CUDA(eng, cudaMemsetAsync(sh.entry, 0, entries * 32, st));
  WG_CUDA(eng, cudaMemsetAsync(sh.uses, 0, lanes / 32 * 8, st));
  WG_CUDA(eng, cudaMemsetAsync(sh.counters, 0, 16 * 8, st));
  WG_CUDA(eng, cudaStreamSynchronize(st));
  return WG_OK;
}

static wg_status shadow_common(wg_engine* e, bool push, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                               wg_verdict* d_out, uint64_t n, wg_mode mode, void* cuda_stream) {
  if (!e || !e->loaded || !e->sh.counters) return WG_ERR_NO_POLICY;
  if (mode != WG_MODE_DETECT && mode != WG_MODE_ENFORCE) return WG_ERR_INVALID_ARG;
  if (n == 0) return WG_OK;
  if (!d_hdr || !d_val || !d_out || n > (1ull << 31)) return WG_ERR_INVALID_ARG;
  if (!aligned(d_hdr, 16) || !aligned(d_val, 16) || !aligned(d_out, 8)) return WG_ERR_INVALID_ARG;
  DeviceGuard g(e->device);
  if (!g.ok) return cuda_fail(e, cudaErrorInvalidDevice);
  wg::Params p = base_params(e);
  p.hdr = reinterpret_cast<const uint4*>(d_hdr);
  p.val = d_val;
  p.out = reinterpret_cast<uint2*>(d_out);
  p.n = n;
  p.mode = static_cast<uint32_t>(mode);
  if (++e->sh.stamp == 0) {  // 2^32 calls later the stamps start over
    WG_CUDA(e, cudaMemsetAsync(e->sh.uses, 0, static_cast<size_t>(e->sh.n_slots ? e->sh.n_slots : 1) * 8,
                               static_cast<cudaStream_t>(cuda_stream)));
    e->sh.stamp = 1;
  }
  WG_CUDA(e, wg::launch_shadow(p, e->sh, push, e->sm_count, static_cast<cudaStream_t>(cuda_stream), &e->launches));
  return WG_OK;
}

wg_status wg_shadow_push(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val, wg_verdict* d_out,
                         uint64_t n, wg_mode mode, void* cuda_stream) {
  return shadow_common(eng, true, d_hdr, d_val, d_out, n, mode, cuda_stream);
}

wg_status wg_shadow_check_ret(wg_engine* eng, const wg_event_hdr* d_hdr, const uint64_t* d_val, wg_verdict* d_out,
                              uint64_t n, wg_mode mode, void* cuda_stream) {
  return shadow_common(eng, false, d_hdr, d_val, d_out, n, mode, cuda_stream);
}

wg_status wg_shadow_read_counters(wg_engine* eng, wg_shadow_counters* h_out, void* cuda_stream) {
  if (!eng || !eng->loaded || !eng->sh.counters) return WG_ERR_NO_POLICY;
  if (!h_out) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  static_assert(sizeof(wg_shadow_counters) == 16 * 8, "wg_shadow_counters layout");
  WG_CUDA(eng, cudaMemcpy(h_out, eng->sh.counters, sizeof(wg_shadow_counters), cudaMemcpyDeviceToHost));
  return WG_OK;
}

wg_status wg_shadow_poke(wg_engine* eng, uint32_t warp_slot, uint32_t lane, uint32_t entry_depth, int field,
                         uint64_t xor_value, void* cuda_stream) {
  if (!eng || !eng->loaded || !eng->sh.counters) return WG_ERR_NO_POLICY;
  if (warp_slot >= eng->sh.n_slots || lane >= 32 || field < 0 || field > 4) return WG_ERR_INVALID_ARG;
  if (field != 4 && entry_depth >= eng->sh.max_depth) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  const size_t li = static_cast<size_t>(warp_slot) * 32 + lane;
  const size_t ei = ((static_cast<size_t>(warp_slot) * eng->sh.max_depth + entry_depth) * 32 + lane) * 4;  // the entry's sector
  void* addr = nullptr;
  size_t bytes = 8;
  switch (field) {
    case 0: addr = eng->sh.entry + ei; break;
    case 1: addr = eng->sh.entry + ei + 1; break;
    case 2: addr = reinterpret_cast<uint32_t*>(eng->sh.entry + ei + 2); bytes = 4; break;
    case 3: addr = reinterpret_cast<uint32_t*>(eng->sh.entry + ei + 2) + 1; bytes = 4; break;
    default: addr = eng->sh.depth_ctr + li; bytes = 4; break;
  }
  uint64_t v = 0;
  WG_CUDA(eng, cudaMemcpy(&v, addr, bytes, cudaMemcpyDeviceToHost));
  v ^= xor_value;
  WG_CUDA(eng, cudaMemcpy(addr, &v, bytes, cudaMemcpyHostToDevice));
  return WG_OK;
}

wg_status wg_shadow_depth(wg_engine* eng, uint32_t warp_slot, uint32_t lane, uint32_t* h_depth, void* cuda_stream) {
  if (!eng || !eng->loaded || !eng->sh.counters) return WG_ERR_NO_POLICY;
  if (warp_slot >= eng->sh.n_slots || lane >= 32 || !h_depth) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  WG_CUDA(eng, cudaMemcpy(h_depth, eng->sh.depth_ctr + static_cast<size_t>(warp_slot) * 32 + lane, 4,
                          cudaMemcpyDeviceToHost));
  return WG_OK;
}

wg_status wg_set_profile(wg_engine* eng, uint32_t flags) {
  if (!eng) return WG_ERR_NO_POLICY;
  if (flags & ~31u) return WG_ERR_INVALID_ARG;
  eng->profile = flags;  // takes effect with the next check call (kernel parameter)
  return WG_OK;
}

wg_status wg_set_skip_sites(wg_engine* eng, const uint8_t* h_skip, void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WG_CUDA(eng, cudaStreamSynchronize(st));  // no launch may still be reading the flags
  if (eng->n_sites == 0) return WG_OK;
  uint8_t* d_skip = nullptr;
  if (h_skip) {
    WG_CUDA(eng, cudaMalloc(&d_skip, eng->n_sites));
    cudaError_t err = cudaMemcpyAsync(d_skip, h_skip, eng->n_sites, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) {
      cudaFree(d_skip);
      return cuda_fail(eng, err);
    }
  }
  cudaError_t err = wg::launch_set_site_flags(eng->d_recs, d_skip, eng->n_sites, st, &eng->launches);
  if (err == cudaSuccess) err = cudaStreamSynchronize(st);
  cudaFree(d_skip);
  if (err != cudaSuccess) return cuda_fail(eng, err);
  return WG_OK;
}

wg_status wg_set_sequence_base(wg_engine* eng, uint64_t base) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (base > (1ull << 58)) return WG_ERR_INVALID_ARG;  // (seq << 5) must not wrap
  eng->seq = base;
  return WG_OK;
}

wg_status wg_get_device_view(wg_engine* eng, wg_device_view* h_view) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (!h_view) return WG_ERR_INVALID_ARG;
  h_view->site_recs = eng->d_recs;
  h_view->targets = eng->d_tgts;
  h_view->n_sites = eng->n_sites;
  h_view->bind_hi = eng->bind_hi;
  for (int i = 0; i < 4; ++i) h_view->v_init[i] = eng->v_init[i];
  return WG_OK;
}

wg_status wg_policy_poke(wg_engine* eng, int what, uint64_t index, uint64_t xor_value, void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (!((what == 0 && index < eng->n_tgts) || (what == 1 && index < eng->n_sites))) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  void* addr = what == 0 ? static_cast<void*>(eng->d_tgts + index) : static_cast<void*>(eng->d_tok + index);
  uint64_t v = 0;
  WG_CUDA(eng, cudaMemcpy(&v, addr, 8, cudaMemcpyDeviceToHost));
  v ^= xor_value;
  WG_CUDA(eng, cudaMemcpy(addr, &v, 8, cudaMemcpyHostToDevice));
  if (what == 0 && eng->d_htab) {
    // the hash index mirrors the target array: rebuild it from what the array holds now (a diagnostic hook: the cost
    // of a full rebuild does not matter), including the all-ones flags of the site records
    const size_t slots = 2 * static_cast<size_t>(eng->n_tgts) + 4 * static_cast<size_t>(eng->n_sites);
    WG_CUDA(eng, cudaMemset(eng->d_htab, 0xff, slots * 8));
    WG_CUDA(eng, wg::launch_clear_allones_flags(eng->d_recs, eng->n_sites, nullptr, &eng->launches));
    WG_CUDA(eng, wg::launch_build_hash(eng->d_htab, eng->d_recs, eng->d_tgts, eng->n_sites, eng->n_tgts, nullptr, &eng->launches));
    WG_CUDA(eng, cudaStreamSynchronize(nullptr));
  }
  return WG_OK;
}

wg_status wg_set_ring_capacity(wg_engine* eng, uint64_t capacity, void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (capacity > (1ull << 28)) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  WG_CUDA(eng, cudaStreamSynchronize(st));  // no launch may still be appending to the old ring
  wg::ViolRec* fresh = nullptr;
  if (capacity) WG_CUDA(eng, cudaMalloc(&fresh, sizeof(wg::ViolRec) * capacity));
  cudaFree(eng->d_ring);
  eng->d_ring = fresh;
  eng->ring_cap = capacity;
  // the ring restarts empty; every other counter keeps running
  WG_CUDA(eng, cudaMemsetAsync(eng->d_glob + wg::C_RING_TOTAL, 0, sizeof(unsigned long long), st));
  WG_CUDA(eng, cudaStreamSynchronize(st));
  return WG_OK;
}

wg_status wg_read_telemetry(wg_engine* eng, wg_telemetry_counters* h_counters, wg_violation_rec* h_first,
                            int* h_have_first, wg_violation_rec* h_ring, uint64_t ring_cap, uint64_t* h_n_ring,
                            void* cuda_stream) {
  if (!eng || !eng->loaded) return WG_ERR_NO_POLICY;
  if (!h_counters) return WG_ERR_INVALID_ARG;
  if ((h_first && !h_have_first) || (h_ring && !h_n_ring)) return WG_ERR_INVALID_ARG;
  DeviceGuard g(eng->device);
  if (!g.ok) return cuda_fail(eng, cudaErrorInvalidDevice);
  WG_CUDA(eng, cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
  unsigned long long w[9];  // words 26 .. 34
  WG_CUDA(eng, cudaMemcpy(w, eng->d_glob + wg::C_SKIP_RET_EVENTS, sizeof w, cudaMemcpyDeviceToHost));
  h_counters->fwd_meta_fail_events = w[wg::C_META_FAIL - wg::C_SKIP_RET_EVENTS];
  const uint64_t total = w[4];
  const uint64_t recorded = total < eng->ring_cap ? total : eng->ring_cap;
  h_counters->skipped_ret_events = w[0];
  h_counters->skipped_ret_lanes = w[1];
  h_counters->skipped_fwd_events = w[2];
  h_counters->skipped_fwd_lanes = w[3];
  h_counters->ring_recorded = recorded;
  h_counters->ring_dropped = total - recorded;
  h_counters->skipped_site_events = w[wg::C_SKIP_SITE_EVENTS - wg::C_SKIP_RET_EVENTS];
  h_counters->skipped_site_lanes = w[wg::C_SKIP_SITE_LANES - wg::C_SKIP_RET_EVENTS];
  h_counters->kernel_launches = eng->launches;
  if (h_first) {
    wg::FirstRec f;
    unsigned long long key = 0;
    WG_CUDA(eng, cudaMemcpy(&f, eng->d_first, sizeof f, cudaMemcpyDeviceToHost));
    WG_CUDA(eng, cudaMemcpy(&key, eng->d_glob + wg::C_FIRST_VIOLATION, sizeof key, cudaMemcpyDeviceToHost));
    static_assert(sizeof(wg_violation_rec) == sizeof(wg::ViolRec), "violation record layout");
    // the record must be the record OF first_violation_key (R29); anything else is an engine bug, reported loudly
    if (f.key != key) return WG_ERR_INTERNAL;
    *h_have_first = f.key != ~0ull;
    if (*h_have_first) std::memcpy(h_first, &f.rec, sizeof(wg_violation_rec));
  }
  if (h_ring) {
    const uint64_t n = recorded < ring_cap ? recorded : ring_cap;
    if (n) WG_CUDA(eng, cudaMemcpy(h_ring, eng->d_ring, sizeof(wg_violation_rec) * n, cudaMemcpyDeviceToHost));
    *h_n_ring = n;
  }
  return WG_OK;
}

wg_status wg_sign_continuations_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                     uint64_t* h_tag, uint64_t n) {
  return host_common(eng, OP_SIGN, h_hdr, h_val, nullptr, h_tag, nullptr, n, WG_MODE_DETECT);
}
wg_status wg_verify_continuations_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                       const uint64_t* h_tag, wg_verdict* h_out, uint64_t n, wg_mode mode) {
  return host_common(eng, OP_VERIFY, h_hdr, h_val, h_tag, nullptr, h_out, n, mode);
}
wg_status wg_check_forward_host(wg_engine* eng, const wg_event_hdr* h_hdr, const uint64_t* h_val,
                                wg_verdict* h_out, uint64_t n, wg_mode mode) {
  return host_common(eng, OP_FORWARD, h_hdr, h_val, nullptr, nullptr, h_out, n, mode);
}

}  // extern "C"

// ---- wg_verify_continuations_static: the verify kernel with its scratch memory in a static device array ------------
// The check kernel's scratch memory — the launch's group ticket, the global counter words it adds into (with the
// first-violation key) and the per-site counters — normally lives in cudaMalloc'ed arrays the engine owns and
// accumulates over calls.  Here it lives in ONE file-scope device array of the library: the call allocates nothing
// (no cudaMalloc / cudaFree, no allocating library routine; only memsets, the launch and device-to-device copies on
// the caller's stream), and it leaves the engine's own counters, sequence numbers, ring and first-violation record
// untouched.  Every GPU that loads the library holds the array (2,098,176 bytes) until the process exits.
namespace {

constexpr uint32_t kStaticMaxSites = WG_STATIC_MAX_SITES;
struct StaticScratch {
  unsigned int ticket[64];                               // the launch's group ticket (256 bytes: its own cache lines)
  unsigned long long glob[64];                           // C_WORDS global counter words, padded
  unsigned long long site[4ull * kStaticMaxSites];       // [n_sites][4] per-site counters
};
static_assert(wg::C_WORDS <= 64, "global counter words");
static_assert(sizeof(StaticScratch) == 256 + 512 + 32ull * kStaticMaxSites, "static scratch layout");
static_assert(WG_STATIC_MAX_EVENTS == kMaxLaunchEvents, "one launch");

// In host code this name is a host-side stand-in for the array, NOT its device address: the address is resolved once
// per device with cudaGetSymbolAddress (that device current) and it is that pointer the kernel is given.
static __device__ __align__(256) unsigned char wg_static_scratch[sizeof(StaticScratch)];

constexpr int kStaticMaxDevices = 64;
StaticScratch* g_static_ptr[kStaticMaxDevices] = {};

// the calling thread's current device must be `device` (the caller holds a DeviceGuard)
cudaError_t static_scratch_for(int device, StaticScratch** out) {
  if (device < 0 || device >= kStaticMaxDevices) return cudaErrorInvalidDevice;
  StaticScratch* ptr = __atomic_load_n(&g_static_ptr[device], __ATOMIC_ACQUIRE);
  if (!ptr) {
    void* a = nullptr;
    const cudaError_t err = cudaGetSymbolAddress(&a, wg_static_scratch);
    if (err != cudaSuccess) return err;
    if (!a) return cudaErrorInvalidSymbol;
    ptr = static_cast<StaticScratch*>(a);
    __atomic_store_n(&g_static_ptr[device], ptr, __ATOMIC_RELEASE);  // (two threads resolve the same address)
  }
  *out = ptr;
  return cudaSuccess;
}

}  // namespace

extern "C" wg_status wg_verify_continuations_static(wg_engine* e, const wg_event_hdr* d_hdr, const uint64_t* d_val,
                                                    const uint64_t* d_tag, wg_verdict* d_out, wg_counters* d_counters,
                                                    wg_site_counters* d_per_site, uint64_t n, wg_mode mode,
                                                    void* cuda_stream) {
  if (!e || !e->loaded) return WG_ERR_NO_POLICY;
  if (mode != WG_MODE_DETECT && mode != WG_MODE_ENFORCE) return WG_ERR_INVALID_ARG;
  if (e->n_sites > kStaticMaxSites || n > WG_STATIC_MAX_EVENTS) return WG_ERR_STATIC_LIMIT;
  if (n != 0 && (!d_hdr || !d_val || !d_tag || !d_out)) return WG_ERR_INVALID_ARG;
  if (!aligned(d_hdr, 16) || !aligned(d_val, 16) || !aligned(d_tag, 16) || !aligned(d_out, 8) ||
      !aligned(d_counters, 8) || !aligned(d_per_site, 8))
    return WG_ERR_INVALID_ARG;
  DeviceGuard g(e->device);
  if (!g.ok) return cuda_fail(e, cudaErrorInvalidDevice);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  StaticScratch* sc = nullptr;
  WG_CUDA(e, static_scratch_for(e->device, &sc));
  // the array keeps the last call's contents: everything the kernel adds into starts at zero (the key at all-ones)
  WG_CUDA(e, cudaMemsetAsync(sc->glob, 0, sizeof(sc->glob), st));
  WG_CUDA(e, cudaMemsetAsync(sc->glob + wg::C_FIRST_VIOLATION, 0xff, sizeof(unsigned long long), st));
  if (e->n_sites) WG_CUDA(e, cudaMemsetAsync(sc->site, 0, sizeof(unsigned long long) * 4 * e->n_sites, st));
  if (n != 0) {
    wg::Params p = base_params(e);
    p.hdr = reinterpret_cast<const uint4*>(d_hdr);
    p.val = d_val;
    p.tag = d_tag;
    p.out = reinterpret_cast<uint2*>(d_out);
    p.n = n;
    p.seq_base = 0;  // the call's own event numbering: first_violation_key counts from this call's first event
    p.mode = static_cast<uint32_t>(mode);
    p.sched = sc->ticket;  // (zeroed by the launcher)
    p.glob = sc->glob;
    p.site = sc->site;
    p.ring = nullptr;  // no violation ring, no first-violation record: diagnostics of the engine's own calls
    p.ring_cap = 0;
    p.first = nullptr;
    WG_CUDA(e, wg::launch_check(p, e->sm_count, st, &e->launches));
  }
  static_assert(sizeof(wg_counters) == 26 * 8 && sizeof(wg_site_counters) == 32, "counter layouts");
  if (d_counters) WG_CUDA(e, cudaMemcpyAsync(d_counters, sc->glob, sizeof(wg_counters), cudaMemcpyDeviceToDevice, st));
  if (d_per_site && e->n_sites)
    WG_CUDA(e, cudaMemcpyAsync(d_per_site, sc->site, sizeof(wg_site_counters) * e->n_sites, cudaMemcpyDeviceToDevice, st));
  return WG_OK;
}
