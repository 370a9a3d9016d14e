// A "protected application kernel" for tests/test_gpu_device_inline.py: it calls the inline device helpers of
// include/warpguard_device.cuh at its own sites, one thread per lane, with the guard applied by the caller
// (a predicated-off lane does not call).  Test code, not part of the library.
#include <cuda_runtime.h>

#include "warpguard_device.cuh"

__global__ void user_kernel(const wg_device_view view, const uint4* hdr, const uint64_t* val, const uint64_t* tag,
                            uint64_t* tag_out, uint32_t* viol_out, uint64_t n, int op) {
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t warp = (static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const uint64_t nwarps = (static_cast<uint64_t>(gridDim.x) * blockDim.x) >> 5;
  for (uint64_t e = warp; e < n; e += nwarps) {
    const uint4 h = hdr[e];
    const bool guard = (h.y >> lane) & 1u;
    const uint64_t ctx = ((static_cast<uint64_t>(h.w) << 32) | h.z) & ~31ull | lane;
    const uint64_t v = val[e * 32 + lane];
    bool bad = false;
    if (op == 0) {  // call site: push
      tag_out[e * 32 + lane] = guard ? wg_dev_sign(view, h.x, v, ctx) : 0ull;
    } else if (op == 1) {  // return site: check_ret
      if (guard) bad = !wg_dev_verify(view, h.x, v, ctx, tag[e * 32 + lane]);
    } else {  // indirect branch: forward check
      if (guard) bad = !wg_dev_check_forward(view, h.x, v);
    }
    const uint32_t mask = __ballot_sync(0xffffffffu, bad);
    if (op != 0 && lane == 0) viol_out[e] = mask;
  }
}

extern "C" int wg_test_run_inline(wg_device_view view, const void* hdr, const void* val, const void* tag, void* tag_out,
                                  void* viol_out, uint64_t n, int op, void* stream) {
  user_kernel<<<148 * 8, 256, 0, static_cast<cudaStream_t>(stream)>>>(
      view, static_cast<const uint4*>(hdr), static_cast<const uint64_t*>(val), static_cast<const uint64_t*>(tag),
      static_cast<uint64_t*>(tag_out), static_cast<uint32_t*>(viol_out), n, op);
  return static_cast<int>(cudaGetLastError());
}

// raw copy of the engine's site records as the view exposes them (tests/test_gpu_device_inline.py checks that
// nothing in them is key-derived)
extern "C" int wg_test_copy_site_recs(wg_device_view view, void* h_out) {
  return static_cast<int>(cudaMemcpy(h_out, view.site_recs, static_cast<size_t>(view.n_sites) * 16, cudaMemcpyDeviceToHost));
}
