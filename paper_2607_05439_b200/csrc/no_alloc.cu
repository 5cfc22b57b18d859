// dcp_pair_bias_attention_no_alloc (include/designcp.h): the layer of dcp_pair_bias_attention for callers that cannot
// allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The
// workspace the layer needs (q, k, v fragments, gate, folded weights, partial online-softmax states; api.cu carve())
// lives in a file-scope device array of DCP_NO_ALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit.
//
// g_scratch is a HOST-SIDE STAND-IN in host code, not a device address: its device address is looked up once per device
// by cudaGetSymbolAddress with that device current, and that pointer is what the kernels get.
//
// Nothing here (or below it: api.cu's launch sequence) calls cudaMalloc, cudaFree or an allocating library routine.
// Every call on a device shares the array, which keeps the previous call's contents: the layer writes each region
// before it reads it (nothing has to start at zero, so nothing is cleared), but two calls that overlap on the GPU --
// different streams, or different host threads on the same device -- race on it.  Calls on one stream are ordered.
#include <mutex>

#include "kernels.h"

namespace {

constexpr size_t kScratchBytes = DCP_NO_ALLOC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {};

// device address of g_scratch on the current device (looked up once per device)
dcp_status scratch_address(void** ptr) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return DCP_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_scratch) != cudaSuccess || !p) return DCP_ERR_CUDA;
    if ((reinterpret_cast<uintptr_t>(p) & 255) != 0) return DCP_ERR_CUDA;
    g_scratch_ptr[dev] = p;
  }
  *ptr = g_scratch_ptr[dev];
  return DCP_OK;
}

}  // namespace

extern "C" {

size_t dcp_no_alloc_scratch_bytes(void) { return kScratchBytes; }

dcp_status dcp_pair_bias_attention_no_alloc(const void* s, const void* z, int64_t ldz, const dcp_weights* w, void* out, int64_t I,
                                            int c_s, int H, int c, int c_z, dcp_dtype dtype, dcp_decomp decomp,
                                            const dcp_plan* plan, void* stream) {
  size_t need = 0;
  dcp_status st = dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, decomp, plan, &need);
  if (st != DCP_OK) return st;
  if (need > kScratchBytes) return DCP_ERR_SCRATCH_LIMIT;
  void* scratch = nullptr;
  st = scratch_address(&scratch);
  if (st != DCP_OK) return st;
  return dcp_pair_bias_attention(s, z, ldz, w, out, I, c_s, H, c, c_z, dtype, decomp, plan, scratch, kScratchBytes, stream);
}

}  // extern "C"
