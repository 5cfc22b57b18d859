// libdesigncp internal header: shared parameter structs and small device helpers.
// Nothing here is shared with oracle/ (the CPU oracle is independent numpy code).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/designcp.h"

namespace dcp {

constexpr int kMaxHeads = 16;     // H <= 16 (RFD3: 16 token heads, 4 atom heads)
constexpr int kMaxD = 768;        // H*c <= 768 = c_token

// Eq. 5: start and length of shard p of n items over `parts` shards.
__host__ __device__ inline void shard_range(int64_t n, int parts, int p, int64_t* start, int64_t* len) {
  int64_t base = n / parts, rem = n % parts;
  *len = base + (p < rem ? 1 : 0);
  *start = (int64_t)p * base + (p < rem ? p : rem);
}

// ---- programmatic dependent launch (sm_90+): a kernel launched with launch_kernel(..., pdl = true) may start while the
// previous kernel in the stream is still draining; everything before pdl_wait() (barrier init, tensor-memory allocation,
// descriptor prefetch) overlaps the predecessor's tail, everything after it sees the predecessor's writes.  Every kernel
// of the chain executes pdl_wait() in every thread before it touches global memory, so completion is transitive: when a
// kernel's pdl_wait() returns, all earlier kernels of the stream have finished.  Both calls are no-ops in a kernel that was
// launched without the attribute.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                 Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__device__ __forceinline__ float to_f32(float x) { return x; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// One sub-problem of the fused (query-tile, key-tile) loop: query rows [q0, q1) against keys [k0, k1),
// the keys cut into `n_chunks` Eq.-5 chunks; chunk cidx writes partial state slot (slot0 + cidx).
// State arrays are indexed [slot][row - state_row0][...], row = absolute token index.
struct FusedParams {
  const void* z;        // [I, I, c_z] storage dtype, z[i, j, :] biases query i <- key j
  int64_t ldz;          // elements between consecutive query rows of z
  const void* q;        // [I, D] storage dtype (workspace)
  const void* k;        // [I, D]
  const void* v;        // [I, D]
  const float* wg;      // [c_z, H] fp32: gamma_k * W_b[k, h]            (folded LayerNorm affine)
  const float* c0;      // [H]      fp32: sum_k beta_k W_b[k, h]
  float* st_m;          // [slots, state_rows, H]
  float* st_l;          // [slots, state_rows, H]
  float* st_acc;        // [slots, state_rows, D]
  int64_t state_rows;   // rows per slot in the state arrays
  int64_t state_row0;   // absolute row of state row 0
  int64_t q0, q1, k0, k1;
  int n_chunks, slot0;
  int I, c_z, H, c, D;
  float eps, scale;     // scale = 1/sqrt(c)
};

struct MergeParams {
  const float* st_m;    // [n_slots, rows, H]
  const float* st_l;
  const float* st_acc;  // [n_slots, rows, D]
  const void* g;        // [rows, D] storage dtype, sigmoid gate (or nullptr: no gate, raw merged state out)
  void* gated;          // [rows, D] storage dtype: g * acc / l            (when g != nullptr)
  float *m_out, *l_out, *acc_out;  // merged state out (when g == nullptr)
  int64_t rows;
  int n_slots, H, c, D;
  bool pdl;             // host only: launch as a programmatic dependent of the previous kernel in the stream
};

}  // namespace dcp
