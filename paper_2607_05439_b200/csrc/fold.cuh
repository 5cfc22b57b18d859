// libdesigncp internal: LayerNorm(z) folded into the bias projection weights (device function shared by the stand-alone
// fold kernel in gemm_mma.cu and by the extra CTA of the tcgen05 GEMM launch in gemm_tc.cu).
//   LN(z) W_b = rstd (z . W' - mu c1) + c0   with W' = diag(gamma) W_b
#pragma once
#include "common.cuh"

namespace dcp {

// wfold[h][k] = bf16(gamma_k W_b[k,h] log2 e)   (K-major rows: the B operand of the projection MMA)
// c1[h] = sum_k wfold[h][k] (the rounded values), c0[h] = log2 e * sum_k beta_k W_b[k,h]
// Executed by the first `nthreads` (a multiple of 32, all of them calling) threads of a CTA.
static __device__ __forceinline__ void fold_ln_z_mma_device(const void* w_b_, const void* gamma_, const void* beta_, void* wfold_, float* c1,
                                     float* c0, int c_z, int H, int H_pad, int tid, int nthreads) {
  const __nv_bfloat16* w_b = reinterpret_cast<const __nv_bfloat16*>(w_b_);
  const __nv_bfloat16* gamma = reinterpret_cast<const __nv_bfloat16*>(gamma_);
  const __nv_bfloat16* beta = reinterpret_cast<const __nv_bfloat16*>(beta_);
  __nv_bfloat16* wfold = reinterpret_cast<__nv_bfloat16*>(wfold_);
  constexpr float kLog2e = 1.4426950408889634f;
  // one warp per head: the warp writes the head's row and sums it (no block-level synchronisation needed)
  for (int h = tid >> 5; h < H_pad; h += nthreads >> 5) {
    float a1 = 0.f, a0 = 0.f;
    for (int k = tid & 31; k < c_z; k += 32) {
      const float v = h < H ? to_f32(gamma[k]) * to_f32(w_b[k * H + h]) * kLog2e : 0.f;
      const __nv_bfloat16 r = __float2bfloat16_rn(v);
      wfold[h * c_z + k] = r;
      a1 += to_f32(r);
      if (h < H) a0 = fmaf(to_f32(beta[k]), to_f32(w_b[k * H + h]), a0);
    }
    a1 = warp_sum(a1);
    a0 = warp_sum(a0);
    if ((tid & 31) == 0) { c1[h] = a1; c0[h] = a0 * kLog2e; }
  }
}

}  // namespace dcp
