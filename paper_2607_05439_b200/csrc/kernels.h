// libdesigncp internal: host-side launchers of every kernel (one translation unit each).
#pragma once
#include "common.cuh"

namespace dcp {

enum GemmEpilogue { EPI_NONE = 0, EPI_SIGMOID = 1 };

// C[M,N] = epi(A[M,K] * W[K,N] + bias[N])  row-major, fp32 accumulate (SIMT; exact-order per element).
// a_is_f32: A is float (LayerNorm'ed s) instead of the storage dtype.  Step a1 / a9 of SURVEY.md section 8(a).
cudaError_t launch_gemm(dcp_dtype dt, bool a_is_f32, const void* A, int64_t lda, const void* W, const void* bias,
                        void* C, int64_t ldc, int64_t M, int N, int K, GemmEpilogue epi, cudaStream_t st);

// Tensor-core (mma.sync bf16) version of the same GEMM for the bf16 path; A, W, C bf16.
cudaError_t launch_gemm_bf16_mma(const void* A, int64_t lda, const void* W, const void* bias, void* C, int64_t ldc,
                                 int64_t M, int N, int K, GemmEpilogue epi, cudaStream_t st);

// s~ = LayerNorm(s; gamma, beta) -> float [rows, width]      (optional LN_s, reading #3 in DESIGN.md)
cudaError_t launch_layernorm_rows(dcp_dtype dt, const void* x, const void* gamma, const void* beta, float* y,
                                  int64_t rows, int width, float eps, cudaStream_t st);

// wg[k,h] = gamma_k * W_b[k,h] (fp32), c0[h] = sum_k beta_k W_b[k,h]
cudaError_t launch_fold_ln_z(dcp_dtype dt, const void* w_b, const void* gamma, const void* beta, float* wg, float* c0,
                             int c_z, int H, cudaStream_t st);

// Generic fp32 CUDA-core fused kernel (steps a2-a7).  Returns cudaErrorInvalidValue for unsupported shapes.
cudaError_t launch_fused_generic(dcp_dtype dt, const FusedParams& p, cudaStream_t st);
bool fused_generic_supports(dcp_dtype dt, int H, int c, int c_z);

// bf16 tensor-core fused kernel (TMA-streamed z).  Workspace for folded bf16 weights is carved by api.cu.
struct MmaAux {
  const void* wfold;    // [H_pad, c_z] bf16: (gamma (.) W_b)^T, K-major
  const float* c1;      // [H] sum_k wfold[h,k]  (for the -mu*c1 term)
  const float* c0;      // [H]
  void* tmap_z;         // host pointer to a CUtensorMap for z (128 B, passed by value into the kernel)
};
cudaError_t launch_fused_mma(const FusedParams& p, const MmaAux& aux, cudaStream_t st);
bool fused_mma_supports(dcp_dtype dt, int H, int c, int c_z);
cudaError_t launch_fold_ln_z_mma(const void* w_b, const void* gamma, const void* beta, void* wfold, float* c1,
                                 float* c0, int c_z, int H, cudaStream_t st);

// Merge (step a8) + normalise + gate (first half of a9); or raw merged state out.
cudaError_t launch_merge(dcp_dtype dt, const MergeParams& p, cudaStream_t st);

}  // namespace dcp
