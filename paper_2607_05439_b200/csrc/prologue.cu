// Single-track projections (step a1) and the output projection (step a9) as a plain fp32-accumulate
// SIMT GEMM, plus the small weight-folding and LayerNorm(s) kernels.
//   PAPER.md:77-81 (sec 3.2): Q^(p) = f_Q(S^(p)); "keys and values are projected from the full single-track S"
//   BASELINE.json config 0:  out = W_o (sigmoid(s W_g) (.) softmax(...) V)
// Every output element is accumulated over k in ascending order by one thread, so a row's result
// does not depend on which tile it falls in (needed for the bitwise row(P) == monolithic contract).
#include "kernels.h"

namespace dcp {

namespace {

constexpr int BM = 64, BN = 64, BK = 16;

template <typename TA, typename TW, typename TC, int EPI>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const TA* __restrict__ A, int64_t lda,
                                                        const TW* __restrict__ W, const TW* __restrict__ bias,
                                                        TC* __restrict__ C, int64_t ldc, int64_t M, int N, int K) {
  __shared__ float As[BK][BM + 4];
  __shared__ float Ws[BK][BN + 4];
  const int tid = threadIdx.x;
  const int tx = tid % 16, ty = tid / 16;
  const int64_t m0 = (int64_t)blockIdx.y * BM;
  const int n0 = blockIdx.x * BN;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < K; k0 += BK) {
    // A tile: 64 rows x 16 k  (1024 elements, 4 per thread)
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      int e = tid + t * 256;
      int r = e / BK, kk = e % BK;
      int64_t gm = m0 + r;
      int gk = k0 + kk;
      As[kk][r] = (gm < M && gk < K) ? to_f32(A[gm * lda + gk]) : 0.f;
    }
    // W tile: 16 k x 64 n
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      int e = tid + t * 256;
      int kk = e / BN, c = e % BN;
      int gk = k0 + kk, gn = n0 + c;
      Ws[kk][c] = (gk < K && gn < N) ? to_f32(W[(int64_t)gk * N + gn]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Ws[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int64_t gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int gn = n0 + tx * 4 + j;
      if (gn >= N) continue;
      float x = acc[i][j];
      if (bias != nullptr) x += to_f32(bias[gn]);
      if (EPI == EPI_SIGMOID) x = 1.f / (1.f + expf(-x));
      C[gm * ldc + gn] = from_f32<TC>(x);
    }
  }
}

template <typename TA, typename TW>
cudaError_t gemm_dispatch(const void* A, int64_t lda, const void* W, const void* bias, void* C, int64_t ldc,
                          int64_t M, int N, int K, GemmEpilogue epi, cudaStream_t st) {
  dim3 grid((N + BN - 1) / BN, (unsigned)((M + BM - 1) / BM));
  if (epi == EPI_SIGMOID)
    gemm_simt_kernel<TA, TW, TW, EPI_SIGMOID><<<grid, 256, 0, st>>>((const TA*)A, lda, (const TW*)W, (const TW*)bias,
                                                                   (TW*)C, ldc, M, N, K);
  else
    gemm_simt_kernel<TA, TW, TW, EPI_NONE><<<grid, 256, 0, st>>>((const TA*)A, lda, (const TW*)W, (const TW*)bias,
                                                                (TW*)C, ldc, M, N, K);
  return cudaGetLastError();
}

template <typename T>
__global__ void layernorm_rows_kernel(const T* __restrict__ x, const T* __restrict__ gamma, const T* __restrict__ beta,
                                      float* __restrict__ y, int64_t rows, int width, float eps) {
  // one warp per row; two-pass (mean, then centred sum of squares), population variance
  int64_t row = (int64_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  int lane = threadIdx.x % 32;
  if (row >= rows) return;
  const T* xr = x + row * width;
  float s = 0.f;
  for (int k = lane; k < width; k += 32) s += to_f32(xr[k]);
  float mu = warp_sum(s) / (float)width;
  float v = 0.f;
  for (int k = lane; k < width; k += 32) {
    float d = to_f32(xr[k]) - mu;
    v = fmaf(d, d, v);
  }
  float rstd = rsqrtf(warp_sum(v) / (float)width + eps);
  for (int k = lane; k < width; k += 32)
    y[row * width + k] = (to_f32(xr[k]) - mu) * rstd * to_f32(gamma[k]) + to_f32(beta[k]);
}

template <typename T>
__global__ void fold_ln_z_kernel(const T* __restrict__ w_b, const T* __restrict__ gamma, const T* __restrict__ beta,
                                 float* __restrict__ wg, float* __restrict__ c0, int c_z, int H) {
  // single block; wg[k,h] = gamma_k W_b[k,h];  c0[h] = sum_k beta_k W_b[k,h] (ascending k)
  for (int e = threadIdx.x; e < c_z * H; e += blockDim.x) wg[e] = to_f32(gamma[e / H]) * to_f32(w_b[e]);
  if (threadIdx.x < H) {
    float a = 0.f;
    for (int k = 0; k < c_z; ++k) a = fmaf(to_f32(beta[k]), to_f32(w_b[k * H + threadIdx.x]), a);
    c0[threadIdx.x] = a;
  }
}

}  // namespace

cudaError_t launch_gemm(dcp_dtype dt, bool a_is_f32, const void* A, int64_t lda, const void* W, const void* bias,
                        void* C, int64_t ldc, int64_t M, int N, int K, GemmEpilogue epi, cudaStream_t st) {
  if (M <= 0 || N <= 0 || K <= 0) return cudaSuccess;
  if (dt == DCP_F32) return gemm_dispatch<float, float>(A, lda, W, bias, C, ldc, M, N, K, epi, st);
  if (a_is_f32) return gemm_dispatch<float, __nv_bfloat16>(A, lda, W, bias, C, ldc, M, N, K, epi, st);
  return gemm_dispatch<__nv_bfloat16, __nv_bfloat16>(A, lda, W, bias, C, ldc, M, N, K, epi, st);
}

cudaError_t launch_layernorm_rows(dcp_dtype dt, const void* x, const void* gamma, const void* beta, float* y,
                                  int64_t rows, int width, float eps, cudaStream_t st) {
  unsigned blocks = (unsigned)((rows + 7) / 8);
  if (dt == DCP_F32)
    layernorm_rows_kernel<float><<<blocks, 256, 0, st>>>((const float*)x, (const float*)gamma, (const float*)beta, y,
                                                         rows, width, eps);
  else
    layernorm_rows_kernel<__nv_bfloat16><<<blocks, 256, 0, st>>>((const __nv_bfloat16*)x, (const __nv_bfloat16*)gamma,
                                                                 (const __nv_bfloat16*)beta, y, rows, width, eps);
  return cudaGetLastError();
}

cudaError_t launch_fold_ln_z(dcp_dtype dt, const void* w_b, const void* gamma, const void* beta, float* wg, float* c0,
                             int c_z, int H, cudaStream_t st) {
  if (dt == DCP_F32)
    fold_ln_z_kernel<float><<<1, 256, 0, st>>>((const float*)w_b, (const float*)gamma, (const float*)beta, wg, c0, c_z, H);
  else
    fold_ln_z_kernel<__nv_bfloat16><<<1, 256, 0, st>>>((const __nv_bfloat16*)w_b, (const __nv_bfloat16*)gamma,
                                                       (const __nv_bfloat16*)beta, wg, c0, c_z, H);
  return cudaGetLastError();
}

}  // namespace dcp
