// Tensor-core GEMMs of the bf16 path: the single-track projections (step a1) and the output projection (step a9).
//   PAPER.md:77-81 (sec 3.2): Q^(p) = f_Q(S^(p)); "keys and values are projected from the full single-track S"
//   BASELINE.json config 0:  out = W_o (sigmoid(s W_g) (.) softmax(...) V)
// C[M, N] = A[M, K] (bf16, row-major) x W[K, N] (bf16, row-major), fp32 accumulate, mma.sync m16n8k16,
// 128 x 128 x 32 CTA tiles, cp.async double buffering.  The four projections run as ONE launch over
// N = 4 D columns; the epilogue writes each segment in the layout the fused kernel reads:
//   q -> qp [I][H][CP]  scaled by log2(e)/sqrt(c) (exp2-domain softmax), head rows zero-padded to CP
//   k -> kfr, v -> vfr  in the MMA B-fragment order of the fused kernel (one coalesced 128-bit load per lane)
//   g -> g  [I][D]      sigmoid gate
// Every output element is accumulated over k in a fixed order that does not depend on the tile it falls in.
#include "kernels.h"
#include "fold.cuh"

namespace dcp {

namespace {

constexpr int BN = 128, BK = 32;   // BM = 32 MI: 128 (MI = 4) or 64 (MI = 2, for grids that would not fill the GPU)
constexpr int LDA_S = BK + 8;    // padded smem rows: conflict-free ldmatrix
constexpr int LDB_S = BN + 8;

__device__ __forceinline__ void cp_async16(void* dst, const void* src, bool ok) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst);
  const int n = ok ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

template <int MI>
__global__ void __launch_bounds__(256) gemm_mma_kernel(const GemmMmaParams p) {
  pdl_trigger();
  pdl_wait();
  constexpr int BM = 32 * MI;
  // pipeline buffers; after the main loop the same memory stages the C tile of the fragment-order outputs
  constexpr int kAElems = 2 * BM * LDA_S, kBElems = 2 * BK * LDB_S, kCElems = BM * LDB_S;
  __shared__ __align__(16) __nv_bfloat16 smem_raw[(kAElems + kBElems) > kCElems ? (kAElems + kBElems) : kCElems];
  __nv_bfloat16 (*As)[BM * LDA_S] = reinterpret_cast<__nv_bfloat16 (*)[BM * LDA_S]>(smem_raw);
  __nv_bfloat16 (*Bs)[BK * LDB_S] = reinterpret_cast<__nv_bfloat16 (*)[BK * LDB_S]>(smem_raw + kAElems);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wm = warp >> 2, wn = warp & 3;            // 2 x 4 warps, warp tile (16 MI) x 32
  const int nb_per_seg = (p.N + BN - 1) / BN;
  const int seg = blockIdx.x / nb_per_seg;
  const int n0 = (blockIdx.x % nb_per_seg) * BN;
  const int64_t m0 = (int64_t)blockIdx.y * BM;
  const __nv_bfloat16* A = reinterpret_cast<const __nv_bfloat16*>(p.A);
  const __nv_bfloat16* W = reinterpret_cast<const __nv_bfloat16*>(p.W[seg]);

  float acc[MI][4][4];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int x = 0; x < 4; ++x) acc[i][j][x] = 0.f;

  auto load_tile = [&](int buf, int k0) {
#pragma unroll
    for (int it = 0; it < 2; ++it) {
      const int e = tid + it * 256;
      if (e < BM * 4) {   // A: BM rows x 4 chunks of 8 elements
        const int r = e >> 2, ch = e & 3;
        const int64_t gm = m0 + r;
        const int gk = k0 + ch * 8;
        const bool ok = gm < p.M && gk < p.K;
        cp_async16(&As[buf][r * LDA_S + ch * 8], ok ? (const void*)(A + gm * p.lda + gk) : (const void*)A, ok);
      }
      {   // W: 32 rows x 16 chunks
        const int r = e >> 4, ch = e & 15;
        const int gk = k0 + r, gn = n0 + ch * 8;
        const bool ok = gk < p.K && gn < p.N;
        cp_async16(&Bs[buf][r * LDB_S + ch * 8], ok ? (const void*)(W + (int64_t)gk * p.N + gn) : (const void*)W, ok);
      }
    }
    cp_async_commit();
  };

  const int nk = (p.K + BK - 1) / BK;
  load_tile(0, 0);
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < nk) { load_tile(buf ^ 1, (kt + 1) * BK); cp_async_wait<1>(); }
    else cp_async_wait<0>();
    __syncthreads();
#pragma unroll
    for (int ks = 0; ks < BK / 16; ++ks) {
      uint32_t af[MI][4], bf[4][2];
#pragma unroll
      for (int i = 0; i < MI; ++i) {
        const int row = wm * (16 * MI) + i * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int col = ks * 16 + (lane >> 4) * 8;
        ldsm_x4((uint32_t)__cvta_generic_to_shared(&As[buf][row * LDA_S + col]), af[i][0], af[i][1], af[i][2], af[i][3]);
      }
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int krow = ks * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int col = wn * 32 + j * 16 + (lane >> 4) * 8;
        ldsm_x4_t((uint32_t)__cvta_generic_to_shared(&Bs[buf][krow * LDB_S + col]), bf[2 * j][0], bf[2 * j][1],
                  bf[2 * j + 1][0], bf[2 * j + 1][1]);
      }
#pragma unroll
      for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) mma16816(acc[i][j], af[i], bf[j][0], bf[j][1]);
    }
    __syncthreads();
  }

  // ---- epilogue, fragment-order outputs (k, v): the C tile goes through shared memory so that the global stores are
  // 8-byte units written in destination order (256 contiguous bytes per warp) instead of scattered 2- / 4-byte stores
  if (p.mode[seg] == GEMM_OUT_KFRAG || p.mode[seg] == GEMM_OUT_VFRAG) {
    __nv_bfloat16* Cs = smem_raw;                       // [BM][LDB_S]; the main loop ended with __syncthreads()
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        const int rl = wm * (16 * MI) + i * 16 + g + 8 * x;
        const bool live = m0 + rl < p.M;                // rows beyond M are written as zeros (0 * finite in PV)
#pragma unroll
        for (int j = 0; j < 4; ++j)
          *reinterpret_cast<__nv_bfloat162*>(Cs + rl * LDB_S + wn * 32 + j * 8 + 2 * t) =
              live ? __floats2bfloat162_rn(acc[i][j][2 * x], acc[i][j][2 * x + 1]) : __floats2bfloat162_rn(0.f, 0.f);
      }
    __syncthreads();
    __nv_bfloat16* C = reinterpret_cast<__nv_bfloat16*>(p.C[seg]);
    const int64_t tile_end = (p.M + 31) / 32 * 2;       // key tiles the fragment buffers hold (mma_frag_elems)
    const bool is_k = p.mode[seg] == GEMM_OUT_KFRAG;
    for (int u = tid; u < BM * BN / 4; u += 256) {
      // unit = [key tile kt][16-column group][g][t][b]: 8 bytes of lane (g, t)'s fragment
      const int b = u & 1, tt = (u >> 1) & 3, gg = (u >> 3) & 7, grp = (u >> 6) & 7, kt = u >> 9;
      const int64_t tile = (m0 >> 4) + kt;
      if (tile >= tile_end) continue;
      uint2 v;
      int col;
      if (is_k) {   // K: 4 head dims of key 4 (g / 2) + g % 2 + 2 b   (b = n-block A / B)
        col = grp * 16 + 4 * tt;
        v = *reinterpret_cast<const uint2*>(Cs + (kt * 16 + 4 * (gg >> 1) + (gg & 1) + 2 * b) * LDB_S + col);
      } else {      // V: keys 4 t .. 4 t + 3 of head dim 8 b + g of the group
        col = grp * 16 + 8 * b + gg;
        const __nv_bfloat16* src = Cs + (kt * 16 + 4 * tt) * LDB_S + col;
        const uint32_t e0 = *reinterpret_cast<const unsigned short*>(src), e1 = *reinterpret_cast<const unsigned short*>(src + LDB_S);
        const uint32_t e2 = *reinterpret_cast<const unsigned short*>(src + 2 * LDB_S), e3 = *reinterpret_cast<const unsigned short*>(src + 3 * LDB_S);
        v = make_uint2(e0 | (e1 << 16), e2 | (e3 << 16));
      }
      const int ca = n0 + col;
      if (ca >= p.N) continue;
      const int h = ca / p.c, d = ca % p.c;
      int64_t idx;
      if (is_k) idx = (((tile * p.H + h) * (p.cp >> 4) + (d >> 4)) * 32 + gg * 4 + ((d & 15) >> 2)) * 8 + b * 4;
      else idx = (((tile * p.H + h) * (p.cp >> 4) + (d >> 4)) * 32 + (d & 7) * 4 + tt) * 8 + ((d >> 3) & 1) * 4;
      *reinterpret_cast<uint2*>(C + idx) = v;
    }
    return;
  }
  // ---- epilogue
  const int g = lane >> 2, t = lane & 3;
  const int mode = p.mode[seg];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int x = 0; x < 2; ++x) {
      const int64_t row = m0 + wm * (16 * MI) + i * 16 + g + 8 * x;
      if (row >= p.M) continue;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int col = n0 + wn * 32 + j * 8 + 2 * t;
        if (col >= p.N) continue;
        float v0 = acc[i][j][2 * x], v1 = acc[i][j][2 * x + 1];
        if (p.bias[seg] != nullptr) {
          const __nv_bfloat16* b = reinterpret_cast<const __nv_bfloat16*>(p.bias[seg]);
          v0 += __bfloat162float(b[col]);
          v1 += __bfloat162float(b[col + 1]);
        }
        __nv_bfloat16* C = reinterpret_cast<__nv_bfloat16*>(p.C[seg]);
        if (mode == GEMM_OUT_PLAIN) {
          *reinterpret_cast<__nv_bfloat162*>(C + row * p.ldc[seg] + col) = __floats2bfloat162_rn(v0, v1);
        } else if (mode == GEMM_OUT_SIGMOID) {
          v0 = 1.f / (1.f + expf(-v0));
          v1 = 1.f / (1.f + expf(-v1));
          *reinterpret_cast<__nv_bfloat162*>(C + row * p.ldc[seg] + col) = __floats2bfloat162_rn(v0, v1);
        } else if (mode == GEMM_OUT_HEADPAD) {
          const int h = col / p.c, d = col % p.c;   // c even, col even: the pair stays inside one head
          *reinterpret_cast<__nv_bfloat162*>(C + (row * p.H + h) * p.cp + d) = __floats2bfloat162_rn(v0 * p.scale[seg], v1 * p.scale[seg]);
        } else {   // GEMM_OUT_TRANSPOSED: vt[col][row]
          C[(int64_t)col * p.ldc[seg] + row] = __float2bfloat16_rn(v0);
          C[(int64_t)(col + 1) * p.ldc[seg] + row] = __float2bfloat16_rn(v1);
        }
      }
    }
}

__global__ void layernorm_rows_bf16_kernel(const __nv_bfloat16* __restrict__ x, const __nv_bfloat16* __restrict__ gamma,
                                           const __nv_bfloat16* __restrict__ beta, __nv_bfloat16* __restrict__ y,
                                           int64_t rows, int width, float eps) {
  // one warp per row; two-pass, population variance (reading #2 in DESIGN.md); output rounded to bf16
  pdl_trigger();
  pdl_wait();
  int64_t row = (int64_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  int lane = threadIdx.x % 32;
  if (row >= rows) return;
  const __nv_bfloat16* xr = x + row * width;
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
    y[row * width + k] = __float2bfloat16_rn((to_f32(xr[k]) - mu) * rstd * to_f32(gamma[k]) + to_f32(beta[k]));
}

// The same for widths that are a multiple of 8 up to 1024 with 16-byte aligned rows: the row lives in registers (up to four
// 128-bit loads per lane), read once
__global__ void __launch_bounds__(256) layernorm_rows_bf16_vec_kernel(const __nv_bfloat16* __restrict__ x, const __nv_bfloat16* __restrict__ gamma,
                                                                      const __nv_bfloat16* __restrict__ beta, __nv_bfloat16* __restrict__ y,
                                                                      int64_t rows, int width, float eps) {
  pdl_trigger();
  pdl_wait();
  const int64_t row = (int64_t)blockIdx.x * 8 + threadIdx.x / 32;
  const int lane = threadIdx.x % 32, nv = width >> 3;
  if (row >= rows) return;
  const uint4* xr = reinterpret_cast<const uint4*>(x + row * width);
  float f[4][8];
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int vi = lane + 32 * i;
    const uint4 u = vi < nv ? xr[vi] : make_uint4(0u, 0u, 0u, 0u);
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      f[i][2 * j] = __uint_as_float(w[j] << 16);
      f[i][2 * j + 1] = __uint_as_float(w[j] & 0xffff0000u);
      s += f[i][2 * j] + f[i][2 * j + 1];
    }
  }
  const float mu = warp_sum(s) / (float)width;
  float v = 0.f;
#pragma unroll
  for (int i = 0; i < 4; ++i)
    if (lane + 32 * i < nv) {
#pragma unroll
      for (int j = 0; j < 8; ++j) { const float d = f[i][j] - mu; v = fmaf(d, d, v); }
    }
  const float rstd = rsqrtf(warp_sum(v) / (float)width + eps);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int vi = lane + 32 * i;
    if (vi < nv) {
      const uint4 g4 = __ldg(reinterpret_cast<const uint4*>(gamma) + vi), b4 = __ldg(reinterpret_cast<const uint4*>(beta) + vi);
      const uint32_t gw[4] = {g4.x, g4.y, g4.z, g4.w}, bw[4] = {b4.x, b4.y, b4.z, b4.w};
      uint32_t o[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float y0 = (f[i][2 * j] - mu) * rstd * __uint_as_float(gw[j] << 16) + __uint_as_float(bw[j] << 16);
        const float y1 = (f[i][2 * j + 1] - mu) * rstd * __uint_as_float(gw[j] & 0xffff0000u) + __uint_as_float(bw[j] & 0xffff0000u);
        o[j] = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(y0)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(y1)) << 16);
      }
      reinterpret_cast<uint4*>(y + row * width)[vi] = make_uint4(o[0], o[1], o[2], o[3]);
    }
  }
}

__global__ void fold_ln_z_mma_kernel(const __nv_bfloat16* __restrict__ w_b, const __nv_bfloat16* __restrict__ gamma,
                                     const __nv_bfloat16* __restrict__ beta, __nv_bfloat16* __restrict__ wfold,
                                     float* __restrict__ c1, float* __restrict__ c0, int c_z, int H, int H_pad) {
  fold_ln_z_mma_device(w_b, gamma, beta, wfold, c1, c0, c_z, H, H_pad, threadIdx.x, blockDim.x);
}

}  // namespace

cudaError_t launch_gemm_mma(const GemmMmaParams& p, cudaStream_t st, bool* fold_done) {
  if (fold_done) *fold_done = false;
  if (p.M <= 0 || p.N <= 0 || p.K <= 0) return cudaSuccess;
  if (gemm_tc_supports(p)) {
    if (fold_done) *fold_done = p.fold_w_b != nullptr;
    return launch_gemm_tc(p, st);
  }
  if (p.K % 8 != 0 || p.N % 8 != 0 || p.lda % 8 != 0 || p.residual != nullptr) return cudaErrorInvalidValue;   // residual: tcgen05 GEMM only
  const int64_t nb = (int64_t)p.nseg * ((p.N + BN - 1) / BN);
  if (nb * ((p.M + 127) / 128) >= 2 * 148) {   // enough 128-row tiles for two CTAs per SM
    dim3 grid((unsigned)nb, (unsigned)((p.M + 127) / 128));
    return launch_kernel(gemm_mma_kernel<4>, grid, dim3(256), 0, st, p.pdl, p);
  } else {
    dim3 grid((unsigned)nb, (unsigned)((p.M + 63) / 64));
    return launch_kernel(gemm_mma_kernel<2>, grid, dim3(256), 0, st, p.pdl, p);
  }
}

cudaError_t launch_layernorm_rows_bf16(const void* x, const void* gamma, const void* beta, void* y, int64_t rows,
                                       int width, float eps, cudaStream_t st) {
  unsigned blocks = (unsigned)((rows + 7) / 8);
  const bool vec = width % 8 == 0 && width <= 1024 &&
                   (((uintptr_t)x | (uintptr_t)y | (uintptr_t)gamma | (uintptr_t)beta) & 15) == 0;
  // a programmatic dependent of the previous kernel in the stream (in a stack: the previous block's output GEMM)
  return launch_kernel(vec ? layernorm_rows_bf16_vec_kernel : layernorm_rows_bf16_kernel, dim3(blocks), dim3(256), 0, st, true,
                       (const __nv_bfloat16*)x, (const __nv_bfloat16*)gamma, (const __nv_bfloat16*)beta, (__nv_bfloat16*)y, rows, width, eps);
}

cudaError_t launch_fold_ln_z_mma(const void* w_b, const void* gamma, const void* beta, void* wfold, float* c1, float* c0,
                                 int c_z, int H, int H_pad, cudaStream_t st) {
  fold_ln_z_mma_kernel<<<1, 256, 0, st>>>((const __nv_bfloat16*)w_b, (const __nv_bfloat16*)gamma,
                                          (const __nv_bfloat16*)beta, (__nv_bfloat16*)wfold, c1, c0, c_z, H, H_pad);
  return cudaGetLastError();
}

}  // namespace dcp
