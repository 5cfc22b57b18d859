// Bias cache for the attention stack on a read-only pair tensor ("cached" mode).
// Every block b of the stack derives its own bias  LN_b(z_ij) W_b^b  from the SAME pair tensor; one pass over z computes
// the biases of up to 23 blocks at once -- LayerNorm statistics once per pair, one tcgen05 projection with
// N = 16 heads x n_blocks + the ones column -- and writes them as fp16 tiles in exactly the layout the attention kernel
// consumes ([query tile of 32][key tile of 16][head pair][32 queries][16 keys] half2, 16 KB per tile), so that each block
// afterwards streams 32 bytes per pair instead of the 256 bytes of z (the paper's own stack materialises
// B in R^{I x I x H} per block).  Values are in the exp2 domain (W' carries log2 e), like the fused kernel's.
//
// One persistent CTA per SM, 12 warps: warp 0 TMA producer (z boxes as in fused_mma.cu), warps 1-2 tcgen05 issuers,
// warps 4-11 statistics + epilogue (thread = pair; warps w and w + 4 of a tensor-memory lane quadrant take every other block).
#include "fold.cuh"
#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int bCz = 128, bH = 16, bTileQ = 32, bTileK = 16, bSubQ = 8, bNZ = 3, bNT = 2;
constexpr int bStageBytes = bSubQ * bTileK * bCz * 2;      // 32 KB
constexpr int bHalfBytes = bStageBytes / 2;
constexpr int bOneBuf = 15;                                 // 16 * 15 + 16 = 256 projection columns: one MMA, two accumulator buffers
constexpr int bMaxBlocks = 23;                              // 16 * 23 + 16 = 384 columns in the X / Y split (below)
constexpr int bMaxN = 384;                                  // rows of W''
constexpr int bThreads = 384;
constexpr int bEpiWarps = 8;                                // warps w and w + 4 share a lane quadrant and alternate blocks
constexpr size_t bSmemZ = 0;
constexpr size_t bSmemWt = bSmemZ + (size_t)bNZ * bStageBytes;            // 2 halves x 384 rows x 128 B = 96 KB
constexpr size_t bSmemC = bSmemWt + 2 * (size_t)bMaxN * 128;              // c1, c0: [23][16] floats each
constexpr size_t bSmemBar = bSmemC + 2 * bMaxBlocks * bH * 4;
constexpr int bNumBars = 2 * bNZ + 2 * bNT + 2;             // z full / empty, X full / empty (two buffers), Y full / empty
constexpr size_t bSmemAlloc = bSmemBar + bNumBars * 8 + 16 + 1024;

// Column plan of a pass of nb blocks.  Up to 15 blocks everything is one region X = [blocks | ones] of 16 nb + 16 <= 256
// columns, double buffered in tensor memory (NY = 0).  16 .. 23 blocks need 272 .. 384 columns, which do not fit twice into
// the 512 columns: the columns are split into Y = [ones | the first blocks] (NY columns, ONE buffer) and X = [the other
// blocks] (NX columns, two buffers), 2 NX + NY <= 512.  Y's MMA is issued first and its columns are read first, so the
// next stage's Y MMA waits only for that part of the epilogue; X stays double buffered.
struct ColPlan { int NX, NY, y_blocks; };
__host__ __device__ inline ColPlan col_plan(int nb) {
  if (nb <= bOneBuf) return ColPlan{16 * nb + 16, 0, 0};
  const int T = 16 * nb + 16;
  const int NX = (512 - T) / 64 * 64;                        // the widest double-buffered part that leaves room for Y; buffers
                                                             // start at multiples of 64 columns
  return ColPlan{NX, T - NX, (T - NX) / 16 - 1};
}

struct BiasTilesParams {
  const void* wfold;       // [n_blocks][16][128] bf16
  const float* c1;         // [n_blocks][16]
  const float* c0;         // [n_blocks][16]
  uint32_t* cache;         // block b: cache + b * block_words; tile (qt, kt): + (qt * KT + kt) * 4096 + ((q / 8) * 8 + hp) * 128 + (q % 8) * 16 + key
  int64_t block_words;
  int I, n_blocks, KT, n_tiles;
  float eps;
};

__global__ void __launch_bounds__(bThreads, 1) bias_tiles_kernel(const __grid_constant__ CUtensorMap tmap_z, const BiasTilesParams p) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
  const uint32_t s_z = smem_u32(smem + bSmemZ), s_wt = smem_u32(smem + bSmemWt), s_bar = smem_u32(smem + bSmemBar);
  float* s_c1 = reinterpret_cast<float*>(smem + bSmemC);
  const uint32_t s_c = smem_u32(smem + bSmemC);
  float* s_c0 = s_c1 + bMaxBlocks * bH;
  const uint32_t bar_zfull = s_bar, bar_zempty = s_bar + 8 * bNZ, bar_tfull = s_bar + 16 * bNZ, bar_tempty = bar_tfull + 8 * bNT;
  const uint32_t bar_yfull = bar_tempty + 8 * bNT, bar_yempty = bar_yfull + 8;
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(smem + bSmemBar + bNumBars * 8);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int NP = 16 * p.n_blocks + 16;                       // projection columns: heads of every block, ones, zero rows
  const ColPlan cp = col_plan(p.n_blocks);
  const int NX = cp.NX, NY = cp.NY, yb = cp.y_blocks;        // Y holds the ones column and blocks [0, yb); X blocks [yb, nb)

  pdl_trigger();
  if (threadIdx.x == 0) {
    // z_empty: the commits of the stage's MMAs (one thread's, or the Y and the X thread's) + the four epilogue warps
    for (int s = 0; s < bNZ; ++s) { mbar_init(bar_zfull + 8 * s, 1); mbar_init(bar_zempty + 8 * s, (NY > 0 ? 2 : 1) + bEpiWarps); }
    for (int b = 0; b < bNT; ++b) { mbar_init(bar_tfull + 8 * b, 1); mbar_init(bar_tempty + 8 * b, bEpiWarps); }
    mbar_init(bar_yfull, 1);
    mbar_init(bar_yempty, bEpiWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), 512);
  pdl_wait();
  // W'' rows in column order, K-major, 128-byte swizzle by hand.  One region: row n < 16 nb = head n % 16 of block n / 16,
  // row 16 nb = ones, others 0.  Split: rows [0, NY) = Y = [ones, 15 zero rows | blocks 0 .. yb), rows [NY, NY + NX) = X.
  for (int e = threadIdx.x; e < NP * (bCz / 8); e += bThreads) {
    const int n = e / (bCz / 8), ch16 = e % (bCz / 8);
    int src = -2;                                            // -2: zero row, -1: ones, >= 0: row of wfold
    if (NY == 0) src = n < 16 * p.n_blocks ? n : (n == 16 * p.n_blocks ? -1 : -2);
    else src = n == 0 ? -1 : (n < 16 ? -2 : n - 16);
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (src >= 0) v = __ldg(reinterpret_cast<const uint4*>(p.wfold) + src * (bCz / 8) + ch16);
    else if (src == -1) v = make_uint4(0x3f803f80u, 0x3f803f80u, 0x3f803f80u, 0x3f803f80u);
    const int half = ch16 >> 3, c = ch16 & 7;
    *reinterpret_cast<uint4*>(smem + bSmemWt + half * (bMaxN * 128) + n * 128 + ((c ^ (n & 7)) << 4)) = v;
  }
  for (int e = threadIdx.x; e < p.n_blocks * bH; e += bThreads) { s_c1[e] = __ldg(p.c1 + e); s_c0[e] = __ldg(p.c0 + e); }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *s_tmem;

  if (warp == 0) {
    if (lane == 0) {
      // =============================================================== TMA producer
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
        const int q0 = (tile / p.KT) * bTileQ, j0 = (tile % p.KT) * bTileK;
        for (int sub = 0; sub < bTileQ / bSubQ; ++sub, ++it) {
          const int stage = it % bNZ;
          mbar_wait(bar_zempty + 8 * stage, ((it / bNZ) & 1) ^ 1);
          mbar_expect_tx(bar_zfull + 8 * stage, bStageBytes);
          const uint32_t dst = s_z + stage * bStageBytes;
          tma_load_3d(dst, &tmap_z, 0, j0, q0 + sub * bSubQ, bar_zfull + 8 * stage, policy);
          tma_load_3d(dst + bHalfBytes, &tmap_z, 64, j0, q0 + sub * bSubQ, bar_zfull + 8 * stage, policy);
        }
      }
    }
  } else if (warp <= 3) {
    if (warp <= 2 && lane == 0) {
      // =============================================================== tcgen05 issuers (stage n -> issuer n % 2: with two
      // accumulator buffers a buffer's consecutive users are then the same thread, so its parity waits cannot alias)
      const uint32_t idesc_x = umma_idesc_bf16(128, NX), idesc_y = umma_idesc_bf16(128, NY > 0 ? NY : 16);
      const uint32_t x_stride = NY == 0 ? 256u : (uint32_t)NX;          // tensor-memory columns between the two X buffers
      const uint32_t me = warp - 1;
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
        for (int sub = 0; sub < bTileQ / bSubQ; ++sub, ++it) {
          const int stage = it % bNZ, tb = it % bNT;
          const uint32_t zs = s_z + stage * bStageBytes;
          if (NY == 0) {
            // one region: stage n -> issuer n % 2 (with two accumulator buffers a buffer's consecutive users are then the
            // same thread, so its parity waits cannot alias)
            if (it % 2 != me) continue;
            mbar_wait(bar_tempty + 8 * tb, ((it / bNT) & 1) ^ 1);
            mbar_wait(bar_zfull + 8 * stage, (it / bNZ) & 1);
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
              umma_bf16(tmem_base + tb * x_stride, umma_desc_sw128(zs + (ks >> 2) * bHalfBytes + (ks & 3) * 32),
                        umma_desc_sw128(s_wt + (ks >> 2) * (bMaxN * 128) + (ks & 3) * 32), idesc_x, ks > 0);
            umma_commit(bar_zempty + 8 * stage);
            umma_commit(bar_tfull + 8 * tb);
          } else if (me == 0) {
            // split columns: this thread issues every stage's Y MMA.  Y has ONE buffer, so its users must be one thread: a
            // thread that alternated stages with another could be two phases ahead of y_empty and its parity wait would
            // pass early.  The buffer is free once the epilogue of the previous stage has read it (completion it - 1).
            mbar_wait(bar_zfull + 8 * stage, (it / bNZ) & 1);
            mbar_wait(bar_yempty, (it & 1) ^ 1);
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
              umma_bf16(tmem_base + 2 * NX, umma_desc_sw128(zs + (ks >> 2) * bHalfBytes + (ks & 3) * 32),
                        umma_desc_sw128(s_wt + (ks >> 2) * (bMaxN * 128) + (ks & 3) * 32), idesc_y, ks > 0);
            umma_commit(bar_zempty + 8 * stage);
            umma_commit(bar_yfull);
          } else {
            // ... and this one every stage's X MMA (two buffers)
            mbar_wait(bar_zfull + 8 * stage, (it / bNZ) & 1);
            mbar_wait(bar_tempty + 8 * tb, ((it / bNT) & 1) ^ 1);
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
              umma_bf16(tmem_base + tb * x_stride, umma_desc_sw128(zs + (ks >> 2) * bHalfBytes + (ks & 3) * 32),
                        umma_desc_sw128(s_wt + (ks >> 2) * (bMaxN * 128) + NY * 128 + (ks & 3) * 32), idesc_x, ks > 0);
            umma_commit(bar_zempty + 8 * stage);
            umma_commit(bar_tfull + 8 * tb);
          }
        }
      }
    }
  } else {
    // =============================================================== LayerNorm statistics + epilogue, thread = pair
    const int pw = warp & 3, par = (warp - 4) >> 2;        // lane quadrant; which of every two blocks this thread writes
    const uint32_t t_lane = tmem_base + ((uint32_t)(pw * 32) << 16);
    const int prow = pw * 32 + lane;
    const uint32_t zrow = s_z + prow * 128, zsw = (uint32_t)(prow & 7);
    uint32_t it = 0;
    for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
      for (int sub = 0; sub < bTileQ / bSubQ; ++sub, ++it) {
        const int stage = it % bNZ, tb = it % bNT;
        mbar_wait(bar_zfull + 8 * stage, (it / bNZ) & 1);
        float sq0 = 0.f, sq1 = 0.f, sq2 = 0.f, sq3 = 0.f;
        const uint32_t zr = zrow + stage * bStageBytes;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint4 w[8];
#pragma unroll
          for (int c = 0; c < 8; ++c) w[c] = lds_u32x4(zr + half * bHalfBytes + ((c ^ zsw) << 4));
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            fma_sq_bf16x2(sq0, sq1, w[c].x); fma_sq_bf16x2(sq2, sq3, w[c].y);
            fma_sq_bf16x2(sq0, sq1, w[c].z); fma_sq_bf16x2(sq2, sq3, w[c].w);
          }
        }
        float zsq = (sq0 + sq1) + (sq2 + sq3);
        asm volatile("" : "+f"(zsq));
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_zempty + 8 * stage);
        // the ones column (sum_k z) comes first: from Y when the columns are split, else from the X buffer
        const uint32_t t_x = t_lane + tb * (NY == 0 ? 256u : (uint32_t)NX), t_y = t_lane + 2 * NX;
        if (NY > 0) mbar_wait(bar_yfull, it & 1); else mbar_wait(bar_tfull + 8 * tb, (it / bNT) & 1);
        tc_fence_after();
        const float zsum = tmem_ld_x1(NY > 0 ? t_y : t_x + 16 * p.n_blocks);
        tmem_ld_wait();
        const float mu = zsum * (1.f / bCz);
        const float var = fmaf(-mu, mu, zsq * (1.f / bCz));      // one rounding; exactly 0 for a constant row (fused_mma.cu)
        const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;
        const float nm = -mu * rstd;
        // tile layout [sub 4][head pair 8][8 queries][16 keys] words: a stage writes one contiguous 4 KB piece per block
        uint32_t* dst = p.cache + (int64_t)tile * (8 * 512) + sub * (8 * bSubQ * bTileK) + prow;
        auto emit = [&](float (&acc)[16], int b) {
#pragma unroll
          for (int i = 0; i < 16; ++i) asm volatile("" : "+f"(acc[i]));        // not before the wait that completes the load
          // explicit ld.shared (generic-pointer loads compiled to LD.E: 16 of them per pair row paced this epilogue)
          const uint32_t c1 = s_c + b * (bH * 4), c0 = c1 + bMaxBlocks * bH * 4;
          uint32_t* d = dst + (int64_t)b * p.block_words;
#pragma unroll
          for (int h4 = 0; h4 < 4; ++h4) {
            const float4 a1 = lds_f32x4(c1 + 16 * h4), a0 = lds_f32x4(c0 + 16 * h4);
            d[(2 * h4) * 128] = pack_f16(fmaf(acc[4 * h4], rstd, fmaf(nm, a1.x, a0.x)), fmaf(acc[4 * h4 + 1], rstd, fmaf(nm, a1.y, a0.y)));
            d[(2 * h4 + 1) * 128] = pack_f16(fmaf(acc[4 * h4 + 2], rstd, fmaf(nm, a1.z, a0.z)), fmaf(acc[4 * h4 + 3], rstd, fmaf(nm, a1.w, a0.w)));
          }
        };
        // blocks [b0, b0 + n) live in 16-column groups from t_col on; block b's columns are processed while block b + 1's are
        // in flight (one tcgen05.ld ahead)
        auto region = [&](uint32_t t_col, int b0, int n) {
          float accA[16], accB[16];
          if (par < n) tmem_ld_x16(t_col + 16 * par, accA);
          for (int j = par; j < n; j += 4) {
            tmem_ld_wait();
            if (j + 2 < n) tmem_ld_x16(t_col + 16 * (j + 2), accB);
            emit(accA, b0 + j);
            if (j + 2 < n) {
              tmem_ld_wait();
              if (j + 4 < n) tmem_ld_x16(t_col + 16 * (j + 4), accA);
              emit(accB, b0 + j + 2);
            }
          }
        };
        if (NY > 0) {
          region(t_y + 16, 0, yb);                               // Y = [ones | blocks 0 .. yb): read first, freed first
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_yempty);
          mbar_wait(bar_tfull + 8 * tb, (it / bNT) & 1);
          tc_fence_after();
        }
        region(t_x, yb, p.n_blocks - yb);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty + 8 * tb);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_base, 512);
  }
}

struct FoldAllParams {
  const void* w_b[bMaxBlocks];
  const void* gamma[bMaxBlocks];
  const void* beta[bMaxBlocks];
  void* wfold;
  float *c1, *c0;
};
__global__ void __launch_bounds__(256) fold_all_kernel(const FoldAllParams f) {
  pdl_trigger();
  pdl_wait();
  const int b = blockIdx.x;
  fold_ln_z_mma_device(f.w_b[b], f.gamma[b], f.beta[b], reinterpret_cast<__nv_bfloat16*>(f.wfold) + (size_t)b * bH * bCz,
                       f.c1 + b * bH, f.c0 + b * bH, bCz, bH, bH, threadIdx.x, 256);
}

}  // namespace

int bias_tiles_max_blocks() { return bMaxBlocks; }
int64_t bias_tiles_block_words(int64_t I) { return ((I + bTileQ - 1) / bTileQ) * ((I + bTileK - 1) / bTileK) * 8 * 512; }
size_t bias_tiles_fold_bytes(int n_blocks) { return (size_t)n_blocks * (bH * bCz * 2 + 2 * bH * 4) + 512; }

// Biases of blocks [0, n_blocks) (n_blocks <= 23) of one pass: fold (one small launch) + the streaming kernel.
cudaError_t launch_bias_tiles(const void* z, int64_t ldz, int64_t I, const dcp_weights* blocks, int n_blocks, float eps,
                              void* fold_ws, void* cache, cudaStream_t st) {
  if (n_blocks < 1 || n_blocks > bMaxBlocks) return cudaErrorInvalidValue;
  PFN_cuTensorMapEncodeTiled enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  FoldAllParams f{};
  for (int b = 0; b < n_blocks; ++b) { f.w_b[b] = blocks[b].w_b; f.gamma[b] = blocks[b].ln_z_gamma; f.beta[b] = blocks[b].ln_z_beta; }
  char* ws = reinterpret_cast<char*>(fold_ws);
  f.wfold = ws;
  f.c1 = reinterpret_cast<float*>(ws + ((size_t)n_blocks * bH * bCz * 2 + 255) / 256 * 256);
  f.c0 = f.c1 + n_blocks * bH;
  cudaError_t e = launch_kernel(fold_all_kernel, dim3(n_blocks), dim3(256), 0, st, true, f);
  if (e != cudaSuccess) return e;
  CUtensorMap tm;
  const cuuint64_t gdim[3] = {(cuuint64_t)bCz, (cuuint64_t)I, (cuuint64_t)I};
  const cuuint64_t gstr[2] = {(cuuint64_t)bCz * 2, (cuuint64_t)ldz * 2};
  const cuuint32_t box[3] = {64, bTileK, bSubQ};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(z), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  BiasTilesParams p{};
  p.wfold = f.wfold; p.c1 = f.c1; p.c0 = f.c0;
  p.cache = reinterpret_cast<uint32_t*>(cache);
  p.block_words = bias_tiles_block_words(I);
  p.I = (int)I; p.n_blocks = n_blocks;
  p.KT = (int)((I + bTileK - 1) / bTileK);
  const int64_t n_tiles = ((I + bTileQ - 1) / bTileQ) * p.KT;
  if (n_tiles > 0x7fffffff) return cudaErrorInvalidValue;
  p.n_tiles = (int)n_tiles;
  p.eps = eps;
  e = cudaFuncSetAttribute(bias_tiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bSmemAlloc);
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (sms <= 0) sms = 148;
  const unsigned grid = (unsigned)(n_tiles < sms ? n_tiles : sms);
  return launch_kernel(bias_tiles_kernel, dim3(grid), dim3(bThreads), bSmemAlloc, st, true, tm, p);
}

}  // namespace dcp
