// tcgen05 GEMMs of the bf16 path: the single-track projections (step a1) and the output projection (step a9).
//   PAPER.md:77-81 (sec 3.2): Q^(p) = f_Q(S^(p)); "keys and values are projected from the full single-track S"
//   BASELINE.json config 0:  out = W_o (sigmoid(s W_g) (.) softmax(...) V)
// C_seg[M, N] = A[M, K] (bf16 row-major = K-major) x W_seg[K, N] (bf16 row-major = MN-major B operand), fp32
// accumulation in tensor memory.  One 128 x TBN output tile per CTA (TBN = 128, or 64 when 128-wide tiles would not
// give every SM two CTAs), K streamed in 64-wide blocks through a 3-stage TMA / mbarrier ring (128-byte swizzle);
// two CTAs per SM overlap one tile's epilogue with the other's main loop.
//   warp 0    TMA producer: A box (64 k, 128 rows), W boxes (64 n, 64 k) x TBN / 64
//   warp 1    tcgen05 issuer (one lane): 4 x tcgen05.mma kind::f16 (M = 128, N = TBN, K = 16) per k-block
//   warps 2-9 epilogue: tcgen05.ld (thread = row, two warps per TMEM lane quadrant) -> bias / scale / sigmoid -> bf16
//             -> shared C tile -> coalesced global stores in the layout the fused kernel reads (gemm_mma.cu lists
//             the output modes)
// The launcher falls back to the mma.sync kernel (gemm_mma.cu) for shapes this tiling does not cover
// (N % 64, K % 64, unaligned pitches).  Every output element is accumulated over k in one fixed order.
#include <cstdlib>

#include "fold.cuh"
#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int TBM = 128, TBK = 64, TST = 3;
constexpr int kABytes = TBM * TBK * 2;                   // 16 KB
constexpr int kTcThreads = 64 + 256;                     // producer warp, issuer warp, 8 epilogue warps
// per output-tile width TBN (128, or 64 for grids that would not fill the GPU)
template <int TBN> struct TcCfg {
  static constexpr int kBBytes = TBN * TBK * 2;          // TBN / 64 boxes of (64 n x 64 k)
  static constexpr int kStage = kABytes + kBBytes;
  static constexpr int kCsPitch = TBN + 8;               // bf16 elements; +8: conflict-free 16-byte row writes
  static constexpr size_t kSmemBar = (size_t)TST * kStage;
  static constexpr size_t kSmemHd = kSmemBar + (2 * TST + 2) * 8 + 16;   // (head, head dim) of the tile's columns
  static constexpr size_t kSmemAlloc = kSmemHd + TBN * 4 + 1024;
  static_assert(TBM * kCsPitch * 2 <= TST * kStage, "C tile is staged in the pipeline buffers");
};

struct GemmTcMaps {
  CUtensorMap a;
  CUtensorMap w[4];
};

// MN-major operand tile (W[K][N], n contiguous), 128-byte swizzle: 64 n x 8 k atoms of 1024 B; atoms along k are
// SBO = 1024 B apart, the second 64-n block of the tile LBO = 64 k-rows * 128 B = 8192 B further
__device__ __forceinline__ uint64_t umma_desc_mn_sw128(uint32_t addr) {
  return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)(8192 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tmap, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld_x32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

template <int TBN>
__global__ void __launch_bounds__(kTcThreads, 2) gemm_tc_kernel(const __grid_constant__ GemmTcMaps maps, const GemmMmaParams p) {
  using Cfg = TcCfg<TBN>;
  constexpr int kTcStage = Cfg::kStage, kCsPitch = Cfg::kCsPitch;
  constexpr size_t kTcSmemBar = Cfg::kSmemBar;
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
  const uint32_t s_base = smem_u32(smem);
  const uint32_t s_bar = smem_u32(smem + kTcSmemBar);
  const uint32_t bar_full = s_bar, bar_empty = s_bar + 8 * TST, bar_acc = s_bar + 16 * TST;
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(smem + kTcSmemBar + (2 * TST + 2) * 8);

  pdl_trigger();
  if (blockIdx.y == gridDim.y - 1 && p.fold_w_b != nullptr) {
    // the extra CTA row of the launch: CTA 0 folds LayerNorm(z) into the bias projection weights, the others leave
    pdl_wait();
    if (blockIdx.x == 0 && threadIdx.x < 256)
      fold_ln_z_mma_device(p.fold_w_b, p.fold_gamma, p.fold_beta, p.fold_wfold, p.fold_c1, p.fold_c0, p.fold_c_z, p.fold_H,
                           p.fold_H_pad, threadIdx.x, 256);
    return;
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nb_per_seg = p.N / TBN;
  const int seg = blockIdx.x / nb_per_seg;
  const int n0 = (blockIdx.x % nb_per_seg) * TBN;
  const int m0 = blockIdx.y * TBM;
  const int nk = p.K / TBK;

  if (threadIdx.x == 0) {
    for (int s = 0; s < TST; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 1); }
    mbar_init(bar_acc, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), TBN);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *s_tmem;
  pdl_wait();                                                // the previous kernel's writes (A, the C buffers) are final

  if (warp == 0) {
    if (lane == 0) {
      // =============================================================== TMA producer
      const CUtensorMap* wmap = &maps.w[seg];
      for (int kb = 0; kb < nk; ++kb) {
        const int stage = kb % TST;
        mbar_wait(bar_empty + 8 * stage, ((kb / TST) & 1) ^ 1);
        mbar_expect_tx(bar_full + 8 * stage, kTcStage);
        const uint32_t dst = s_base + stage * kTcStage;
        tma_load_2d(dst, &maps.a, kb * TBK, m0, bar_full + 8 * stage);
#pragma unroll
        for (int nb = 0; nb < TBN / 64; ++nb)
          tma_load_2d(dst + kABytes + nb * 8192, wmap, n0 + 64 * nb, kb * TBK, bar_full + 8 * stage);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // =============================================================== tcgen05 issuer
      // instruction descriptor: D = f32, A = B = bf16, A K-major, B MN-major (bit 16), M = 128, N = 128
      constexpr uint32_t idesc = umma_idesc_bf16(TBM, TBN) | (1u << 16);
      for (int kb = 0; kb < nk; ++kb) {
        const int stage = kb % TST;
        mbar_wait(bar_full + 8 * stage, (kb / TST) & 1);
        tc_fence_after();
        const uint32_t a0 = s_base + stage * kTcStage, b0 = a0 + kABytes;
#pragma unroll
        for (int ks = 0; ks < TBK / 16; ++ks)
          umma_bf16(tmem_base, umma_desc_sw128(a0 + ks * 32), umma_desc_mn_sw128(b0 + ks * 2048), idesc, (kb | ks) != 0);
        umma_commit(bar_empty + 8 * stage);
      }
      umma_commit(bar_acc);
    }
  } else {
    // =============================================================== epilogue (warps 2-9: TMEM lane quadrant = warp % 4,
    // the two warps of a quadrant take one half of the tile's columns each)
    const int quad = warp & 3, half = (warp - 2) >> 2, et = threadIdx.x - 64;   // et: 0..255 among the epilogue threads
    const int row = quad * 32 + lane;                       // tile row of this thread = its TMEM lane
    const int mode = p.mode[seg];
    // C tile [128][kCsPitch] bf16, aliases the drained pipeline stages; (head, head dim) table of the tile's columns.
    // Both are read and written with explicit shared-memory instructions (generic loads of shared memory are slower).
    const uint32_t s_cs = s_base, s_hd = smem_u32(smem + Cfg::kSmemHd);
    short2* hd = reinterpret_cast<short2*>(smem + Cfg::kSmemHd);
    if (et < TBN && p.c > 0) hd[et] = make_short2((short)((n0 + et) / p.c), (short)((n0 + et) % p.c));   // one division per column
    mbar_wait(bar_acc, 0);
    tc_fence_after();
    const __nv_bfloat16* bias = reinterpret_cast<const __nv_bfloat16*>(p.bias[seg]);
    const float scale = mode == GEMM_OUT_HEADPAD ? p.scale[seg] : 1.f;
#pragma unroll
    for (int c32 = 0; c32 < TBN / 64; ++c32) {
      const int ch = half * (TBN / 64) + c32;               // 32-column chunk of the tile
      float v[32];
      tmem_ld_x32(tmem_base + ((uint32_t)(quad * 32) << 16) + ch * 32, v);
      tmem_ld_wait();
      if (bias != nullptr) {
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] += __bfloat162float(bias[n0 + ch * 32 + i]);
      }
      if (mode == GEMM_OUT_SIGMOID) {
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = 1.f / (1.f + expf(-v[i]));
      }
      if (mode == GEMM_OUT_PLAIN && p.residual != nullptr && m0 + row < p.M) {
        const uint4* rp = reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(p.residual) +
                                                         (int64_t)(m0 + row) * p.ldr + n0 + ch * 32);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const uint4 r = rp[i];                              // plain load: the buffer may be this kernel's own output
          const uint32_t rw[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            v[8 * i + 2 * j] += __uint_as_float(rw[j] << 16);
            v[8 * i + 2 * j + 1] += __uint_as_float(rw[j] & 0xffff0000u);
          }
        }
      }
      const uint32_t dst = s_cs + (row * kCsPitch + ch * 32) * 2;
#pragma unroll
      for (int i = 0; i < 4; ++i)
        sts_u32x4(dst + 16 * i,
                  make_uint4(pack_bf16(v[8 * i] * scale, v[8 * i + 1] * scale), pack_bf16(v[8 * i + 2] * scale, v[8 * i + 3] * scale),
                             pack_bf16(v[8 * i + 4] * scale, v[8 * i + 5] * scale), pack_bf16(v[8 * i + 6] * scale, v[8 * i + 7] * scale)));
    }
    tc_fence_before();
    asm volatile("bar.sync 1, 256;" ::: "memory");
    __nv_bfloat16* C = reinterpret_cast<__nv_bfloat16*>(p.C[seg]);
    if (mode == GEMM_OUT_PLAIN || mode == GEMM_OUT_SIGMOID || (mode == GEMM_OUT_HEADPAD && p.cp == p.c)) {
      // row-major rows (HEADPAD without padding is [row][H * c]): TBN / 8 lanes store one row segment of the tile
      const int64_t ldc = mode == GEMM_OUT_HEADPAD ? (int64_t)p.H * p.c : p.ldc[seg];
      for (int u = et; u < TBM * (TBN / 8); u += 256) {
        const int r = u / (TBN / 8), c8 = u % (TBN / 8);
        if (m0 + r < p.M)
          *reinterpret_cast<uint4*>(C + (int64_t)(m0 + r) * ldc + n0 + c8 * 8) = lds_u32x4(s_cs + (r * kCsPitch + c8 * 8) * 2);
      }
    } else if (mode == GEMM_OUT_HEADPAD) {
      for (int u = et; u < TBM * (TBN / 2); u += 256) {
        const int r = u / (TBN / 2), col = (u % (TBN / 2)) * 2;
        if (m0 + r < p.M) {
          const uint32_t hw = lds_u32(s_hd + col * 4);
          const int h = (short)(hw & 0xffffu), d = (short)(hw >> 16);  // c even, col even: the pair stays inside one head
          *reinterpret_cast<uint32_t*>(C + ((int64_t)(m0 + r) * p.H + h) * p.cp + d) = lds_u32(s_cs + (r * kCsPitch + col) * 2);
        }
      }
    } else {
      // K / V in the MMA B-fragment order of the fused kernels (see gemm_mma.cu): 8-byte units in destination order
      const int64_t tile_end = (p.M + 31) / 32 * 2;
      const bool is_k = mode == GEMM_OUT_KFRAG;
      for (int u = et; u < TBM * TBN / 4; u += 256) {
        const int b = u & 1, tt = (u >> 1) & 3, gg = (u >> 3) & 7, grp = (u >> 6) % (TBN / 16), kt = u / (TBN * 4);
        const int64_t tile = (m0 >> 4) + kt;
        if (tile >= tile_end) continue;
        uint2 v;
        int col;
        if (is_k) {
          col = grp * 16 + 4 * tt;
          v = lds_u32x2(s_cs + ((kt * 16 + 4 * (gg >> 1) + (gg & 1) + 2 * b) * kCsPitch + col) * 2);
        } else {
          col = grp * 16 + 8 * b + gg;
          const uint32_t src = s_cs + ((kt * 16 + 4 * tt) * kCsPitch + col) * 2;
          const uint32_t e0 = lds_u16(src), e1 = lds_u16(src + 2 * kCsPitch), e2 = lds_u16(src + 4 * kCsPitch), e3 = lds_u16(src + 6 * kCsPitch);
          v = make_uint2(e0 | (e1 << 16), e2 | (e3 << 16));
        }
        const uint32_t hw = lds_u32(s_hd + col * 4);
        const int h = (short)(hw & 0xffffu), d = (short)(hw >> 16);
        int64_t idx;
        if (is_k) idx = (((tile * p.H + h) * (p.cp >> 4) + (d >> 4)) * 32 + gg * 4 + ((d & 15) >> 2)) * 8 + b * 4;
        else idx = (((tile * p.H + h) * (p.cp >> 4) + (d >> 4)) * 32 + (d & 7) * 4 + tt) * 8 + ((d >> 3) & 1) * 4;
        *reinterpret_cast<uint2*>(C + idx) = v;
      }
    }
  }
  // teardown: the epilogue has drained tensor memory before the allocating warp frees it
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_base, TBN);
  }
}

}  // namespace

bool gemm_tc_supports(const GemmMmaParams& p) {
  if (p.M <= 0 || p.N % 64 != 0 || p.K % TBK != 0 || p.lda % 8 != 0 || ((uintptr_t)p.A & 15) != 0) return false;
  for (int s = 0; s < p.nseg; ++s) {
    if (((uintptr_t)p.W[s] & 15) != 0 || ((uintptr_t)p.C[s] & 15) != 0) return false;
    if ((p.mode[s] == GEMM_OUT_PLAIN || p.mode[s] == GEMM_OUT_SIGMOID) && p.ldc[s] % 8 != 0) return false;
    if (p.mode[s] == GEMM_OUT_TRANSPOSED) return false;
  }
  if (p.residual != nullptr && (p.ldr % 8 != 0 || ((uintptr_t)p.residual & 15) != 0)) return false;
  return get_encode_fn() != nullptr;
}

cudaError_t launch_gemm_tc(const GemmMmaParams& p, cudaStream_t st) {
  PFN_cuTensorMapEncodeTiled enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  GemmTcMaps maps;
  const cuuint32_t estr[2] = {1, 1};
  {
    const cuuint64_t gdim[2] = {(cuuint64_t)p.K, (cuuint64_t)p.M};
    const cuuint64_t gstr[1] = {(cuuint64_t)p.lda * 2};
    const cuuint32_t box[2] = {TBK, TBM};
    if (enc(&maps.a, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(p.A), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  for (int s = 0; s < 4; ++s) {
    const void* w = p.W[s < p.nseg ? s : 0];
    const cuuint64_t gdim[2] = {(cuuint64_t)p.N, (cuuint64_t)p.K};
    const cuuint64_t gstr[1] = {(cuuint64_t)p.N * 2};
    const cuuint32_t box[2] = {64, TBK};
    if (enc(&maps.w[s], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(w), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {   // per-device function attribute: set on every launch (cheap), so a process may use several GPUs
    cudaError_t e = cudaFuncSetAttribute(gemm_tc_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TcCfg<128>::kSmemAlloc);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(gemm_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TcCfg<64>::kSmemAlloc);
    if (e != cudaSuccess) return e;
  }
  const unsigned mt_tiles = (unsigned)((p.M + TBM - 1) / TBM);
  const unsigned mt = mt_tiles + (p.fold_w_b != nullptr ? 1u : 0u);     // + the row that carries the LayerNorm(z) fold
  // 128-wide tiles when they give every SM two CTAs (or N does not split into 64s evenly enough to matter)
  static const int force = [] { const char* e = getenv("DCP_GEMM_TBN"); return e ? atoi(e) : 0; }();
  if (force != 64 && p.N % 128 == 0 && (force == 128 || (int64_t)p.nseg * (p.N / 128) * mt_tiles >= 2 * 148)) {
    dim3 grid((unsigned)(p.nseg * (p.N / 128)), mt);
    return launch_kernel(gemm_tc_kernel<128>, grid, dim3(kTcThreads), TcCfg<128>::kSmemAlloc, st, p.pdl, maps, p);
  } else {
    dim3 grid((unsigned)(p.nseg * (p.N / 64)), mt);
    return launch_kernel(gemm_tc_kernel<64>, grid, dim3(kTcThreads), TcCfg<64>::kSmemAlloc, st, p.pdl, maps, p);
  }
}

}  // namespace dcp
