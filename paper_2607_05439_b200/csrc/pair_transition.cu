// Pairwise SwiGLU transition on the pair tensor, bf16, c_z = 128, hidden 4 c_z = 512.
//   PAPER.md:381-385 (Eq. 6)   Transition(Z) = W_3 ( SiLU(W_1 LN(Z)) (.) W_2 LN(Z) ),  Z <- Z + Transition(Z)
//   PAPER.md:387-409 (Alg. 1)  the memory-friendly order N, A, B, SiLU, (.), W_3, residual -- here per 128-pair tile,
//                              so the 4 c_z-wide intermediates never leave the SM at all.
// ~393 kflop per pair over 512 bytes of traffic (read + write z): tensor bound.
//
// LayerNorm is folded into the first GEMM:
//   LN(z) W = rstd (z . W' - mu c1 + (1 / rstd) c0),  W' = diag(gamma) W, c1[j] = sum_k W'[k][j], c0[j] = sum_k beta_k W[k][j]
// The raw z tile, as TMA wrote it (K-major, 128-byte swizzle), is the A operand of 8 k-steps; a ninth k-step multiplies
// the K extension [-mu, 1 / rstd, 0 ...] (written per row by the epilogue warps) with the weight rows [c1; c0; 0 ...],
// so the accumulator only has to be scaled by the row's rstd: no per-column constants in the epilogue.
//
// One persistent CTA per SM, 10 warps, CTAs launched as clusters of two that walk the weight chunks in lockstep:
//   warp 0     TMA producer: z tiles (128 pairs x 128 ch = 32 KB, double buffered) and, per 128-wide hidden chunk c,
//              the weight tiles W1'[:, c], W2'[:, c] (two 64-row k-blocks of 32 KB in a three-slot ring, refilled in the
//              order in which the tensor pipe frees them) and W3[c, :] (32 KB) -- row-major weights are MN-major B
//              operands.  Each CTA of the pair fetches half of every weight tile and multicasts it to both, so a weight
//              byte leaves L2 once per tile pair; the slot-free barriers collect one tcgen05.commit from each CTA.
//   warp 1     tcgen05 issuer: G1(c): [A1 | A2] (128 x 256, TMEM) = [z | -mu, 1/rstd] . [W1'c | W2'c ; c1 ; c0]  (9 k-steps)
//                              G2(c): OUT (128 x 128, TMEM) += H_c . W3_c   (8 k-steps, H_c read from TMEM: A-in-TMEM form)
//              issued as G1(0), G1(1), G2(0), G1(2), G2(1), G1(3), G2(2), G2(3): the tensor pipe works on the next
//              chunk while the epilogue warps turn the previous one into H
//   warps 2-9  epilogue (TMEM lane quadrant = warp % 4, two warps per quadrant = two 64-column halves): per chunk
//              tcgen05.ld A1, A2 -> h = SiLU(rstd A1) rstd A2 -> bf16x2 -> tcgen05.st into the H columns of TMEM
//              (lane = row, one column = two hidden units; double buffered); per tile OUT + z -> bf16, written over
//              the thread's own bytes of the z tile -> TMA store from there.
// TMEM: A1 [0,128) A2 [128,256) OUT [256,384) H [384,448) [448,512).  Shared memory: z 64 KB, W12 ring 96 KB, W3 32 KB,
// K extension 8 + 16 KB.  What limits it (what-if builds): the weight bytes every SM has to take in per
// tile (416 KB) and the accumulator hand-offs between the tensor pipe and the epilogue warps.
#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int tCz = 128, tHid = 512, tNC = 128, tChunks = tHid / tNC, tM = 128;
constexpr int tThreads = 64 + 256 + 128;     // producer, issuer, 8 epilogue warps, 4 output warps
constexpr int tCluster = 2;                    // CTA pair: every weight tile is read from L2 once and multicast to both
constexpr uint16_t tClusterMask = (1u << tCluster) - 1;
constexpr int tZBytes = tM * tCz * 2;          // 32 KB, two 64-channel halves of 16 KB
constexpr int tW12Bytes = 2 * tCz * tNC * 2;   // 64 KB: per k-block of 64: [W1 n-half 0][W1 n-half 1][W2 n-half 0][W2 n-half 1]
constexpr int tW3Bytes = tNC * tCz * 2;        // 32 KB: per k-block of 64: [n-half 0][n-half 1]
constexpr int tKx = 16;                        // the K extension: channels 128..133 (-mu terms), 134..136 (1 / rstd terms), zeros
constexpr int tZxBytes = tM * tKx * 2;         // 4 KB per z buffer, K-major, 32-byte swizzle
constexpr int tW12xBytes = 4 * 64 * tKx * 2;   // 8 KB: rows k = 128..143 of [W1'c | W2'c], four 64-n blocks of 2 KB
constexpr size_t tSmemZ = 0;
constexpr int tW12Slot = tW12Bytes / 2;         // 32 KB: one k-block of a chunk; a ring of three slots
constexpr size_t tSmemW12 = tSmemZ + 2 * (size_t)tZBytes;
constexpr size_t tSmemW3 = tSmemW12 + 3 * (size_t)tW12Slot;
constexpr size_t tSmemZx = tSmemW3 + tW3Bytes;
constexpr size_t tSmemW12x = tSmemZx + 2 * (size_t)tZxBytes;
constexpr size_t tSmemBar = tSmemW12x + 2 * (size_t)tW12xBytes;
constexpr size_t tSmemAlloc = tSmemBar + 24 * 8 + 1024;
constexpr int tColA1 = 0, tColOut = 256, tColH = 384;       // TMEM columns: A1 [0,128) A2 [128,256) OUT [256,384)
                                                            // H (bf16x2, the A operand of G2) [384,448) and [448,512)

struct TransMaps {
  CUtensorMap z_in, z_out, w1, w2, w3, w1x, w2x;   // w1x / w2x: the same folded weights with a (64 n, 16 k) box
};

// K-major A tile, 32-byte swizzle (rows of 16 bf16, 8-row groups 256 B apart): the K extension of the z tile
__device__ __forceinline__ uint64_t umma_desc_k_sw32(uint32_t addr) {
  return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)6 << 61);
}

// MN-major B tile, 128-byte swizzle, 64-n blocks `lbo` bytes apart, 8-k-row atoms 1024 B apart
__device__ __forceinline__ uint64_t umma_desc_mn(uint32_t addr, uint32_t lbo) {
  return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void tma_load_2d_t(uint32_t dst, const CUtensorMap* tmap, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
// the same load written to the same shared-memory offset (and signalled on the same barrier offset) of every CTA in cta_mask
__device__ __forceinline__ void tma_load_2d_mc(uint32_t dst, const CUtensorMap* tmap, int c0, int c1, uint32_t bar, uint16_t cta_mask) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;"
               ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar), "h"(cta_mask) : "memory");
}
// tcgen05.commit arriving on the barrier at this offset in every CTA of cta_mask
__device__ __forceinline__ void umma_commit_mc(uint32_t bar, uint16_t cta_mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(cta_mask) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tmap, int c0, int c1, uint32_t src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
               ::"l"(tmap), "r"(c0), "r"(c1), "r"(src) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
// 16 consecutive 32-bit columns of the thread's TMEM lane
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
// D[tmem] (+)= A[tmem: lane = row, one column = two consecutive k] . B[smem]
__device__ __forceinline__ void umma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ float tanh_fast(float x) {
  float y;
  asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// acc_s += lo(w) + hi(w), acc_q += lo(w)^2 + hi(w)^2  (bf16x2 word, mixed-precision FMAs)
__device__ __forceinline__ void stats_bf16x2(float& acc_s, float& acc_q, uint32_t w) {
  asm("{\n\t.reg .b16 l, h, o;\n\t"
      "mov.b32 {l, h}, %2;\n\t"
      "mov.b16 o, 0x3f80;\n\t"
      "fma.rn.f32.bf16 %0, l, o, %0;\n\t"
      "fma.rn.f32.bf16 %0, h, o, %0;\n\t"
      "fma.rn.f32.bf16 %1, l, l, %1;\n\t"
      "fma.rn.f32.bf16 %1, h, h, %1;\n\t}"
      : "+f"(acc_s), "+f"(acc_q) : "r"(w));
}

__global__ void __cluster_dims__(tCluster, 1, 1) __launch_bounds__(tThreads, 1) pair_transition_kernel(const __grid_constant__ TransMaps maps,
                                                                      int64_t n_pairs, float eps) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
  const uint32_t s_z = smem_u32(smem + tSmemZ), s_w12 = smem_u32(smem + tSmemW12), s_w3 = smem_u32(smem + tSmemW3);
  const uint32_t s_bar = smem_u32(smem + tSmemBar);
  const uint32_t s_zx = smem_u32(smem + tSmemZx), s_w12x = smem_u32(smem + tSmemW12x);
  // barriers
  // (8 bytes each; z, x, h: one per buffer; w12: one per ring slot)
  const uint32_t b_zfull = s_bar, b_zempty = s_bar + 16, b_w12full = s_bar + 32, b_w12empty = s_bar + 56, b_w3full = s_bar + 80,
                 b_w3empty = s_bar + 88, b_afull = s_bar + 96, b_aempty = s_bar + 104, b_hfull = s_bar + 112,
                 b_hempty = s_bar + 128, b_ofull = s_bar + 144, b_oempty = s_bar + 152, b_xfull = s_bar + 160;
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(smem + tSmemBar + 22 * 8);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int b = 0; b < 2; ++b) { mbar_init(b_zfull + 8 * b, 1); mbar_init(b_zempty + 8 * b, 1); }
    for (int b = 0; b < 3; ++b) { mbar_init(b_w12full + 8 * b, 1); mbar_init(b_w12empty + 8 * b, tCluster); }
    mbar_init(b_w3full, 1); mbar_init(b_w3empty, tCluster);
    mbar_init(b_afull, 1); mbar_init(b_aempty, 8);
    for (int b = 0; b < 2; ++b) { mbar_init(b_hfull + 8 * b, 8); mbar_init(b_hempty + 8 * b, 1); }
    mbar_init(b_ofull, 1); mbar_init(b_oempty, 4);
    mbar_init(b_xfull, 4); mbar_init(b_xfull + 8, 4);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                        // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  const uint32_t tmem_base = *s_tmem;
  // Tiles go to CTA pairs: pair p of tiles (2 p, 2 p + 1) to cluster p % n_clusters, tile 2 p + rank to the CTA of
  // that rank, so that both CTAs of a cluster walk the weight chunks in lockstep.  A tile index == n_tiles (odd tile
  // count) is a phantom: its loads are zero-filled and its store is clipped by the tensor map.
  const int64_t n_tiles = (n_pairs + tM - 1) / tM;
  uint32_t rank;
  asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
  const int64_t n_clusters = gridDim.x / tCluster, cid = blockIdx.x / tCluster, n_tpairs = (n_tiles + tCluster - 1) / tCluster;
  const int n_it = cid < n_tpairs ? (int)((n_tpairs - cid + n_clusters - 1) / n_clusters) : 0;
  auto tile_of = [&](int it) -> int64_t { return (cid + (int64_t)it * n_clusters) * tCluster + rank; };

  if (warp == 0) {
    if (lane == 0) {
      // =============================================================== TMA producer
      auto load_z = [&](int64_t tile, int it) {
        const int zb = it & 1;
        mbar_wait(b_zempty + 8 * zb, ((it >> 1) & 1) ^ 1);
        mbar_expect_tx(b_zfull + 8 * zb, tZBytes);
        tma_load_2d_t(s_z + zb * tZBytes, &maps.z_in, 0, (int)(tile * tM), b_zfull + 8 * zb);
        tma_load_2d_t(s_z + zb * tZBytes + tZBytes / 2, &maps.z_in, 64, (int)(tile * tM), b_zfull + 8 * zb);
      };
      // The CTA's chunks are numbered g = 4 it + c across its tiles; the weights of chunk g are those of c = g & 3.
      // k-block j = 2 g + kb of [W1'c | W2'c] goes to ring slot j % 3 (use number j / 3); the K-extension rows of chunk g
      // ride on the kb = 1 load (buffer g & 1: free because slot j - 3's release follows every MMA of chunk g - 2).
      const uint32_t n_kblocks = (uint32_t)n_it * tChunks * 2;
      auto load_w12 = [&](uint32_t j) {
        if (j >= n_kblocks) return;
        const uint32_t g = j >> 1, kb = j & 1, c = g & 3, slot = j % 3, use = j / 3;
        mbar_wait(b_w12empty + 8 * slot, (use & 1) ^ 1);
        mbar_expect_tx(b_w12full + 8 * slot, tW12Slot + (kb ? tW12xBytes : 0));
        const uint32_t base = s_w12 + slot * tW12Slot;
        // rank 0 fetches the W1' boxes, rank 1 the W2' boxes, each for both CTAs
        const CUtensorMap* wm = rank ? &maps.w2 : &maps.w1;
        const CUtensorMap* wxm = rank ? &maps.w2x : &maps.w1x;
#pragma unroll
        for (int nh = 0; nh < 2; ++nh)
          tma_load_2d_mc(base + rank * 16384 + nh * 8192, wm, c * tNC + 64 * nh, 64 * kb, b_w12full + 8 * slot, tClusterMask);
        if (kb) {
          const uint32_t xb = s_w12x + (g & 1) * tW12xBytes;
#pragma unroll
          for (int nh = 0; nh < 2; ++nh)
            tma_load_2d_mc(xb + rank * 4096 + nh * 2048, wxm, c * tNC + 64 * nh, tCz, b_w12full + 8 * slot, tClusterMask);
        }
      };
      if (n_it) load_z(tile_of(0), 0);
      load_w12(0); load_w12(1); load_w12(2);
      uint32_t g = 0;
      for (int it = 0; it < n_it; ++it) {
        for (int c = 0; c < tChunks; ++c, ++g) {
          // in the order in which the tensor pipe frees the buffers: k-block (g, 0) -> (g + 1, 1), (g, 1) -> (g + 2, 0),
          // G2(g - 1) -> W3(g)
          load_w12(2 * g + 3);
          load_w12(2 * g + 4);
          mbar_wait(b_w3empty, (g & 1) ^ 1);
          mbar_expect_tx(b_w3full, tW3Bytes);
#pragma unroll
          for (int nh = 0; nh < 2; ++nh)                     // k-block `rank` of W3's chunk, for both CTAs
            tma_load_2d_mc(s_w3 + rank * 16384 + nh * 8192, &maps.w3, 64 * nh, c * tNC + 64 * (int)rank, b_w3full, tClusterMask);
          if (c == 1 && it + 1 < n_it) load_z(tile_of(it + 1), it + 1);
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // =============================================================== tcgen05 issuer
      constexpr uint32_t idesc1 = umma_idesc_bf16(tM, 256) | (1u << 16);     // B MN-major
      constexpr uint32_t idesc2 = umma_idesc_bf16(tM, 128) | (1u << 16);
      const uint32_t n_chunks = (uint32_t)n_it * tChunks;
      // G1 of the CTA's chunk number g (tile g / 4): [A1 | A2] = [z | -mu, 1 / rstd] . [W1'c | W2'c ; c1 ; c0], k-block by k-block
      auto g1 = [&](uint32_t g) {
        const uint32_t it = g / tChunks, zb = it & 1;
        const uint32_t zs = s_z + zb * tZBytes;
        if ((g & (tChunks - 1)) == 0) {
          mbar_wait(b_zfull + 8 * zb, (it >> 1) & 1);
          mbar_wait(b_xfull + 8 * zb, (it >> 1) & 1);        // the epilogue has written this tile's K extension
        }
#pragma unroll
        for (int kb = 0; kb < 2; ++kb) {
          const uint32_t j = 2 * g + kb, slot = j % 3, use = j / 3;
          mbar_wait(b_w12full + 8 * slot, use & 1);
          if (kb == 0) mbar_wait(b_aempty, (g & 1) ^ 1);
          tc_fence_after();
          const uint32_t wb = s_w12 + slot * tW12Slot;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            umma_bf16(tmem_base + tColA1, umma_desc_sw128(zs + kb * (tZBytes / 2) + ks * 32), umma_desc_mn(wb + ks * 2048, 8192),
                      idesc1, (kb | ks) != 0);
          if (kb == 1) {
            umma_bf16(tmem_base + tColA1, umma_desc_k_sw32(s_zx + zb * tZxBytes), umma_desc_mn(s_w12x + (g & 1) * tW12xBytes, 2048),
                      idesc1, 1);
            umma_commit(b_afull);
          }
          umma_commit_mc(b_w12empty + 8 * slot, tClusterMask);   // both CTAs write into this slot
        }
      };
      // G2 of chunk g: OUT (+)= H . W3[rows of the chunk]
      auto g2 = [&](uint32_t g) {
        const uint32_t hb = g & 1, c = g & (tChunks - 1);
        mbar_wait(b_hfull + 8 * hb, (g >> 1) & 1);
        mbar_wait(b_w3full, g & 1);
        if (c == 0) mbar_wait(b_oempty, ((g / tChunks) & 1) ^ 1);   // the output warps have read the previous tile's OUT
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)
          umma_bf16_ts(tmem_base + tColOut, tmem_base + tColH + 64 * hb + 8 * ks,
                       umma_desc_mn(s_w3 + (ks >> 2) * 16384 + (ks & 3) * 2048, 8192), idesc2, (c | ks) != 0);
        umma_commit(b_hempty + 8 * hb);
        umma_commit_mc(b_w3empty, tClusterMask);
        if (c == tChunks - 1) umma_commit(b_ofull);
      };
      // G1(g + 1) ahead of G2(g), across tile boundaries too: the tensor pipe works on the next chunk while the
      // epilogue warps turn the previous one into H
      if (n_chunks) g1(0);
      for (uint32_t g = 0; g < n_chunks; ++g) {
        if (g + 1 < n_chunks) g1(g + 1);
        g2(g);
      }
    }
  } else if (warp >= 10) {
    // =============================================================== output warps (one per TMEM lane quadrant)
    // residual: z + OUT -> bf16, written over the thread's own row of the z tile (every G1 of the tile is complete
    // once out_full is, and the epilogue warps read a z tile only before its first G1) -> TMA store from there
    const int quad = warp & 3, ot = threadIdx.x - 320;
    const int r = quad * 32 + lane;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16);
    const uint32_t sw = (uint32_t)(r & 7);
    for (int it = 0; it < n_it; ++it) {
      const int64_t tile = tile_of(it);
      const int zb = it & 1;
      const uint32_t zrow = s_z + zb * tZBytes + r * 128;   // row base inside a 64-channel half
      mbar_wait(b_ofull, it & 1);
      tc_fence_after();
#pragma unroll
      for (int sb = 0; sb < 4; ++sb) {                       // 32 channels at a time
        uint32_t o[32];
        tmem_ld32(t_lane + tColOut + sb * 32, o);
        tmem_ld_wait();
        if (sb == 3) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(b_oempty);              // OUT is in registers: the next tile's G2 may overwrite it
        }
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          const uint32_t addr = zrow + (sb >> 1) * (tZBytes / 2) + ((((sb & 1) * 4 + ch) ^ sw) << 4);
          const uint4 zv = lds_u32x4(addr);
          const uint32_t zw[4] = {zv.x, zv.y, zv.z, zv.w};
          uint32_t ow[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const float z0 = __uint_as_float(zw[q] << 16), z1 = __uint_as_float(zw[q] & 0xffff0000u);
            ow[q] = pack_bf16(z0 + __uint_as_float(o[ch * 8 + 2 * q]), z1 + __uint_as_float(o[ch * 8 + 2 * q + 1]));
          }
          asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(ow[0]), "r"(ow[1]), "r"(ow[2]), "r"(ow[3]) : "memory");
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (ot == 0) {
        tma_store_2d(&maps.z_out, 0, (int)(tile * tM), s_z + zb * tZBytes);
        tma_store_2d(&maps.z_out, 64, (int)(tile * tM), s_z + zb * tZBytes + tZBytes / 2);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the store has read the buffer: free for z
        mbar_arrive(b_zempty + 8 * zb);
      }
    }
    if (ot == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  } else {
    // =============================================================== epilogue warps
    const int quad = warp & 3, half = (warp - 2) >> 2;
    const int r = quad * 32 + lane;                         // tile row = TMEM lane of this thread
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16);
    const uint32_t sw = (uint32_t)(r & 7);
    uint32_t na = 0, nh = 0;
    // LayerNorm statistics of the thread's pair of tile number `jt` (fp32: mu = sum / c_z, var = sum z^2 / c_z - mu^2)
    // and the K extension row [-mu, 1 / rstd, 0 ...] of that z buffer (32-byte swizzle: 16-byte chunk ^ bit 2 of the
    // row); returns rstd.  Called one tile ahead, so that the issuer never waits for it.
    auto prepare = [&](int jt) -> float {
      const int zb = jt & 1;
      const uint32_t zrow = s_z + zb * tZBytes + r * 128;
      mbar_wait(b_zfull + 8 * zb, (jt >> 1) & 1);
      float sm = 0.f, sq = 0.f;
#pragma unroll
      for (int hf = 0; hf < 2; ++hf)
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
          const uint4 w = lds_u32x4(zrow + hf * (tZBytes / 2) + ((ch ^ sw) << 4));
          stats_bf16x2(sm, sq, w.x); stats_bf16x2(sm, sq, w.y); stats_bf16x2(sm, sq, w.z); stats_bf16x2(sm, sq, w.w);
        }
      // var with ONE rounding: sum z^2 / c_z is exact (c_z is a power of two) and the FMA subtracts the unrounded mu^2
      const float mu = sm * (1.f / tCz);
      const float vpe = fmaxf(fmaf(-mu, mu, sq * (1.f / tCz)), 0.f) + eps;
      if (half == 0) {
        // -mu and 1 / rstd travel through the bf16 tensor pipe as sums of bf16 terms (hi + lo + lo2, hi + lo) against the
        // weight rows [c1h, c1l, c1l2, c1h, c1l, c1h | c0h, c0l, c0h] (transition_fold_kernel): every product of the
        // expansion down to 2^-16 of mu c1 is there, so z.W' - mu c1 cancels to fp32 accuracy however large |mu| / sigma is.
        const float nm = -mu, sd = sqrtf(vpe);
        const float mh = bf16_round(nm), ml = bf16_round(nm - mh), ml2 = bf16_round((nm - mh) - ml);
        const float rh = bf16_round(sd), rl = bf16_round(sd - rh);
        const uint32_t xrow = s_zx + zb * tZxBytes + r * 32;
        const uint32_t c0 = ((uint32_t)(r >> 2) & 1u) << 4;
        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(xrow + c0), "r"(pack_bf16(mh, mh)), "r"(pack_bf16(mh, ml)),
                     "r"(pack_bf16(ml, ml2)), "r"(pack_bf16(rh, rh)) : "memory");
        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %2, %2};" ::"r"(xrow + (c0 ^ 16u)), "r"(pack_bf16(rl, 0.f)), "r"(0u) : "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(b_xfull + 8 * zb);
      }
      return rsqrtf(vpe);
    };
    int it = 0;
    float rstd_next = n_it ? prepare(0) : 0.f;
    for (; it < n_it; ++it) {
      const float rstd = rstd_next, hrstd = 0.5f * rstd_next;

      for (int c = 0; c < tChunks; ++c) {
        mbar_wait(b_afull, na & 1);
        tc_fence_after();
        const uint32_t hb = nh & 1;                          // H buffer of this chunk: TMEM columns tColH + 64 hb ..
#pragma unroll
        for (int sb = 0; sb < 2; ++sb) {
          uint32_t hw[16];                                   // 32 h values of the thread's row, bf16x2
          uint32_t a1[32], a2[32];
          tmem_ld32(t_lane + tColA1 + half * 64 + sb * 32, a1);
          tmem_ld32(t_lane + tColA1 + 128 + half * 64 + sb * 32, a2);
          tmem_ld_wait();
          if (sb == 1) {                                     // A1 / A2 are in registers: the next G1 may overwrite them
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(b_aempty);
          }
#pragma unroll
          for (int i = 0; i < 32; i += 2) {
            float hv[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              // a = rstd * accumulator (the K extension carried -mu c1 + c0 / rstd);  SiLU(x) = 0.5 x (1 + tanh(x / 2))
              const float hx = __uint_as_float(a1[i + e]) * hrstd;
              hv[e] = fmaf(hx, tanh_fast(hx), hx) * (__uint_as_float(a2[i + e]) * rstd);
            }
            hw[i >> 1] = pack_bf16(hv[0], hv[1]);
          }
          // ---- H (the A operand of G2, read from TMEM): lane = row, column = two consecutive hidden units
          if (sb == 0) mbar_wait(b_hempty + 8 * hb, ((nh >> 1) & 1) ^ 1);   // G2 two chunks back has finished reading it
          tmem_st16(t_lane + tColH + 64 * hb + half * 32 + sb * 16, hw);
        }
        ++na;
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(b_hfull + 8 * hb);
        ++nh;
        if (c == 2 && it + 1 < n_it) rstd_next = prepare(it + 1);   // the next tile's statistics, early
      }

    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                        // no CTA leaves while its peer may still signal its barriers
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_base, 512);
  }
}

// Folded weights [c_z + 16][4 c_z] for W1 and W2: rows k < c_z: bf16(gamma_k W[k][j]); rows c_z ..: the K extension of the
// first GEMM -- c1[j] = sum_k of those rounded values and c0[j] = sum_k beta_k W[k][j], each split into bf16 terms
__global__ void __launch_bounds__(32) transition_fold_kernel(const __nv_bfloat16* __restrict__ w1, const __nv_bfloat16* __restrict__ w2,
                                                             const __nv_bfloat16* __restrict__ gamma, const __nv_bfloat16* __restrict__ beta,
                                                             __nv_bfloat16* __restrict__ w1f, __nv_bfloat16* __restrict__ w2f) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= tHid) return;
  float c11 = 0.f, c01 = 0.f, c12 = 0.f, c02 = 0.f;
#pragma unroll 16
  for (int k = 0; k < tCz; ++k) {
    const float g = to_f32(gamma[k]), b = to_f32(beta[k]);
    const float a = to_f32(w1[k * tHid + j]), c = to_f32(w2[k * tHid + j]);
    const __nv_bfloat16 af = __float2bfloat16_rn(g * a), cf = __float2bfloat16_rn(g * c);
    w1f[k * tHid + j] = af;
    w2f[k * tHid + j] = cf;
    c11 += to_f32(af); c12 += to_f32(cf);
    c01 = fmaf(b, a, c01); c02 = fmaf(b, c, c02);
  }
  // K-extension rows, matching the columns [mh, mh, mh, ml, ml, ml2 | rh, rh, rl | 0 ...] the kernel writes per pair
  auto ext = [&](__nv_bfloat16* wf, float c1, float c0) {
    const __nv_bfloat16 c1h = __float2bfloat16_rn(c1), c1l = __float2bfloat16_rn(c1 - to_f32(c1h)),
                        c1l2 = __float2bfloat16_rn((c1 - to_f32(c1h)) - to_f32(c1l));
    const __nv_bfloat16 c0h = __float2bfloat16_rn(c0), c0l = __float2bfloat16_rn(c0 - to_f32(c0h));
    const __nv_bfloat16 rows[tKx] = {c1h, c1l, c1l2, c1h, c1l, c1h, c0h, c0l, c0h};
    for (int k = 0; k < tKx; ++k) wf[(tCz + k) * tHid + j] = k < 9 ? rows[k] : __float2bfloat16_rn(0.f);
  };
  ext(w1f, c11, c01);
  ext(w2f, c12, c02);
}

CUresult encode2d(PFN_cuTensorMapEncodeTiled enc, CUtensorMap* m, const void* base, uint64_t d0, uint64_t d1, uint32_t b0,
                  uint32_t b1) {
  const cuuint64_t gdim[2] = {d0, d1};
  const cuuint64_t gstr[1] = {d0 * 2};
  const cuuint32_t box[2] = {b0, b1};
  const cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstr, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

}  // namespace

bool pair_transition_supports(dcp_dtype dt, int c_z) { return dt == DCP_BF16 && c_z == tCz; }
size_t pair_transition_workspace_bytes() { return (size_t)2 * (tCz + tKx) * tHid * 2; }

cudaError_t launch_pair_transition(const void* z_in, void* z_out, int64_t n_pairs, const void* w1, const void* w2,
                                   const void* w3, const void* gamma, const void* beta, float eps, void* workspace,
                                   cudaStream_t st) {
  if (n_pairs <= 0) return cudaSuccess;
  PFN_cuTensorMapEncodeTiled enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  __nv_bfloat16* w1f = reinterpret_cast<__nv_bfloat16*>(workspace);
  __nv_bfloat16* w2f = w1f + (tCz + tKx) * tHid;
  transition_fold_kernel<<<tHid / 32, 32, 0, st>>>((const __nv_bfloat16*)w1, (const __nv_bfloat16*)w2,
                                                     (const __nv_bfloat16*)gamma, (const __nv_bfloat16*)beta, w1f, w2f);
  TransMaps maps;
  if (encode2d(enc, &maps.z_in, z_in, tCz, (uint64_t)n_pairs, 64, tM) != CUDA_SUCCESS ||
      encode2d(enc, &maps.z_out, z_out, tCz, (uint64_t)n_pairs, 64, tM) != CUDA_SUCCESS ||
      encode2d(enc, &maps.w1, w1f, tHid, tCz + tKx, 64, 64) != CUDA_SUCCESS ||
      encode2d(enc, &maps.w2, w2f, tHid, tCz + tKx, 64, 64) != CUDA_SUCCESS ||
      encode2d(enc, &maps.w1x, w1f, tHid, tCz + tKx, 64, tKx) != CUDA_SUCCESS ||
      encode2d(enc, &maps.w2x, w2f, tHid, tCz + tKx, 64, tKx) != CUDA_SUCCESS ||
      encode2d(enc, &maps.w3, w3, tCz, tHid, 64, 64) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(pair_transition_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tSmemAlloc);
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (sms <= 0) sms = 148;
  const int64_t n_tiles = (n_pairs + tM - 1) / tM;
  const int64_t n_tpairs = (n_tiles + tCluster - 1) / tCluster, max_clusters = sms / tCluster;
  const unsigned grid = (unsigned)((n_tpairs < max_clusters ? n_tpairs : max_clusters) * tCluster);
  pair_transition_kernel<<<grid, tThreads, tSmemAlloc, st>>>(maps, n_pairs, eps);
  return cudaGetLastError();
}

}  // namespace dcp
