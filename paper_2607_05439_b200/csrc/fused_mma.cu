// bf16 tensor-core fused kernel (steps a2-a7 of SURVEY.md section 8(a)) for c_z = 128, H = 16 heads.
//   per pair (i, j):  LayerNorm(z_ij) -> bias_h = zhat . W_b[:,h]          ("learned projection of Z")
//   logit_h = q_i^h . k_j^h / sqrt(c) + bias_h                             (PAPER.md:83 Eq. 2; i = row of z, :81)
//   online softmax over keys with running (m, l, acc)
// z is streamed from HBM exactly once by TMA (cp.async.bulk.tensor, 128-byte swizzle, evict_first) through a 3-stage
// mbarrier ring; the I*I*H logits and the LayerNorm output never leave the SM.
//
// One persistent CTA per SM, 16 warps, warp-specialised (register budgets moved with setmaxnreg 24 / 104 / 192):
//   warp 0        TMA producer: z boxes of (64 ch, 16 keys, 8 queries) x 2 channel halves = 32 KB per stage
//   warps 1-3     tcgen05 issuers (one lane each, stage n -> issuer n % 3): per stage 8 x tcgen05.mma kind::f16
//                 (M = 128 pair rows exactly as TMA wrote them, N = 32, K = 16) against W'' = [(gamma (.) W_b log2 e)^T ;
//                 ones ; 0] -> z.W' for 16 heads and sum_k z, accumulated in tensor memory (4 buffers of 32 columns)
//   warps 4-7     LayerNorm statistics + bias epilogue, thread = pair: sum_k z^2 from the thread's own 256-byte row of
//                 the swizzled stage (exact bf16 x bf16 products, fp32 sums: fma.rn.f32.bf16), z.W' and sum z by
//                 tcgen05.ld; bias = rstd (z.W' - mu c1) + c0 -> double-buffered shared tile bias[h][32 queries][16 keys]
//                 fp32 (the layout change "row = pair" -> "row = query")
//   warps 8-15    attention: warp w owns heads 2w, 2w+1 for the tile's 32 queries (two m16 blocks): the mma.sync
//                 accumulator is initialised with the bias, S += Q K^T (Q fragments by conflict-free LDS.64 from a padded
//                 shared Q tile), online softmax in the exp2 domain with a lazily moving reference (q is pre-scaled by
//                 log2 e / sqrt(c)), P (bf16) feeds PV straight from registers, K / V fragments are single coalesced
//                 128-bit loads from L2 (MMA B-fragment order, written by the prologue GEMM), O stays in registers
//                 (96 per thread) and leaves as a partial state through a shared-memory slab.
// Why QK^T / PV stay on mma.sync: what-if builds (profiles/r02_fused_c2_ncu_full.txt) show that removing every
// attention MMA changes the kernel time by 1-2 %; what paced the kernel was the issue rate of the projection MMAs.
#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int kCz = 128;
constexpr int kH = 16;
constexpr int kTileQ = 32;          // queries per work unit
constexpr int kTileK = 16;          // keys per attention tile
constexpr int kSubQ = 8;            // queries per z stage
constexpr int kNZ = 3;              // z stages
constexpr int kStageBytes = kSubQ * kTileK * kCz * 2;   // 32 KB
constexpr int kHalfBytes = kStageBytes / 2;
constexpr int kBiasHeadPitch = kTileQ * kTileK + 4;     // floats; +4: conflict-free projection stores
constexpr int kBiasBufFloats = kH * kBiasHeadPitch;
constexpr int kThreads = 512;
constexpr int kProjWarp0 = 4, kNumProjWarps = 4, kAttnWarp0 = 8, kNumAttnWarps = 8;
constexpr int kNumIssuers = 3;      // tcgen05 issuing threads (lane 0 of warps 1..3)

constexpr size_t kSmemZ = 0;
constexpr size_t kSmemBias = kSmemZ + (size_t)kNZ * kStageBytes;
constexpr int kProjN = 32;                               // projection MMA N: 16 heads, the ones row (sum z), zero rows
constexpr int kWtHalfBytes = kProjN * 128;               // W'' tile: 32 rows x 64 channels bf16 per channel half
constexpr int kNT = 4;                                   // TMEM accumulator buffers
constexpr int kTmemBufCols = 32;                         // projection columns per buffer
constexpr int kTmemCols = kNT * kTmemBufCols;            // 128 (a power of two >= 32)
constexpr size_t kSmemWt = (kSmemBias + 2 * (size_t)kBiasBufFloats * 4 + 1023) / 1024 * 1024;   // 1024-aligned (swizzle)
constexpr size_t kSmemBar = kSmemWt + 2 * (size_t)kWtHalfBytes;
constexpr size_t kSmemQ = (kSmemBar + (2 * kNZ + 4 + 2 * kNT) * 8 + 16 + 15) / 16 * 16;   // Q tile [32 rows][H][CP] bf16, padded rows
__host__ __device__ constexpr int q_pitch(int CP) { return kH * CP * 2 + 32; }      // bytes; +32: conflict-free 64-bit loads
__host__ __device__ constexpr size_t smem_alloc(int CP) { return kSmemQ + (size_t)kTileQ * q_pitch(CP) + 1024; }  // + alignment slack

// ------------------------------------------------------------------ the kernel
// C = head dim, CP = C rounded up to a multiple of 16 (q/k rows are zero-padded to CP by the prologue)
template <int C, int CP>
__global__ void __launch_bounds__(kThreads, 1) fused_mma_kernel(const __grid_constant__ CUtensorMap tmap_z,
                                                                const __grid_constant__ CUtensorMap tmap_tail, const MmaParams p) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
  const uint32_t s_z = smem_u32(smem + kSmemZ);
  float* s_bias = reinterpret_cast<float*>(smem + kSmemBias);
  const uint32_t s_wt = smem_u32(smem + kSmemWt);
  const uint32_t s_bar = smem_u32(smem + kSmemBar);
  const uint32_t s_q = smem_u32(smem + kSmemQ);
  const uint32_t bar_zfull = s_bar, bar_zempty = s_bar + 8 * kNZ, bar_bfull = s_bar + 16 * kNZ,
                 bar_bempty = s_bar + 16 * kNZ + 16, bar_tfull = s_bar + 16 * kNZ + 32, bar_tempty = bar_tfull + 8 * kNT;
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(smem + kSmemBar + (2 * kNZ + 4 + 2 * kNT) * 8);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;

  pdl_trigger();
  if (threadIdx.x == 0) {
    // zempty / tfull are arrived on by tcgen05.commit (the MMAs that read the stage / wrote the accumulators are done)
    for (int s = 0; s < kNZ; ++s) { mbar_init(bar_zfull + 8 * s, 1); mbar_init(bar_zempty + 8 * s, 1 + kNumProjWarps); }
    for (int b = 0; b < 2; ++b) { mbar_init(bar_bfull + 8 * b, kNumProjWarps); mbar_init(bar_bempty + 8 * b, kNumAttnWarps); }
    for (int b = 0; b < kNT; ++b) { mbar_init(bar_tfull + 8 * b, 1); mbar_init(bar_tempty + 8 * b, kNumProjWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), kTmemCols);
  pdl_wait();          // the prologue's q / k / v / folded weights are final (and so is everything before it in the stream)
  // W'' = B operand of the projection MMA, K-major, 128-byte swizzled by hand: row n < 16 = head n of
  // (gamma (.) W_b log2 e)^T, row 16 = ones (its accumulator column is sum_k z), rows 17..31 = 0.
  for (int e = threadIdx.x; e < kProjN * (kCz / 8); e += kThreads) {
    const int n = e / (kCz / 8), ch16 = e % (kCz / 8);          // 16-byte chunk = 8 channels
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (n < kH) v = __ldg(reinterpret_cast<const uint4*>(p.wfold) + n * (kCz / 8) + ch16);
    else if (n == kH) v = make_uint4(0x3f803f80u, 0x3f803f80u, 0x3f803f80u, 0x3f803f80u);
    const int half = ch16 >> 3, c = ch16 & 7;
    *reinterpret_cast<uint4*>(smem + kSmemWt + half * kWtHalfBytes + n * 128 + ((c ^ (n & 7)) << 4)) = v;
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to TMA / tcgen05
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *s_tmem;

  const int n_units = (int)mma_num_units<0>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg, p.tile_h);

  if (warp < kProjWarp0) {
    // =============================================================== TMA producer (warp 0, one lane)
    reg_dec<24>();
    if (warp == 0 && lane == 0) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      int stage = 0;
      uint32_t phase = 0;
      const int tail_rows = p.tile_h % kSubQ;               // 0: every stage is a full box
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const Unit un = decode_unit<0, kTileK>(p, u);
        const int rows = (un.q_end - un.q0) < p.tile_h ? (un.q_end - un.q0) : p.tile_h;
        const int nsub = (rows + kSubQ - 1) / kSubQ;
        for (int j0 = un.ks & ~(kTileK - 1); j0 < un.ke; j0 += kTileK) {
          for (int sub = 0; sub < nsub; ++sub) {
            mbar_wait(bar_zempty + 8 * stage, phase ^ 1);
            // the last stage of a tile whose height is not a multiple of 8 fetches only the tile's own rows (box of
            // tail_rows queries; the stage's remaining pair rows keep stale data, their results are never stored)
            const bool tail = sub == nsub - 1 && rows - sub * kSubQ == tail_rows;
            const CUtensorMap* tm = tail ? &tmap_tail : &tmap_z;
            const uint32_t half_bytes = tail ? tail_rows * (kHalfBytes / kSubQ) : kHalfBytes;
            mbar_expect_tx(bar_zfull + 8 * stage, 2 * half_bytes);
            const uint32_t dst = s_z + stage * kStageBytes;
            const int qrow = un.q0 + sub * kSubQ;
            tma_load_3d(dst, tm, 0, j0, qrow, bar_zfull + 8 * stage, policy);
            tma_load_3d(dst + kHalfBytes, tm, 64, j0, qrow, bar_zfull + 8 * stage, policy);
            if (++stage == kNZ) { stage = 0; phase ^= 1; }
          }
        }
      }
    } else if (warp >= 1 && warp <= kNumIssuers && lane == 0) {
      // ============================================================= tcgen05 issuers (one thread each, warps 1..3)
      // A K = 16 projection MMA costs its issuing thread ~130 cycles whatever N is (the 4 KB A-operand fetch), eight of
      // them per 32 KB stage: one thread alone needs ~1050 of the ~1450 cycles a stage may take at the HBM bound, and
      // with the attention warps competing for issue slots it became the kernel's pacemaker (what-if: half the MMAs
      // -> -9.5 % kernel time).  Several threads' MMAs overlap in the tensor pipe, so stage n goes to issuer n % 3.
      // Per z stage (128 pair rows = 8 queries x 16 keys, K-major, exactly as TMA wrote it) two accumulator chains
      // over the 8 K = 16 steps:   P[128 x 32]  = z . W''^T   (a3: 16 heads; column 16 = sum_k z)
      //                            G[128 x 128] = z . z^T     (a2: its diagonal is sum_k z^2)
      // into TMEM buffer tb; tcgen05.commit then releases the smem stage and publishes the accumulators.
      constexpr uint32_t idesc_p = umma_idesc_bf16(128, kProjN);
      const int me = warp - 1;
      int stage = 0, tb = 0, turn = 0;
      uint32_t phase = 0, tphase = 0;
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const Unit un = decode_unit<0, kTileK>(p, u);
        const int rows = (un.q_end - un.q0) < p.tile_h ? (un.q_end - un.q0) : p.tile_h;
        const int nsub = (rows + kSubQ - 1) / kSubQ;
        for (int j0 = un.ks & ~(kTileK - 1); j0 < un.ke; j0 += kTileK) {
          for (int sub = 0; sub < nsub; ++sub) {
            const bool mine = turn == me;
            if (++turn == kNumIssuers) turn = 0;
            if (!mine) {
              if (++stage == kNZ) { stage = 0; phase ^= 1; }
              if (++tb == kNT) { tb = 0; tphase ^= 1; }
              continue;
            }
            mbar_wait(bar_tempty + 8 * tb, tphase ^ 1);
            mbar_wait(bar_zfull + 8 * stage, phase);
            tc_fence_after();
            const uint32_t zs = s_z + stage * kStageBytes;
            const uint32_t d_p = tmem_base + tb * kTmemBufCols;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              const uint64_t a = umma_desc_sw128(zs + (ks >> 2) * kHalfBytes + (ks & 3) * 32);
              const uint64_t b = umma_desc_sw128(s_wt + (ks >> 2) * kWtHalfBytes + (ks & 3) * 32);
              umma_bf16(d_p, a, b, idesc_p, ks > 0);
            }
            umma_commit(bar_zempty + 8 * stage);
            umma_commit(bar_tfull + 8 * tb);
            if (++stage == kNZ) { stage = 0; phase ^= 1; }
            if (++tb == kNT) { tb = 0; tphase ^= 1; }
          }
        }
      }
    }
  } else if (warp < kAttnWarp0) {
    // =============================================================== LayerNorm statistics + bias epilogue (TMEM -> smem)
    // Thread = one pair row of the stage: TMEM lane 32*pw + lane = (query 2pw + lane/16 of the stage, key lane%16).
    // sum_k z^2 comes from the thread's own 256-byte row of the swizzled stage (16 conflict-free LDS.128, fp32 FMAs);
    // sum_k z (the ones row of W'') and z.W' come from the tcgen05 accumulators.
    reg_dec<104>();
    const int pw = warp - kProjWarp0;                       // == warp % 4: the TMEM lane quadrant this warp may read
    float c1h[kH], c0h[kH];
#pragma unroll
    for (int h = 0; h < kH; ++h) { c1h[h] = __ldg(p.c1 + h); c0h[h] = __ldg(p.c0 + h); }
    const uint32_t t_lane = tmem_base + ((uint32_t)(pw * 32) << 16);
    const int prow = pw * 32 + lane;                        // pair row inside the stage
    const uint32_t zrow = s_z + prow * 128;                 // row base inside a channel half (128-byte swizzle atom rows)
    const uint32_t zsw = (uint32_t)(prow & 7);
    int tb = 0, bbuf = 0, stage = 0;
    uint32_t tphase = 0, bphase = 0, zphase = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const Unit un = decode_unit<0, kTileK>(p, u);
      const int rows = (un.q_end - un.q0) < p.tile_h ? (un.q_end - un.q0) : p.tile_h;
      const int nsub = (rows + kSubQ - 1) / kSubQ;
      for (int j0 = un.ks & ~(kTileK - 1); j0 < un.ke; j0 += kTileK) {
        mbar_wait(bar_bempty + 8 * bbuf, bphase ^ 1);
        const uint32_t bias_buf = smem_u32(s_bias) + bbuf * (kBiasBufFloats * 4);
        for (int sub = 0; sub < nsub; ++sub) {
          // ---- a2: sum_k z^2 of this pair straight from the TMA stage
          mbar_wait(bar_zfull + 8 * stage, zphase);
          float sq0 = 0.f, sq1 = 0.f, sq2 = 0.f, sq3 = 0.f;
          const uint32_t zr = zrow + stage * kStageBytes;
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            uint4 w[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) w[c] = lds_u32x4(zr + half * kHalfBytes + ((c ^ zsw) << 4));
#pragma unroll
            for (int c = 0; c < 8; ++c) {
              fma_sq_bf16x2(sq0, sq1, w[c].x); fma_sq_bf16x2(sq2, sq3, w[c].y);
              fma_sq_bf16x2(sq0, sq1, w[c].z); fma_sq_bf16x2(sq2, sq3, w[c].w);
            }
          }
          float zsq = (sq0 + sq1) + (sq2 + sq3);
          asm volatile("" : "+f"(zsq));                       // the row has been consumed before the stage is released
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_zempty + 8 * stage);
          if (++stage == kNZ) { stage = 0; zphase ^= 1; }
          // ---- a3: z.W' (16 heads) and sum_k z from tensor memory
          mbar_wait(bar_tfull + 8 * tb, tphase);
          tc_fence_after();
          const uint32_t t_p = t_lane + tb * kTmemBufCols;
          float acc[16];
          tmem_ld_x16(t_p, acc);
          const float zsum = tmem_ld_x1(t_p + kH);
          tmem_ld_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_tempty + 8 * tb);    // accumulators are in registers: buffer free
          if (++tb == kNT) { tb = 0; tphase ^= 1; }
          // LayerNorm statistics (fp32): mu = sum / c_z, var = sum z^2 / c_z - mu^2 with ONE rounding: c_z is a power of
          // two, so sum z^2 / c_z is exact, and the FMA subtracts the unrounded mu^2.  The sums themselves are exact
          // whenever the row's values span few binades (bf16 x bf16 products have 16 significant bits), which is exactly
          // when |mu| >> sigma makes the subtraction cancel; a constant row gives var == 0 exactly, and then LN(z) = beta:
          // rstd = 0 keeps the tensor pipe's rounding residue of z.W' - mu c1 from being amplified by 1 / sqrt(eps).
          const float mu = zsum * (1.f / kCz);
          const float var = fmaf(-mu, mu, zsq * (1.f / kCz));
          const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;
          const float nm = -mu * rstd;
          // ---- LN(z) W_b = rstd * (z.W' - mu * c1) + c0 ; store to bias[h][query][key] (32 lanes = 128 contiguous bytes)
          const uint32_t brow = bias_buf + ((sub * kSubQ) * kTileK + prow) * 4;
#pragma unroll
          for (int h = 0; h < kH; ++h)
            sts_f32(brow + h * (kBiasHeadPitch * 4), fmaf(acc[h], rstd, fmaf(nm, c1h[h], c0h[h])));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_bfull + 8 * bbuf);
        bbuf ^= 1;
        if (bbuf == 0) bphase ^= 1;
      }
    }
  } else {
    // =============================================================== attention: QK^T + bias, online softmax, PV
    reg_inc<192>();
    const int aw = warp - kAttnWarp0;
    constexpr int KK = CP / 16;     // k-steps of QK^T
    constexpr int ND = C / 8;       // n-blocks of PV
    const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.qp);
    const uint4* kfr = reinterpret_cast<const uint4*>(p.kfr);
    const uint4* vfr = reinterpret_cast<const uint4*>(p.vfr);
    int bbuf = 0;
    uint32_t bphase = 0;
    // K / V fragments of (key tile j, head h) are read from L2 into the registers the previous block just released:
    // K right after the last QK^T MMA that used it, V right after the last PV MMA (software pipelining, no extra
    // registers).  Both live in MMA B-fragment order (gemm_mma.cu), so every load is one coalesced 128-bit access per
    // lane: K k-step kk -> (n-block A, n-block B) fragments, V n-block pair ndp -> fragments of nd = 2 ndp, 2 ndp + 1.
    // key of S column: n-block A col c <-> j + 4*(c/2) + c%2, n-block B col c <-> that + 2
    constexpr int NDP = CP / 16;
    uint4 kq[KK], vq[NDP];
    auto load_k = [&](int j, int h) {
      const uint4* src = kfr + ((int64_t)((j >> 4) * kH + h) * KK) * 32 + lane;
#pragma unroll
      for (int kk = 0; kk < KK; ++kk) kq[kk] = __ldg(src + kk * 32);
    };
    auto load_v = [&](int j, int h) {
      const uint4* src = vfr + ((int64_t)((j >> 4) * kH + h) * NDP) * 32 + lane;
#pragma unroll
      for (int ndp = 0; ndp < NDP; ++ndp) vq[ndp] = __ldg(src + ndp * 32);
    };
    // The first K / V tile of a unit is requested during the last tile of the previous one (the slot that would re-read
    // the tile itself), so a unit change costs one L2 round trip (the Q tile) instead of two.
    if ((int)blockIdx.x < n_units) {
      const Unit u0 = decode_unit<0, kTileK>(p, blockIdx.x);
      load_k(u0.ks & ~(kTileK - 1), 2 * aw);
      load_v(u0.ks & ~(kTileK - 1), 2 * aw);
    }
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const Unit un = decode_unit<0, kTileK>(p, u);
      const int next_first = u + (int)gridDim.x < n_units ? (decode_unit<0, kTileK>(p, u + gridDim.x).ks & ~(kTileK - 1)) : -1;
      // Q tile -> shared memory (rows of the tile, all heads), shared by the 8 attention warps; row pitch padded so the
      // per-thread 64-bit fragment loads are conflict-free.  Named barrier 1 = the 256 attention threads.
      constexpr int kQP = q_pitch(CP);
      constexpr int kQRowChunks = kH * CP * 2 / 16;
      // All of a thread's chunks are requested before the barrier and stored after it: the unit change costs one L2 round
      // trip, not one per chunk (kTileQ * kQRowChunks is a multiple of the 256 attention threads for every CP).
      {
        constexpr int kQIter = kTileQ * kQRowChunks / (kNumAttnWarps * 32);
        static_assert(kQIter * kNumAttnWarps * 32 == kTileQ * kQRowChunks, "Q tile chunks per thread");
        uint4 qv[kQIter];
#pragma unroll
        for (int i = 0; i < kQIter; ++i) {
          const int e = threadIdx.x - kAttnWarp0 * 32 + i * (kNumAttnWarps * 32);
          const int r = e / kQRowChunks, ch = e - r * kQRowChunks;
          const int64_t row = (un.q0 + r) < p.I ? (un.q0 + r) : p.I - 1;
          qv[i] = __ldg(reinterpret_cast<const uint4*>(qp + row * (kH * CP)) + ch);
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");        // every warp is done with the previous unit's Q
#pragma unroll
        for (int i = 0; i < kQIter; ++i) {
          const int e = threadIdx.x - kAttnWarp0 * 32 + i * (kNumAttnWarps * 32);
          const int r = e / kQRowChunks, ch = e - r * kQRowChunks;
          *reinterpret_cast<uint4*>(smem + kSmemQ + r * kQP + ch * 16) = qv[i];
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
      // fragment address of (row g, head 2aw, k-step 0): + mb*16*kQP (+8 rows: +8*kQP), + hh*CP*2, + kk*32
      const uint32_t q_frag = s_q + g * kQP + (2 * aw) * (CP * 2) + 8 * t;
      float o[2][2][ND][4];
      float m_run[2][2][2], l_run[2][2][2];
#pragma unroll
      for (int hh = 0; hh < 2; ++hh)
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          m_run[hh][mb][0] = m_run[hh][mb][1] = -INFINITY;
          l_run[hh][mb][0] = l_run[hh][mb][1] = 0.f;
#pragma unroll
          for (int nd = 0; nd < ND; ++nd)
#pragma unroll
            for (int x = 0; x < 4; ++x) o[hh][mb][nd][x] = 0.f;
        }


      for (int j0 = un.ks & ~(kTileK - 1); j0 < un.ke; j0 += kTileK) {
        const bool partial = (j0 < un.ks) || (j0 + kTileK > un.ke);
        // next tile; the unit's last tile fetches the next unit's first one (or re-reads itself at the very end: harmless)
        const int jn = j0 + kTileK < un.ke ? j0 + kTileK : (next_first >= 0 ? next_first : j0);
        mbar_wait(bar_bfull + 8 * bbuf, bphase);
        const uint32_t bias_buf = smem_u32(s_bias) + bbuf * (kBiasBufFloats * 4) + (g * kTileK + 4 * t) * 4;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int h = 2 * aw + hh;
          // ---- a4: S = bias + Q K^T for both 16-row blocks (four independent accumulator chains)
          float sA[2][4], sB[2][4];
#pragma unroll
          for (int mb = 0; mb < 2; ++mb) {
            const float4 b0 = lds_f32x4(bias_buf + (h * kBiasHeadPitch + mb * 16 * kTileK) * 4);
            const float4 b1 = lds_f32x4(bias_buf + (h * kBiasHeadPitch + (mb * 16 + 8) * kTileK) * 4);
            sA[mb][0] = b0.x; sA[mb][1] = b0.y; sA[mb][2] = b1.x; sA[mb][3] = b1.y;
            sB[mb][0] = b0.z; sB[mb][1] = b0.w; sB[mb][2] = b1.z; sB[mb][3] = b1.w;
          }
#pragma unroll
          for (int kk = 0; kk < KK; ++kk)
#pragma unroll
            for (int mb = 0; mb < 2; ++mb) {
              const uint2 qa = lds_u32x2(q_frag + (mb * 16) * kQP + hh * (CP * 2) + kk * 32);
              const uint2 qb = lds_u32x2(q_frag + (mb * 16 + 8) * kQP + hh * (CP * 2) + kk * 32);
              mma_bf16(sA[mb], qa.x, qb.x, qa.y, qb.y, kq[kk].x, kq[kk].y);
              mma_bf16(sB[mb], qa.x, qb.x, qa.y, qb.y, kq[kk].z, kq[kk].w);
            }
          if (hh == 0) load_k(j0, h + 1); else load_k(jn, h - 1);
          uint32_t pf[2][4];
#pragma unroll
          for (int mb = 0; mb < 2; ++mb) {
            if (partial) {
              const int k0 = j0 + 4 * t;
              if (k0 < un.ks || k0 >= un.ke) { sA[mb][0] = -INFINITY; sA[mb][2] = -INFINITY; }
              if (k0 + 1 < un.ks || k0 + 1 >= un.ke) { sA[mb][1] = -INFINITY; sA[mb][3] = -INFINITY; }
              if (k0 + 2 < un.ks || k0 + 2 >= un.ke) { sB[mb][0] = -INFINITY; sB[mb][2] = -INFINITY; }
              if (k0 + 3 < un.ks || k0 + 3 >= un.ke) { sB[mb][1] = -INFINITY; sB[mb][3] = -INFINITY; }
            }
            // ---- a5: online softmax (exp2 domain), rows g (x = 0) and g+8 (x = 1).  The reference m of a row moves only
            // when the tile maximum exceeds it by more than kLazy (P <= 2^kLazy stays well inside bf16 / fp32 range); a
            // state (m, l, acc) is defined up to its reference (reading 19).  Rows that keep their reference
            // have alpha == 1 exactly, so skipping the rescale when no row of the warp moved changes no bit.
            constexpr float kLazy = 8.f;
            const float mx0 = quad_max(fmaxf(fmaxf(sA[mb][0], sA[mb][1]), fmaxf(sB[mb][0], sB[mb][1])));
            const float mx1 = quad_max(fmaxf(fmaxf(sA[mb][2], sA[mb][3]), fmaxf(sB[mb][2], sB[mb][3])));
            const float mo0 = m_run[hh][mb][0], mo1 = m_run[hh][mb][1];
            const bool mv0 = mx0 > mo0 + kLazy, mv1 = mx1 > mo1 + kLazy;
            const float mn0 = mv0 ? mx0 : mo0, mn1 = mv1 ? mx1 : mo1;
            m_run[hh][mb][0] = mn0;
            m_run[hh][mb][1] = mn1;
            sA[mb][0] = fast_exp2(sA[mb][0] - mn0); sA[mb][1] = fast_exp2(sA[mb][1] - mn0);
            sB[mb][0] = fast_exp2(sB[mb][0] - mn0); sB[mb][1] = fast_exp2(sB[mb][1] - mn0);
            sA[mb][2] = fast_exp2(sA[mb][2] - mn1); sA[mb][3] = fast_exp2(sA[mb][3] - mn1);
            sB[mb][2] = fast_exp2(sB[mb][2] - mn1); sB[mb][3] = fast_exp2(sB[mb][3] - mn1);
            const float sum0 = (sA[mb][0] + sA[mb][1]) + (sB[mb][0] + sB[mb][1]);
            const float sum1 = (sA[mb][2] + sA[mb][3]) + (sB[mb][2] + sB[mb][3]);
            if (__any_sync(0xffffffffu, mv0 || mv1)) {
              const float al0 = mv0 ? fast_exp2(mo0 - mn0) : 1.f, al1 = mv1 ? fast_exp2(mo1 - mn1) : 1.f;
              l_run[hh][mb][0] *= al0;
              l_run[hh][mb][1] *= al1;
#pragma unroll
              for (int nd = 0; nd < ND; ++nd) {
                o[hh][mb][nd][0] *= al0; o[hh][mb][nd][1] *= al0;
                o[hh][mb][nd][2] *= al1; o[hh][mb][nd][3] *= al1;
              }
            }
            l_run[hh][mb][0] += sum0;
            l_run[hh][mb][1] += sum1;
            pf[mb][0] = pack_bf16(sA[mb][0], sA[mb][1]); pf[mb][1] = pack_bf16(sA[mb][2], sA[mb][3]);
            pf[mb][2] = pack_bf16(sB[mb][0], sB[mb][1]); pf[mb][3] = pack_bf16(sB[mb][2], sB[mb][3]);
          }
          // ---- a6: acc += P V
#pragma unroll
          for (int nd = 0; nd < ND; ++nd)
#pragma unroll
            for (int mb = 0; mb < 2; ++mb)
              mma_bf16(o[hh][mb][nd], pf[mb][0], pf[mb][1], pf[mb][2], pf[mb][3],
                       (nd & 1) ? vq[nd >> 1].z : vq[nd >> 1].x, (nd & 1) ? vq[nd >> 1].w : vq[nd >> 1].y);
          if (hh == 0) load_v(j0, h + 1); else load_v(jn, h - 1);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_bempty + 8 * bbuf);
        bbuf ^= 1;
        if (bbuf == 0) bphase ^= 1;
      }

      // ---- a7: partial state of (rows, key segment) -> slot   (m back in natural-log units).
      // acc goes through shared memory: in the MMA fragment layout a store instruction touches 8 rows (8 lines of 32
      // useful bytes; the unit's 96 KB cost ~7 us of LSU wavefronts, a what-if without them showed); staged per
      // (head, 16-row block) in the warp's slab of the Q tile's buffer -- free once every warp has finished the unit's
      // last QK^T -- and written back as 128-bit row pieces, a row's C floats contiguous.
      constexpr float kLn2 = 0.6931471805599453f;
      constexpr int kOPitch = C == 24 ? 40 : C + 8;            // floats; conflict-free 64-bit fragment writes
      static_assert(8 * 16 * kOPitch * 4 <= kTileQ * q_pitch(CP), "O staging fits the Q tile buffer");
      const uint32_t slab = s_q + aw * (16 * kOPitch * 4);
      asm volatile("bar.sync 1, 256;" ::: "memory");          // nobody reads this unit's Q tile any more
#pragma unroll
      for (int hh = 0; hh < 2; ++hh)
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          const int h = 2 * aw + hh;
#pragma unroll
          for (int x = 0; x < 2; ++x) {
            const float l = quad_sum(l_run[hh][mb][x]);
            const int row = un.q0 + mb * 16 + g + 8 * x;
            if (row < un.q_end && t == 0) {
              const int64_t srow = (int64_t)un.slot * p.state_rows + (row - p.state_row0);
              p.st_m[srow * kH + h] = m_run[hh][mb][x] * kLn2;
              p.st_l[srow * kH + h] = l;
            }
#pragma unroll
            for (int nd = 0; nd < ND; ++nd)
              asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(slab + ((g + 8 * x) * kOPitch + nd * 8 + 2 * t) * 4),
                           "f"(o[hh][mb][nd][2 * x]), "f"(o[hh][mb][nd][2 * x + 1]) : "memory");
          }
          __syncwarp();
#pragma unroll
          for (int i = 0; i < 16 * (C / 4) / 32; ++i) {
            const int e = i * 32 + lane, r = e / (C / 4), c4 = e - r * (C / 4);
            const int row = un.q0 + mb * 16 + r;
            const float4 v = lds_f32x4(slab + (r * kOPitch + c4 * 4) * 4);
            if (row < un.q_end) {
              const int64_t srow = (int64_t)un.slot * p.state_rows + (row - p.state_row0);
              *reinterpret_cast<float4*>(p.st_acc + srow * (kH * C) + h * C + c4 * 4) = v;
            }
          }
          __syncwarp();
        }
    }
  }
  // teardown: every role is done with tensor memory before the allocating warp frees it
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_base, kTmemCols);
  }
}

// ------------------------------------------------------------------ host side
template <int C, int CP>
cudaError_t launch_c(const CUtensorMap& tm, const CUtensorMap& tm_tail, const MmaParams& p, int64_t units, cudaStream_t st) {
  {   // per-device function attribute: set on every launch (cheap), so a process may use several GPUs
    cudaError_t e = cudaFuncSetAttribute(fused_mma_kernel<C, CP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_alloc(CP));
    if (e != cudaSuccess) return e;
  }
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (sms <= 0) sms = 148;
  const unsigned grid = (unsigned)(units < sms ? units : sms);
  return launch_kernel(fused_mma_kernel<C, CP>, dim3(grid), dim3(kThreads), smem_alloc(CP), st, p.pdl, tm, tm_tail, p);
}

}  // namespace

bool fused_mma_supports(dcp_dtype dt, int H, int c, int c_z) {
  return (dt == DCP_BF16 && H == kH && c_z == kCz && (c == 24 || c == 32 || c == 48)) || fused_atom_supports(dt, H, c, c_z);
}

int mma_head_pad(int c) { return (c + 15) / 16 * 16; }
// keys rounded up to 32: the atom kernel reads K / V two 16-key blocks at a time
int64_t mma_frag_elems(int64_t I, int H, int c) { return (I + 31) / 32 * 2 * H * (mma_head_pad(c) / 16) * 256; }

// Work units of the tensor-core kernels.  Cost model (in key tiles of one SM): waves x (tile height / 32) x (key tiles of
// a unit + kUnitOverhead) x (1 + the partial-state round trip, ~25 * slots / I of the z bytes), waves = ceil(units / 148).
// nseg is picked for the MONOLITHIC row count, so that it depends on (I, n_kparts) only -- every decomposition then cuts
// a row's keys alike (bitwise contract); the tile height (fused_mma_kernel only: a trimmed last TMA box makes a tile of
// h rows cost h / 32 of a full one) is picked afterwards for the actual row partition and changes no row's arithmetic.
namespace {
constexpr double kUnitOverhead = 1.5;    // key tiles: state write + Q reload + pipeline restart, measured ~5 us at C2
int64_t count_tiles(int64_t n, int parts, int h) {
  const int64_t base = n / parts, rem = n % parts;
  return rem * ((base + 1 + h - 1) / h) + (parts - rem) * ((base + h - 1) / h);
}
double unit_cost(int64_t I, int n_qparts, int n_kparts, int s, int h, int h_full, int tile_k) {
  const int64_t units = count_tiles(I, n_qparts, h) * n_kparts * s;
  const int64_t waves = (units + 147) / 148;
  const double key_tiles = (double)I / n_kparts / s / tile_k;
  // a lower tile streams fewer bytes but repeats the tile's fixed work (K / V fragments, attention MMAs over all 32 rows)
  const double fixed = 1.0 + 0.1 * (h_full - h) / 8.0;
  return (double)waves * ((double)h / h_full) * fixed * (key_tiles + kUnitOverhead) * (1.0 + 25.0 * s * n_kparts / (double)I);
}
}  // namespace

void mma_pick_units(int64_t I, int H, int n_qparts, int n_kparts, int force_nseg, int force_tile_h, int* nseg, int* tile_h) {
  const bool token = H == kH;
  const int h_full = token ? kTileQ : fused_atom_tile_q(), tile_k = token ? kTileK : 32;
  const int h_min = token ? 25 : h_full;
  const int64_t chunk = I / n_kparts;
  int best_s = 1;
  if (force_nseg > 0) best_s = force_nseg;
  else {
    double best = 1e300;
    for (int s = 1; s <= 16; ++s) {
      if (s > 1 && chunk / s < 64) break;
      for (int h = h_full; h >= h_min; --h) {
        const double c = unit_cost(I, 1, n_kparts, s, h, h_full, tile_k);
        if (c < best * (1.0 - 1e-9)) { best = c; best_s = s; }
      }
    }
  }
  int best_h = h_full;
  if (force_tile_h > 0) best_h = force_tile_h;
  else {
    double best = 1e300;
    for (int h = h_full; h >= h_min; --h) {
      const double c = unit_cost(I, n_qparts, n_kparts, best_s, h, h_full, tile_k);
      if (c < best * (1.0 - 1e-9)) { best = c; best_h = h; }
    }
  }
  *nseg = best_s;
  *tile_h = best_h;
}

cudaError_t launch_fused_mma(const MmaParams& p, const void* z, int64_t ldz, cudaStream_t st) {
  if (p.H != kH) return launch_fused_atom(p, z, ldz, st);
  if (p.bias_cache) return launch_cached_attn(p, st);      // cached_attn.cu: the bias comes from a cache, z is not read
  if (p.q_end <= p.q_begin || p.k_end <= p.k_begin) return cudaSuccess;
  PFN_cuTensorMapEncodeTiled enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tm;
  const cuuint64_t gdim[3] = {(cuuint64_t)kCz, (cuuint64_t)p.I, (cuuint64_t)p.I};
  const cuuint64_t gstr[2] = {(cuuint64_t)kCz * 2, (cuuint64_t)ldz * 2};
  const cuuint32_t box[3] = {64, kTileK, kSubQ};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(z), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  if (p.tile_h < 1 || p.tile_h > kTileQ) return cudaErrorInvalidValue;
  CUtensorMap tm_tail = tm;                                  // tile heights that are not a multiple of 8: the tile's last box
  if (p.tile_h % kSubQ != 0) {
    const cuuint32_t box_t[3] = {64, kTileK, (cuuint32_t)(p.tile_h % kSubQ)};
    r = enc(&tm_tail, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(z), gdim, gstr, box_t, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  }
  const int64_t units = mma_num_units<0>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg, p.tile_h);
  if (units > 0x7fffffff) return cudaErrorInvalidValue;
  switch (p.c) {
    case 24: return launch_c<24, 32>(tm, tm_tail, p, units, st);
    case 32: return launch_c<32, 32>(tm, tm_tail, p, units, st);
    case 48: return launch_c<48, 48>(tm, tm_tail, p, units, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace dcp
