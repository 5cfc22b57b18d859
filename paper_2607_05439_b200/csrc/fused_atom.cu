// bf16 tensor-core fused kernel for the atom-level layer (steps a2-a7 of SURVEY.md section 8(a), BASELINE.json config 4):
// c_atompair = 16 channels per pair, H = 4 heads, head dim c = 32.  Same computation as fused_mma.cu
//   LayerNorm(p_lm) -> bias_h -> logit = q_l^h . k_m^h / sqrt(c) + bias_h -> online softmax -> acc += P V
//   (PAPER.md:58 "learned projection of Z"; :83 Eq. 2; :40, :90 running softmax statistics)
// in the low-c_z regime: 32 bytes of p per pair, so the per-pair instruction budget (not the tensor pipe) is what
// has to be watched.  p is streamed from HBM exactly once by TMA (32-byte swizzle) through a 3-stage mbarrier ring.
//
// One persistent CTA per SM, 16 warps, warp-specialised:
//   warp 0        TMA producer: one box (16 ch, 32 keys, 32 queries) = 1024 pairs = 32 KB per stage
//   warp 1        tcgen05 issuer: per stage 8 MMAs (M = 128 pairs, N = 16, K = 16): z . W''^T with W'' rows 0-3 =
//                 (gamma (.) W_b log2 e)^T, row 4 = ones (sum_k z), accumulators in tensor memory (2 x 128 columns)
//   warps 4-7     LayerNorm statistics + bias epilogue: thread = pair; sum_k z^2 from the thread's own 32-byte row of
//                 the stage (2 LDS.128, 16 mixed-precision FMAs), z.W' and sum_k z from TMEM;
//                 bias = rstd*(z.W' - mu*c1) + c0 -> shared tile bias[h][64 queries][32 keys] fp32 (double buffered)
//   warps 8-15    attention: warp = (head, 32-query half): S = bias + Q K^T (mma.sync m16n8k16), online softmax in the
//                 exp2 domain with a lazy reference, P (bf16) feeds PV from registers; Q and O live in registers,
//                 K / V fragments (MMA B-fragment order, gemm_mma.cu) are 128-bit L2 / L1 loads
// Work unit = (64-query tile) x (key segment); key tiles are aligned to absolute multiples of 32 and a row's arithmetic
// depends only on its key segments.  No atomics.
#include <cstdlib>

#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int aCz = 16, aH = 4, aC = 32;
constexpr int aTileQ = 64;           // queries per work unit
constexpr int aTileK = 32;           // keys per attention tile
constexpr int aSubQ = 32;            // queries per p stage
constexpr int aNZ = 3;               // p stages
constexpr int aStageBytes = aSubQ * aTileK * aCz * 2;    // 32 KB
constexpr int aMmaPerStage = aSubQ * aTileK / 128;       // 8
constexpr int aThreads = 512;
constexpr int aProjWarp0 = 4, aNumProjWarps = 4, aAttnWarp0 = 8, aNumAttnWarps = 8;
constexpr int aProjN = 16;                               // projection MMA N: 4 heads, the ones row, zero rows
constexpr int aTmemBufCols = aMmaPerStage * aProjN;      // 128
constexpr int aTmemCols = 2 * aTmemBufCols;              // 256
constexpr int aBiasBufFloats = aH * aTileQ * aTileK;     // 8192 floats = 32 KB

constexpr size_t aSmemZ = 0;
constexpr size_t aSmemBias = aSmemZ + (size_t)aNZ * aStageBytes;
constexpr size_t aSmemWt = aSmemBias + 2 * (size_t)aBiasBufFloats * 4;     // 512 B, 1024-aligned
constexpr size_t aSmemBar = aSmemWt + 512;
constexpr size_t aSmemTotal = aSmemBar + (2 * aNZ + 8) * 8 + 16;
constexpr size_t aSmemAlloc = aSmemTotal + 1024;         // slack for 1024-byte alignment

// K-major operand tile, 32-byte swizzle: rows of 16 bf16 (32 B), 8-row groups 256 B apart (SBO), descriptor version 1
// (sm_100), layout type 6 = SWIZZLE_32B.  K = 16 is one MMA k-step: no advance inside the atom.
__device__ __forceinline__ uint64_t umma_desc_sw32(uint32_t addr) {
  return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)6 << 61);
}
__device__ __forceinline__ void tmem_ld_x8(uint32_t taddr, float (&v)[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}

// kWide (L % 4 == 0): p is viewed as [L queries][L / 4 key groups][4 keys x 16 ch = 128 bytes] and fetched with 128-byte
// TMA rows (128-byte swizzle): a 32 KB stage is 256 TMA rows instead of 1024 -- with 32-byte rows the TMA engine, not HBM,
// capped the stream at 5.8 TB/s.  Stage row = 8 q + key group; MMA (b, s), b = 128-row block, s = key
// inside the group, reads the 32 bytes at offset 32 s of every row (the K = 16 slice of the swizzle atom): its TMEM lane r
// is the pair (query 16 b + r / 8, key 4 (r % 8) + s) of the stage.  Otherwise (any L): 32-byte rows, stage row = 32 q +
// key, MMA m covers queries 4 m .. 4 m + 3.
template <bool kWide>
__global__ void __launch_bounds__(aThreads, 1) fused_atom_kernel(const __grid_constant__ CUtensorMap tmap_z,
                                                                 const MmaParams p) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
  const uint32_t s_z = smem_u32(smem + aSmemZ);
  const uint32_t s_bias = smem_u32(smem + aSmemBias);
  const uint32_t s_wt = smem_u32(smem + aSmemWt);
  const uint32_t s_bar = smem_u32(smem + aSmemBar);
  const uint32_t bar_zfull = s_bar, bar_zempty = s_bar + 8 * aNZ, bar_bfull = s_bar + 16 * aNZ,
                 bar_bempty = s_bar + 16 * aNZ + 16, bar_tfull = s_bar + 16 * aNZ + 32, bar_tempty = s_bar + 16 * aNZ + 48;
  volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(smem + aSmemBar + (2 * aNZ + 8) * 8);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;

  pdl_trigger();
  if (threadIdx.x == 0) {
    // zempty: the tcgen05.commit of the stage's MMAs + the four epilogue warps that read the rows with LDS
    for (int s = 0; s < aNZ; ++s) { mbar_init(bar_zfull + 8 * s, 1); mbar_init(bar_zempty + 8 * s, 1 + aNumProjWarps); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar_bfull + 8 * b, aNumProjWarps); mbar_init(bar_bempty + 8 * b, aNumAttnWarps);
      mbar_init(bar_tfull + 8 * b, 1); mbar_init(bar_tempty + 8 * b, aNumProjWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), aTmemCols);
  pdl_wait();          // the prologue's q / k / v / folded weights are final (and so is everything before it in the stream)
  // W'' = B operand of the projection MMA: 16 rows (n) x 16 channels, K-major, 32-byte swizzle by hand (16-byte chunk
  // index ^ bit 2 of the row): row n < 4 = head n of (gamma (.) W_b log2 e)^T, row 4 = ones, rows 5..15 = 0.
  if (threadIdx.x < aProjN * 2) {
    const int n = threadIdx.x >> 1, ch = threadIdx.x & 1;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (n < aH) v = __ldg(reinterpret_cast<const uint4*>(p.wfold) + n * 2 + ch);
    else if (n == aH) v = make_uint4(0x3f803f80u, 0x3f803f80u, 0x3f803f80u, 0x3f803f80u);
    *reinterpret_cast<uint4*>(smem + aSmemWt + n * 32 + ((ch ^ ((n >> 2) & 1)) << 4)) = v;
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to tcgen05
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *s_tmem;

  const int n_units = (int)mma_num_units<aTileQ>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg);

  if (warp < aProjWarp0) {
    reg_dec<24>();
    if (warp == 0 && lane == 0) {
      // =============================================================== TMA producer
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      int stage = 0;
      uint32_t phase = 0;
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const Unit un = decode_unit<aTileQ, aTileK>(p, u);
        const int rows = (un.q_end - un.q0) < aTileQ ? (un.q_end - un.q0) : aTileQ;
        const int nsub = (rows + aSubQ - 1) / aSubQ;
        for (int j0 = un.ks & ~(aTileK - 1); j0 < un.ke; j0 += aTileK) {
          for (int sub = 0; sub < nsub; ++sub) {
            mbar_wait(bar_zempty + 8 * stage, phase ^ 1);
            mbar_expect_tx(bar_zfull + 8 * stage, aStageBytes);
            tma_load_3d(s_z + stage * aStageBytes, &tmap_z, 0, kWide ? j0 >> 2 : j0, un.q0 + sub * aSubQ, bar_zfull + 8 * stage, policy);
            if (++stage == aNZ) { stage = 0; phase ^= 1; }
          }
        }
      }
    } else if (warp == 1 && lane == 0) {
      // =============================================================== tcgen05 issuer
      // stage row 32 q + key (q = query of the stage, key = key of the tile); MMA m covers rows 128 m .. 128 m + 127
      constexpr uint32_t idesc = umma_idesc_bf16(128, aProjN);
      const uint64_t bdesc = umma_desc_sw32(s_wt);
      int stage = 0, tb = 0;
      uint32_t phase = 0, tphase = 0;
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const Unit un = decode_unit<aTileQ, aTileK>(p, u);
        const int rows = (un.q_end - un.q0) < aTileQ ? (un.q_end - un.q0) : aTileQ;
        const int nsub = (rows + aSubQ - 1) / aSubQ;
        for (int j0 = un.ks & ~(aTileK - 1); j0 < un.ke; j0 += aTileK) {
          for (int sub = 0; sub < nsub; ++sub) {
            mbar_wait(bar_tempty + 8 * tb, tphase ^ 1);
            mbar_wait(bar_zfull + 8 * stage, phase);
            tc_fence_after();
            const uint32_t zs = s_z + stage * aStageBytes;
#pragma unroll
            for (int m = 0; m < aMmaPerStage; ++m)
              umma_bf16(tmem_base + tb * aTmemBufCols + m * aProjN,
                        kWide ? umma_desc_sw128(zs + (m >> 2) * 16384 + (m & 3) * 32) : umma_desc_sw32(zs + m * 4096), bdesc, idesc, 0);
            umma_commit(bar_zempty + 8 * stage);
            umma_commit(bar_tfull + 8 * tb);
            if (++stage == aNZ) { stage = 0; phase ^= 1; }
            tb ^= 1;
            if (tb == 0) tphase ^= 1;
          }
        }
      }
    }
  } else if (warp < aAttnWarp0) {
    // =============================================================== LayerNorm statistics + bias epilogue (TMEM -> smem)
    // Thread = one pair row of each MMA: TMEM lane 32 pw + lane of MMA m = (query 4 m + pw of the stage, key lane).
    reg_dec<104>();
    const int pw = warp - aProjWarp0;                       // == warp % 4: the TMEM lane quadrant this warp may read
    float c1h[aH], c0h[aH];
#pragma unroll
    for (int h = 0; h < aH; ++h) { c1h[h] = __ldg(p.c1 + h); c0h[h] = __ldg(p.c0 + h); }
    const uint32_t t_lane = tmem_base + ((uint32_t)(pw * 32) << 16);
    // the thread's 32-byte row; lanes 4..7 (mod 8) read the second 16-byte chunk first: conflict-free LDS.128, and the
    // sum of squares does not care about the order (nor about the 32-byte swizzle, which only swaps the two chunks)
    const uint32_t zrow = s_z + (pw * 32 + lane) * 32 + ((lane >> 2) & 1) * 16;
    const uint32_t zrow2 = s_z + (pw * 32 + lane) * 32 + (((lane >> 2) & 1) ^ 1) * 16;
    int tb = 0, bbuf = 0, stage = 0;
    uint32_t tphase = 0, bphase = 0, zphase = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const Unit un = decode_unit<aTileQ, aTileK>(p, u);
      const int rows = (un.q_end - un.q0) < aTileQ ? (un.q_end - un.q0) : aTileQ;
      const int nsub = (rows + aSubQ - 1) / aSubQ;
      for (int j0 = un.ks & ~(aTileK - 1); j0 < un.ke; j0 += aTileK) {
        mbar_wait(bar_bempty + 8 * bbuf, bphase ^ 1);
        const uint32_t bias_buf = s_bias + bbuf * (aBiasBufFloats * 4);
        for (int sub = 0; sub < nsub; ++sub) {
          // ---- a2: sum_k z^2 of the thread's 8 pairs straight from the TMA stage
          mbar_wait(bar_zfull + 8 * stage, zphase);
          float zsq[aMmaPerStage];
          if constexpr (kWide) {
            // the thread's two 128-byte rows (one per block b): key s of the group = 16-byte chunks 2 s, 2 s + 1, each at
            // (chunk ^ row % 8): eight conflict-free LDS.128 per row
            const uint32_t rp = pw * 32 + lane, sw = rp & 7;
#pragma unroll
            for (int b = 0; b < 2; ++b) {
              const uint32_t base = s_z + stage * aStageBytes + (128 * b + rp) * 128;
              uint4 w[8];
#pragma unroll
              for (int c = 0; c < 8; ++c) w[c] = lds_u32x4(base + ((c ^ sw) << 4));
#pragma unroll
              for (int sk = 0; sk < 4; ++sk) {
                float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
                fma_sq_bf16x2(s0, s1, w[2 * sk].x); fma_sq_bf16x2(s2, s3, w[2 * sk].y);
                fma_sq_bf16x2(s0, s1, w[2 * sk].z); fma_sq_bf16x2(s2, s3, w[2 * sk].w);
                fma_sq_bf16x2(s0, s1, w[2 * sk + 1].x); fma_sq_bf16x2(s2, s3, w[2 * sk + 1].y);
                fma_sq_bf16x2(s0, s1, w[2 * sk + 1].z); fma_sq_bf16x2(s2, s3, w[2 * sk + 1].w);
                zsq[4 * b + sk] = (s0 + s1) + (s2 + s3);
              }
            }
          } else {
#pragma unroll
          for (int m = 0; m < aMmaPerStage; ++m) {
            const uint4 w0 = lds_u32x4(zrow + stage * aStageBytes + m * 4096);
            const uint4 w1 = lds_u32x4(zrow2 + stage * aStageBytes + m * 4096);
            float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
            fma_sq_bf16x2(s0, s1, w0.x); fma_sq_bf16x2(s2, s3, w0.y);
            fma_sq_bf16x2(s0, s1, w0.z); fma_sq_bf16x2(s2, s3, w0.w);
            fma_sq_bf16x2(s0, s1, w1.x); fma_sq_bf16x2(s2, s3, w1.y);
            fma_sq_bf16x2(s0, s1, w1.z); fma_sq_bf16x2(s2, s3, w1.w);
            zsq[m] = (s0 + s1) + (s2 + s3);
          }
          }
#pragma unroll
          for (int m = 0; m < aMmaPerStage; ++m) asm volatile("" : "+f"(zsq[m]));   // rows consumed before the release
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_zempty + 8 * stage);
          if (++stage == aNZ) { stage = 0; zphase ^= 1; }
          // ---- a3: z.W' (4 heads) and sum_k z from tensor memory, four MMAs at a time
          mbar_wait(bar_tfull + 8 * tb, tphase);
          tc_fence_after();
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            float v[4][8];
#pragma unroll
            for (int i = 0; i < 4; ++i) tmem_ld_x8(t_lane + tb * aTmemBufCols + (half * 4 + i) * aProjN, v[i]);
            tmem_ld_wait();
            if (half == 1) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive(bar_tempty + 8 * tb);    // accumulators are in registers: buffer free
            }
            if constexpr (kWide) {
              // the four MMAs of this block are the four keys of the thread's group: one 128-bit store per head
              float bv[aH][4];
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const float mu = v[i][aH] * (1.f / aCz);
                const float var = fmaf(-mu, mu, zsq[half * 4 + i] * (1.f / aCz));
                const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;
                const float nm = -mu * rstd;
#pragma unroll
                for (int h = 0; h < aH; ++h) bv[h][i] = fmaf(v[i][h], rstd, fmaf(nm, c1h[h], c0h[h]));
              }
              const int ql = sub * aSubQ + 16 * half + 4 * pw + (lane >> 3);
              const uint32_t brow = bias_buf + (ql * aTileK + ((4 * (lane & 7)) ^ ((ql & 1) << 4))) * 4;
#pragma unroll
              for (int h = 0; h < aH; ++h)
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(brow + h * (aTileQ * aTileK * 4)), "f"(bv[h][0]),
                             "f"(bv[h][1]), "f"(bv[h][2]), "f"(bv[h][3]) : "memory");
            } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int m = half * 4 + i;
              // LayerNorm statistics (fp32): mu = sum/c_z, var = sum z^2 / c_z - mu^2
              const float mu = v[i][aH] * (1.f / aCz);
              const float var = fmaf(-mu, mu, zsq[m] * (1.f / aCz));   // one rounding; == 0 exactly for a constant row
              const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;  // (fused_mma.cu has the argument)
              const float nm = -mu * rstd;
              // bias[h][query][key ^ 16 (query odd)]: the XOR makes the attention warps' 128-bit reads conflict-free
              const int ql = sub * aSubQ + 4 * m + pw;
              const uint32_t brow = bias_buf + (ql * aTileK + (lane ^ ((ql & 1) << 4))) * 4;
#pragma unroll
              for (int h = 0; h < aH; ++h)
                sts_f32(brow + h * (aTileQ * aTileK * 4), fmaf(v[i][h], rstd, fmaf(nm, c1h[h], c0h[h])));
            }
            }
          }
          tb ^= 1;
          if (tb == 0) tphase ^= 1;
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
    const int aw = warp - aAttnWarp0;
    const int h = aw & 3, qhalf = aw >> 2;        // this warp: head h, tile rows 32 qhalf .. 32 qhalf + 31
    constexpr int KK = aC / 16;                   // k-steps of QK^T (2)
    constexpr int ND = aC / 8;                    // n-blocks of PV (4)
    constexpr int NDP = aC / 16;                  // 128-bit V fragment loads per 16-key block (2)
    const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.qp);
    const uint4* kfr = reinterpret_cast<const uint4*>(p.kfr);
    const uint4* vfr = reinterpret_cast<const uint4*>(p.vfr);
    int bbuf = 0;
    uint32_t bphase = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const Unit un = decode_unit<aTileQ, aTileK>(p, u);
      // Q fragments (registers): [m-block][k-step] -> (a0, a2) of row g and (a1, a3) of row g + 8
      uint2 qa[2][KK], qb[2][KK];
#pragma unroll
      for (int mb = 0; mb < 2; ++mb) {
        const int r0i = un.q0 + 32 * qhalf + mb * 16 + g, r1i = r0i + 8;
        const int64_t r0 = r0i < p.I ? r0i : p.I - 1;
        const int64_t r1 = r1i < p.I ? r1i : p.I - 1;
#pragma unroll
        for (int kk = 0; kk < KK; ++kk) {
          qa[mb][kk] = ldg_u2(qp + (r0 * aH + h) * aC + kk * 16 + 4 * t);
          qb[mb][kk] = ldg_u2(qp + (r1 * aH + h) * aC + kk * 16 + 4 * t);
        }
      }
      float o[2][ND][4];
      float m_run[2][2], l_run[2][2];
#pragma unroll
      for (int mb = 0; mb < 2; ++mb) {
        m_run[mb][0] = m_run[mb][1] = -INFINITY;
        l_run[mb][0] = l_run[mb][1] = 0.f;
#pragma unroll
        for (int nd = 0; nd < ND; ++nd)
#pragma unroll
          for (int x = 0; x < 4; ++x) o[mb][nd][x] = 0.f;
      }
      // K / V fragments of the tile's two 16-key blocks T = 0, 1 (MMA B-fragment order: one 128-bit load per lane);
      // the next tile's K is requested right after the last QK^T MMA, its V right after the last PV MMA.
      // key of S column: block T, n-block A col c <-> j + 16 T + 4 (c / 2) + c % 2, n-block B col c <-> that + 2
      uint4 kq[2][KK], vq[2][NDP];
      auto load_k = [&](int j) {
#pragma unroll
        for (int T = 0; T < 2; ++T) {
          const uint4* src = kfr + ((int64_t)(((j >> 4) + T) * aH + h) * KK) * 32 + lane;
#pragma unroll
          for (int kk = 0; kk < KK; ++kk) kq[T][kk] = __ldg(src + kk * 32);
        }
      };
      auto load_v = [&](int j) {
#pragma unroll
        for (int T = 0; T < 2; ++T) {
          const uint4* src = vfr + ((int64_t)(((j >> 4) + T) * aH + h) * NDP) * 32 + lane;
#pragma unroll
          for (int ndp = 0; ndp < NDP; ++ndp) vq[T][ndp] = __ldg(src + ndp * 32);
        }
      };
      load_k(un.ks & ~(aTileK - 1));
      load_v(un.ks & ~(aTileK - 1));

      for (int j0 = un.ks & ~(aTileK - 1); j0 < un.ke; j0 += aTileK) {
        const bool partial = (j0 < un.ks) || (j0 + aTileK > un.ke);
        const int jn = j0 + aTileK < un.ke ? j0 + aTileK : j0;     // next tile (the last one re-reads itself: harmless)
        mbar_wait(bar_bfull + 8 * bbuf, bphase);
        // bias[h][row][key ^ 16 (row odd)]; tile row of (mb, x) = 32 qhalf + 16 mb + g + 8 x, odd iff g is odd
        const uint32_t bias_row = s_bias + bbuf * (aBiasBufFloats * 4) + ((h * aTileQ + 32 * qhalf + g) * aTileK + 4 * t) * 4;
        // ---- a4: S = bias + Q K^T: [m-block][key block T] x (n-block A, n-block B)
        float sA[2][2][4], sB[2][2][4];
#pragma unroll
        for (int mb = 0; mb < 2; ++mb)
#pragma unroll
          for (int T = 0; T < 2; ++T) {
            const int col = 16 * (T ^ (g & 1));      // the row's keys 16 T + 4 t .. + 3 after the XOR swizzle
            const float4 b0 = lds_f32x4(bias_row + ((mb * 16) * aTileK + col) * 4);
            const float4 b1 = lds_f32x4(bias_row + ((mb * 16 + 8) * aTileK + col) * 4);
            sA[mb][T][0] = b0.x; sA[mb][T][1] = b0.y; sA[mb][T][2] = b1.x; sA[mb][T][3] = b1.y;
            sB[mb][T][0] = b0.z; sB[mb][T][1] = b0.w; sB[mb][T][2] = b1.z; sB[mb][T][3] = b1.w;
          }
#pragma unroll
        for (int kk = 0; kk < KK; ++kk)
#pragma unroll
          for (int mb = 0; mb < 2; ++mb)
#pragma unroll
            for (int T = 0; T < 2; ++T) {
              mma_bf16(sA[mb][T], qa[mb][kk].x, qb[mb][kk].x, qa[mb][kk].y, qb[mb][kk].y, kq[T][kk].x, kq[T][kk].y);
              mma_bf16(sB[mb][T], qa[mb][kk].x, qb[mb][kk].x, qa[mb][kk].y, qb[mb][kk].y, kq[T][kk].z, kq[T][kk].w);
            }
        load_k(jn);
        if (partial) {
#pragma unroll
          for (int T = 0; T < 2; ++T) {
            const int k0 = j0 + 16 * T + 4 * t;
#pragma unroll
            for (int mb = 0; mb < 2; ++mb) {
              if (k0 < un.ks || k0 >= un.ke) { sA[mb][T][0] = -INFINITY; sA[mb][T][2] = -INFINITY; }
              if (k0 + 1 < un.ks || k0 + 1 >= un.ke) { sA[mb][T][1] = -INFINITY; sA[mb][T][3] = -INFINITY; }
              if (k0 + 2 < un.ks || k0 + 2 >= un.ke) { sB[mb][T][0] = -INFINITY; sB[mb][T][2] = -INFINITY; }
              if (k0 + 3 < un.ks || k0 + 3 >= un.ke) { sB[mb][T][1] = -INFINITY; sB[mb][T][3] = -INFINITY; }
            }
          }
        }
        // ---- a5: online softmax (exp2 domain), rows g (x = 0) and g + 8 (x = 1) of each m-block, 32 keys at once.
        // The reference m of a row moves only when the tile maximum exceeds it by more than kLazy (P <= 2^kLazy stays
        // well inside bf16 / fp32 range); a state (m, l, acc) is defined up to its reference (reading 19).
        // Rows that keep their reference have alpha == 1 exactly, so skipping the rescale when no row of the warp moved
        // changes no bit.
        constexpr float kLazy = 8.f;
        uint32_t pf[2][2][4];
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          float mx0 = fmaxf(fmaxf(sA[mb][0][0], sA[mb][0][1]), fmaxf(sB[mb][0][0], sB[mb][0][1]));
          float mx1 = fmaxf(fmaxf(sA[mb][0][2], sA[mb][0][3]), fmaxf(sB[mb][0][2], sB[mb][0][3]));
          mx0 = fmaxf(mx0, fmaxf(fmaxf(sA[mb][1][0], sA[mb][1][1]), fmaxf(sB[mb][1][0], sB[mb][1][1])));
          mx1 = fmaxf(mx1, fmaxf(fmaxf(sA[mb][1][2], sA[mb][1][3]), fmaxf(sB[mb][1][2], sB[mb][1][3])));
          mx0 = quad_max(mx0);
          mx1 = quad_max(mx1);
          const float mo0 = m_run[mb][0], mo1 = m_run[mb][1];
          const bool mv0 = mx0 > mo0 + kLazy, mv1 = mx1 > mo1 + kLazy;
          const float mn0 = mv0 ? mx0 : mo0, mn1 = mv1 ? mx1 : mo1;
          m_run[mb][0] = mn0;
          m_run[mb][1] = mn1;
          float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
          for (int T = 0; T < 2; ++T) {
            sA[mb][T][0] = fast_exp2(sA[mb][T][0] - mn0); sA[mb][T][1] = fast_exp2(sA[mb][T][1] - mn0);
            sB[mb][T][0] = fast_exp2(sB[mb][T][0] - mn0); sB[mb][T][1] = fast_exp2(sB[mb][T][1] - mn0);
            sA[mb][T][2] = fast_exp2(sA[mb][T][2] - mn1); sA[mb][T][3] = fast_exp2(sA[mb][T][3] - mn1);
            sB[mb][T][2] = fast_exp2(sB[mb][T][2] - mn1); sB[mb][T][3] = fast_exp2(sB[mb][T][3] - mn1);
            sum0 += (sA[mb][T][0] + sA[mb][T][1]) + (sB[mb][T][0] + sB[mb][T][1]);
            sum1 += (sA[mb][T][2] + sA[mb][T][3]) + (sB[mb][T][2] + sB[mb][T][3]);
            pf[mb][T][0] = pack_bf16(sA[mb][T][0], sA[mb][T][1]); pf[mb][T][1] = pack_bf16(sA[mb][T][2], sA[mb][T][3]);
            pf[mb][T][2] = pack_bf16(sB[mb][T][0], sB[mb][T][1]); pf[mb][T][3] = pack_bf16(sB[mb][T][2], sB[mb][T][3]);
          }
          if (__any_sync(0xffffffffu, mv0 || mv1)) {
            const float al0 = mv0 ? fast_exp2(mo0 - mn0) : 1.f, al1 = mv1 ? fast_exp2(mo1 - mn1) : 1.f;
            l_run[mb][0] *= al0;
            l_run[mb][1] *= al1;
#pragma unroll
            for (int nd = 0; nd < ND; ++nd) {
              o[mb][nd][0] *= al0; o[mb][nd][1] *= al0;
              o[mb][nd][2] *= al1; o[mb][nd][3] *= al1;
            }
          }
          l_run[mb][0] += sum0;
          l_run[mb][1] += sum1;
        }
        // ---- a6: acc += P V
#pragma unroll
        for (int T = 0; T < 2; ++T)
#pragma unroll
          for (int nd = 0; nd < ND; ++nd)
#pragma unroll
            for (int mb = 0; mb < 2; ++mb)
              mma_bf16(o[mb][nd], pf[mb][T][0], pf[mb][T][1], pf[mb][T][2], pf[mb][T][3],
                       (nd & 1) ? vq[T][nd >> 1].z : vq[T][nd >> 1].x, (nd & 1) ? vq[T][nd >> 1].w : vq[T][nd >> 1].y);
        load_v(jn);
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_bempty + 8 * bbuf);
        bbuf ^= 1;
        if (bbuf == 0) bphase ^= 1;
      }

      // ---- a7: partial state of (rows, key segment) -> slot   (m back in natural-log units)
      constexpr float kLn2 = 0.6931471805599453f;
#pragma unroll
      for (int mb = 0; mb < 2; ++mb)
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          const float l = quad_sum(l_run[mb][x]);
          const int row = un.q0 + 32 * qhalf + mb * 16 + g + 8 * x;
          if (row < un.q_end) {
            const int64_t srow = (int64_t)un.slot * p.state_rows + (row - p.state_row0);
            if (t == 0) {
              p.st_m[srow * aH + h] = m_run[mb][x] * kLn2;
              p.st_l[srow * aH + h] = l;
            }
            float* dst = p.st_acc + srow * (aH * aC) + h * aC + 2 * t;
#pragma unroll
            for (int nd = 0; nd < ND; ++nd)
              *reinterpret_cast<float2*>(dst + nd * 8) = make_float2(o[mb][nd][2 * x], o[mb][nd][2 * x + 1]);
          }
        }
    }
  }
  // teardown: every role is done with tensor memory before the allocating warp frees it
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_base, aTmemCols);
  }
}

}  // namespace

bool fused_atom_supports(dcp_dtype dt, int H, int c, int c_z) { return dt == DCP_BF16 && H == aH && c == aC && c_z == aCz; }
int fused_atom_tile_q() { return aTileQ; }

cudaError_t launch_fused_atom(const MmaParams& p, const void* z, int64_t ldz, cudaStream_t st) {
  if (p.q_end <= p.q_begin || p.k_end <= p.k_begin) return cudaSuccess;
  PFN_cuTensorMapEncodeTiled enc = get_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tm;
  static const bool narrow_only = [] { const char* e = getenv("DCP_ATOM_NARROW"); return e && e[0] == '1'; }();   // A-B timing switch
  const bool wide = p.I % 4 == 0 && !narrow_only;          // whole key groups of 4: 128-byte TMA rows
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r;
  if (wide) {
    const cuuint64_t gdim[3] = {(cuuint64_t)4 * aCz, (cuuint64_t)p.I / 4, (cuuint64_t)p.I};
    const cuuint64_t gstr[2] = {(cuuint64_t)4 * aCz * 2, (cuuint64_t)ldz * 2};
    const cuuint32_t box[3] = {4 * aCz, aTileK / 4, aSubQ};
    r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(z), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  } else {
    const cuuint64_t gdim[3] = {(cuuint64_t)aCz, (cuuint64_t)p.I, (cuuint64_t)p.I};
    const cuuint64_t gstr[2] = {(cuuint64_t)aCz * 2, (cuuint64_t)ldz * 2};
    const cuuint32_t box[3] = {aCz, aTileK, aSubQ};
    r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(z), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  const int64_t units = mma_num_units<aTileQ>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg);
  if (units > 0x7fffffff) return cudaErrorInvalidValue;
  {   // per-device function attribute: set on every launch (cheap), so a process may use several GPUs
    cudaError_t e = cudaFuncSetAttribute(fused_atom_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)aSmemAlloc);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(fused_atom_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)aSmemAlloc);
    if (e != cudaSuccess) return e;
  }
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (sms <= 0) sms = 148;
  const unsigned grid = (unsigned)(units < sms ? units : sms);
  return wide ? launch_kernel(fused_atom_kernel<true>, dim3(grid), dim3(aThreads), aSmemAlloc, st, p.pdl, tm, p)
              : launch_kernel(fused_atom_kernel<false>, dim3(grid), dim3(aThreads), aSmemAlloc, st, p.pdl, tm, p);
}

}  // namespace dcp
