// Attention over a bias cache (steps a4-a7 of SURVEY.md section 8(a) for the blocks of dcp_attention_stack_cached;
// DESIGN.md 6.8): the bias of every (block, head, pair) was written once by bias_tiles_kernel (bias_tiles.cu) as fp16
// tiles, so a block reads 32 bytes per pair instead of the 256 bytes of z and no LayerNorm / projection runs here.
//   logit_h = q_i^h . k_j^h / sqrt(c) + bias_h (Eq. 2), online softmax with running (m, l, acc)
// With the z side gone the kernel is paced by the attention warps themselves (mma.sync + softmax at the issue rate of two
// warps per scheduler in fused_mma_kernel), so this kernel spends the registers the projection warps held there on twice
// as many attention warps: one persistent CTA per SM, 16 warps of 128 registers, warp = head.  For the unit's 32 queries
// (two m16 blocks) S = bias + Q K^T, online softmax in the exp2 domain with the lazily moving reference of fused_mma.cu
// (same arithmetic, same order), P (bf16) feeds PV from registers, O stays in registers (48 per thread).
//   packages     per key tile {bias tile 16 KB [8-query block][head pair][8 queries][16 keys] half2, K fragments, V
//                fragments of all heads}, three bulk copies (cp.async.bulk) on one mbarrier into a ring of pkg_count
//                buffers: fragments are read by conflict-free 128-bit shared loads, no warp waits on an L2 round trip
//   refill       there is no producer warp (a 17th warp would cap every thread at 96 registers): the warp that finishes
//                a buffer LAST (shared-memory atomic counter per buffer) issues the copies of the tile pkg_count ahead
//   Q tile       kept in shared memory in A-fragment order ([m16 block][k-step][head][lane] x 16 bytes), so one 128-bit
//                load delivers the four MMA operand registers in place
// Work units, key segments and the partial-state slots are those of fused_mma_kernel (mma_ptx.cuh decode_unit), so the
// merge kernel and the bitwise decomposition contract are unchanged.
#include <type_traits>

#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int cH = 16;
constexpr int cTileQ = 32;
constexpr int cTileK = 16;
constexpr int cSubQ = 8;
constexpr int cAttnWarps = 16;
constexpr int cThreads = cAttnWarps * 32;
constexpr int cBiasBytes = (cH / 2) * cTileQ * cTileK * 4;                       // 16 KB
__host__ __device__ constexpr int c_frag_bytes(int CP) { return cH * (CP / 16) * 512; }
__host__ __device__ constexpr int c_pkg_bytes(int CP) { return cBiasBytes + 2 * c_frag_bytes(CP); }
__host__ __device__ constexpr int c_q_bytes(int CP) { return 2 * (CP / 16) * cH * 512; }   // A-fragment order
__host__ __device__ constexpr int c_o_pitch(int C) { return C == 24 ? 40 : C + 8; }   // floats
__host__ __device__ constexpr int c_qo_bytes(int C, int CP) {
  return c_q_bytes(CP) > cAttnWarps * 16 * c_o_pitch(C) * 4 ? c_q_bytes(CP) : cAttnWarps * 16 * c_o_pitch(C) * 4;
}
__host__ __device__ constexpr int c_pkg_count(int C, int CP) {
  return (220 * 1024 - c_qo_bytes(C, CP)) / c_pkg_bytes(CP) < 4 ? (220 * 1024 - c_qo_bytes(C, CP)) / c_pkg_bytes(CP) : 4;
}
__host__ __device__ constexpr size_t c_smem_alloc(int C, int CP) {
  return (size_t)c_pkg_count(C, CP) * c_pkg_bytes(CP) + c_qo_bytes(C, CP) + 2 * 8 * 8 + 128;   // + full[], done[] + alignment
}

// C = head dim, CP = C rounded up to a multiple of 16 (q / k rows are zero-padded to CP by the prologue)
template <int C, int CP>
__global__ void __launch_bounds__(cThreads, 1) cached_attn_kernel(const MmaParams p) {
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 127) & ~(uintptr_t)127);
  constexpr int kNC = c_pkg_count(C, CP), kPkg = c_pkg_bytes(CP), kFragBytes = c_frag_bytes(CP);
  static_assert(kNC >= 2, "two packages must fit shared memory");
  const uint32_t s_pkg = smem_u32(smem);
  const uint32_t s_q = s_pkg + kNC * kPkg;
  const uint32_t s_bar = s_q + c_qo_bytes(C, CP);            // full[kNC] mbarriers, then done[kNC] counters (u32)
  const uint32_t s_done = s_bar + 8 * kNC;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;
  const int n_units = (int)mma_num_units<0>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg, p.tile_h);
  const int KT = (p.I + cTileK - 1) / cTileK;

  // the CTA's tile sequence (unit by unit, key tile by key tile), walked kNC tiles ahead of the consumers by `nx`
  struct TileIt { int u, j, ke, qt; };
  auto it_unit = [&](TileIt& it) {
    if (it.u < n_units) {
      const Unit un = decode_unit<0, cTileK>(p, it.u);
      it.j = un.ks & ~(cTileK - 1); it.ke = un.ke; it.qt = un.q0 / cTileQ;
    }
  };
  auto it_next = [&](TileIt& it) {
    it.j += cTileK;
    if (it.j >= it.ke) { it.u += gridDim.x; it_unit(it); }
  };
  // one package -> buffer b (one thread): the full barrier's single arrival + the three copies' bytes
  auto fetch = [&](const TileIt& it, int b) {
    if (it.u >= n_units) return;
    const uint32_t bar = s_bar + 8 * b, dst = s_pkg + b * kPkg;
    const int kt = it.j / cTileK;
    mbar_expect_tx(bar, kPkg);
    bulk_copy_g2s(dst, p.bias_cache + ((int64_t)it.qt * KT + kt) * (cBiasBytes / 4), cBiasBytes, bar);
    bulk_copy_g2s(dst + cBiasBytes, reinterpret_cast<const char*>(p.kfr) + (int64_t)kt * kFragBytes, kFragBytes, bar);
    bulk_copy_g2s(dst + cBiasBytes + kFragBytes, reinterpret_cast<const char*>(p.vfr) + (int64_t)kt * kFragBytes, kFragBytes, bar);
  };

  pdl_trigger();
  TileIt nx{(int)blockIdx.x, 0, 0, 0};
  it_unit(nx);
  if (threadIdx.x == 0) {
    for (int b = 0; b < kNC; ++b) {
      mbar_init(s_bar + 8 * b, 1);
      asm volatile("st.shared.u32 [%0], %1;" ::"r"(s_done + 4 * b), "r"(0) : "memory");
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    pdl_wait();        // the prologue's q / k / v fragments and the bias cache are final
    TileIt it = nx;
    for (int b = 0; b < kNC; ++b) { fetch(it, b); it_next(it); }
  } else {
    pdl_wait();
  }
  for (int b = 0; b < kNC; ++b) it_next(nx);
  __syncthreads();

  // ================================================================= attention, warp = head
  const int h = warp;
  constexpr int KK = CP / 16;     // k-steps of QK^T
  constexpr int ND = C / 8;       // n-blocks of PV
  constexpr int NDP = CP / 16;    // V fragment pairs
  constexpr int kQRowChunks = cH * CP * 2 / 16;
  constexpr int kQIter = cTileQ * kQRowChunks / (cAttnWarps * 32);
  static_assert(kQIter * cAttnWarps * 32 == cTileQ * kQRowChunks, "Q tile chunks per thread");
  const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.qp);
  // A fragment of (m16 block mb, k-step kk, head h) for this lane: + (mb * KK + kk) * (cH * 512)
  const uint32_t q_frag = s_q + h * 512 + lane * 16;
  // this head's half of the bias words of rows g + 8 s, keys 4 t .. 4 t + 3: + s * (cBiasBytes / 4)
  const uint32_t bias_off = ((h >> 1) * (cSubQ * cTileK) + g * cTileK + 4 * t) * 4;
  const uint32_t k_off = cBiasBytes + ((h * KK) * 32 + lane) * 16, v_off = cBiasBytes + kFragBytes + ((h * NDP) * 32 + lane) * 16;
  int bbuf = 0;
  uint32_t bphase = 0;

  // The loop is compiled once per head parity (which half of a bias word the warp reads): a scheduler's four warps have
  // the same parity, so each runs one copy, with half the conversions of a run-time select.
  auto run = [&](auto HI) {
  constexpr int kHi = decltype(HI)::value;
  for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
    const Unit un = decode_unit<0, cTileK>(p, u);
    {
      // Q tile -> shared memory in A-fragment order; every chunk is requested before the barrier and stored after it:
      // the unit change costs one L2 round trip.  A 16-byte chunk = 8 consecutive k of (row r, head hd) = the (a0 | a1,
      // a2 | a3) words of lanes t = 2 (c & 1), + 1 of the row's group (k order within a 16-step: fused_mma.cu).
      uint4 qv[kQIter];
#pragma unroll
      for (int i = 0; i < kQIter; ++i) {
        const int e = threadIdx.x + i * (cAttnWarps * 32);
        const int r = e / kQRowChunks, ch = e - r * kQRowChunks;
        const int64_t row = (un.q0 + r) < p.I ? (un.q0 + r) : p.I - 1;
        qv[i] = __ldg(reinterpret_cast<const uint4*>(qp + row * (cH * CP)) + ch);
      }
      __syncthreads();                                        // every warp is done with the previous unit's O staging
#pragma unroll
      for (int i = 0; i < kQIter; ++i) {
        const int e = threadIdx.x + i * (cAttnWarps * 32);
        const int r = e / kQRowChunks, ch = e - r * kQRowChunks;
        const int hd = ch / (CP / 8), c8 = ch - hd * (CP / 8);
        const int mb = r >> 4, x = (r >> 3) & 1, gg = r & 7;
        const uint32_t dst = s_q + ((mb * KK + (c8 >> 1)) * cH + hd) * 512 + (gg * 4 + 2 * (c8 & 1)) * 16 + x * 4;
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst), "r"(qv[i].x) : "memory");
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + 8), "r"(qv[i].y) : "memory");
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + 16), "r"(qv[i].z) : "memory");
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + 24), "r"(qv[i].w) : "memory");
      }
    }
    __syncthreads();
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

    // one key tile; compiled twice: tiles cut by the segment's ends (at most the first and the last of a unit) mask
    // their foreign keys, the others carry no select at all
    auto tile = [&](const int j0, auto PART) {
      constexpr bool partial = decltype(PART)::value;
      mbar_wait(s_bar + 8 * bbuf, bphase);
      const uint32_t pkg = s_pkg + bbuf * kPkg;
      // ---- a4: S = bias + Q K^T for both 16-row blocks (four independent accumulator chains).  Column c of n-block A is
      // key j0 + 4 (c / 2) + c % 2, of n-block B that + 2 (the K fragment order of gemm_mma.cu).
      float sA[2][4], sB[2][4];
#pragma unroll
      for (int mb = 0; mb < 2; ++mb) {
        // word j of the 16 bytes = heads (2 (h / 2), 2 (h / 2) + 1) of key 4 t + j, fp16
        const uint4 b0 = lds_u32x4(pkg + bias_off + (2 * mb) * (cBiasBytes / 4));
        const uint4 b1 = lds_u32x4(pkg + bias_off + (2 * mb + 1) * (cBiasBytes / 4));
        sA[mb][0] = f16_half(b0.x, kHi); sA[mb][1] = f16_half(b0.y, kHi); sA[mb][2] = f16_half(b1.x, kHi); sA[mb][3] = f16_half(b1.y, kHi);
        sB[mb][0] = f16_half(b0.z, kHi); sB[mb][1] = f16_half(b0.w, kHi); sB[mb][2] = f16_half(b1.z, kHi); sB[mb][3] = f16_half(b1.w, kHi);
      }
#pragma unroll
      for (int kk = 0; kk < KK; ++kk) {
        const uint4 kq = lds_u32x4(pkg + k_off + kk * 512);
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          const uint4 qa = lds_u32x4(q_frag + (mb * KK + kk) * (cH * 512));
          mma_bf16(sA[mb], qa.x, qa.y, qa.z, qa.w, kq.x, kq.y);
          mma_bf16(sB[mb], qa.x, qa.y, qa.z, qa.w, kq.z, kq.w);
        }
      }
      uint32_t pf[2][4];
      if (partial) {
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          const int k0 = j0 + 4 * t;
          if (k0 < un.ks || k0 >= un.ke) { sA[mb][0] = -INFINITY; sA[mb][2] = -INFINITY; }
          if (k0 + 1 < un.ks || k0 + 1 >= un.ke) { sA[mb][1] = -INFINITY; sA[mb][3] = -INFINITY; }
          if (k0 + 2 < un.ks || k0 + 2 >= un.ke) { sB[mb][0] = -INFINITY; sB[mb][2] = -INFINITY; }
          if (k0 + 3 < un.ks || k0 + 3 >= un.ke) { sB[mb][1] = -INFINITY; sB[mb][3] = -INFINITY; }
        }
      }
      // ---- a5: online softmax (exp2 domain), rows g (x = 0) and g + 8 (x = 1); the reference m of a row moves only when
      // the tile maximum exceeds it by more than kLazy (reading 19; fused_mma.cu).  After the first tiles that is
      // rare, so the common tile only ASKS whether any logit exceeds its row's reference + kLazy (sixteen compares, one
      // vote) and skips the maxima, their two shuffle rounds and the rescale; the answer is the same predicate the maxima
      // would give, so no bit changes.
      constexpr float kLazy = 8.f;
      bool exceed = false;
#pragma unroll
      for (int mb = 0; mb < 2; ++mb) {
        const float t0 = m_run[mb][0] + kLazy, t1 = m_run[mb][1] + kLazy;
        exceed = exceed || sA[mb][0] > t0 || sA[mb][1] > t0 || sB[mb][0] > t0 || sB[mb][1] > t0 ||
                 sA[mb][2] > t1 || sA[mb][3] > t1 || sB[mb][2] > t1 || sB[mb][3] > t1;
      }
      const bool moved = __any_sync(0xffffffffu, exceed);
#pragma unroll
      for (int mb = 0; mb < 2; ++mb) {
        float mn0 = m_run[mb][0], mn1 = m_run[mb][1];
        if (moved) {
          const float mx0 = quad_max(fmaxf(fmaxf(sA[mb][0], sA[mb][1]), fmaxf(sB[mb][0], sB[mb][1])));
          const float mx1 = quad_max(fmaxf(fmaxf(sA[mb][2], sA[mb][3]), fmaxf(sB[mb][2], sB[mb][3])));
          const float mo0 = mn0, mo1 = mn1;
          const bool mv0 = mx0 > mo0 + kLazy, mv1 = mx1 > mo1 + kLazy;
          mn0 = mv0 ? mx0 : mo0;
          mn1 = mv1 ? mx1 : mo1;
          m_run[mb][0] = mn0;
          m_run[mb][1] = mn1;
          const float al0 = mv0 ? fast_exp2(mo0 - mn0) : 1.f, al1 = mv1 ? fast_exp2(mo1 - mn1) : 1.f;   // rows that stay: x 1
          l_run[mb][0] *= al0;
          l_run[mb][1] *= al1;
#pragma unroll
          for (int nd = 0; nd < ND; ++nd) {
            o[mb][nd][0] *= al0; o[mb][nd][1] *= al0;
            o[mb][nd][2] *= al1; o[mb][nd][3] *= al1;
          }
        }
        sA[mb][0] = fast_exp2(sA[mb][0] - mn0); sA[mb][1] = fast_exp2(sA[mb][1] - mn0);
        sB[mb][0] = fast_exp2(sB[mb][0] - mn0); sB[mb][1] = fast_exp2(sB[mb][1] - mn0);
        sA[mb][2] = fast_exp2(sA[mb][2] - mn1); sA[mb][3] = fast_exp2(sA[mb][3] - mn1);
        sB[mb][2] = fast_exp2(sB[mb][2] - mn1); sB[mb][3] = fast_exp2(sB[mb][3] - mn1);
        l_run[mb][0] += (sA[mb][0] + sA[mb][1]) + (sB[mb][0] + sB[mb][1]);
        l_run[mb][1] += (sA[mb][2] + sA[mb][3]) + (sB[mb][2] + sB[mb][3]);
        pf[mb][0] = pack_bf16(sA[mb][0], sA[mb][1]); pf[mb][1] = pack_bf16(sA[mb][2], sA[mb][3]);
        pf[mb][2] = pack_bf16(sB[mb][0], sB[mb][1]); pf[mb][3] = pack_bf16(sB[mb][2], sB[mb][3]);
      }
      // ---- a6: acc += P V
#pragma unroll
      for (int ndp = 0; ndp < NDP; ++ndp) {
        const uint4 vq = lds_u32x4(pkg + v_off + ndp * 512);
#pragma unroll
        for (int mb = 0; mb < 2; ++mb) {
          if (2 * ndp < ND) mma_bf16(o[mb][2 * ndp], pf[mb][0], pf[mb][1], pf[mb][2], pf[mb][3], vq.x, vq.y);
          if (2 * ndp + 1 < ND) mma_bf16(o[mb][2 * ndp + 1], pf[mb][0], pf[mb][1], pf[mb][2], pf[mb][3], vq.z, vq.w);
        }
      }
      // the warp that finishes the buffer last refills it with the tile kNC ahead (every warp's shared loads of the
      // buffer have returned before its increment; acq_rel orders them before the last finisher's copies)
      __syncwarp();
      if (lane == 0) {
        uint32_t old;
        asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(s_done + 4 * bbuf) : "memory");
        if ((old & (cAttnWarps - 1)) == cAttnWarps - 1) fetch(nx, bbuf);
      }
      it_next(nx);
      if (++bbuf == kNC) { bbuf = 0; bphase ^= 1; }
    };
    for (int j0 = un.ks & ~(cTileK - 1); j0 < un.ke; j0 += cTileK) {
      if ((j0 < un.ks) || (j0 + cTileK > un.ke)) tile(j0, std::true_type{});
      else tile(j0, std::false_type{});
    }

    // ---- a7: partial state of (rows, key segment) -> slot (m back in natural-log units).  acc is staged per 16-row block
    // in the warp's slab of the Q tile's buffer -- free once every warp has finished the unit's last QK^T -- and written
    // back as 128-bit row pieces, a row's C floats contiguous (fused_mma.cu).
    constexpr float kLn2 = 0.6931471805599453f;
    constexpr int kOPitch = c_o_pitch(C);
    const uint32_t slab = s_q + h * (16 * kOPitch * 4);
    __syncthreads();                                          // nobody reads this unit's Q tile any more
#pragma unroll
    for (int mb = 0; mb < 2; ++mb) {
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        const float l = quad_sum(l_run[mb][x]);
        const int row = un.q0 + mb * 16 + g + 8 * x;
        if (row < un.q_end && t == 0) {
          const int64_t srow = (int64_t)un.slot * p.state_rows + (row - p.state_row0);
          p.st_m[srow * cH + h] = m_run[mb][x] * kLn2;
          p.st_l[srow * cH + h] = l;
        }
#pragma unroll
        for (int nd = 0; nd < ND; ++nd)
          asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(slab + ((g + 8 * x) * kOPitch + nd * 8 + 2 * t) * 4),
                       "f"(o[mb][nd][2 * x]), "f"(o[mb][nd][2 * x + 1]) : "memory");
      }
      __syncwarp();
#pragma unroll
      for (int i = 0; i < 16 * (C / 4) / 32; ++i) {
        const int e = i * 32 + lane, r = e / (C / 4), c4 = e - r * (C / 4);
        const int row = un.q0 + mb * 16 + r;
        const float4 v = lds_f32x4(slab + (r * kOPitch + c4 * 4) * 4);
        if (row < un.q_end) {
          const int64_t srow = (int64_t)un.slot * p.state_rows + (row - p.state_row0);
          *reinterpret_cast<float4*>(p.st_acc + srow * (cH * C) + h * C + c4 * 4) = v;
        }
      }
      __syncwarp();
    }
  }
  };
  if (h & 1) run(std::integral_constant<int, 1>{}); else run(std::integral_constant<int, 0>{});
}

template <int C, int CP>
cudaError_t launch_c(const MmaParams& p, int64_t units, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(cached_attn_kernel<C, CP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c_smem_alloc(C, CP));
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (sms <= 0) sms = 148;
  const unsigned grid = (unsigned)(units < sms ? units : sms);
  return launch_kernel(cached_attn_kernel<C, CP>, dim3(grid), dim3(cThreads), c_smem_alloc(C, CP), st, p.pdl, p);
}

}  // namespace

// p as for launch_fused_mma with p.bias_cache set: whole-tensor rows (q_begin = 0, one row part), tile height 32
cudaError_t launch_cached_attn(const MmaParams& p, cudaStream_t st) {
  if (p.H != cH || !p.bias_cache || p.q_begin != 0 || p.n_qparts != 1 || p.tile_h != cTileQ) return cudaErrorInvalidValue;
  if (p.q_end <= p.q_begin || p.k_end <= p.k_begin) return cudaSuccess;
  const int64_t units = mma_num_units<0>(p.q_end - p.q_begin, p.n_qparts, p.n_kparts, p.nseg, p.tile_h);
  if (units > 0x7fffffff) return cudaErrorInvalidValue;
  switch (p.c) {
    case 24: return launch_c<24, 32>(p, units, st);
    case 32: return launch_c<32, 32>(p, units, st);
    case 48: return launch_c<48, 48>(p, units, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace dcp
