// libdesigncp internal: inline-PTX helpers shared by the sm_100a fused kernels (mbarrier, TMA, tcgen05 / TMEM,
// mma.sync, shared-memory vector accesses).  Everything has internal linkage (anonymous namespace inside dcp).
#pragma once
#include <cuda.h>
#include <cudaTypedefs.h>

#include <type_traits>

#include "kernels.h"

namespace dcp {
namespace {

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  uint32_t spins = 0;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    // watchdog: a pipeline bug must surface as a CUDA error, never as a hung GPU (each failed try_wait already
    // sleeps for the hardware time limit, so 2^24 failures is seconds)
    if (!done && ++spins == (1u << 24)) __trap();
  } while (!done);
}
// ---- tcgen05 / TMEM (5th-generation tensor cores): single-thread MMA issue, accumulators in tensor memory
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// K-major operand tile, 128-byte swizzle: rows of 64 bf16 (128 B), 8-row groups 1024 B apart (SBO), descriptor
// version 1 (sm_100), layout type 2 = SWIZZLE_128B.  `addr` may be advanced by 32 B per K = 16 step inside the atom.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t addr) {
  return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
// instruction descriptor, kind::f16: D = f32, A = B = bf16, both K-major, M x N
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld_x16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float tmem_ld_x1(uint32_t taddr) {
  uint32_t r;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r) : "r"(taddr));
  return __uint_as_float(r);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// plain bulk copy global -> shared (16-byte aligned, size a multiple of 16), bytes counted on an mbarrier
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tmap, int c0, int c1, int c2, uint32_t bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void mma_bf16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                         uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void sts_f32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ float4 lds_f32x4(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint4 lds_u32x4(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint2 lds_u32x2(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
  uint16_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts_u32x4(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// acc_lo += lo(w)^2, acc_hi += hi(w)^2 for a bf16x2 word: mixed-precision FMA (bf16 x bf16 + f32, PTX ISA 8.6, sm_100:
// SASS FHFMA.BF16 with .H0/.H1 operand selectors), exact products, fp32 accumulation, no unpacking instructions
__device__ __forceinline__ void fma_sq_bf16x2(float& acc_lo, float& acc_hi, uint32_t w) {
  asm("{\n\t.reg .b16 l, h;\n\t"
      "mov.b32 {l, h}, %2;\n\t"
      "fma.rn.f32.bf16 %0, l, l, %0;\n\t"
      "fma.rn.f32.bf16 %1, h, h, %1;\n\t}"
      : "+f"(acc_lo), "+f"(acc_hi) : "r"(w));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// (lo, hi) -> packed fp16x2; and one half of such a word back to fp32
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ float f16_half(uint32_t w, int hi) {
  float f;
  if (hi) asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %1;\n\tcvt.f32.f16 %0, h;\n\t}" : "=f"(f) : "r"(w));
  else asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %1;\n\tcvt.f32.f16 %0, l;\n\t}" : "=f"(f) : "r"(w));
  return f;
}
// x rounded to the nearest bf16, as a float
__device__ __forceinline__ float bf16_round(float x) { return __bfloat162float(__float2bfloat16_rn(x)); }
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint2 ldg_u2(const void* p) { return __ldg(reinterpret_cast<const uint2*>(p)); }
__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v + __shfl_xor_sync(0xffffffffu, v, 2);
}

template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
inline PFN_cuTensorMapEncodeTiled get_encode_fn() {
  static PFN_cuTensorMapEncodeTiled fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(ptr);
  }
  return fn;
}

// ------------------------------------------------------------------ work units
struct Unit {
  int q0;      // first query row of the TQ-row tile
  int q_end;   // end of the tile's own rows (rows >= q_end are not stored)
  int ks, ke;  // key segment
  int slot;    // partial-state slot
};

// Eq. 5 in 32-bit (I <= 2^30)
__device__ __forceinline__ void shard32(int n, int parts, int p, int* start, int* len) {
  const int base = n / parts, rem = n % parts;
  *len = base + (p < rem ? 1 : 0);
  *start = p * base + (p < rem ? p : rem);
}

// kTileQ > 0: compile-time tile height; kTileQ == 0: run-time height `tq_rt` (fused_mma_kernel: MmaParams.tile_h)
template <int kTileQ>
__host__ __device__ inline int64_t mma_num_units(int n, int n_qparts, int n_kparts, int nseg, int tq_rt = 0) {
  const int tq = kTileQ > 0 ? kTileQ : tq_rt;
  // query parts have sizes floor(n/P) or floor(n/P)+1 (Eq. 5): count their TQ-row tiles in closed form
  const int base = n / n_qparts, rem = n % n_qparts;
  const int t_big = (base + 1 + tq - 1) / tq, t_small = (base + tq - 1) / tq;
  return ((int64_t)rem * t_big + (int64_t)(n_qparts - rem) * t_small) * n_kparts * nseg;
}

// Key chunk cb (Eq. 5 over the keys: the decomposition contract's chunks) is cut into nseg segments along the kTileK-key
// tiles that overlap it (Eq. 5 over those tiles), so that only chunk boundaries -- never segment boundaries -- fall
// inside a tile: a boundary tile would be streamed and projected twice.  A pure function of (I, chunks, segments).
template <int kTileQ, int kTileK>
__device__ __forceinline__ Unit decode_unit(const MmaParams& p, int u) {
  const int tq = kTileQ > 0 ? kTileQ : p.tile_h;
  const int n = p.q_end - p.q_begin;
  const int base = n / p.n_qparts, rem = n % p.n_qparts;
  const int t_big = (base + 1 + tq - 1) / tq, t_small = (base + tq - 1) / tq;
  const int per_tile = p.n_kparts * p.nseg;
  int tile = u / per_tile;
  const int r = u - tile * per_tile;
  int part, tile_i;
  if (tile < rem * t_big) { part = tile / t_big; tile_i = tile - part * t_big; }
  else { tile -= rem * t_big; part = tile / t_small; tile_i = tile - part * t_small; part += rem; }
  int ps, pl;
  shard32(n, p.n_qparts, part, &ps, &pl);
  Unit un;
  un.q0 = p.q_begin + ps + tile_i * tq;
  un.q_end = p.q_begin + ps + pl;                             // end of the part ...
  if (un.q_end > un.q0 + tq) un.q_end = un.q0 + tq;           // ... or of the tile (tile heights below the kernel's 32 / 64 rows)
  const int cb = r / p.nseg, sg = r - cb * p.nseg;
  int cs, cl, ts, tl;
  shard32(p.k_end - p.k_begin, p.n_kparts, cb, &cs, &cl);
  cs += p.k_begin;
  const int t0 = cs / kTileK, t1 = (cs + cl + kTileK - 1) / kTileK;     // tiles [t0, t1) overlap the chunk
  shard32(t1 - t0, p.nseg, sg, &ts, &tl);
  const int a = (t0 + ts) * kTileK, b = (t0 + ts + tl) * kTileK;
  un.ks = a > cs ? a : cs;
  un.ke = b < cs + cl ? b : cs + cl;
  un.slot = p.slot0 + r;
  return un;
}



}  // namespace
}  // namespace dcp
