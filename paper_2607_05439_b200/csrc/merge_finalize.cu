// Merge of partial online-softmax states (step a8) and the normalise + gate half of step a9.
//   PAPER.md:90  "merges the partial output into a running total via an online softmax"
//   PAPER.md:446 Fold-CP's tiled_softmax_attention_update; PAPER.md:40 running softmax statistics.
// Left fold over the key-block slots 0..n-1 with  m' = max(m_a, m_b),
//   l' = l_a e^{m_a-m'} + l_b e^{m_b-m'},  acc' = acc_a e^{m_a-m'} + acc_b e^{m_b-m'}.
// The first slot initialises the state (no arithmetic on -inf).  No atomics, fixed order: run-to-run
// bitwise repeatable (the lesson of PAPER.md:362).  One thread per (row, channel).
#include "kernels.h"

namespace dcp {

namespace {

template <typename T>
__global__ void __launch_bounds__(256) merge_kernel(const MergeParams p) {
  pdl_trigger();
  pdl_wait();
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = p.rows * p.D;
  if (idx >= total) return;
  const int64_t row = idx / p.D;
  const int e = (int)(idx % p.D);
  const int h = e / p.c;
  float m = p.st_m[row * p.H + h];
  float l = p.st_l[row * p.H + h];
  float a = p.st_acc[row * p.D + e];
  for (int s = 1; s < p.n_slots; ++s) {
    const int64_t srow = (int64_t)s * p.rows + row;
    const float mb = p.st_m[srow * p.H + h];
    const float lb = p.st_l[srow * p.H + h];
    const float ab = p.st_acc[srow * p.D + e];
    const float mn = fmaxf(m, mb);
    const float fa = mn == -INFINITY ? 0.f : expf(m - mn), fb = mn == -INFINITY ? 0.f : expf(mb - mn);   // empty (+) empty
    l = l * fa + lb * fb;
    a = a * fa + ab * fb;
    m = mn;
  }
  if (p.g != nullptr) {
    const float o = a / l;
    const float g = to_f32(reinterpret_cast<const T*>(p.g)[row * p.D + e]);
    reinterpret_cast<T*>(p.gated)[row * p.D + e] = from_f32<T>(g * o);
  } else {
    p.acc_out[row * p.D + e] = a;
    if (e % p.c == 0) { p.m_out[row * p.H + h] = m; p.l_out[row * p.H + h] = l; }
  }
}

// Same fold, four consecutive channels of one head per thread (c % 4 == 0): 128-bit state loads, the rescale
// factors e^{m_a-m'}, e^{m_b-m'} computed once per thread instead of once per channel.  Element arithmetic and
// order are identical to merge_kernel, so both produce the same bits.
// NS > 0: the slot count is a compile-time constant, so all slots' loads are issued before the fold (the fold itself,
// its order and every operation are the same as in the runtime-count version: same bits).
template <typename T, int NS>
__global__ void __launch_bounds__(256) merge_vec4_kernel(const MergeParams p) {
  pdl_trigger();
  pdl_wait();
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int dq = p.D >> 2;
  if (idx >= p.rows * dq) return;
  const int64_t row = idx / dq;
  const int e = (int)(idx - row * dq) << 2;
  const int h = e / p.c;
  float m, l;
  float4 a;
  if constexpr (NS > 0) {
    float ms[NS], ls[NS];
    float4 as[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const int64_t srow = (int64_t)s * p.rows + row;
      ms[s] = p.st_m[srow * p.H + h];
      ls[s] = p.st_l[srow * p.H + h];
      as[s] = *reinterpret_cast<const float4*>(p.st_acc + srow * p.D + e);
    }
    m = ms[0]; l = ls[0]; a = as[0];
#pragma unroll
    for (int s = 1; s < NS; ++s) {
      const float mn = fmaxf(m, ms[s]);
      const float fa = mn == -INFINITY ? 0.f : expf(m - mn), fb = mn == -INFINITY ? 0.f : expf(ms[s] - mn);
      l = l * fa + ls[s] * fb;
      a.x = a.x * fa + as[s].x * fb; a.y = a.y * fa + as[s].y * fb;
      a.z = a.z * fa + as[s].z * fb; a.w = a.w * fa + as[s].w * fb;
      m = mn;
    }
  } else {
    m = p.st_m[row * p.H + h];
    l = p.st_l[row * p.H + h];
    a = *reinterpret_cast<const float4*>(p.st_acc + row * p.D + e);
    for (int s = 1; s < p.n_slots; ++s) {
      const int64_t srow = (int64_t)s * p.rows + row;
      const float mb = p.st_m[srow * p.H + h];
      const float lb = p.st_l[srow * p.H + h];
      const float4 ab = *reinterpret_cast<const float4*>(p.st_acc + srow * p.D + e);
      const float mn = fmaxf(m, mb);
      const float fa = mn == -INFINITY ? 0.f : expf(m - mn), fb = mn == -INFINITY ? 0.f : expf(mb - mn);
      l = l * fa + lb * fb;
      a.x = a.x * fa + ab.x * fb; a.y = a.y * fa + ab.y * fb;
      a.z = a.z * fa + ab.z * fb; a.w = a.w * fa + ab.w * fb;
      m = mn;
    }
  }
  if (p.g != nullptr) {
    const T* gp = reinterpret_cast<const T*>(p.g) + row * p.D + e;
    T* out = reinterpret_cast<T*>(p.gated) + row * p.D + e;
    if constexpr (sizeof(T) == 2) {
      // bf16: the four gates and the four results as one 8-byte access each (e % 4 == 0, rows are 8-byte aligned)
      const uint2 gw = *reinterpret_cast<const uint2*>(gp);
      const float g0 = __uint_as_float(gw.x << 16), g1 = __uint_as_float(gw.x & 0xffff0000u);
      const float g2 = __uint_as_float(gw.y << 16), g3 = __uint_as_float(gw.y & 0xffff0000u);
      const __nv_bfloat162 o01 = __floats2bfloat162_rn(g0 * (a.x / l), g1 * (a.y / l));
      const __nv_bfloat162 o23 = __floats2bfloat162_rn(g2 * (a.z / l), g3 * (a.w / l));
      *reinterpret_cast<uint2*>(out) = make_uint2(*reinterpret_cast<const uint32_t*>(&o01), *reinterpret_cast<const uint32_t*>(&o23));
    } else {
      out[0] = from_f32<T>(to_f32(gp[0]) * (a.x / l));
      out[1] = from_f32<T>(to_f32(gp[1]) * (a.y / l));
      out[2] = from_f32<T>(to_f32(gp[2]) * (a.z / l));
      out[3] = from_f32<T>(to_f32(gp[3]) * (a.w / l));
    }
  } else {
    *reinterpret_cast<float4*>(p.acc_out + row * p.D + e) = a;
    if (e % p.c == 0) { p.m_out[row * p.H + h] = m; p.l_out[row * p.H + h] = l; }
  }
}

template <typename T, int NS>
cudaError_t launch_vec4_n(const MergeParams& p, unsigned blocks, cudaStream_t st) {
  return launch_kernel(merge_vec4_kernel<T, NS>, dim3(blocks), dim3(256), 0, st, p.pdl, p);
}
template <typename T>
cudaError_t launch_vec4(const MergeParams& p, unsigned blocks, cudaStream_t st) {
  switch (p.n_slots) {
    case 1: return launch_vec4_n<T, 1>(p, blocks, st);
    case 2: return launch_vec4_n<T, 2>(p, blocks, st);
    case 3: return launch_vec4_n<T, 3>(p, blocks, st);
    case 4: return launch_vec4_n<T, 4>(p, blocks, st);
    case 5: return launch_vec4_n<T, 5>(p, blocks, st);
    case 6: return launch_vec4_n<T, 6>(p, blocks, st);
    case 7: return launch_vec4_n<T, 7>(p, blocks, st);
    case 8: return launch_vec4_n<T, 8>(p, blocks, st);
    case 9: return launch_vec4_n<T, 9>(p, blocks, st);
    case 12: return launch_vec4_n<T, 12>(p, blocks, st);
    case 16: return launch_vec4_n<T, 16>(p, blocks, st);
    default: return launch_vec4_n<T, 0>(p, blocks, st);
  }
}

}  // namespace

cudaError_t launch_merge(dcp_dtype dt, const MergeParams& p, cudaStream_t st) {
  const int64_t total = p.rows * p.D;
  if (total <= 0) return cudaSuccess;
  if (p.c % 4 == 0 && ((uintptr_t)p.st_acc & 15) == 0 &&
      (p.g != nullptr ? (((uintptr_t)p.g | (uintptr_t)p.gated) & 7) == 0 : ((uintptr_t)p.acc_out & 15) == 0)) {
    const unsigned vblocks = (unsigned)((total / 4 + 255) / 256);
    return dt == DCP_F32 ? launch_vec4<float>(p, vblocks, st) : launch_vec4<__nv_bfloat16>(p, vblocks, st);
  }
  unsigned blocks = (unsigned)((total + 255) / 256);
  return dt == DCP_F32 ? launch_kernel(merge_kernel<float>, dim3(blocks), dim3(256), 0, st, p.pdl, p)
                       : launch_kernel(merge_kernel<__nv_bfloat16>, dim3(blocks), dim3(256), 0, st, p.pdl, p);
}

}  // namespace dcp
