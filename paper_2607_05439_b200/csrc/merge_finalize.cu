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
    const float fa = expf(m - mn), fb = expf(mb - mn);
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

}  // namespace

cudaError_t launch_merge(dcp_dtype dt, const MergeParams& p, cudaStream_t st) {
  const int64_t total = p.rows * p.D;
  if (total <= 0) return cudaSuccess;
  unsigned blocks = (unsigned)((total + 255) / 256);
  if (dt == DCP_F32) merge_kernel<float><<<blocks, 256, 0, st>>>(p);
  else merge_kernel<__nv_bfloat16><<<blocks, 256, 0, st>>>(p);
  return cudaGetLastError();
}

}  // namespace dcp
