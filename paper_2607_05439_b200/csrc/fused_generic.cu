// Generic fp32 CUDA-core fused kernel: steps a2-a7 of SURVEY.md section 8(a) for any shape.
//   per pair (i, j):  LayerNorm(z_ij) -> bias_h = zhat . W_b[:,h]           ("learned projection of Z")
//   logit_h = q_i^h . k_j^h / sqrt(c) + bias_h                              (PAPER.md:83 Eq. 2; i = row of z, :81)
//   online softmax over keys with running (m, l, acc)
// The I*I*H logits live only in registers / shared memory.  One warp owns one query row, its 32 lanes
// own 32 consecutive keys of the current key tile; a row's arithmetic never depends on its neighbours,
// and key tiles start at the chunk's first key, so row(P) == monolithic bitwise and
// grid(G x G) == monolithic(key_split = G) bitwise.
// This is the fp32 path of config 0 (max-abs <= 1e-5) and the fallback / cross-check for the MMA kernel.
#include "kernels.h"

namespace dcp {

namespace {

constexpr int kWarps = 8;          // query rows per CTA
constexpr int kKeys = 32;          // keys per tile (one per lane)

template <typename T> struct Vec16;   // 16-byte global loads of z
template <> struct Vec16<float> { static constexpr int N = 4; };
template <> struct Vec16<__nv_bfloat16> { static constexpr int N = 8; };

template <typename T>
__device__ __forceinline__ void load16(const T* p, float* out);
template <>
__device__ __forceinline__ void load16<float>(const float* p, float* out) {
  float4 v = __ldg(reinterpret_cast<const float4*>(p));
  out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
}
template <>
__device__ __forceinline__ void load16<__nv_bfloat16>(const __nv_bfloat16* p, float* out) {
  uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
  uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    out[2 * t] = __uint_as_float(w[t] << 16);
    out[2 * t + 1] = __uint_as_float(w[t] & 0xffff0000u);
  }
}

// NR = D / 32: accumulator elements per lane (element e = lane + 32 r of the row's [D] accumulator)
template <typename T, int NR>
__global__ void __launch_bounds__(kWarps * 32) fused_generic_kernel(const FusedParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int D = p.D, H = p.H, c = p.c, c_z = p.c_z;
  const int ldk = D + (sizeof(T) == 2 ? 2 : 1);       // padded K row: conflict-free lane-per-key reads
  T* Ks = reinterpret_cast<T*>(smem_raw);             // [32][ldk]
  T* Vs = Ks + kKeys * ldk;                           // [32][D]
  float* fbase = reinterpret_cast<float*>(smem_raw + (((size_t)(kKeys * ldk + kKeys * D) * sizeof(T) + 15) / 16) * 16);
  float* qs = fbase;                                  // [kWarps][D]
  float* wgs = qs + kWarps * D;                       // [c_z][H]
  float* c0s = wgs + c_z * H;                         // [kMaxHeads]
  float* Ps = c0s + kMaxHeads;                        // [kWarps][H][32]
  float* als = Ps + kWarps * H * kKeys;               // [kWarps][kMaxHeads]

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const T* zg = reinterpret_cast<const T*>(p.z);
  const T* qg = reinterpret_cast<const T*>(p.q);
  const T* kg = reinterpret_cast<const T*>(p.k);
  const T* vg = reinterpret_cast<const T*>(p.v);

  // key chunk of this CTA (Eq. 5 over [k0, k1))
  int64_t cs, cl;
  shard_range(p.k1 - p.k0, p.n_chunks, blockIdx.y, &cs, &cl);
  const int64_t ks = p.k0 + cs, ke = ks + cl;
  const int64_t i = p.q0 + (int64_t)blockIdx.x * kWarps + warp;
  const bool row_ok = i < p.q1;

  for (int e = threadIdx.x; e < c_z * H; e += blockDim.x) wgs[e] = p.wg[e];
  if (threadIdx.x < kMaxHeads) c0s[threadIdx.x] = threadIdx.x < H ? p.c0[threadIdx.x] : 0.f;
  if (row_ok)
    for (int e = lane; e < D; e += 32) qs[warp * D + e] = to_f32(qg[i * D + e]);

  float m_run[kMaxHeads], l_run[kMaxHeads];
#pragma unroll
  for (int h = 0; h < kMaxHeads; ++h) { m_run[h] = -INFINITY; l_run[h] = 0.f; }
  float acc[NR];
  int hr[NR];
#pragma unroll
  for (int r = 0; r < NR; ++r) { acc[r] = 0.f; hr[r] = (lane + 32 * r) / c; }

  for (int64_t j0 = ks; j0 < ke; j0 += kKeys) {
    const int nk = (int)((ke - j0) < kKeys ? (ke - j0) : kKeys);
    __syncthreads();   // previous tile's K/V fully consumed (also orders the prologue stores above)
    for (int e = threadIdx.x; e < kKeys * D; e += blockDim.x) {
      int r = e / D, cc = e % D;
      bool ok = r < nk;
      Ks[r * ldk + cc] = ok ? kg[(j0 + r) * D + cc] : from_f32<T>(0.f);
      Vs[r * D + cc] = ok ? vg[(j0 + r) * D + cc] : from_f32<T>(0.f);
    }
    __syncthreads();
    if (!row_ok) continue;     // warp-uniform

    const bool valid = lane < nk;
    float b[kMaxHeads];
#pragma unroll
    for (int h = 0; h < kMaxHeads; ++h) b[h] = 0.f;
    if (valid) {
      // ---- a2: LayerNorm statistics of z[i, j, :] (two-pass, fp32), a3: bias projection
      const T* zp = zg + i * p.ldz + (j0 + lane) * (int64_t)c_z;
      constexpr int VN = Vec16<T>::N;
      float sum = 0.f;
      for (int k = 0; k < c_z; k += VN) {
        float x[VN];
        load16<T>(zp + k, x);
#pragma unroll
        for (int t = 0; t < VN; ++t) sum += x[t];
      }
      const float mu = sum / (float)c_z;
      float var = 0.f;
      for (int k = 0; k < c_z; k += VN) {
        float x[VN];
        load16<T>(zp + k, x);
#pragma unroll
        for (int t = 0; t < VN; ++t) { float d = x[t] - mu; var = fmaf(d, d, var); }
      }
      const float rstd = rsqrtf(var / (float)c_z + p.eps);
      for (int k = 0; k < c_z; k += VN) {
        float x[VN];
        load16<T>(zp + k, x);
#pragma unroll
        for (int t = 0; t < VN; ++t) {
          const float d = x[t] - mu;
          const float* wrow = wgs + (k + t) * H;
#pragma unroll
          for (int h = 0; h < kMaxHeads; ++h)
            if (h < H) b[h] = fmaf(d, wrow[h], b[h]);
        }
      }
#pragma unroll
      for (int h = 0; h < kMaxHeads; ++h) b[h] = fmaf(b[h], rstd, c0s[h]);
    }

    // ---- a4: logits, a5: online softmax (per head, reductions across the 32 keys of the tile)
    const float* qrow = qs + warp * D;
    const T* krow = Ks + lane * ldk;
#pragma unroll
    for (int h = 0; h < kMaxHeads; ++h) {
      if (h < H) {
        float dot = 0.f;
        for (int d = 0; d < c; ++d) dot = fmaf(qrow[h * c + d], to_f32(krow[h * c + d]), dot);
        const float lg = valid ? fmaf(dot, p.scale, b[h]) : -INFINITY;
        const float m_new = fmaxf(m_run[h], warp_max(lg));
        const float pe = valid ? expf(lg - m_new) : 0.f;
        const float alpha = expf(m_run[h] - m_new);        // first tile: exp(-inf) = 0
        l_run[h] = fmaf(l_run[h], alpha, warp_sum(pe));
        m_run[h] = m_new;
        Ps[(warp * H + h) * kKeys + lane] = pe;
        if (lane == 0) als[warp * kMaxHeads + h] = alpha;
      }
    }
    __syncwarp();
    // ---- a6: acc = acc * alpha + P V   (lane owns channels e = lane + 32 r)
#pragma unroll
    for (int r = 0; r < NR; ++r) acc[r] *= als[warp * kMaxHeads + hr[r]];
    for (int jj = 0; jj < nk; ++jj) {
#pragma unroll
      for (int r = 0; r < NR; ++r)
        acc[r] = fmaf(Ps[(warp * H + hr[r]) * kKeys + jj], to_f32(Vs[jj * D + lane + 32 * r]), acc[r]);
    }
    __syncwarp();
  }

  if (!row_ok) return;
  // ---- a7: partial state of (row i, key chunk blockIdx.y) -> slot
  const int64_t slot = p.slot0 + blockIdx.y;
  const int64_t srow = slot * p.state_rows + (i - p.state_row0);
#pragma unroll
  for (int h = 0; h < kMaxHeads; ++h)
    if (h < H && lane == 0) { p.st_m[srow * H + h] = m_run[h]; p.st_l[srow * H + h] = l_run[h]; }
#pragma unroll
  for (int r = 0; r < NR; ++r) p.st_acc[srow * D + lane + 32 * r] = acc[r];
}

size_t generic_smem_bytes(int elt, int D, int c_z, int H) {
  int ldk = D + (elt == 2 ? 2 : 1);
  size_t b = (((size_t)(kKeys * ldk + kKeys * D) * elt + 15) / 16) * 16;
  b += sizeof(float) * ((size_t)kWarps * D + (size_t)c_z * H + kMaxHeads + (size_t)kWarps * H * kKeys +
                        kWarps * kMaxHeads);
  return b;
}

template <typename T, int NR>
cudaError_t launch_nr(const FusedParams& p, cudaStream_t st) {
  size_t smem = generic_smem_bytes(sizeof(T), p.D, p.c_z, p.H);
  cudaError_t e = cudaFuncSetAttribute(fused_generic_kernel<T, NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int64_t nq = p.q1 - p.q0;
  dim3 grid((unsigned)((nq + kWarps - 1) / kWarps), p.n_chunks);
  fused_generic_kernel<T, NR><<<grid, kWarps * 32, smem, st>>>(p);
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_t(const FusedParams& p, cudaStream_t st) {
  switch (p.D / 32) {
    case 1: return launch_nr<T, 1>(p, st);
    case 2: return launch_nr<T, 2>(p, st);
    case 3: return launch_nr<T, 3>(p, st);
    case 4: return launch_nr<T, 4>(p, st);
    case 6: return launch_nr<T, 6>(p, st);
    case 8: return launch_nr<T, 8>(p, st);
    case 12: return launch_nr<T, 12>(p, st);
    case 16: return launch_nr<T, 16>(p, st);
    case 24: return launch_nr<T, 24>(p, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

bool fused_generic_supports(dcp_dtype dt, int H, int c, int c_z) {
  int D = H * c;
  if (H < 1 || H > kMaxHeads || c < 1 || D % 32 != 0 || D > kMaxD) return false;
  int nr = D / 32;
  if (!(nr == 1 || nr == 2 || nr == 3 || nr == 4 || nr == 6 || nr == 8 || nr == 12 || nr == 16 || nr == 24)) return false;
  int elt = dt == DCP_F32 ? 4 : 2;
  if ((c_z * elt) % 16 != 0) return false;
  return generic_smem_bytes(elt, D, c_z, H) <= 227 * 1024;
}

cudaError_t launch_fused_generic(dcp_dtype dt, const FusedParams& p, cudaStream_t st) {
  if (p.q1 <= p.q0 || p.k1 <= p.k0) return cudaSuccess;
  if (dt == DCP_F32) return launch_t<float>(p, st);
  return launch_t<__nv_bfloat16>(p, st);
}

}  // namespace dcp
