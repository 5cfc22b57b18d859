// Sparse (k-neighbour) atom-level attention with pair bias, bf16.
//   PAPER.md:58  "each query atom attends to a budget of k neighbours ... The relevant slice of P is gathered at
//                those k indices and then projected to the per-head bias, so the attention computation itself is O(L k)"
//   PAPER.md:303 the block consumes a [L, k, c_atompair] slice;  PAPER.md:456 K/V/B entries are gathered at the indices
// Per query atom l and head h:  logit_j = q_l^h . k_{idx[l,j]}^h / sqrt(c) + LN(p_slice[l,j,:]) . W_b[:,h],
// softmax over the valid slots j (idx >= 0), o = sum_j a_j v_{idx[l,j]}^h, gated by sigmoid(a_l W_g).
//
// Every query has its own key set, so there is no key tile to share between queries: the work is a gather of
// k x 2 x 64-byte head slices of the (L2-resident) K / V rows per (atom, head) plus ~100 FMAs per gathered row,
// not a contraction the tensor pipe could batch.  One warp per (atom, head), the four heads of an atom in one CTA
// (they read adjacent 64-byte slices of the same 256-byte rows: L1 hits); lane = slot (32 slots per pass):
//   * the lane reads its neighbour's 64-byte K slice (4 x 128-bit) and dots it with q (mixed-precision
//     fma.rn.f32.bf16: bf16 products are exact, fp32 accumulation, no unpacking),
//   * LayerNorm statistics and the bias projection of its 32-byte p row the same way (the rows of a warp are 1 KB
//     contiguous), folded as in the dense kernels: bias = rstd (p.W' - mu c1) + c0,
//   * softmax over the warp (shuffle max / sum, exp2 domain), P rounded to bf16 like the dense kernels,
//   * acc[32] += P v over the lane's slots, then a 31-shuffle reduce-scatter leaves head dim d on lane d.
#include "kernels.h"
#include "mma_ptx.cuh"

namespace dcp {

namespace {

constexpr int sC = 32;          // head dim
constexpr int sCz = 16;         // c_atompair
constexpr int sMaxPass = 16;    // k <= 512

// acc += lo(a) lo(b) + hi(a) hi(b)  (bf16x2 words; SASS FHFMA.BF16 with .H0/.H1 selectors)
__device__ __forceinline__ void dot_bf16x2(float& acc, uint32_t a, uint32_t b) {
  asm("{\n\t.reg .b16 al, ah, bl, bh;\n\t"
      "mov.b32 {al, ah}, %1;\n\t"
      "mov.b32 {bl, bh}, %2;\n\t"
      "fma.rn.f32.bf16 %0, al, bl, %0;\n\t"
      "fma.rn.f32.bf16 %0, ah, bh, %0;\n\t}"
      : "+f"(acc) : "r"(a), "r"(b));
}
// (acc_lo, acc_hi) += s * (lo(v), hi(v))  with s a bf16 scalar in the low half of `s16`
__device__ __forceinline__ void axpy_bf16x2(float& acc_lo, float& acc_hi, uint32_t v, uint32_t s16) {
  asm("{\n\t.reg .b16 vl, vh, sl, sh;\n\t"
      "mov.b32 {vl, vh}, %2;\n\t"
      "mov.b32 {sl, sh}, %3;\n\t"
      "fma.rn.f32.bf16 %0, vl, sl, %0;\n\t"
      "fma.rn.f32.bf16 %1, vh, sl, %1;\n\t}"
      : "+f"(acc_lo), "+f"(acc_hi) : "r"(v), "r"(s16));
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

struct SparseParams {
  const __nv_bfloat16* q;      // [L][H*32], scaled by log2(e)/sqrt(c)
  const __nv_bfloat16* k;      // [L][H*32]
  const __nv_bfloat16* v;      // [L][H*32]
  const __nv_bfloat16* g;      // [L][H*32] sigmoid gate
  const __nv_bfloat16* p;      // [L][k][16]
  const int32_t* idx;          // [L][k]
  const __nv_bfloat16* wfold;  // [16][16]: row h = (gamma (.) W_b[:,h] log2 e), bf16
  const float* c1;             // [16]
  const float* c0;             // [16]
  __nv_bfloat16* gated;        // [L][H*32]
  int64_t L;
  int kn, H;
  float eps;
};

__global__ void __launch_bounds__(128) sparse_atom_kernel(const SparseParams p) {
  const int lane = threadIdx.x & 31;
  const int64_t wg = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  const int64_t l = wg / p.H;
  const int h = (int)(wg - l * p.H);
  if (l >= p.L) return;
  const int D = p.H * sC;
  // q_l^h (every lane holds all 32 dims) and the folded projection row of head h
  uint4 qv[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) qv[i] = __ldg(reinterpret_cast<const uint4*>(p.q + l * D + h * sC) + i);
  const uint4 wf0 = __ldg(reinterpret_cast<const uint4*>(p.wfold + h * sCz));
  const uint4 wf1 = __ldg(reinterpret_cast<const uint4*>(p.wfold + h * sCz) + 1);
  const float c1 = __ldg(p.c1 + h), c0 = __ldg(p.c0 + h);
  const int npass = (p.kn + 31) >> 5;
  const uint32_t ones = 0x3f803f80u;

  // ---- logits of the lane's slots (slot j = 32 pass + lane)
  float s[sMaxPass];
  int nb[sMaxPass];
  float mx = -INFINITY;
#pragma unroll
  for (int ps = 0; ps < sMaxPass; ++ps) {
    s[ps] = -INFINITY;
    nb[ps] = -1;
    if (ps < npass) {
      const int j = ps * 32 + lane;
      int m = j < p.kn ? __ldg(p.idx + l * p.kn + j) : -1;
      if ((unsigned)m >= (unsigned)p.L) m = -1;          // negative or >= L: unused slot
      nb[ps] = m;
      if (m >= 0) {
        const uint4* kr = reinterpret_cast<const uint4*>(p.k + (int64_t)m * D + h * sC);
        float d0 = 0.f, d1 = 0.f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const uint4 kv = __ldg(kr + i);
          dot_bf16x2(d0, kv.x, qv[i].x); dot_bf16x2(d1, kv.y, qv[i].y);
          dot_bf16x2(d0, kv.z, qv[i].z); dot_bf16x2(d1, kv.w, qv[i].w);
        }
        const uint4* pr = reinterpret_cast<const uint4*>(p.p + (l * p.kn + j) * sCz);
        const uint4 p0 = __ldg(pr), p1 = __ldg(pr + 1);
        float sm = 0.f, sq = 0.f, pw = 0.f;
        const uint32_t pw_[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
        const uint32_t wf_[8] = {wf0.x, wf0.y, wf0.z, wf0.w, wf1.x, wf1.y, wf1.z, wf1.w};
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          dot_bf16x2(sm, pw_[i], ones);
          dot_bf16x2(sq, pw_[i], pw_[i]);
          dot_bf16x2(pw, pw_[i], wf_[i]);
        }
        const float mu = sm * (1.f / sCz);
        const float var = fmaf(-mu, mu, sq * (1.f / sCz));      // one rounding (c_z is a power of two); 0 for a constant row
        const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;
        s[ps] = (d0 + d1) + fmaf(rstd, fmaf(-mu, c1, pw), c0);
        mx = fmaxf(mx, s[ps]);
      }
    }
  }
  mx = warp_max(mx);
  __nv_bfloat16* out = p.gated + l * D + h * sC;
  if (mx == -INFINITY) {            // no valid neighbour: o = 0 (oracle reading)
    out[lane] = __float2bfloat16_rn(0.f);
    return;
  }
  // ---- softmax numerators, PV over the lane's slots
  float acc[sC];
#pragma unroll
  for (int d = 0; d < sC; ++d) acc[d] = 0.f;
  float lsum = 0.f;
#pragma unroll
  for (int ps = 0; ps < sMaxPass; ++ps) {
    if (ps < npass && nb[ps] >= 0) {
      const float pe = fast_exp2(s[ps] - mx);
      lsum += pe;
      const uint32_t pb = pack_bf16(pe, 0.f);          // P rounded to bf16 for PV, like the dense kernels
      const uint4* vr = reinterpret_cast<const uint4*>(p.v + (int64_t)nb[ps] * D + h * sC);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint4 vv = __ldg(vr + i);
        axpy_bf16x2(acc[8 * i + 0], acc[8 * i + 1], vv.x, pb); axpy_bf16x2(acc[8 * i + 2], acc[8 * i + 3], vv.y, pb);
        axpy_bf16x2(acc[8 * i + 4], acc[8 * i + 5], vv.z, pb); axpy_bf16x2(acc[8 * i + 6], acc[8 * i + 7], vv.w, pb);
      }
    }
  }
  lsum = warp_sum(lsum);
  // ---- reduce-scatter over the warp: after the step with offset `off` a lane keeps the half of its values whose
  // index bit equals its own lane bit; after five steps lane d holds the warp total of head dim d
#pragma unroll
  for (int off = 16, n = sC; off >= 1; off >>= 1, n >>= 1) {
    const bool upper = (lane & off) != 0;
#pragma unroll
    for (int i = 0; i < n / 2; ++i) {
      const float send = upper ? acc[i] : acc[i + n / 2];
      const float keep = upper ? acc[i + n / 2] : acc[i];
      acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
    }
  }
  const float gate = __bfloat162float(p.g[l * D + h * sC + lane]);
  out[lane] = __float2bfloat16_rn(gate * (acc[0] / lsum));
}

// ---- row-coalesced variant for H in {2, 4, 8}: one warp per atom, ALL heads.  A K / V row of the atom's neighbour is
// H * 64 bytes; LPR = 4 H lanes read it as 16-byte chunks (lane chunk ch -> head ch / 4, head dims 8 (ch % 4) .. + 7), so
// one warp-level load covers 32 / LPR whole rows = a few fully used 128-byte lines.  The slot-per-lane kernel above
// touches 32 different lines per load instruction and is bound by L1 tag throughput (one wavefront per line); this one
// needs ~8x fewer wavefronts.  Per warp: (A) lane = slot: bias of all heads from the p row -> shared logits[slot][h];
// (B) QK^T row by row, 4-lane shuffle reduction per head, added to the logits; (C) softmax statistics over the slots;
// (D) acc += P v row by row, the partial sums of the 32 / LPR row groups combined by shuffles at the end.
template <int H>
__global__ void __launch_bounds__(128) sparse_atom_rows_kernel(const SparseParams p) {
  constexpr int LPR = 4 * H;            // lanes per K / V row
  constexpr int RPL = 32 / LPR;         // rows per warp-level load
  constexpr int D = H * sC;
  extern __shared__ float smem_f[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int kpad = (p.kn + 31) & ~31;
  float* s_logit = smem_f + (size_t)wib * kpad * (H + 1);          // [kpad][H]
  int* s_idx = reinterpret_cast<int*>(s_logit + (size_t)kpad * H);  // [kpad]
  const int64_t l = (int64_t)blockIdx.x * 4 + wib;
  if (l >= p.L) return;
  const int ch = lane % LPR, grp = lane / LPR, hd = ch >> 2;        // chunk of the row, row group, head of the chunk
  const uint4 qv = __ldg(reinterpret_cast<const uint4*>(p.q + l * D) + ch);
  const uint32_t ones = 0x3f803f80u;

  // ---- (A) lane = slot: neighbour index, LayerNorm statistics of the p row, bias of every head
  for (int j0 = 0; j0 < kpad; j0 += 32) {
    const int j = j0 + lane;
    int m = j < p.kn ? __ldg(p.idx + l * p.kn + j) : -1;
    if ((unsigned)m >= (unsigned)p.L) m = -1;            // negative or >= L: unused slot
    s_idx[j] = m;
    if (m >= 0) {
      const uint4* pr = reinterpret_cast<const uint4*>(p.p + (l * p.kn + j) * sCz);
      const uint4 p0 = __ldg(pr), p1 = __ldg(pr + 1);
      const uint32_t pw_[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
      float sm = 0.f, sq = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) { dot_bf16x2(sm, pw_[i], ones); dot_bf16x2(sq, pw_[i], pw_[i]); }
      const float mu = sm * (1.f / sCz);
      const float var = fmaf(-mu, mu, sq * (1.f / sCz));        // one rounding (c_z is a power of two); 0 for a constant row
      const float rstd = var > 0.f ? rsqrtf(var + p.eps) : 0.f;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        const uint4 w0 = __ldg(reinterpret_cast<const uint4*>(p.wfold + h * sCz));
        const uint4 w1 = __ldg(reinterpret_cast<const uint4*>(p.wfold + h * sCz) + 1);
        const uint32_t wf_[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
        float pw = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) dot_bf16x2(pw, pw_[i], wf_[i]);
        s_logit[j * H + h] = fmaf(rstd, fmaf(-mu, __ldg(p.c1 + h), pw), __ldg(p.c0 + h));
      }
    } else {
#pragma unroll
      for (int h = 0; h < H; ++h) s_logit[j * H + h] = -INFINITY;
    }
  }
  __syncwarp();
  // ---- (B) logits += q . k, RPL rows per load, four loads in flight
  for (int j0 = 0; j0 < p.kn; j0 += 4 * RPL) {
    uint4 kv[4];
    int mm[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int j = j0 + u * RPL + grp;
      mm[u] = j < p.kn ? s_idx[j] : -1;
      if (mm[u] >= 0) kv[u] = __ldg(reinterpret_cast<const uint4*>(p.k + (int64_t)mm[u] * D) + ch);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      float d0 = 0.f, d1 = 0.f;
      if (mm[u] >= 0) {
        dot_bf16x2(d0, kv[u].x, qv.x); dot_bf16x2(d1, kv[u].y, qv.y);
        dot_bf16x2(d0, kv[u].z, qv.z); dot_bf16x2(d1, kv[u].w, qv.w);
      }
      float d = d0 + d1;
      d += __shfl_xor_sync(0xffffffffu, d, 1);
      d += __shfl_xor_sync(0xffffffffu, d, 2);
      if (mm[u] >= 0 && (ch & 3) == 0) s_logit[(j0 + u * RPL + grp) * H + hd] += d;
    }
  }
  __syncwarp();
  // ---- (C) softmax statistics per head over the slots (lane = slot), numerators back to shared memory
  float mx[H], sum[H];
#pragma unroll
  for (int h = 0; h < H; ++h) { mx[h] = -INFINITY; sum[h] = 0.f; }
  for (int j = lane; j < kpad; j += 32)
#pragma unroll
    for (int h = 0; h < H; ++h) mx[h] = fmaxf(mx[h], s_logit[j * H + h]);
#pragma unroll
  for (int h = 0; h < H; ++h) mx[h] = warp_max(mx[h]);
  if (mx[0] == -INFINITY) {             // no valid neighbour (a slot is valid for all heads or for none): o = 0
    for (int e = lane; e < D; e += 32) p.gated[l * D + e] = __float2bfloat16_rn(0.f);
    return;
  }
  for (int j = lane; j < kpad; j += 32)
#pragma unroll
    for (int h = 0; h < H; ++h) {
      const float pe = fast_exp2(s_logit[j * H + h] - mx[h]);    // exp2(-inf) = 0 for unused slots
      sum[h] += pe;
      s_logit[j * H + h] = pe;
    }
#pragma unroll
  for (int h = 0; h < H; ++h) sum[h] = warp_sum(sum[h]);
  __syncwarp();
  // ---- (D) acc += P v, RPL rows per load, four loads in flight
  float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  for (int j0 = 0; j0 < p.kn; j0 += 4 * RPL) {
    uint4 vv[4];
    int mm[4];
    float pe[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int j = j0 + u * RPL + grp;
      mm[u] = j < p.kn ? s_idx[j] : -1;
      if (mm[u] >= 0) {
        vv[u] = __ldg(reinterpret_cast<const uint4*>(p.v + (int64_t)mm[u] * D) + ch);
        pe[u] = s_logit[j * H + hd];
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (mm[u] >= 0) {
        const uint32_t pb = pack_bf16(pe[u], 0.f);     // P rounded to bf16 for PV, like the dense kernels
        axpy_bf16x2(acc[0], acc[1], vv[u].x, pb); axpy_bf16x2(acc[2], acc[3], vv[u].y, pb);
        axpy_bf16x2(acc[4], acc[5], vv[u].z, pb); axpy_bf16x2(acc[6], acc[7], vv[u].w, pb);
      }
  }
  // the RPL row groups hold partial sums of the same output chunk
#pragma unroll
  for (int off = LPR; off < 32; off <<= 1)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], off);
  if (grp == 0) {
    float lh = sum[0];
#pragma unroll
    for (int h = 1; h < H; ++h) lh = hd == h ? sum[h] : lh;
    const float inv = 1.f / lh;
    const uint4 gv = __ldg(reinterpret_cast<const uint4*>(p.g + l * D) + ch);
    const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
    uint32_t ow[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float g0 = __uint_as_float(gw[i] << 16), g1 = __uint_as_float(gw[i] & 0xffff0000u);
      ow[i] = pack_bf16(g0 * (acc[2 * i] * inv), g1 * (acc[2 * i + 1] * inv));
    }
    *reinterpret_cast<uint4*>(p.gated + l * D + ch * 8) = make_uint4(ow[0], ow[1], ow[2], ow[3]);
  }
}

// p_slice[l, j, :] = P[l, idx[l, j], :]  ("The relevant slice of P is gathered at those k indices"):
// 16-byte chunks, the chunks of one slot on adjacent lanes; unused slots (idx < 0) are filled with zeros.
__global__ void __launch_bounds__(256) gather_pair_slice_kernel(const uint4* __restrict__ P, int64_t ldp16,
                                                                const int32_t* __restrict__ idx, uint4* __restrict__ out,
                                                                int64_t L, int kn, int chunks) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = L * kn * chunks;
  if (e >= total) return;
  const int ch = (int)(e % chunks);
  const int64_t slot = e / chunks;
  const int64_t l = slot / kn;
  const int m = __ldg(idx + slot);
  out[e] = (unsigned)m < (unsigned)L ? __ldg(P + l * ldp16 + (int64_t)m * chunks + ch) : make_uint4(0u, 0u, 0u, 0u);
}

}  // namespace

bool sparse_atom_supports(dcp_dtype dt, int H, int c, int c_z, int kn) {
  return dt == DCP_BF16 && c == sC && c_z == sCz && H >= 1 && H <= 16 && kn >= 1 && kn <= 32 * sMaxPass;
}

cudaError_t launch_sparse_atom(const void* q, const void* k, const void* v, const void* g, const void* p_slice,
                               const int32_t* idx, const void* wfold, const float* c1, const float* c0, void* gated,
                               int64_t L, int kn, int H, float eps, cudaStream_t st) {
  if (L <= 0) return cudaSuccess;
  SparseParams sp;
  sp.q = (const __nv_bfloat16*)q; sp.k = (const __nv_bfloat16*)k; sp.v = (const __nv_bfloat16*)v;
  sp.g = (const __nv_bfloat16*)g; sp.p = (const __nv_bfloat16*)p_slice; sp.idx = idx;
  sp.wfold = (const __nv_bfloat16*)wfold; sp.c1 = c1; sp.c0 = c0; sp.gated = (__nv_bfloat16*)gated;
  sp.L = L; sp.kn = kn; sp.H = H; sp.eps = eps;
  if (H == 2 || H == 4 || H == 8) {   // row-coalesced kernel: one warp per atom, dynamic smem = logits + indices
    const int kpad = (kn + 31) & ~31;
    const size_t smem = (size_t)4 * kpad * (H + 1) * sizeof(float);
    const unsigned blocks = (unsigned)((L + 3) / 4);
    cudaError_t e = cudaSuccess;
    if (H == 2) {
      e = cudaFuncSetAttribute(sparse_atom_rows_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e == cudaSuccess) sparse_atom_rows_kernel<2><<<blocks, 128, smem, st>>>(sp);
    } else if (H == 4) {
      e = cudaFuncSetAttribute(sparse_atom_rows_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e == cudaSuccess) sparse_atom_rows_kernel<4><<<blocks, 128, smem, st>>>(sp);
    } else {
      e = cudaFuncSetAttribute(sparse_atom_rows_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e == cudaSuccess) sparse_atom_rows_kernel<8><<<blocks, 128, smem, st>>>(sp);
    }
    return e != cudaSuccess ? e : cudaGetLastError();
  }
  const int64_t warps = L * H;
  sparse_atom_kernel<<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(sp);
  return cudaGetLastError();
}

}  // namespace dcp

namespace dcp {
cudaError_t launch_gather_pair_slice(const void* P, int64_t ldp_bytes, const int32_t* idx, void* out, int64_t L, int kn,
                                     int row_bytes, cudaStream_t st) {
  const int chunks = row_bytes / 16;
  const int64_t total = L * kn * chunks;
  if (total <= 0) return cudaSuccess;
  gather_pair_slice_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>((const uint4*)P, ldp_bytes / 16, idx, (uint4*)out,
                                                                            L, kn, chunks);
  return cudaGetLastError();
}
}  // namespace dcp
