// k-nearest-neighbour lists for the sparse atom attention: the one-GPU core of the
// paper's chunked cdist + running top-k.
//   PAPER.md:303  "The kNN indices are computed once per denoising step from the current noised coordinates X^(t) via a
//                 single cdist call ... until the per-query budget k = n_attn-keys (default k = 128) is filled"
//   PAPER.md:454  "A naive implementation computes an [L, L] distance matrix and takes the top-k per row" -- here the
//                 distance row never exists: candidates stream past a running sorted top-k list (the single-device
//                 form of the ring_topk merge).
// idx[l, :] = the k atoms m with the smallest d2(l, m) = (x_m0-x_l0)^2 + (x_m1-x_l1)^2 + (x_m2-x_l2)^2, ordered by
// (d2, m) ascending; the query itself is part of its list.  Floating point decides an integer here, so the distance
// arithmetic is pinned: IEEE binary32, round to nearest, NO fused multiply-add, t = x_m - x_l per coordinate,
// d2 = (t0 t0 + t1 t1) + t2 t2 -- the oracle (oracle/knn.py) uses the same operations and the result is bit-exact.
//
// One warp per query.  The list of k (d2, index) pairs, sorted lexicographically, lives in registers, NR = k / 32
// (rounded up) consecutive positions per lane.  Candidates are visited 128 at a time; a ballot picks those that beat
// the current k-th entry, and each is inserted by a ballot-count of its position and a one-place shift (register
// moves + one shuffle).  A window of indices around the query is scanned first, which tightens the k-th distance
// early (same-chain atoms are close in space), so that few of the remaining L candidates are ever inserted and the
// scan (about a dozen instructions per 32 candidates) dominates.
#include "kernels.h"

namespace dcp {

namespace {

constexpr float kInf = __builtin_huge_valf();
constexpr int kTile = 2048;   // candidates per shared-memory tile (3 x 8 KB)

template <int NR>
__global__ void __launch_bounds__(256) knn_kernel(const float* __restrict__ x, int32_t* __restrict__ idx, int L, int k) {
  const int lane = threadIdx.x & 31;
  __shared__ float sx[kTile], sy[kTile], sz[kTile];
  const int lq = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const bool active = lq < L;                           // inactive warps still help staging the tiles
  const int l = active ? lq : L - 1;
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  float ld[NR];       // list position lane * NR + r, sorted by (d2, index)
  int li[NR];
#pragma unroll
  for (int r = 0; r < NR; ++r) { ld[r] = kInf; li[r] = 0x7fffffff; }
  const int last_lane = (k - 1) / NR, last_r = (k - 1) % NR;
  float tau = kInf;   // (d2, index) of list position k - 1: the current k-th best
  int tau_i = 0x7fffffff;

  // insert the candidates of one 32-wide chunk that beat the k-th entry, in increasing index
  auto insert_chunk = [&](int c0, float d, unsigned mask) {
    while (mask) {
      const int b = __ffs(mask) - 1;
      mask &= mask - 1;
      const float dn = __shfl_sync(0xffffffffu, d, b);
      const int mn = c0 + b;
      if (!(dn < tau || (dn == tau && mn < tau_i))) continue;      // the k-th entry moved meanwhile (warp-uniform)
      // position = number of entries that come before (dn, mn) in (d2, index) order
      int pos = 0;
#pragma unroll
      for (int r = 0; r < NR; ++r) pos += __popc(__ballot_sync(0xffffffffu, ld[r] < dn || (ld[r] == dn && li[r] < mn)));
      const int pl = pos / NR, pr = pos % NR;
      // shift positions pos .. one place to the right (the old k-th entry falls off), insert at pos
      const float up_d = __shfl_up_sync(0xffffffffu, ld[NR - 1], 1);
      const int up_i = __shfl_up_sync(0xffffffffu, li[NR - 1], 1);
      if (lane > pl) {
#pragma unroll
        for (int r = NR - 1; r > 0; --r) { ld[r] = ld[r - 1]; li[r] = li[r - 1]; }
        ld[0] = up_d; li[0] = up_i;
      } else if (lane == pl) {
#pragma unroll
        for (int r = NR - 1; r > 0; --r)
          if (r > pr) { ld[r] = ld[r - 1]; li[r] = li[r - 1]; }
#pragma unroll
        for (int r = 0; r < NR; ++r)
          if (r == pr) { ld[r] = dn; li[r] = mn; }
      }
      float tl = ld[0];
      int ti = li[0];
#pragma unroll
      for (int r = 1; r < NR; ++r) { tl = r == last_r ? ld[r] : tl; ti = r == last_r ? li[r] : ti; }
      tau = __shfl_sync(0xffffffffu, tl, last_lane);
      tau_i = __shfl_sync(0xffffffffu, ti, last_lane);
    }
  };
  // The 8 queries of a block scan the same candidates: tiles of kTile atoms are staged once per block in shared memory
  // as three coordinate planes (conflict-free reads; the [L][3] rows in global memory cost 3-4 L1 wavefronts per
  // 32-candidate load and made the scan L1-bound).  Tile order: the tile of the block's own atoms first (atoms close
  // in index are mostly close in space, so the k-th distance tightens early and few later candidates are inserted),
  // then the others; the (d2, index) order of the list makes the result independent of the visiting order.
  const int n_tiles = (L + kTile - 1) / kTile;
  const int own = (blockIdx.x * (blockDim.x >> 5)) / kTile;
  for (int tt = 0; tt < n_tiles; ++tt) {
    const int tile = tt == 0 ? own : (tt <= own ? tt - 1 : tt);
    const int t0 = tile * kTile;
    __syncthreads();                                   // every warp is done with the previous tile
    for (int e = threadIdx.x; e < kTile; e += blockDim.x) {
      const int m = t0 + e;
      sx[e] = m < L ? __ldg(x + 3 * (int64_t)m) : 0.f;
      sy[e] = m < L ? __ldg(x + 3 * (int64_t)m + 1) : 0.f;
      sz[e] = m < L ? __ldg(x + 3 * (int64_t)m + 2) : 0.f;
    }
    __syncthreads();
    if (!active) continue;
    const int n_here = (L - t0 < kTile ? L - t0 : kTile);
    for (int c0 = 0; c0 < n_here; c0 += 128) {          // four chunks per step: independent loads and arithmetic
      float d[4];
      unsigned mk[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int e = (c0 + 32 * u + lane) & (kTile - 1);   // c0 + 128 may run past the tile when n_here is ragged
        const float a0 = __fsub_rn(sx[e], q0), a1 = __fsub_rn(sy[e], q1), a2 = __fsub_rn(sz[e], q2);
        const float dd = __fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2));
        d[u] = c0 + 32 * u + lane < n_here ? dd : kInf;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int m = t0 + c0 + 32 * u + lane;
        mk[u] = __ballot_sync(0xffffffffu, d[u] < tau || (d[u] == tau && m < tau_i));
      }
      if ((mk[0] | mk[1] | mk[2] | mk[3]) == 0) continue;
#pragma unroll 1
      for (int u = 0; u < 4; ++u)
        if (mk[u]) insert_chunk(t0 + c0 + 32 * u, d[u], mk[u]);
    }
  }
  if (!active) return;
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const int pos = lane * NR + r;
    if (pos < k) idx[(int64_t)l * k + pos] = li[r];
  }
}

}  // namespace

bool knn_supports(int64_t L, int k) { return L >= 1 && L <= 0x7fffffff && k >= 1 && k <= 512 && k <= L; }

cudaError_t launch_knn(const float* x, int32_t* idx, int64_t L, int k, cudaStream_t st) {
  const int nr = (k + 31) / 32;
  const unsigned blocks = (unsigned)((L + 7) / 8);
  if (nr <= 1) knn_kernel<1><<<blocks, 256, 0, st>>>(x, idx, (int)L, k);
  else if (nr <= 2) knn_kernel<2><<<blocks, 256, 0, st>>>(x, idx, (int)L, k);
  else if (nr <= 4) knn_kernel<4><<<blocks, 256, 0, st>>>(x, idx, (int)L, k);
  else if (nr <= 8) knn_kernel<8><<<blocks, 256, 0, st>>>(x, idx, (int)L, k);
  else knn_kernel<16><<<blocks, 256, 0, st>>>(x, idx, (int)L, k);
  return cudaGetLastError();
}

}  // namespace dcp
