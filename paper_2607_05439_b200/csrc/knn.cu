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
// One warp per query, 8 queries per CTA sharing shared-memory tiles of 2048 candidates (three coordinate planes:
// conflict-free reads; the [L][3] rows in global memory cost 3-4 L1 wavefronts per 32-candidate load).  The tile of the
// CTA's own atoms comes first (atoms close in index are mostly close in space, so the bound on the k-th distance tightens
// early); the (d2, index) order makes the result independent of the visiting order.
//   knn_select_kernel      threshold select with candidate buffers (below)
//   knn_insert_global      exact fallback of a single query: the sorted list of k (d2, index) pairs lives in registers
//                          (NR = k / 32 per lane); candidates that beat the k-th entry (one ballot per 32) are inserted by a
//                          ballot-count of their position and a one-place shift.  Round 1's first kernel worked this way for
//                          every query (2.81 ms at L = 24000, k = 128).
#include <type_traits>

#include "kernels.h"

namespace dcp {

namespace {

constexpr float kInf = __builtin_huge_valf();
constexpr int kTile = 2048;   // candidates per shared-memory tile (3 x 8 KB)

// ---- threshold select (k <= 512): no sorted list is maintained while scanning.
//   1. own tile (2048 atoms): each lane keeps the r = ceil(k / 32) smallest of its 64 distances while they stream past
//      (nothing else stays in registers); the largest of the lanes' r-th smallest is a bound T1 with at least k of the
//      tile's distances <= T1.  A second pass appends the tile's entries <= T1 to the per-warp shared-memory buffer,
//      a bisection of the binary32 bit pattern over the BUFFER (16 values per lane, counted with ballots) tightens the
//      bound to a threshold T a few percent above the tile's own k-th distance, and the buffer is compacted to <= T;
//   2. one scan over the other tiles appends every (d2, index) with d2 <= T (one ballot + one prefix popcount per 32
//      candidates; typically 1.5 k .. 2 k entries in the end) -- but only over the 128-atom chunks whose bounding box
//      reaches within T: the bound applies the pinned arithmetic to the query-to-box gaps, rounding is monotone, so a
//      skipped chunk provably holds no candidate; a buffer about to overflow is re-bounded by its own k-th distance;
//   3. a full bisection over the buffer finds the exact k-th distance D, the entries <= D (k of them unless distances
//      tie) are compacted and sorted by (d2, index) with a bitonic network: the first k are the answer.
// Same distances, same (d2, index) order as knn_kernel: the result is identical.  A query whose buffer overflows
// (more than kCap candidates within the bound: a very dense neighbourhood) falls back to the insertion scan over global
// memory.  Round 1's version held the own tile's 64 distances per lane in registers (128 registers, 16 warps per SM) and
// sorted the whole buffer.

template <int NR>
__device__ __noinline__ void knn_insert_global(const float* __restrict__ x, int32_t* __restrict__ idx, int L, int k, int l,
                                               int lane) {
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  float ld[NR];
  int li[NR];
#pragma unroll
  for (int r = 0; r < NR; ++r) { ld[r] = kInf; li[r] = 0x7fffffff; }
  const int last_lane = (k - 1) / NR, last_r = (k - 1) % NR;
  float tau = kInf;
  int tau_i = 0x7fffffff;
  for (int c0 = 0; c0 < L; c0 += 32) {
    const int m = c0 + lane;
    float d = kInf;
    if (m < L) {
      const float a0 = __fsub_rn(__ldg(x + 3 * (int64_t)m), q0), a1 = __fsub_rn(__ldg(x + 3 * (int64_t)m + 1), q1);
      const float a2 = __fsub_rn(__ldg(x + 3 * (int64_t)m + 2), q2);
      d = __fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2));
    }
    unsigned mask = __ballot_sync(0xffffffffu, d < tau || (d == tau && m < tau_i));
    while (mask) {
      const int b = __ffs(mask) - 1;
      mask &= mask - 1;
      const float dn = __shfl_sync(0xffffffffu, d, b);
      const int mn = c0 + b;
      if (!(dn < tau || (dn == tau && mn < tau_i))) continue;
      int pos = 0;
#pragma unroll
      for (int r = 0; r < NR; ++r) pos += __popc(__ballot_sync(0xffffffffu, ld[r] < dn || (ld[r] == dn && li[r] < mn)));
      const int pl = pos / NR, pr = pos % NR;
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
  }
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const int pos = lane * NR + r;
    if (pos < k) idx[(int64_t)l * k + pos] = li[r];
  }
}

// kCap = candidate-buffer entries per warp; NRF = list registers per lane of the exact fallback
template <int kCap, int NRF>
__global__ void __launch_bounds__(256) knn_select_kernel(const float* __restrict__ x, int32_t* __restrict__ idx, int L, int k) {
  extern __shared__ float smem_knn[];
  float* sx = smem_knn;
  float* sy = sx + kTile;
  float* sz = sy + kTile;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  unsigned* bd = reinterpret_cast<unsigned*>(sz + kTile) + wib * (2 * kCap);   // per-warp buffer: kCap distances (bit patterns),
  int* bi = reinterpret_cast<int*>(bd + kCap);                                 // kCap indices
  constexpr int kPer = kCap / 32;                              // buffer entries per lane
  constexpr int NS = kCap / 64;                                // per-lane smallest-values slots of step 1a: >= ceil(k / 32)
  float* box = sz + kTile + 8 * (2 * kCap);                    // per tile: bounding boxes of its 16 chunks of 128 atoms, [16][lo xyz, hi xyz]
  constexpr unsigned kInfBits = 0x7f800000u;
  const int lq = blockIdx.x * 8 + wib;
  const bool active = lq < L;
  const int l = active ? lq : L - 1;
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  const int n_tiles = (L + kTile - 1) / kTile;
  const int own = (blockIdx.x * 8) / kTile;
  unsigned thr = kInfBits;                                     // bit pattern of the threshold T
  int cnt = 0;
  const unsigned lt_mask = (1u << lane) - 1u;
  auto dist_bits = [&](int e) {
    const float a0 = __fsub_rn(sx[e], q0), a1 = __fsub_rn(sy[e], q1), a2 = __fsub_rn(sz[e], q2);
    return __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2)));
  };
  // smallest pattern T in [0, hi0] with #{buffer entries <= T} >= need, to `iters` bisection steps (hi stays a valid bound)
  auto bisect = [&](const unsigned (&bv)[kPer], unsigned hi0, int need, int iters) {
    unsigned lo = 0u, hi = hi0;
    for (int it = 0; it < iters && lo < hi; ++it) {
      const unsigned mid = lo + ((hi - lo) >> 1);
      int c = 0;
#pragma unroll
      for (int j = 0; j < kPer; ++j) c += __popc(__ballot_sync(0xffffffffu, bv[j] <= mid));
      if (c >= need) hi = mid; else lo = mid + 1;
      if (c == need) break;                                    // exactly `need` entries are <= mid: the set is settled
    }
    return hi;
  };
  // keep the buffer entries <= t, in order; returns the new count
  auto compact = [&](const unsigned (&bv)[kPer], unsigned t, int n) {
    int nc = 0;
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
      if (32 * j >= n) break;                                  // warp-uniform
      const int e = 32 * j + lane;
      const int iv = e < n ? bi[e] : 0;
      const bool pass = e < n && bv[j] <= t;
      const unsigned mask = __ballot_sync(0xffffffffu, pass);  // every lane has read chunk j before any lane overwrites it
      if (pass) { const int slot = nc + __popc(mask & lt_mask); bd[slot] = bv[j]; bi[slot] = iv; }
      nc += __popc(mask);
      __syncwarp();
    }
    return nc;
  };
  auto load_buffer = [&](unsigned (&bv)[kPer], int n) {
#pragma unroll
    for (int j = 0; j < kPer; ++j) bv[j] = 32 * j + lane < n ? bd[32 * j + lane] : 0xffffffffu;
  };

  bool over = false;                                           // more than kCap entries tie within the bound: exact fallback
  // the buffer's own k-th distance is a bound too: when the buffer is about to overflow (a dense neighbourhood), bisect
  // it, keep the entries within the new bound and go on (the buffer holds >= k entries then: kCap >= 2 k)
  auto tighten = [&]() {
    __syncwarp();
    unsigned bv[kPer];
    load_buffer(bv, cnt);
    thr = bisect(bv, thr, k, 32);
    cnt = compact(bv, thr, cnt);
  };
  // append the lanes' candidates (d2 bits v, atom m) that pass
  auto append = [&](unsigned v, int m, bool pass) {
    if (over) return;
    unsigned mask = __ballot_sync(0xffffffffu, pass);
    if (cnt + __popc(mask) > kCap) {
      tighten();
      pass = pass && v <= thr;
      mask = __ballot_sync(0xffffffffu, pass);
      if (cnt + __popc(mask) > kCap) { over = true; return; }
    }
    if (pass) { const int slot = cnt + __popc(mask & lt_mask); bd[slot] = v; bi[slot] = m; }
    cnt += __popc(mask);
  };

  for (int tt = 0; tt < n_tiles; ++tt) {
    const int tile = tt == 0 ? own : (tt <= own ? tt - 1 : tt);
    const int t0 = tile * kTile;
    __syncthreads();
    for (int e = threadIdx.x; e < kTile; e += blockDim.x) {
      const int m = t0 + e;
      sx[e] = m < L ? __ldg(x + 3 * (int64_t)m) : 0.f;
      sy[e] = m < L ? __ldg(x + 3 * (int64_t)m + 1) : 0.f;
      sz[e] = m < L ? __ldg(x + 3 * (int64_t)m + 2) : 0.f;
    }
    __syncthreads();
    const int n_here = (L - t0 < kTile ? L - t0 : kTile);
    {
      // bounding boxes of the tile's 128-atom chunks (atoms close in index are mostly close in space): warp w takes
      // chunks 2 w and 2 w + 1; an empty chunk gets lo = +inf, hi = -inf
#pragma unroll
      for (int cc = 0; cc < 2; ++cc) {
        const int ch = 2 * wib + cc;
        float lo0 = kInf, lo1 = kInf, lo2 = kInf, hi0 = -kInf, hi1 = -kInf, hi2 = -kInf;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int e = ch * 128 + 32 * i + lane;
          if (e < n_here) {
            lo0 = fminf(lo0, sx[e]); hi0 = fmaxf(hi0, sx[e]);
            lo1 = fminf(lo1, sy[e]); hi1 = fmaxf(hi1, sy[e]);
            lo2 = fminf(lo2, sz[e]); hi2 = fmaxf(hi2, sz[e]);
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          lo0 = fminf(lo0, __shfl_xor_sync(0xffffffffu, lo0, o)); hi0 = fmaxf(hi0, __shfl_xor_sync(0xffffffffu, hi0, o));
          lo1 = fminf(lo1, __shfl_xor_sync(0xffffffffu, lo1, o)); hi1 = fmaxf(hi1, __shfl_xor_sync(0xffffffffu, hi1, o));
          lo2 = fminf(lo2, __shfl_xor_sync(0xffffffffu, lo2, o)); hi2 = fmaxf(hi2, __shfl_xor_sync(0xffffffffu, hi2, o));
        }
        if (lane == 0) {
          box[ch * 6] = lo0; box[ch * 6 + 1] = lo1; box[ch * 6 + 2] = lo2;
          box[ch * 6 + 3] = hi0; box[ch * 6 + 4] = hi1; box[ch * 6 + 5] = hi2;
        }
      }
      __syncthreads();
    }
    unsigned skip = 0u;                                        // chunks of this tile that step 1 has already taken
    if (tt == 0) {
      // ---- 1a. the home window: the kWin chunks of the own tile around the query (the whole tile when the window does not
      // hold k atoms); the r smallest distances of each lane's share of it
      constexpr int kWin = kCap <= 512 ? 4 : 16;               // 4 chunks = 512 atoms >= 2 k (k <= 256); larger k: the whole tile
      int h0 = ((lq - t0) >> 7) - kWin / 2;
      h0 = h0 < 0 ? 0 : (h0 > 16 - kWin ? 16 - kWin : h0);
      int e0 = h0 * 128, e1 = e0 + kWin * 128;
      e1 = e1 < n_here ? e1 : n_here;
      if (e1 - e0 < k) { e0 = 0; e1 = n_here; }                // ragged tile end: take everything the tile has
      const int n_win = e1 - e0;
      skip = e1 - e0 == n_here ? 0xffffu : (((1u << kWin) - 1u) << h0);
      const int need = k < n_win ? k : n_win;
      const int r = (need + 31) >> 5;                          // <= NS (k <= kCap / 2)
      unsigned sm[NS];
#pragma unroll
      for (int j = 0; j < NS; ++j) sm[j] = kInfBits;
      for (int eb = e0; eb < e1; eb += 32) {
        const int e = eb + lane;
        unsigned v = e < e1 ? dist_bits(e) : kInfBits;
        if (__any_sync(0xffffffffu, v < sm[NS - 1])) {
#pragma unroll
          for (int j = 0; j < NS; ++j) { const unsigned lo = min(sm[j], v); v = max(sm[j], v); sm[j] = lo; }
        }
      }
      unsigned sr = sm[0];
#pragma unroll
      for (int j = 1; j < NS; ++j) sr = j == r - 1 ? sm[j] : sr;
      thr = n_win >= k ? __reduce_max_sync(0xffffffffu, sr) : kInfBits;   // T1; fewer than k atoms: no bound
      // ---- 1b. the window's entries <= T1 -> buffer
      for (int eb = e0; eb < e1; eb += 32) {
        const int e = eb + lane;
        const unsigned v = e < e1 ? dist_bits(e) : kInfBits;
        append(v, t0 + e, e < e1 && v <= thr);
      }
      __syncwarp();
      if (!over && thr != kInfBits) {
        // ---- 1c. tighten the bound over the buffer, keep what is within it
        unsigned bv[kPer];
        load_buffer(bv, cnt);
        thr = bisect(bv, thr, need, 14);
        cnt = compact(bv, thr, cnt);
      }
    }
    {
      // ---- 2. the chunks (of the own tile: the ones outside the home window) whose bounding box reaches within the bound,
      // four 32-candidate pieces per step.
      // Lane c < 16 takes chunk c: lb = the pinned distance arithmetic applied to the per-axis gaps between the query and
      // the box (sub, mul, add, add, each rounded to nearest, no FMA).  Rounding is monotone, so every atom of the chunk has
      // a computed d2 >= lb: a chunk with lb > T holds no candidate, and skipping it changes no bit of the result.
      float lb = kInf;
      if (lane < 16) {
        const float* bx = box + lane * 6;
        const float g0 = fmaxf(fmaxf(__fsub_rn(bx[0], q0), __fsub_rn(q0, bx[3])), 0.f);
        const float g1 = fmaxf(fmaxf(__fsub_rn(bx[1], q1), __fsub_rn(q1, bx[4])), 0.f);
        const float g2 = fmaxf(fmaxf(__fsub_rn(bx[2], q2), __fsub_rn(q2, bx[5])), 0.f);
        lb = __fadd_rn(__fadd_rn(__fmul_rn(g0, g0), __fmul_rn(g1, g1)), __fmul_rn(g2, g2));
      }
      unsigned todo = __ballot_sync(0xffffffffu, lane < 16 && __float_as_uint(lb) <= thr) & ~skip;
      while (todo) {
        const int c0 = (__ffs(todo) - 1) * 128;
        todo &= todo - 1;
        unsigned dbv[4], mk[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int e = c0 + 32 * u + lane;
          dbv[u] = dist_bits(e);
          mk[u] = __ballot_sync(0xffffffffu, dbv[u] <= thr && e < n_here);
        }
        if ((mk[0] | mk[1] | mk[2] | mk[3]) == 0) continue;
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (mk[u]) append(dbv[u], t0 + c0 + 32 * u + lane, (mk[u] >> lane) & 1u);
      }
    }
  }
  if (!active) return;
  if (over) {                                                  // > kCap entries tie within the bound: exact fallback
    knn_insert_global<NRF>(x, idx, L, k, l, lane);
    return;
  }
  // ---- 3. the exact k-th distance over the buffer, then a sort of the entries within it (k of them unless distances tie)
  __syncwarp();
  {
    unsigned bv[kPer];
    load_buffer(bv, cnt);
    const unsigned dk = bisect(bv, thr, k < cnt ? k : cnt, 32);
    cnt = compact(bv, dk, cnt);
  }
  int P = 32;
  while (P < cnt) P <<= 1;
  for (int e = cnt + lane; e < P; e += 32) { bd[e] = 0xffffffffu; bi[e] = 0x7fffffff; }
  __syncwarp();
  for (int size = 2; size <= P; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = lane; i < (P >> 1); i += 32) {
        const int pos = 2 * i - (i & (stride - 1));
        const int par = pos + stride;
        const bool asc = (pos & size) == 0;
        const unsigned da = bd[pos], dbb = bd[par];
        const int ia = bi[pos], ib = bi[par];
        const bool a_after_b = da > dbb || (da == dbb && ia > ib);
        if (a_after_b == asc) { bd[pos] = dbb; bd[par] = da; bi[pos] = ib; bi[par] = ia; }
      }
      __syncwarp();
    }
  }
  for (int j = lane; j < k; j += 32) idx[(int64_t)l * k + j] = bi[j];
}

// ---- structured neighbour budget (reading 26; oracle/knn_budget.py)
// One warp per query, the insertion scan of knn_kernel with TWO sorted register lists: the own chain (class A; with at
// most three chains: every atom) ordered by (not sequence-local, d2, index) -- the flag rides in bit 31 of the
// non-negative distance's bit pattern, so sequence-local atoms come first -- and the other chains (class B) ordered by
// (d2, index).  After the scan the quotas are arithmetic on the class sizes; the chosen prefixes of the two lists are
// sorted together by (d2, index) in shared memory (bitonic) and written out.
template <int NR>
struct TopList {
  unsigned key[NR];
  int li[NR];
  unsigned tau;
  int tau_i;
  int last_lane, last_r;
  __device__ __forceinline__ void init(int cap) {
#pragma unroll
    for (int r = 0; r < NR; ++r) { key[r] = 0xffffffffu; li[r] = 0x7fffffff; }
    tau = 0xffffffffu; tau_i = 0x7fffffff;
    last_lane = (cap - 1) / NR; last_r = (cap - 1) % NR;
  }
  __device__ __forceinline__ bool beats(unsigned kk, int m) const { return kk < tau || (kk == tau && m < tau_i); }
  // insert the candidates of `mask` (lane b holds key kk of atom c0 + b), in increasing index
  __device__ __forceinline__ void insert_chunk(int c0, unsigned kk, unsigned mask, int lane) {
    while (mask) {
      const int b = __ffs(mask) - 1;
      mask &= mask - 1;
      const unsigned kn = __shfl_sync(0xffffffffu, kk, b);
      const int mn = c0 + b;
      if (!beats(kn, mn)) continue;                            // the last entry moved meanwhile (warp-uniform)
      int pos = 0;
#pragma unroll
      for (int r = 0; r < NR; ++r) pos += __popc(__ballot_sync(0xffffffffu, key[r] < kn || (key[r] == kn && li[r] < mn)));
      const int pl = pos / NR, pr = pos % NR;
      const unsigned up_k = __shfl_up_sync(0xffffffffu, key[NR - 1], 1);
      const int up_i = __shfl_up_sync(0xffffffffu, li[NR - 1], 1);
      if (lane > pl) {
#pragma unroll
        for (int r = NR - 1; r > 0; --r) { key[r] = key[r - 1]; li[r] = li[r - 1]; }
        key[0] = up_k; li[0] = up_i;
      } else if (lane == pl) {
#pragma unroll
        for (int r = NR - 1; r > 0; --r)
          if (r > pr) { key[r] = key[r - 1]; li[r] = li[r - 1]; }
#pragma unroll
        for (int r = 0; r < NR; ++r)
          if (r == pr) { key[r] = kn; li[r] = mn; }
      }
      unsigned tk = key[0];
      int ti = li[0];
#pragma unroll
      for (int r = 1; r < NR; ++r) { tk = r == last_r ? key[r] : tk; ti = r == last_r ? li[r] : ti; }
      tau = __shfl_sync(0xffffffffu, tk, last_lane);
      tau_i = __shfl_sync(0xffffffffu, ti, last_lane);
    }
  }
};

template <int NR>
__global__ void __launch_bounds__(256) knn_budget_kernel(const float* __restrict__ x, const int32_t* __restrict__ rid,
                                                         const int32_t* __restrict__ cid, int32_t* __restrict__ idx, int L, int k,
                                                         int n_seq, int split, int q_out) {
  extern __shared__ float smem_knn[];
  float* sx = smem_knn;
  float* sy = sx + kTile;
  float* sz = sy + kTile;
  int* sr = reinterpret_cast<int*>(sz + kTile);
  int* sc = sr + kTile;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  unsigned* bk = reinterpret_cast<unsigned*>(sc + kTile) + wib * (2 * 512);   // per-warp sort buffer: 512 keys, 512 indices
  int* bi = reinterpret_cast<int*>(bk + 512);
  const int lq = blockIdx.x * 8 + wib;
  const bool active = lq < L;
  const int l = active ? lq : L - 1;
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  const int qr = __ldg(rid + l), qc = __ldg(cid + l), win = n_seq - 1;
  TopList<NR> la, lb;
  la.init(k);
  lb.init(k);
  int cnt_a = 0, cnt_b = 0;
  const int n_tiles = (L + kTile - 1) / kTile;
  const int own = (blockIdx.x * 8) / kTile;
  for (int tt = 0; tt < n_tiles; ++tt) {
    const int tile = tt == 0 ? own : (tt <= own ? tt - 1 : tt);
    const int t0 = tile * kTile;
    __syncthreads();
    for (int e = threadIdx.x; e < kTile; e += blockDim.x) {
      const int m = t0 + e;
      sx[e] = m < L ? __ldg(x + 3 * (int64_t)m) : 0.f;
      sy[e] = m < L ? __ldg(x + 3 * (int64_t)m + 1) : 0.f;
      sz[e] = m < L ? __ldg(x + 3 * (int64_t)m + 2) : 0.f;
      sr[e] = m < L ? __ldg(rid + m) : 0;
      sc[e] = m < L ? __ldg(cid + m) : -1;
    }
    __syncthreads();
    if (!active) continue;
    const int n_here = (L - t0 < kTile ? L - t0 : kTile);
    for (int c0 = 0; c0 < n_here; c0 += 32) {
      const int e = c0 + lane;
      const bool valid = e < n_here;
      const float a0 = __fsub_rn(sx[e & (kTile - 1)], q0), a1 = __fsub_rn(sy[e & (kTile - 1)], q1), a2 = __fsub_rn(sz[e & (kTile - 1)], q2);
      const unsigned db = __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2)));
      const bool same = sc[e & (kTile - 1)] == qc;
      int dr = sr[e & (kTile - 1)] - qr;
      dr = dr < 0 ? -dr : dr;
      const bool local = same && dr <= win;
      const bool in_a = valid && (same || !split);
      const bool in_b = valid && !same && split;
      const unsigned ka = db | (local ? 0u : 0x80000000u);
      const int m = t0 + e;
      cnt_a += __popc(__ballot_sync(0xffffffffu, in_a));
      cnt_b += __popc(__ballot_sync(0xffffffffu, in_b));
      const unsigned mka = __ballot_sync(0xffffffffu, in_a && la.beats(ka, m));
      const unsigned mkb = __ballot_sync(0xffffffffu, in_b && lb.beats(db, m));
      if (mka) la.insert_chunk(t0 + c0, ka, mka, lane);
      if (mkb) lb.insert_chunk(t0 + c0, db, mkb, lane);
    }
  }
  if (!active) return;
  // quotas (oracle/knn_budget.py): the foreign quota first, the own chain gets the rest, leftovers go back
  int n_out = cnt_b < q_out ? cnt_b : q_out;
  const int n_in = cnt_a < k - n_out ? cnt_a : k - n_out;
  n_out = cnt_b < k - n_in ? cnt_b : k - n_in;
  int P = 32;
  while (P < k) P <<= 1;
  for (int e = lane; e < P; e += 32) { bk[e] = 0xffffffffu; bi[e] = 0x7fffffff; }
  __syncwarp();
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const int pos = lane * NR + r;
    if (pos < n_in) { bk[pos] = la.key[r] & 0x7fffffffu; bi[pos] = la.li[r]; }
    if (pos < n_out) { bk[n_in + pos] = lb.key[r]; bi[n_in + pos] = lb.li[r]; }
  }
  __syncwarp();
  for (int size = 2; size <= P; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = lane; i < (P >> 1); i += 32) {
        const int pos = 2 * i - (i & (stride - 1));
        const int par = pos + stride;
        const bool asc = (pos & size) == 0;
        const unsigned da = bk[pos], dbb = bk[par];
        const int ia = bi[pos], ib = bi[par];
        const bool a_after_b = da > dbb || (da == dbb && ia > ib);
        if (a_after_b == asc) { bk[pos] = dbb; bk[par] = da; bi[pos] = ib; bi[par] = ia; }
      }
      __syncwarp();
    }
  }
  for (int j = lane; j < k; j += 32) idx[(int64_t)l * k + j] = bi[j];
}

// ---- structured budget, threshold-select variant (k <= 256): the two classes keep candidate BUFFERS instead of sorted
// register lists.  A buffer starts unbounded; when it is about to overflow, the k-th smallest key it holds becomes the
// class's bound (exact bisection of the 32-bit key over the buffer, counted with ballots) and only the entries within it
// stay -- the own tile is visited first, so the bounds settle after a few such steps and the scan appends little.  After
// the scan the quotas are known; each class keeps the entries within its exact n-th key, sorts them by (key, index),
// and the chosen prefixes are sorted together by (d2, index).  More than kCap entries tying within a bound (coincident
// atoms) send the query to the register-list scan over global memory, which fills the same buffers.
template <int kPer>
__device__ __forceinline__ void buf_load(unsigned (&bv)[kPer], const unsigned* key, int n, int lane) {
#pragma unroll
  for (int j = 0; j < kPer; ++j) bv[j] = 32 * j + lane < n ? key[32 * j + lane] : 0xffffffffu;
}
// smallest key T <= hi0 with #{entries <= T} >= need (hi0 itself must satisfy it)
template <int kPer>
__device__ __forceinline__ unsigned buf_bisect(const unsigned (&bv)[kPer], unsigned hi0, int need) {
  unsigned lo = 0u, hi = hi0;
  while (lo < hi) {
    const unsigned mid = lo + ((hi - lo) >> 1);
    int c = 0;
#pragma unroll
    for (int j = 0; j < kPer; ++j) c += __popc(__ballot_sync(0xffffffffu, bv[j] <= mid));
    if (c >= need) hi = mid; else lo = mid + 1;
    if (c == need) break;                                      // exactly `need` entries are <= mid: the set is settled
  }
  return hi;
}
// keep the entries <= t, in order; returns the new count
template <int kPer>
__device__ __forceinline__ int buf_compact(const unsigned (&bv)[kPer], unsigned* key, int* id, unsigned t, int n, int lane) {
  int nc = 0;
#pragma unroll
  for (int j = 0; j < kPer; ++j) {
    if (32 * j >= n) break;                                    // warp-uniform
    const int e = 32 * j + lane;
    const int iv = e < n ? id[e] : 0;
    const bool pass = e < n && bv[j] <= t;
    const unsigned mask = __ballot_sync(0xffffffffu, pass);    // every lane has read chunk j before any lane overwrites it
    if (pass) { const int slot = nc + __popc(mask & ((1u << lane) - 1u)); key[slot] = bv[j]; id[slot] = iv; }
    nc += __popc(mask);
    __syncwarp();
  }
  return nc;
}
// bitonic sort of n entries by (key, index), padded to a power of two (the buffer has room for it)
__device__ __forceinline__ void buf_sort(unsigned* key, int* id, int n, int lane) {
  int P = 32;
  while (P < n) P <<= 1;
  for (int e = n + lane; e < P; e += 32) { key[e] = 0xffffffffu; id[e] = 0x7fffffff; }
  __syncwarp();
  for (int size = 2; size <= P; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = lane; i < (P >> 1); i += 32) {
        const int pos = 2 * i - (i & (stride - 1));
        const int par = pos + stride;
        const bool asc = (pos & size) == 0;
        const unsigned da = key[pos], dbb = key[par];
        const int ia = id[pos], ib = id[par];
        const bool a_after_b = da > dbb || (da == dbb && ia > ib);
        if (a_after_b == asc) { key[pos] = dbb; key[par] = da; id[pos] = ib; id[par] = ia; }
      }
      __syncwarp();
    }
  }
}

// exact fallback of one query: the two-list insertion scan over global memory; leaves each class's first min(k, size)
// entries, sorted, in its buffer
template <int NR>
__device__ __noinline__ void budget_insert_global(const float* __restrict__ x, const int32_t* __restrict__ rid,
                                                  const int32_t* __restrict__ cid, int L, int k, int l, int n_seq, int split,
                                                  int lane, unsigned* ak, int* ai, unsigned* bk, int* bi, int* na, int* nb) {
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  const int qr = __ldg(rid + l), qc = __ldg(cid + l), win = n_seq - 1;
  TopList<NR> la, lb;
  la.init(k);
  lb.init(k);
  int cnt_a = 0, cnt_b = 0;
  for (int c0 = 0; c0 < L; c0 += 32) {
    const int m = c0 + lane;
    const bool valid = m < L;
    const int mm = valid ? m : L - 1;
    const float a0 = __fsub_rn(__ldg(x + 3 * (int64_t)mm), q0), a1 = __fsub_rn(__ldg(x + 3 * (int64_t)mm + 1), q1);
    const float a2 = __fsub_rn(__ldg(x + 3 * (int64_t)mm + 2), q2);
    const unsigned db = __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2)));
    const bool same = __ldg(cid + mm) == qc;
    int dr = __ldg(rid + mm) - qr;
    dr = dr < 0 ? -dr : dr;
    const bool local = same && dr <= win;
    const bool in_a = valid && (same || !split), in_b = valid && !same && split;
    const unsigned ka = db | (local ? 0u : 0x80000000u);
    cnt_a += __popc(__ballot_sync(0xffffffffu, in_a));
    cnt_b += __popc(__ballot_sync(0xffffffffu, in_b));
    const unsigned mka = __ballot_sync(0xffffffffu, in_a && la.beats(ka, m));
    const unsigned mkb = __ballot_sync(0xffffffffu, in_b && lb.beats(db, m));
    if (mka) la.insert_chunk(c0, ka, mka, lane);
    if (mkb) lb.insert_chunk(c0, db, mkb, lane);
  }
  *na = cnt_a < k ? cnt_a : k;
  *nb = cnt_b < k ? cnt_b : k;
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const int pos = lane * NR + r;
    if (pos < *na) { ak[pos] = la.key[r]; ai[pos] = la.li[r]; }
    if (pos < *nb) { bk[pos] = lb.key[r]; bi[pos] = lb.li[r]; }
  }
  __syncwarp();
}

template <int kCap, int NRF>
__global__ void __launch_bounds__(256) knn_budget_select_kernel(const float* __restrict__ x, const int32_t* __restrict__ rid,
                                                                const int32_t* __restrict__ cid, int32_t* __restrict__ idx,
                                                                int L, int k, int n_seq, int split, int q_out) {
  extern __shared__ float smem_knn[];
  float* sx = smem_knn;
  float* sy = sx + kTile;
  float* sz = sy + kTile;
  int2* scr = reinterpret_cast<int2*>(sz + kTile);             // (chain id, residue id) per candidate: one 64-bit load
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  constexpr int kPer = kCap / 32;
  unsigned* ak = reinterpret_cast<unsigned*>(scr + kTile) + wib * (4 * kCap);   // per warp: class A keys, indices, class B keys, indices
  int* ai = reinterpret_cast<int*>(ak + kCap);
  unsigned* bk = ak + 2 * kCap;
  int* bi = reinterpret_cast<int*>(bk + kCap);
  // per tile: its 16 chunks of 128 atoms -- bounding box [lo xyz, hi xyz], chain-id range, residue-id range
  float* box = reinterpret_cast<float*>(scr + kTile) + 8 * (4 * kCap);
  int* meta = reinterpret_cast<int*>(box + 16 * 6);
  const int lq = blockIdx.x * 8 + wib;
  const bool active = lq < L;
  const int l = active ? lq : L - 1;
  const float q0 = __ldg(x + 3 * (int64_t)l), q1 = __ldg(x + 3 * (int64_t)l + 1), q2 = __ldg(x + 3 * (int64_t)l + 2);
  const int qr = __ldg(rid + l), qc = __ldg(cid + l), win = n_seq - 1;
  const unsigned lt_mask = (1u << lane) - 1u;
  unsigned thr_a = 0xffffffffu, thr_b = 0xffffffffu;           // the classes' bounds (keys <= bound are kept)
  int na = 0, nb = 0;                                          // buffer fill
  int cs = 0;                                                  // this lane's share of the own chain's size
  int cs_w = 0;                                                // ... and the part counted per chunk (warp-uniform)
  const bool has_win = win >= 0;                               // n_seq = 0: no atom is sequence-local
  const unsigned win2 = has_win ? 2u * (unsigned)win : 0u;
  bool over = false;
  // append the lanes' candidates (key v, atom m) of `mask` to a class buffer; re-bound the buffer when it would overflow
  // A class never contributes more than k entries; the foreign class B no more than max(q_out, k - |own chain|) (the
  // quota arithmetic at the end), and the part of the own chain counted so far bounds that from above: once the own tile
  // has shown k - q_out own atoms, B's bound is its q_out-th (32nd) key instead of its k-th -- a much shorter radius, so
  // most foreign chunks are skipped afterwards.
  auto append = [&](unsigned* key, int* id, int& n, unsigned& thr, unsigned mask, bool pass, unsigned v, int m, bool class_b) {
    if (over) return;
    if (n + __popc(mask) > kCap) {
      __syncwarp();
      int need = k;
      if (class_b) {
        const int own_lb = __reduce_add_sync(0xffffffffu, cs) + cs_w;        // own-chain atoms seen so far
        need = k - own_lb > q_out ? k - own_lb : q_out;
        need = need < k ? need : k;
      }
      unsigned bv[kPer];
      buf_load(bv, key, n, lane);
      thr = buf_bisect(bv, thr, need);                         // the buffer holds more than kCap - 32 >= k >= need entries
      n = buf_compact(bv, key, id, thr, n, lane);
      pass = pass && v <= thr;
      mask = __ballot_sync(0xffffffffu, pass);
      if (n + __popc(mask) > kCap) { over = true; return; }
    }
    if (pass) { const int slot = n + __popc(mask & lt_mask); key[slot] = v; id[slot] = m; }
    n += __popc(mask);
  };
  const int n_tiles = (L + kTile - 1) / kTile;
  const int own = (blockIdx.x * 8) / kTile;
  for (int tt = 0; tt < n_tiles; ++tt) {
    const int tile = tt == 0 ? own : (tt <= own ? tt - 1 : tt);
    const int t0 = tile * kTile;
    __syncthreads();
    for (int e = threadIdx.x; e < kTile; e += blockDim.x) {
      const int m = t0 + e;
      sx[e] = m < L ? __ldg(x + 3 * (int64_t)m) : 0.f;
      sy[e] = m < L ? __ldg(x + 3 * (int64_t)m + 1) : 0.f;
      sz[e] = m < L ? __ldg(x + 3 * (int64_t)m + 2) : 0.f;
      scr[e] = m < L ? make_int2(__ldg(cid + m), __ldg(rid + m)) : make_int2(-1, 0);
    }
    __syncthreads();
    const int n_here = (L - t0 < kTile ? L - t0 : kTile);
    {
      // chunk metadata: warp w takes chunks 2 w and 2 w + 1; an empty chunk gets an empty box and empty id ranges
#pragma unroll
      for (int cc = 0; cc < 2; ++cc) {
        const int ch = 2 * wib + cc;
        float lo0 = kInf, lo1 = kInf, lo2 = kInf, hi0 = -kInf, hi1 = -kInf, hi2 = -kInf;
        int cmin = 0x7fffffff, cmax = (int)0x80000000, rmin = 0x7fffffff, rmax = (int)0x80000000;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int e = ch * 128 + 32 * i + lane;
          if (e < n_here) {
            lo0 = fminf(lo0, sx[e]); hi0 = fmaxf(hi0, sx[e]);
            lo1 = fminf(lo1, sy[e]); hi1 = fmaxf(hi1, sy[e]);
            lo2 = fminf(lo2, sz[e]); hi2 = fmaxf(hi2, sz[e]);
            const int2 cr = scr[e];
            cmin = min(cmin, cr.x); cmax = max(cmax, cr.x);
            rmin = min(rmin, cr.y); rmax = max(rmax, cr.y);
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          lo0 = fminf(lo0, __shfl_xor_sync(0xffffffffu, lo0, o)); hi0 = fmaxf(hi0, __shfl_xor_sync(0xffffffffu, hi0, o));
          lo1 = fminf(lo1, __shfl_xor_sync(0xffffffffu, lo1, o)); hi1 = fmaxf(hi1, __shfl_xor_sync(0xffffffffu, hi1, o));
          lo2 = fminf(lo2, __shfl_xor_sync(0xffffffffu, lo2, o)); hi2 = fmaxf(hi2, __shfl_xor_sync(0xffffffffu, hi2, o));
        }
        cmin = __reduce_min_sync(0xffffffffu, cmin); cmax = __reduce_max_sync(0xffffffffu, cmax);
        rmin = __reduce_min_sync(0xffffffffu, rmin); rmax = __reduce_max_sync(0xffffffffu, rmax);
        if (lane == 0) {
          box[ch * 6] = lo0; box[ch * 6 + 1] = lo1; box[ch * 6 + 2] = lo2;
          box[ch * 6 + 3] = hi0; box[ch * 6 + 4] = hi1; box[ch * 6 + 5] = hi2;
          meta[ch * 4] = cmin; meta[ch * 4 + 1] = cmax; meta[ch * 4 + 2] = rmin; meta[ch * 4 + 3] = rmax;
        }
      }
      __syncthreads();
    }
    if (!active) continue;
    // Which chunks to scan (lane c < 16 decides for chunk c).  A chunk can be skipped when none of its atoms can enter a
    // buffer: no atom can be sequence-local (those pass whatever their distance) and the pinned distance arithmetic applied
    // to the query-to-box gaps -- a lower bound of every atom's computed d2, rounding being monotone -- exceeds both
    // classes' distance bounds.  The own chain's size is then counted per chunk: all of it, none of it, or (a chunk that
    // straddles chains) by a pass over the chain ids alone.
    // The own tile goes in two rounds: the four chunks around the query first, so that both bounds are tight before the
    // rest of the tile (and every other tile) is tested.
    unsigned home = 0xffffu;
    if (tt == 0) {
      int h0 = ((lq - t0) >> 7) - 2;
      h0 = h0 < 0 ? 0 : (h0 > 12 ? 12 : h0);
      home = 0xfu << h0;
    }
    for (int round = 0; round < (tt == 0 ? 2 : 1); ++round) {
    const unsigned allowed = round == 0 ? home : ~home;
    unsigned todo, count_only, pure_b;
    {
      bool scan_it = false, count_it = false, foreign = false;
      int whole = 0;
      if (lane < 16 && lane * 128 < n_here && ((allowed >> lane) & 1u)) {
        const float* bx = box + lane * 6;
        const float g0 = fmaxf(fmaxf(__fsub_rn(bx[0], q0), __fsub_rn(q0, bx[3])), 0.f);
        const float g1 = fmaxf(fmaxf(__fsub_rn(bx[1], q1), __fsub_rn(q1, bx[4])), 0.f);
        const float g2 = fmaxf(fmaxf(__fsub_rn(bx[2], q2), __fsub_rn(q2, bx[5])), 0.f);
        const unsigned lb = __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(g0, g0), __fmul_rn(g1, g1)), __fmul_rn(g2, g2)));
        const int cmin = meta[lane * 4], cmax = meta[lane * 4 + 1], rmin = meta[lane * 4 + 2], rmax = meta[lane * 4 + 3];
        const bool may_same = cmin <= qc && qc <= cmax, all_same = cmin == qc && cmax == qc;
        const bool may_local = may_same && has_win && (int64_t)rmin <= (int64_t)qr + win && (int64_t)rmax >= (int64_t)qr - win;
        const unsigned lim_a = thr_a & 0x7fffffffu, lim_b = split ? thr_b : 0u;
        // class A lives only in chunks that hold own-chain atoms (every chunk without a split), class B in the others
        scan_it = may_local || ((may_same || !split) && lb <= lim_a) || (split && !all_same && lb <= lim_b);
        count_it = !scan_it && may_same && !all_same;
        foreign = split && !may_same;                          // no own-chain atom in the chunk: every atom is class B
        const int n_ch = n_here - lane * 128 < 128 ? n_here - lane * 128 : 128;
        whole = (!scan_it && all_same) ? n_ch : 0;
      }
      todo = __ballot_sync(0xffffffffu, scan_it);
      count_only = __ballot_sync(0xffffffffu, count_it);
      pure_b = __ballot_sync(0xffffffffu, foreign);
      cs_w += __reduce_add_sync(0xffffffffu, whole);
    }
    while (count_only) {
      const int c0 = (__ffs(count_only) - 1) * 128;
      count_only &= count_only - 1;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int e = c0 + 32 * u + lane;
        cs += (e < n_here && scr[e].x == qc) ? 1 : 0;
      }
    }
    // four 32-candidate pieces per step: independent loads and arithmetic; only the last tile can be ragged
    auto scan = [&](auto RAGGED) {
      while (todo) {
        const int ch = __ffs(todo) - 1, c0 = ch * 128;
        todo &= todo - 1;
        if ((pure_b >> ch) & 1u) {
          // a chunk of foreign atoms only (most of them): distances and one compare, no ids, no class A
          unsigned dbf[4], mf[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int e = c0 + 32 * u + lane;
            const float a0 = __fsub_rn(sx[e], q0), a1 = __fsub_rn(sy[e], q1), a2 = __fsub_rn(sz[e], q2);
            dbf[u] = __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2)));
            mf[u] = __ballot_sync(0xffffffffu, dbf[u] <= thr_b && (!decltype(RAGGED)::value || e < n_here));
          }
          if ((mf[0] | mf[1] | mf[2] | mf[3]) == 0) continue;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (mf[u]) append(bk, bi, nb, thr_b, mf[u], (mf[u] >> lane) & 1u, dbf[u], t0 + c0 + 32 * u + lane, true);
          continue;
        }
        unsigned db[4], ka[4], ma[4], mb[4];
        bool pa[4], pb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int e = c0 + 32 * u + lane;                     // < kTile
          const float a0 = __fsub_rn(sx[e], q0), a1 = __fsub_rn(sy[e], q1), a2 = __fsub_rn(sz[e], q2);
          db[u] = __float_as_uint(__fadd_rn(__fadd_rn(__fmul_rn(a0, a0), __fmul_rn(a1, a1)), __fmul_rn(a2, a2)));
          const int2 cr = scr[e];
          const bool valid = !decltype(RAGGED)::value || e < n_here;
          const bool same = cr.x == qc && valid;
          const bool local = same && has_win && (unsigned)(cr.y - qr + win) <= win2;   // |residue - query's| <= win
          cs += same ? 1 : 0;
          ka[u] = local ? db[u] : (db[u] | 0x80000000u);
          pa[u] = valid && (same || !split) && ka[u] <= thr_a;
          pb[u] = valid && !same && split && db[u] <= thr_b;
          ma[u] = __ballot_sync(0xffffffffu, pa[u]);
          mb[u] = __ballot_sync(0xffffffffu, pb[u]);
        }
        if (((ma[0] | ma[1]) | (ma[2] | ma[3]) | (mb[0] | mb[1]) | (mb[2] | mb[3])) == 0) continue;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int m = t0 + c0 + 32 * u + lane;
          if (ma[u]) append(ak, ai, na, thr_a, ma[u], pa[u], ka[u], m, false);
          if (mb[u]) append(bk, bi, nb, thr_b, mb[u], pb[u], db[u], m, true);
        }
      }
    };
    if (n_here == kTile) scan(std::false_type{}); else scan(std::true_type{});
    }
  }
  if (!active) return;
  __syncwarp();
  // class sizes: the own chain's count; every atom without a split
  int n_same = cs;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_same += __shfl_xor_sync(0xffffffffu, n_same, o);
  n_same += cs_w;
  const int cnt_a = split ? n_same : L, cnt_b = split ? L - n_same : 0;
  if (over) budget_insert_global<NRF>(x, rid, cid, L, k, l, n_seq, split, lane, ak, ai, bk, bi, &na, &nb);
  // quotas (oracle/knn_budget.py): the foreign quota first, the own chain gets the rest, leftovers go back
  int n_out = cnt_b < q_out ? cnt_b : q_out;
  const int n_in = cnt_a < k - n_out ? cnt_a : k - n_out;
  n_out = cnt_b < k - n_in ? cnt_b : k - n_in;
  // each class: the entries within its exact n-th key, sorted by (key, index); the first n are the class's share
  if (n_in > 0) {
    unsigned bv[kPer];
    buf_load(bv, ak, na, lane);
    const unsigned t = buf_bisect(bv, thr_a, n_in);
    na = buf_compact(bv, ak, ai, t, na, lane);
    buf_sort(ak, ai, na, lane);
  }
  if (n_out > 0) {
    unsigned bv[kPer];
    buf_load(bv, bk, nb, lane);
    const unsigned t = buf_bisect(bv, thr_b, n_out);
    nb = buf_compact(bv, bk, bi, t, nb, lane);
    buf_sort(bk, bi, nb, lane);
  }
  // the two prefixes together, by (d2, index): class A loses its flag bit, class B follows it in A's buffer
  for (int j = lane; j < n_in; j += 32) ak[j] &= 0x7fffffffu;
  for (int j = lane; j < n_out; j += 32) { ak[n_in + j] = bk[j]; ai[n_in + j] = bi[j]; }
  __syncwarp();
  buf_sort(ak, ai, n_in + n_out, lane);
  for (int j = lane; j < k; j += 32) idx[(int64_t)l * k + j] = ai[j];
}

template <int kCap, int NRF>
cudaError_t launch_budget_select(const float* x, const int32_t* rid, const int32_t* cid, int32_t* idx, int L, int k, int n_seq,
                                 int split, int q_out, cudaStream_t st) {
  const size_t smem = (size_t)(5 * kTile + 8 * 4 * kCap + 16 * 10) * 4;
  cudaError_t e = cudaFuncSetAttribute(knn_budget_select_kernel<kCap, NRF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  knn_budget_select_kernel<kCap, NRF><<<(unsigned)((L + 7) / 8), 256, smem, st>>>(x, rid, cid, idx, L, k, n_seq, split, q_out);
  return cudaGetLastError();
}

template <int NR>
cudaError_t launch_budget(const float* x, const int32_t* rid, const int32_t* cid, int32_t* idx, int L, int k, int n_seq, int split,
                          int q_out, cudaStream_t st) {
  const size_t smem = (size_t)(5 * kTile + 8 * 2 * 512) * 4;
  cudaError_t e = cudaFuncSetAttribute(knn_budget_kernel<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  knn_budget_kernel<NR><<<(unsigned)((L + 7) / 8), 256, smem, st>>>(x, rid, cid, idx, L, k, n_seq, split, q_out);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_knn_budget(const float* x, const int32_t* rid, const int32_t* cid, int32_t* idx, int64_t L, int k, int n_seq,
                              int n_chains, cudaStream_t st) {
  const int split = n_chains > 3 ? 1 : 0;
  int q_out = k / 4 > 32 ? k / 4 : 32;
  if (q_out > k - 1) q_out = k - 1;
  const int nr = (k + 31) / 32;
  // threshold-select kernel (candidate buffers of >= 2 k entries per class); larger k: the register-list kernel
  if (k <= 128) return launch_budget_select<256, 4>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  if (k <= 256) return launch_budget_select<512, 8>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  if (nr <= 1) return launch_budget<1>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  if (nr <= 2) return launch_budget<2>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  if (nr <= 4) return launch_budget<4>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  if (nr <= 8) return launch_budget<8>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
  return launch_budget<16>(x, rid, cid, idx, (int)L, k, n_seq, split, q_out, st);
}

bool knn_supports(int64_t L, int k) { return L >= 1 && L <= 0x7fffffff && k >= 1 && k <= 512 && k <= L; }

cudaError_t launch_knn(const float* x, int32_t* idx, int64_t L, int k, cudaStream_t st) {
  const int nr = (k + 31) / 32;
  const unsigned blocks = (unsigned)((L + 7) / 8);
  // threshold-select kernel: shared tiles (24 KB) + 8 per-warp candidate buffers (8 bytes per entry)
  if (k <= 256) {
    const size_t smem = (size_t)(3 * kTile + 8 * 2 * 512 + 96) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(knn_select_kernel<512, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    knn_select_kernel<512, 8><<<blocks, 256, smem, st>>>(x, idx, (int)L, k);
    return cudaGetLastError();
  }
  {   // k <= 512: 1024-entry buffers (88 KB per CTA)
    const size_t smem = (size_t)(3 * kTile + 8 * 2 * 1024 + 96) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(knn_select_kernel<1024, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    knn_select_kernel<1024, 16><<<blocks, 256, smem, st>>>(x, idx, (int)L, k);
    return cudaGetLastError();
  }
}

}  // namespace dcp
