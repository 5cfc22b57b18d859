// libdesigncp C ABI (include/designcp.h): validation, the Eq.-5 planner, workspace carving and the
// launch sequence  prologue (a1) -> fused kernel per sub-problem (a2-a7) -> merge + gate (a8) -> W_o (a9).
// Decomposition emulation (PAPER.md:72-86 row stripes, :90 grid): one fused launch per stripe / quadrant on a
// strided view of z (a base-pointer offset, no copy), partial states merged left to right by one kernel.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "kernels.h"

namespace dcp {
namespace {

thread_local int g_launches = 0;

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Programmatic dependent launch between the kernels of a call (common.cuh) is on unless DCP_PDL=0 is set in the
// environment (a debugging / A-B timing switch, read once).
bool pdl_enabled() {
  static const bool on = [] { const char* e = getenv("DCP_PDL"); return !(e && e[0] == '0'); }();
  return on;
}
inline int elt_size(dcp_dtype dt) { return dt == DCP_F32 ? 4 : 2; }

struct Carve {
  size_t q, k, v, g, gated, s_ln, wg, c0, wfold, c1, st_m, st_l, st_acc, total;
};

Carve carve(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dt, int slots) {
  Carve w{};
  const size_t D = (size_t)H * c, e = elt_size(dt);
  // the tensor-core path keeps q, k zero-padded per head ([I][H][cp]) and v transposed ([D][ldv])
  const size_t Dp = (size_t)H * mma_head_pad(c), frag = (size_t)mma_frag_elems(I, H, c);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  w.q = take((size_t)I * Dp * e);
  w.k = take(std::max((size_t)I * Dp, frag) * e);
  w.v = take(std::max((size_t)I * D, frag) * e);
  w.g = take((size_t)I * D * e);
  w.gated = take((size_t)I * D * e);
  w.s_ln = take((size_t)I * c_s * sizeof(float));
  w.wg = take((size_t)c_z * H * sizeof(float));
  w.c0 = take(32 * sizeof(float));
  w.wfold = take((size_t)32 * c_z * 2);
  w.c1 = take(32 * sizeof(float));
  w.st_m = take((size_t)slots * I * H * sizeof(float));
  w.st_l = take((size_t)slots * I * H * sizeof(float));
  w.st_acc = take((size_t)slots * I * D * sizeof(float));
  w.total = off;
  return w;
}

int isqrt_exact(int p) {
  int g = 0;
  while ((int64_t)(g + 1) * (g + 1) <= p) ++g;
  return (g * g == p) ? g : -1;
}

struct Plan {
  dcp_decomp decomp;
  int parts, key_split, slots, G, kernel;
  bool use_mma;   // bf16 tensor-core path (fused_mma.cu) instead of the generic fp32 CUDA-core kernel
  int nseg;       // tensor-core path: Eq.-5 segments per key chunk (a pure function of I and the chunk count)
  int tile_h;     // tensor-core path: query rows per work unit
  cudaEvent_t ev_begin, ev_end;
};

dcp_status make_plan(int64_t I, int H, int c, int c_z, dcp_dtype dt, dcp_decomp decomp, const dcp_plan* in, Plan* out) {
  Plan p{};
  p.decomp = decomp;
  p.parts = in ? in->parts : 1;
  p.key_split = (in && in->key_split > 0) ? in->key_split : 1;
  p.kernel = in ? in->kernel : DCP_KERNEL_AUTO;
  p.ev_begin = in ? (cudaEvent_t)in->ev_fused_begin : nullptr;
  p.ev_end = in ? (cudaEvent_t)in->ev_fused_end : nullptr;
  p.G = 1;
  if (p.kernel < DCP_KERNEL_AUTO || p.kernel > DCP_KERNEL_MMA) return DCP_ERR_INVALID_ARG;
  switch (decomp) {
    case DCP_MONOLITHIC:
      p.parts = 1;
      break;
    case DCP_ROW:
      if (p.parts < 1 || p.parts > I) return DCP_ERR_INVALID_ARG;
      break;
    case DCP_GRID:
      // "this 2D grid scheme applies only when the available GPU count P is a perfect square"
      if (p.parts < 1) return DCP_ERR_INVALID_ARG;
      p.G = isqrt_exact(p.parts);
      if (p.G < 1 || p.G > I) return DCP_ERR_INVALID_ARG;
      p.key_split = p.G;
      break;
    default:
      return DCP_ERR_INVALID_ARG;
  }
  if (p.key_split > I) return DCP_ERR_INVALID_ARG;
  const bool mma_ok = fused_mma_supports(dt, H, c, c_z);
  if (p.kernel == DCP_KERNEL_MMA && !mma_ok) return DCP_ERR_UNSUPPORTED;
  if (p.kernel == DCP_KERNEL_GENERIC && !fused_generic_supports(dt, H, c, c_z)) return DCP_ERR_UNSUPPORTED;
  p.use_mma = mma_ok && p.kernel != DCP_KERNEL_GENERIC;
  if (in && (in->tile_q < 0 || in->tile_k < 0 || in->key_segments < 0 || in->key_segments > 64)) return DCP_ERR_INVALID_ARG;
  if (in && (in->tile_q || in->tile_k)) {
    // one tiling per kernel: a non-zero request must name it (include/designcp.h)
    int tq, tk;
    if (p.use_mma) { tq = H == 16 ? 32 : fused_atom_tile_q(); tk = H == 16 ? 16 : 32; }
    else { tq = 8; tk = 32; }
    // fused_mma_kernel takes any query-tile height 25..32 (a trimmed last TMA box); the others have one tiling
    const bool tq_ok = in->tile_q == 0 || in->tile_q == tq || (p.use_mma && H == 16 && in->tile_q >= 25 && in->tile_q <= 32);
    if (!tq_ok || (in->tile_k && in->tile_k != tk)) return DCP_ERR_UNSUPPORTED;
  }
  p.nseg = 1;
  p.tile_h = 0;
  if (p.use_mma) {
    int force_s = 0;
    if (in && in->key_segments > 0) {
      // never more segments than whole key tiles in the smallest chunk: every segment keeps at least one key
      const int64_t tile_k = H == 16 ? 16 : 32;
      force_s = (int)std::min<int64_t>(in->key_segments, std::max<int64_t>(1, (I / p.key_split) / tile_k));
    }
    const int n_qparts = decomp == DCP_GRID ? p.G : p.parts;
    mma_pick_units(I, H, n_qparts, p.key_split, force_s, (in && H == 16) ? in->tile_q : 0, &p.nseg, &p.tile_h);
  }
  p.slots = p.key_split * p.nseg;
  *out = p;
  return DCP_OK;
}

dcp_status check_shape(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dt) {
  if (I <= 0 || c_s <= 0 || H <= 0 || c <= 0 || c_z <= 0) return DCP_ERR_INVALID_ARG;
  if (dt != DCP_F32 && dt != DCP_BF16) return DCP_ERR_INVALID_ARG;
  if (I > (int64_t)1 << 30) return DCP_ERR_INVALID_ARG;
  if ((c_z * elt_size(dt)) % 16 != 0) return DCP_ERR_INVALID_ARG;
  if (!fused_generic_supports(dt, H, c, c_z) && !fused_mma_supports(dt, H, c, c_z)) return DCP_ERR_UNSUPPORTED;
  // the tensor-core path's GEMMs move 16-byte row pieces of s, the projections and out
  if (fused_mma_supports(dt, H, c, c_z) && c_s % 8 != 0) return DCP_ERR_UNSUPPORTED;
  return DCP_OK;
}

inline bool misaligned(const void* p, size_t a = 16) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

#define DCP_CUDA(expr)                         \
  do {                                         \
    cudaError_t _e = (expr);                   \
    if (_e != cudaSuccess) return DCP_ERR_CUDA; \
    ++g_launches;                              \
  } while (0)

struct Ctx {
  int64_t I;
  int c_s, H, c, c_z, D;
  dcp_dtype dt;
  const dcp_weights* w;
  float eps;
  char* ws;
  Carve cv;
  cudaStream_t st;
  bool use_mma;
};

// a1: (optional LN_s) + q, k, v, g projections for ALL rows (keys/values come from the full S),
// plus the folded LayerNorm(z) affine.
dcp_status run_prologue(const Ctx& x, const void* s) {
  const void* a = s;
  bool a_f32 = false;
  if (x.w->ln_s_gamma != nullptr) {
    DCP_CUDA(launch_layernorm_rows(x.dt, s, x.w->ln_s_gamma, x.w->ln_s_beta, (float*)(x.ws + x.cv.s_ln), x.I, x.c_s,
                                   x.eps, x.st));
    a = x.ws + x.cv.s_ln;
    a_f32 = x.dt != DCP_F32;
  }
  DCP_CUDA(launch_gemm(x.dt, a_f32, a, x.c_s, x.w->w_q, x.w->b_q, x.ws + x.cv.q, x.D, x.I, x.D, x.c_s, EPI_NONE, x.st));
  DCP_CUDA(launch_gemm(x.dt, a_f32, a, x.c_s, x.w->w_k, nullptr, x.ws + x.cv.k, x.D, x.I, x.D, x.c_s, EPI_NONE, x.st));
  DCP_CUDA(launch_gemm(x.dt, a_f32, a, x.c_s, x.w->w_v, nullptr, x.ws + x.cv.v, x.D, x.I, x.D, x.c_s, EPI_NONE, x.st));
  DCP_CUDA(launch_gemm(x.dt, a_f32, a, x.c_s, x.w->w_g, nullptr, x.ws + x.cv.g, x.D, x.I, x.D, x.c_s, EPI_SIGMOID, x.st));
  DCP_CUDA(launch_fold_ln_z(x.dt, x.w->w_b, x.w->ln_z_gamma, x.w->ln_z_beta, (float*)(x.ws + x.cv.wg),
                            (float*)(x.ws + x.cv.c0), x.c_z, x.H, x.st));
  return DCP_OK;
}

FusedParams base_params(const Ctx& x, const void* z, int64_t ldz) {
  FusedParams p{};
  p.z = z;
  p.ldz = ldz;
  p.q = x.ws + x.cv.q;
  p.k = x.ws + x.cv.k;
  p.v = x.ws + x.cv.v;
  p.wg = (const float*)(x.ws + x.cv.wg);
  p.c0 = (const float*)(x.ws + x.cv.c0);
  p.I = (int)x.I;
  p.c_z = x.c_z;
  p.H = x.H;
  p.c = x.c;
  p.D = x.D;
  p.eps = x.eps;
  p.scale = 1.0f / sqrtf((float)x.c);
  return p;
}

// a1 on tensor cores (bf16 path): one GEMM launch for q, k, v, g in the layouts the fused MMA kernel reads.
dcp_status run_prologue_mma(const Ctx& x, const void* s) {
  const void* a = s;
  if (x.w->ln_s_gamma != nullptr) {
    DCP_CUDA(launch_layernorm_rows_bf16(s, x.w->ln_s_gamma, x.w->ln_s_beta, x.ws + x.cv.s_ln, x.I, x.c_s, x.eps, x.st));
    a = x.ws + x.cv.s_ln;
  }
  const int cp = mma_head_pad(x.c);
  const size_t frag = (size_t)mma_frag_elems(x.I, x.H, x.c);
  if (cp != x.c) {   // zero the per-head padding of q
    if (cudaMemsetAsync(x.ws + x.cv.q, 0, (size_t)x.I * x.H * cp * 2, x.st) != cudaSuccess) return DCP_ERR_CUDA;
  }
  if (cp != x.c) {   // zero the head-dim padding of the K / V fragments (keys beyond I are zero-filled by the GEMM)
    if (cudaMemsetAsync(x.ws + x.cv.k, 0, frag * 2, x.st) != cudaSuccess) return DCP_ERR_CUDA;
    if (cudaMemsetAsync(x.ws + x.cv.v, 0, frag * 2, x.st) != cudaSuccess) return DCP_ERR_CUDA;
  }
  GemmMmaParams gp{};
  gp.A = a; gp.lda = x.c_s; gp.M = x.I; gp.N = x.D; gp.K = x.c_s; gp.nseg = 4;
  gp.W[0] = x.w->w_q; gp.W[1] = x.w->w_k; gp.W[2] = x.w->w_v; gp.W[3] = x.w->w_g;
  gp.bias[0] = x.w->b_q;
  gp.C[0] = x.ws + x.cv.q; gp.C[1] = x.ws + x.cv.k; gp.C[2] = x.ws + x.cv.v; gp.C[3] = x.ws + x.cv.g;
  gp.mode[0] = GEMM_OUT_HEADPAD; gp.mode[1] = GEMM_OUT_KFRAG; gp.mode[2] = GEMM_OUT_VFRAG; gp.mode[3] = GEMM_OUT_SIGMOID;
  gp.scale[0] = 1.4426950408889634f / sqrtf((float)x.c);   // log2(e)/sqrt(c): the softmax runs in the exp2 domain
  gp.scale[1] = 1.f;
  gp.ldc[3] = x.D;
  gp.H = x.H; gp.c = x.c; gp.cp = cp;
  gp.fold_w_b = x.w->w_b; gp.fold_gamma = x.w->ln_z_gamma; gp.fold_beta = x.w->ln_z_beta;
  gp.fold_wfold = x.ws + x.cv.wfold; gp.fold_c1 = (float*)(x.ws + x.cv.c1); gp.fold_c0 = (float*)(x.ws + x.cv.c0);
  gp.fold_c_z = x.c_z; gp.fold_H = x.H; gp.fold_H_pad = 16;
  gp.pdl = pdl_enabled();   // programmatic dependent of whatever kernel precedes the call in the stream (common.cuh)
  bool folded = false;
  DCP_CUDA(launch_gemm_mma(gp, x.st, &folded));
  if (!folded)
    DCP_CUDA(launch_fold_ln_z_mma(x.w->w_b, x.w->ln_z_gamma, x.w->ln_z_beta, x.ws + x.cv.wfold, (float*)(x.ws + x.cv.c1),
                                  (float*)(x.ws + x.cv.c0), x.c_z, x.H, 16, x.st));
  return DCP_OK;
}

MmaParams base_params_mma(const Ctx& x) {
  MmaParams p{};
  p.qp = x.ws + x.cv.q;
  p.kfr = x.ws + x.cv.k;
  p.vfr = x.ws + x.cv.v;
  p.wfold = x.ws + x.cv.wfold;
  p.c1 = (const float*)(x.ws + x.cv.c1);
  p.c0 = (const float*)(x.ws + x.cv.c0);
  p.I = (int)x.I;
  p.H = x.H;
  p.c = x.c;
  p.c_z = x.c_z;
  p.eps = x.eps;
  return p;
}

dcp_status run_fused(const Ctx& x, const FusedParams& p) {
  DCP_CUDA(launch_fused_generic(x.dt, p, x.st));
  return DCP_OK;
}

dcp_status validate_weights(const dcp_weights* w) {
  if (!w || !w->w_q || !w->w_k || !w->w_v || !w->w_g || !w->w_b || !w->w_o || !w->ln_z_gamma || !w->ln_z_beta)
    return DCP_ERR_INVALID_ARG;
  if ((w->ln_s_gamma == nullptr) != (w->ln_s_beta == nullptr)) return DCP_ERR_INVALID_ARG;
  return DCP_OK;
}

dcp_status layer(const void* s, const void* z, int64_t ldz, const dcp_weights* w, void* out, int64_t I, int c_s, int H,
                 int c, int c_z, dcp_dtype dt, dcp_decomp decomp, const dcp_plan* plan_in, void* workspace,
                 size_t workspace_bytes, void* stream, const void* residual = nullptr, const uint32_t* bias_cache = nullptr) {
  // bias_cache != nullptr: this block's bias tiles (bias_tiles.cu) replace the LayerNorm + projection of z (token kernel,
  // MONOLITHIC, 32-row tiles)
  // residual != nullptr: out = storage(residual + layer output), added in fp32 inside the W_o GEMM's epilogue (tensor-core
  // path with a tcgen05-shaped W_o only: DCP_ERR_UNSUPPORTED otherwise); residual may be `out`
  g_launches = 0;
  if (!s || !z || !out || !workspace) return DCP_ERR_INVALID_ARG;
  dcp_status st = validate_weights(w);
  if (st != DCP_OK) return st;
  st = check_shape(I, c_s, H, c, c_z, dt);
  if (st != DCP_OK) return st;
  Plan plan;
  st = make_plan(I, H, c, c_z, dt, decomp, plan_in, &plan);
  if (st != DCP_OK) return st;
  const int e = elt_size(dt);
  if (ldz == 0) ldz = I * (int64_t)c_z;
  if (ldz < I * (int64_t)c_z) return DCP_ERR_INVALID_ARG;
  if (misaligned(s) || misaligned(z) || misaligned(out) || misaligned(workspace, 256) || (ldz * e) % 16 != 0)
    return DCP_ERR_INVALID_ARG;
  Ctx x{};
  x.I = I; x.c_s = c_s; x.H = H; x.c = c; x.c_z = c_z; x.D = H * c; x.dt = dt; x.w = w;
  x.eps = w->ln_eps > 0.f ? w->ln_eps : 1e-5f;
  x.ws = (char*)workspace;
  x.cv = carve(I, c_s, H, c, c_z, dt, plan.slots);
  x.st = (cudaStream_t)stream;
  if (workspace_bytes < x.cv.total) return DCP_ERR_WORKSPACE;

  float* st_m = (float*)(x.ws + x.cv.st_m);
  float* st_l = (float*)(x.ws + x.cv.st_l);
  float* st_acc = (float*)(x.ws + x.cv.st_acc);

  if (plan.use_mma) {
    st = run_prologue_mma(x, s);
    if (st != DCP_OK) return st;
    // ONE persistent launch over every (stripe | grid row block, 32-query tile, key chunk, segment) unit; each unit
    // reads only its own block of z and writes its own partial state (no cross-unit communication).
    MmaParams mp = base_params_mma(x);
    mp.st_m = st_m; mp.st_l = st_l; mp.st_acc = st_acc;
    mp.state_rows = I; mp.state_row0 = 0;
    mp.q_begin = 0; mp.q_end = (int)I; mp.n_qparts = plan.decomp == DCP_GRID ? plan.G : plan.parts;
    mp.k_begin = 0; mp.k_end = (int)I; mp.n_kparts = plan.key_split;
    mp.nseg = plan.nseg; mp.slot0 = 0; mp.tile_h = plan.tile_h;
    mp.bias_cache = bias_cache;
    mp.pdl = pdl_enabled() && plan.ev_begin == nullptr;   // an event record between two launches would serialise them anyway
    if (plan.ev_begin && cudaEventRecord(plan.ev_begin, x.st) != cudaSuccess) return DCP_ERR_CUDA;
    DCP_CUDA(launch_fused_mma(mp, z, ldz, x.st));
  } else {
  if (bias_cache != nullptr) return DCP_ERR_UNSUPPORTED;
  st = run_prologue(x, s);
  if (st != DCP_OK) return st;

  FusedParams bp = base_params(x, z, ldz);
  bp.st_m = st_m;
  bp.st_l = st_l;
  bp.st_acc = st_acc;
  bp.state_rows = I;
  bp.state_row0 = 0;

  if (plan.ev_begin && cudaEventRecord(plan.ev_begin, x.st) != cudaSuccess) return DCP_ERR_CUDA;
  if (plan.decomp == DCP_GRID) {
    // quadrant (r, cb): rows of block r against keys of block cb, bias from Z^(r,cb) only; slot = cb
    for (int r = 0; r < plan.G; ++r) {
      for (int cb = 0; cb < plan.G; ++cb) {
        FusedParams p = bp;
        int64_t len;
        shard_range(I, plan.G, r, &p.q0, &len);
        p.q1 = p.q0 + len;
        shard_range(I, plan.G, cb, &p.k0, &len);
        p.k1 = p.k0 + len;
        p.n_chunks = 1;
        p.slot0 = cb;
        st = run_fused(x, p);
        if (st != DCP_OK) return st;
      }
    }
  } else {
    // stripe p: its query rows against ALL keys (cross-attention); MONOLITHIC is one stripe
    for (int sp = 0; sp < plan.parts; ++sp) {
      FusedParams p = bp;
      int64_t len;
      shard_range(I, plan.parts, sp, &p.q0, &len);
      p.q1 = p.q0 + len;
      p.k0 = 0;
      p.k1 = I;
      p.n_chunks = plan.key_split;
      p.slot0 = 0;
      st = run_fused(x, p);
      if (st != DCP_OK) return st;
    }
  }
  }

  if (plan.ev_end && cudaEventRecord(plan.ev_end, x.st) != cudaSuccess) return DCP_ERR_CUDA;

  MergeParams mp{};
  mp.st_m = st_m; mp.st_l = st_l; mp.st_acc = st_acc;
  mp.g = x.ws + x.cv.g;
  mp.gated = x.ws + x.cv.gated;
  mp.rows = I; mp.n_slots = plan.slots; mp.H = H; mp.c = c; mp.D = x.D;
  mp.pdl = pdl_enabled() && plan.use_mma && plan.ev_end == nullptr;
  DCP_CUDA(launch_merge(dt, mp, x.st));
  if (plan.use_mma) {
    GemmMmaParams gp{};
    gp.A = x.ws + x.cv.gated; gp.lda = x.D; gp.M = I; gp.N = c_s; gp.K = x.D; gp.nseg = 1;
    gp.W[0] = w->w_o; gp.C[0] = out; gp.mode[0] = GEMM_OUT_PLAIN; gp.ldc[0] = c_s;
    gp.pdl = pdl_enabled();
    if (residual != nullptr) {
      gp.residual = residual; gp.ldr = c_s;
      if (!gemm_tc_supports(gp)) return DCP_ERR_UNSUPPORTED;
    }
    DCP_CUDA(launch_gemm_mma(gp, x.st));
  } else {
    if (residual != nullptr) return DCP_ERR_UNSUPPORTED;
    DCP_CUDA(launch_gemm(dt, false, x.ws + x.cv.gated, x.D, w->w_o, nullptr, out, c_s, I, c_s, x.D, EPI_NONE, x.st));
  }
  return DCP_OK;
}

}  // namespace
}  // namespace dcp

using namespace dcp;

extern "C" {

dcp_status dcp_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, dcp_decomp decomp,
                               const dcp_plan* plan_in, size_t* bytes) {
  if (!bytes) return DCP_ERR_INVALID_ARG;
  dcp_status st = check_shape(I, c_s, H, c, c_z, dtype);
  if (st != DCP_OK) return st;
  Plan plan;
  st = make_plan(I, H, c, c_z, dtype, decomp, plan_in, &plan);
  if (st != DCP_OK) return st;
  *bytes = carve(I, c_s, H, c, c_z, dtype, plan.slots).total;
  return DCP_OK;
}

dcp_status dcp_pair_bias_attention(const void* s, const void* z, int64_t ldz, const dcp_weights* w, void* out, int64_t I,
                                   int c_s, int H, int c, int c_z, dcp_dtype dtype, dcp_decomp decomp,
                                   const dcp_plan* plan, void* workspace, size_t workspace_bytes, void* stream) {
  return layer(s, z, ldz, w, out, I, c_s, H, c, c_z, dtype, decomp, plan, workspace, workspace_bytes, stream);
}

dcp_status dcp_atom_pair_bias_attention(const void* a, const void* p, int64_t ldp, const dcp_weights* w, void* out,
                                        int64_t L, int c_atom, int H, int c, int c_atompair, dcp_dtype dtype,
                                        dcp_decomp decomp, const dcp_plan* plan, void* workspace,
                                        size_t workspace_bytes, void* stream) {
  return layer(a, p, ldp, w, out, L, c_atom, H, c, c_atompair, dtype, decomp, plan, workspace, workspace_bytes, stream);
}

// ---- sparse k-neighbour atom attention
namespace {
struct SparseCarve { size_t q, k, v, g, gated, s_ln, wfold, c1, c0, total; };
SparseCarve sparse_carve(int64_t L, int c_atom, int H, int c) {
  SparseCarve w{};
  const size_t D = (size_t)H * c;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  w.q = take((size_t)L * D * 2); w.k = take((size_t)L * D * 2); w.v = take((size_t)L * D * 2);
  w.g = take((size_t)L * D * 2); w.gated = take((size_t)L * D * 2);
  w.s_ln = take((size_t)L * c_atom * 2);
  w.wfold = take(16 * 16 * 2); w.c1 = take(16 * sizeof(float)); w.c0 = take(16 * sizeof(float));
  w.total = off;
  return w;
}
}  // namespace

dcp_status dcp_sparse_atom_workspace_bytes(int64_t L, int c_atom, int H, int c, dcp_dtype dtype, size_t* bytes) {
  if (!bytes || L <= 0 || c_atom <= 0 || H <= 0 || c <= 0) return DCP_ERR_INVALID_ARG;
  if (dtype != DCP_BF16) return DCP_ERR_UNSUPPORTED;
  *bytes = sparse_carve(L, c_atom, H, c).total;
  return DCP_OK;
}

dcp_status dcp_sparse_atom_attention(const void* a, const void* p_slice, const int32_t* idx, const dcp_weights* w,
                                     void* out, int64_t L, int k, int c_atom, int H, int c, int c_atompair,
                                     dcp_dtype dtype, const dcp_plan* plan, void* workspace, size_t workspace_bytes,
                                     void* stream) {
  g_launches = 0;
  if (!a || !p_slice || !idx || !out || !workspace) return DCP_ERR_INVALID_ARG;
  if (!w || !w->w_q || !w->w_k || !w->w_v || !w->w_g || !w->w_b || !w->w_o || !w->ln_z_gamma || !w->ln_z_beta)
    return DCP_ERR_INVALID_ARG;
  if ((w->ln_s_gamma == nullptr) != (w->ln_s_beta == nullptr)) return DCP_ERR_INVALID_ARG;
  if (L <= 0 || k <= 0 || c_atom <= 0 || H <= 0 || c <= 0 || c_atompair <= 0 || L > 0x7fffffff) return DCP_ERR_INVALID_ARG;
  if (dtype != DCP_BF16 || !sparse_atom_supports(dtype, H, c, c_atompair, k) || c_atom % 8 != 0) return DCP_ERR_UNSUPPORTED;
  if ((((uintptr_t)a | (uintptr_t)p_slice | (uintptr_t)out | (uintptr_t)workspace) & 15) != 0) return DCP_ERR_INVALID_ARG;
  const SparseCarve cv = sparse_carve(L, c_atom, H, c);
  if (workspace_bytes < cv.total) return DCP_ERR_WORKSPACE;
  char* ws = (char*)workspace;
  cudaStream_t st = (cudaStream_t)stream;
  const float eps = w->ln_eps > 0.f ? w->ln_eps : 1e-5f;
  const int D = H * c;
  const void* x = a;
  if (w->ln_s_gamma != nullptr) {
    DCP_CUDA(launch_layernorm_rows_bf16(a, w->ln_s_gamma, w->ln_s_beta, ws + cv.s_ln, L, c_atom, eps, st));
    x = ws + cv.s_ln;
  }
  GemmMmaParams gp{};
  gp.A = x; gp.lda = c_atom; gp.M = L; gp.N = D; gp.K = c_atom; gp.nseg = 4;
  gp.W[0] = w->w_q; gp.W[1] = w->w_k; gp.W[2] = w->w_v; gp.W[3] = w->w_g;
  gp.bias[0] = w->b_q;
  gp.C[0] = ws + cv.q; gp.C[1] = ws + cv.k; gp.C[2] = ws + cv.v; gp.C[3] = ws + cv.g;
  gp.mode[0] = GEMM_OUT_HEADPAD; gp.mode[1] = GEMM_OUT_PLAIN; gp.mode[2] = GEMM_OUT_PLAIN; gp.mode[3] = GEMM_OUT_SIGMOID;
  gp.scale[0] = 1.4426950408889634f / sqrtf((float)c);   // exp2-domain softmax
  gp.ldc[1] = D; gp.ldc[2] = D; gp.ldc[3] = D;
  gp.H = H; gp.c = c; gp.cp = c;
  gp.fold_w_b = w->w_b; gp.fold_gamma = w->ln_z_gamma; gp.fold_beta = w->ln_z_beta;
  gp.fold_wfold = ws + cv.wfold; gp.fold_c1 = (float*)(ws + cv.c1); gp.fold_c0 = (float*)(ws + cv.c0);
  gp.fold_c_z = c_atompair; gp.fold_H = H; gp.fold_H_pad = 16;
  bool folded = false;
  DCP_CUDA(launch_gemm_mma(gp, st, &folded));
  if (!folded)
    DCP_CUDA(launch_fold_ln_z_mma(w->w_b, w->ln_z_gamma, w->ln_z_beta, ws + cv.wfold, (float*)(ws + cv.c1),
                                  (float*)(ws + cv.c0), c_atompair, H, 16, st));
  if (plan && plan->ev_fused_begin && cudaEventRecord((cudaEvent_t)plan->ev_fused_begin, st) != cudaSuccess) return DCP_ERR_CUDA;
  DCP_CUDA(launch_sparse_atom(ws + cv.q, ws + cv.k, ws + cv.v, ws + cv.g, p_slice, idx, ws + cv.wfold,
                              (const float*)(ws + cv.c1), (const float*)(ws + cv.c0), ws + cv.gated, L, k, H, eps, st));
  if (plan && plan->ev_fused_end && cudaEventRecord((cudaEvent_t)plan->ev_fused_end, st) != cudaSuccess) return DCP_ERR_CUDA;
  GemmMmaParams go{};
  go.A = ws + cv.gated; go.lda = D; go.M = L; go.N = c_atom; go.K = D; go.nseg = 1;
  go.W[0] = w->w_o; go.C[0] = out; go.mode[0] = GEMM_OUT_PLAIN; go.ldc[0] = c_atom;
  DCP_CUDA(launch_gemm_mma(go, st));
  return DCP_OK;
}

dcp_status dcp_gather_pair_slice(const void* p, int64_t ldp, const int32_t* idx, void* p_slice, int64_t L, int k,
                                 int c_atompair, dcp_dtype dtype, void* stream) {
  g_launches = 0;
  if (!p || !idx || !p_slice || L <= 0 || k <= 0 || c_atompair <= 0 || L > 0x7fffffff) return DCP_ERR_INVALID_ARG;
  if (dtype != DCP_F32 && dtype != DCP_BF16) return DCP_ERR_INVALID_ARG;
  const int64_t e = elt_size(dtype);
  if (ldp == 0) ldp = L * (int64_t)c_atompair;
  if ((c_atompair * e) % 16 != 0 || (ldp * e) % 16 != 0 || (((uintptr_t)p | (uintptr_t)p_slice) & 15) != 0)
    return DCP_ERR_INVALID_ARG;
  DCP_CUDA(launch_gather_pair_slice(p, ldp * e, idx, p_slice, L, k, (int)(c_atompair * e), (cudaStream_t)stream));
  return DCP_OK;
}

dcp_status dcp_pair_transition_workspace_bytes(int c_z, dcp_dtype dtype, size_t* bytes) {
  if (!bytes || c_z <= 0) return DCP_ERR_INVALID_ARG;
  if (!pair_transition_supports(dtype, c_z)) return DCP_ERR_UNSUPPORTED;
  *bytes = align_up(pair_transition_workspace_bytes());
  return DCP_OK;
}

dcp_status dcp_pair_transition(const void* z, void* z_out, int64_t n_pairs, int c_z, const void* w1, const void* w2,
                               const void* w3, const void* ln_gamma, const void* ln_beta, float ln_eps, dcp_dtype dtype,
                               void* workspace, size_t workspace_bytes, void* stream) {
  g_launches = 0;
  if (!z || !z_out || !w1 || !w2 || !w3 || !ln_gamma || !ln_beta || !workspace || n_pairs <= 0 || c_z <= 0)
    return DCP_ERR_INVALID_ARG;
  if (!pair_transition_supports(dtype, c_z)) return DCP_ERR_UNSUPPORTED;
  if (n_pairs > 0x7fffff00ll) return DCP_ERR_INVALID_ARG;
  if ((((uintptr_t)z | (uintptr_t)z_out | (uintptr_t)w1 | (uintptr_t)w2 | (uintptr_t)w3 | (uintptr_t)workspace) & 15) != 0)
    return DCP_ERR_INVALID_ARG;
  if (workspace_bytes < pair_transition_workspace_bytes()) return DCP_ERR_WORKSPACE;
  DCP_CUDA(launch_pair_transition(z, z_out, n_pairs, w1, w2, w3, ln_gamma, ln_beta, ln_eps > 0.f ? ln_eps : 1e-5f, workspace,
                                  (cudaStream_t)stream));
  ++g_launches;   // the weight-fold launch
  return DCP_OK;
}

// s <- bf16(s + o), eight elements per thread
static __global__ void __launch_bounds__(256) residual_add_bf16_kernel(__nv_bfloat16* __restrict__ s, const __nv_bfloat16* __restrict__ o,
                                                                int64_t n8) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n8) return;
  uint4 a = reinterpret_cast<const uint4*>(s)[i];
  const uint4 b = reinterpret_cast<const uint4*>(o)[i];
  __nv_bfloat162* pa = reinterpret_cast<__nv_bfloat162*>(&a);
  const __nv_bfloat162* pb = reinterpret_cast<const __nv_bfloat162*>(&b);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float2 x = __bfloat1622float2(pa[j]), y = __bfloat1622float2(pb[j]);
    pa[j] = __floats2bfloat162_rn(x.x + y.x, x.y + y.y);
  }
  reinterpret_cast<uint4*>(s)[i] = a;
}
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

dcp_status dcp_pairformer_stack_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t* bytes) {
  if (!bytes) return DCP_ERR_INVALID_ARG;
  size_t attn = 0;
  dcp_status st = dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, &attn);
  if (st != DCP_OK) return st;
  if (!pair_transition_supports(dtype, c_z)) return DCP_ERR_UNSUPPORTED;
  *bytes = align256(attn) + align256((size_t)I * c_s * elt_size(dtype)) + align256(pair_transition_workspace_bytes());
  return DCP_OK;
}

dcp_status dcp_pairformer_stack(void* s, void* z, const dcp_block_weights* blocks, int n_blocks, int64_t I, int c_s, int H,
                                int c, int c_z, dcp_dtype dtype, void* workspace, size_t workspace_bytes, void* stream) {
  g_launches = 0;
  if (!s || !z || !blocks || !workspace || n_blocks <= 0) return DCP_ERR_INVALID_ARG;
  size_t need = 0, attn = 0;
  dcp_status st = dcp_pairformer_stack_workspace_bytes(I, c_s, H, c, c_z, dtype, &need);
  if (st != DCP_OK) return st;
  if (workspace_bytes < need) return DCP_ERR_WORKSPACE;
  if (((uintptr_t)workspace & 255) != 0 || (((uintptr_t)s | (uintptr_t)z) & 15) != 0 || (I * c_s) % 8 != 0) return DCP_ERR_INVALID_ARG;
  if (I * I > 0x7fffff00ll) return DCP_ERR_INVALID_ARG;
  dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, &attn);
  char* ws = reinterpret_cast<char*>(workspace);
  void* ws_attn = ws;
  void* o = ws + align256(attn);
  void* ws_tr = ws + align256(attn) + align256((size_t)I * c_s * elt_size(dtype));
  int launches = 0;
  for (int b = 0; b < n_blocks; ++b) {
    const dcp_block_weights& w = blocks[b];
    st = layer(s, z, 0, &w.attn, o, I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, ws_attn, attn, stream);   // AttentionPairBias
    if (st != DCP_OK) return st;
    launches += g_launches;
    const int64_t n8 = I * c_s / 8;
    residual_add_bf16_kernel<<<(unsigned)((n8 + 255) / 256), 256, 0, (cudaStream_t)stream>>>((__nv_bfloat16*)s, (const __nv_bfloat16*)o, n8);
    if (cudaGetLastError() != cudaSuccess) return DCP_ERR_CUDA;
    st = dcp_pair_transition(z, z, I * I, c_z, w.w1, w.w2, w.w3, w.ln_gamma, w.ln_beta, w.ln_eps, dtype, ws_tr,
                             pair_transition_workspace_bytes(), stream);                                       // Transition, Eq. 6
    if (st != DCP_OK) return st;
    launches += 1 + g_launches;
  }
  g_launches = launches;
  return DCP_OK;
}

// ---- attention stack on a read-only pair tensor (reading 25)
dcp_status dcp_attention_stack_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t* bytes) {
  if (!bytes) return DCP_ERR_INVALID_ARG;
  size_t attn = 0;
  dcp_status st = dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, &attn);
  if (st != DCP_OK) return st;
  if (dtype != DCP_BF16 || !fused_mma_supports(dtype, H, c, c_z)) return DCP_ERR_UNSUPPORTED;
  *bytes = align256(attn) + align256((size_t)I * c_s * elt_size(dtype));
  return DCP_OK;
}

dcp_status dcp_attention_stack(void* a, const void* z, int64_t ldz, const dcp_weights* blocks, int n_blocks, int64_t I,
                               int c_s, int H, int c, int c_z, dcp_dtype dtype, void* workspace, size_t workspace_bytes,
                               void* stream) {
  g_launches = 0;
  if (!a || !z || !blocks || !workspace || n_blocks <= 0) return DCP_ERR_INVALID_ARG;
  size_t need = 0, attn = 0;
  dcp_status st = dcp_attention_stack_workspace_bytes(I, c_s, H, c, c_z, dtype, &need);
  if (st != DCP_OK) return st;
  if (workspace_bytes < need) return DCP_ERR_WORKSPACE;
  if (((uintptr_t)workspace & 255) != 0 || (I * c_s) % 8 != 0) return DCP_ERR_INVALID_ARG;
  dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, &attn);
  char* ws = reinterpret_cast<char*>(workspace);
  void* o = ws + align256(attn);
  int launches = 0;
  for (int b = 0; b < n_blocks; ++b) {
    // A <- A + AttentionPairBias_b(A, Z): the residual rides in the output GEMM's epilogue (one rounding per block)
    st = layer(a, z, ldz, &blocks[b], a, I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, ws, attn, stream, a);
    if (st == DCP_ERR_UNSUPPORTED) {   // W_o not tcgen05-shaped: layer output to scratch, then the residual kernel
      st = layer(a, z, ldz, &blocks[b], o, I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, ws, attn, stream);
      if (st != DCP_OK) return st;
      const int64_t n8 = I * c_s / 8;
      residual_add_bf16_kernel<<<(unsigned)((n8 + 255) / 256), 256, 0, (cudaStream_t)stream>>>((__nv_bfloat16*)a, (const __nv_bfloat16*)o, n8);
      if (cudaGetLastError() != cudaSuccess) return DCP_ERR_CUDA;
      ++launches;
    }
    if (st != DCP_OK) return st;
    launches += g_launches;
  }
  g_launches = launches;
  return DCP_OK;
}

// ---- the same stack with a bias cache: one pass over z per 23 blocks writes every block's bias tiles, then each block
// streams 32 bytes per pair instead of 256
dcp_status dcp_attention_stack_cache_bytes(int64_t I, int n_blocks, size_t* bytes) {
  if (!bytes || I <= 0 || n_blocks <= 0) return DCP_ERR_INVALID_ARG;
  *bytes = (size_t)n_blocks * (size_t)bias_tiles_block_words(I) * 4;
  return DCP_OK;
}

dcp_status dcp_attention_stack_cached_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t* bytes) {
  size_t base = 0;
  dcp_status st = dcp_attention_stack_workspace_bytes(I, c_s, H, c, c_z, dtype, &base);
  if (st != DCP_OK) return st;
  if (H != 16 || c_z != 128) return DCP_ERR_UNSUPPORTED;
  *bytes = base + align256(bias_tiles_fold_bytes(bias_tiles_max_blocks()));
  return DCP_OK;
}

dcp_status dcp_attention_stack_cached(void* a, const void* z, int64_t ldz, const dcp_weights* blocks, int n_blocks, int64_t I,
                                      int c_s, int H, int c, int c_z, dcp_dtype dtype, void* bias_cache, size_t bias_cache_bytes,
                                      void* workspace, size_t workspace_bytes, void* stream) {
  g_launches = 0;
  if (!a || !z || !blocks || !workspace || !bias_cache || n_blocks <= 0) return DCP_ERR_INVALID_ARG;
  size_t need = 0, base = 0, attn = 0, cache_need = 0;
  dcp_status st = dcp_attention_stack_cached_workspace_bytes(I, c_s, H, c, c_z, dtype, &need);
  if (st != DCP_OK) return st;
  dcp_attention_stack_cache_bytes(I, n_blocks, &cache_need);
  if (workspace_bytes < need || bias_cache_bytes < cache_need) return DCP_ERR_WORKSPACE;
  if (((uintptr_t)workspace & 255) != 0 || ((uintptr_t)bias_cache & 15) != 0 || ((uintptr_t)z & 15) != 0 || (I * c_s) % 8 != 0)
    return DCP_ERR_INVALID_ARG;
  if (ldz == 0) ldz = I * (int64_t)c_z;
  if (ldz < I * (int64_t)c_z || (ldz * 2) % 16 != 0) return DCP_ERR_INVALID_ARG;
  for (int b = 0; b < n_blocks; ++b) {
    if (validate_weights(&blocks[b]) != DCP_OK) return DCP_ERR_INVALID_ARG;
    if ((blocks[b].ln_eps > 0.f ? blocks[b].ln_eps : 1e-5f) != (blocks[0].ln_eps > 0.f ? blocks[0].ln_eps : 1e-5f))
      return DCP_ERR_UNSUPPORTED;                            // one set of LayerNorm statistics serves every block of a pass
  }
  dcp_attention_stack_workspace_bytes(I, c_s, H, c, c_z, dtype, &base);
  dcp_workspace_bytes(I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, nullptr, &attn);
  char* ws = reinterpret_cast<char*>(workspace);
  void* fold_ws = ws + base;
  const float eps = blocks[0].ln_eps > 0.f ? blocks[0].ln_eps : 1e-5f;
  const int64_t bw = bias_tiles_block_words(I);
  int launches = 0;
  for (int b0 = 0; b0 < n_blocks; b0 += bias_tiles_max_blocks()) {
    const int nb = std::min(n_blocks - b0, bias_tiles_max_blocks());
    if (launch_bias_tiles(z, ldz, I, blocks + b0, nb, eps, fold_ws, reinterpret_cast<uint32_t*>(bias_cache) + (int64_t)b0 * bw,
                          (cudaStream_t)stream) != cudaSuccess)
      return DCP_ERR_CUDA;
    launches += 2;
  }
  dcp_plan plan{};
  plan.parts = 1; plan.key_split = 1; plan.kernel = DCP_KERNEL_MMA; plan.tile_q = 32;   // tiles aligned with the cache's
  for (int b = 0; b < n_blocks; ++b) {
    st = layer(a, z, ldz, &blocks[b], a, I, c_s, H, c, c_z, dtype, DCP_MONOLITHIC, &plan, ws, attn, stream, a,
               reinterpret_cast<const uint32_t*>(bias_cache) + (int64_t)b * bw);
    if (st != DCP_OK) return st;
    launches += g_launches;
  }
  g_launches = launches;
  return DCP_OK;
}

dcp_status dcp_knn(const float* x, int32_t* idx, int64_t L, int k, void* stream) {
  g_launches = 0;
  if (!x || !idx || L <= 0 || k <= 0 || k > L) return DCP_ERR_INVALID_ARG;
  if (!knn_supports(L, k)) return DCP_ERR_UNSUPPORTED;
  DCP_CUDA(launch_knn(x, idx, L, k, (cudaStream_t)stream));
  return DCP_OK;
}

dcp_status dcp_knn_budget(const float* x, const int32_t* residue_id, const int32_t* chain_id, int32_t* idx, int64_t L, int k,
                          int n_seq, int n_chains, void* stream) {
  g_launches = 0;
  if (!x || !residue_id || !chain_id || !idx || L <= 0 || k <= 0 || k > L || n_seq < 0 || n_chains < 1) return DCP_ERR_INVALID_ARG;
  if (!knn_supports(L, k)) return DCP_ERR_UNSUPPORTED;
  DCP_CUDA(launch_knn_budget(x, residue_id, chain_id, idx, L, k, n_seq, n_chains, (cudaStream_t)stream));
  return DCP_OK;
}

dcp_status dcp_pair_bias_attention_host(const void* s_host, const void* z_host, const dcp_weights* w, void* out_host,
                                        void* s_dev, void* z_dev, void* out_dev, int64_t I, int c_s, int H, int c,
                                        int c_z, dcp_dtype dtype, dcp_decomp decomp, const dcp_plan* plan,
                                        void* workspace, size_t workspace_bytes, void* stream) {
  if (!s_host || !z_host || !out_host || !s_dev || !z_dev || !out_dev) return DCP_ERR_INVALID_ARG;
  dcp_status st = check_shape(I, c_s, H, c, c_z, dtype);
  if (st != DCP_OK) return st;
  const size_t e = elt_size(dtype);
  cudaStream_t cs = (cudaStream_t)stream;
  if (cudaMemcpyAsync(s_dev, s_host, (size_t)I * c_s * e, cudaMemcpyHostToDevice, cs) != cudaSuccess) return DCP_ERR_CUDA;
  if (cudaMemcpyAsync(z_dev, z_host, (size_t)I * I * c_z * e, cudaMemcpyHostToDevice, cs) != cudaSuccess)
    return DCP_ERR_CUDA;
  st = layer(s_dev, z_dev, 0, w, out_dev, I, c_s, H, c, c_z, dtype, decomp, plan, workspace, workspace_bytes, stream);
  if (st != DCP_OK) return st;
  if (cudaMemcpyAsync(out_host, out_dev, (size_t)I * c_s * e, cudaMemcpyDeviceToHost, cs) != cudaSuccess)
    return DCP_ERR_CUDA;
  return DCP_OK;
}

dcp_status dcp_partial_states(const void* s, const void* z, int64_t ldz, const dcp_weights* w, int64_t I, int c_s, int H,
                              int c, int c_z, dcp_dtype dtype, int kernel, int64_t q0, int64_t q1, int64_t k0,
                              int64_t k1, float* m, float* l, float* acc, void* workspace, size_t workspace_bytes,
                              void* stream) {
  g_launches = 0;
  if (!s || !z || !m || !l || !acc || !workspace) return DCP_ERR_INVALID_ARG;
  dcp_status st = validate_weights(w);
  if (st != DCP_OK) return st;
  st = check_shape(I, c_s, H, c, c_z, dtype);
  if (st != DCP_OK) return st;
  if (q0 < 0 || q1 > I || q0 >= q1 || k0 < 0 || k1 > I || k0 >= k1) return DCP_ERR_INVALID_ARG;
  const bool mma_ok = fused_mma_supports(dtype, H, c, c_z);
  if (kernel == DCP_KERNEL_MMA && !mma_ok) return DCP_ERR_UNSUPPORTED;
  if (kernel == DCP_KERNEL_GENERIC && !fused_generic_supports(dtype, H, c, c_z)) return DCP_ERR_UNSUPPORTED;
  const bool use_mma = mma_ok && kernel != DCP_KERNEL_GENERIC;
  if (ldz == 0) ldz = I * (int64_t)c_z;
  if (ldz < I * (int64_t)c_z || (ldz * elt_size(dtype)) % 16 != 0) return DCP_ERR_INVALID_ARG;
  if (misaligned(s) || misaligned(z) || misaligned(workspace, 256) || misaligned(m) || misaligned(l) || misaligned(acc))
    return DCP_ERR_INVALID_ARG;
  Ctx x{};
  x.I = I; x.c_s = c_s; x.H = H; x.c = c; x.c_z = c_z; x.D = H * c; x.dt = dtype; x.w = w;
  x.eps = w->ln_eps > 0.f ? w->ln_eps : 1e-5f;
  x.ws = (char*)workspace;
  x.cv = carve(I, c_s, H, c, c_z, dtype, 1);
  x.st = (cudaStream_t)stream;
  if (workspace_bytes < x.cv.total) return DCP_ERR_WORKSPACE;
  if (use_mma) {
    st = run_prologue_mma(x, s);
    if (st != DCP_OK) return st;
    MmaParams mp = base_params_mma(x);
    mp.st_m = m; mp.st_l = l; mp.st_acc = acc;
    mp.state_rows = q1 - q0; mp.state_row0 = q0;
    mp.q_begin = (int)q0; mp.q_end = (int)q1; mp.n_qparts = 1;
    mp.k_begin = (int)k0; mp.k_end = (int)k1; mp.n_kparts = 1;
    mp.nseg = 1; mp.slot0 = 0; mp.tile_h = 32;
    DCP_CUDA(launch_fused_mma(mp, z, ldz, x.st));
    return DCP_OK;
  }
  st = run_prologue(x, s);
  if (st != DCP_OK) return st;
  FusedParams p = base_params(x, z, ldz);
  p.st_m = m; p.st_l = l; p.st_acc = acc;
  p.state_rows = q1 - q0;
  p.state_row0 = q0;
  p.q0 = q0; p.q1 = q1; p.k0 = k0; p.k1 = k1;
  p.n_chunks = 1;
  p.slot0 = 0;
  return run_fused(x, p);
}

dcp_status dcp_merge_states(int n_parts, int64_t rows, int H, int c, const float* m, const float* l, const float* acc,
                            float* m_out, float* l_out, float* acc_out, void* stream) {
  if (n_parts < 1 || rows < 1 || H < 1 || c < 1 || !m || !l || !acc || !m_out || !l_out || !acc_out)
    return DCP_ERR_INVALID_ARG;
  MergeParams mp{};
  mp.st_m = m; mp.st_l = l; mp.st_acc = acc;
  mp.g = nullptr;
  mp.m_out = m_out; mp.l_out = l_out; mp.acc_out = acc_out;
  mp.rows = rows; mp.n_slots = n_parts; mp.H = H; mp.c = c; mp.D = H * c;
  if (launch_merge(DCP_F32, mp, (cudaStream_t)stream) != cudaSuccess) return DCP_ERR_CUDA;
  return DCP_OK;
}

dcp_status dcp_shard_range(int64_t n, int parts, int p, int64_t* start, int64_t* len) {
  if (n < 0 || parts < 1 || p < 0 || p >= parts || !start || !len) return DCP_ERR_INVALID_ARG;
  shard_range(n, parts, p, start, len);
  return DCP_OK;
}

dcp_status dcp_plan_units(int64_t I, int H, int c, int c_z, dcp_dtype dtype, dcp_decomp decomp, const dcp_plan* plan_in,
                          int* key_segments, int* tile_q, int* slots) {
  if (!key_segments || !tile_q || !slots || I <= 0) return DCP_ERR_INVALID_ARG;
  if (!fused_generic_supports(dtype, H, c, c_z) && !fused_mma_supports(dtype, H, c, c_z)) return DCP_ERR_UNSUPPORTED;
  Plan plan;
  dcp_status st = make_plan(I, H, c, c_z, dtype, decomp, plan_in, &plan);
  if (st != DCP_OK) return st;
  *key_segments = plan.nseg;
  *tile_q = plan.tile_h;
  *slots = plan.slots;
  return DCP_OK;
}

int dcp_kernel_supported(int kernel, dcp_dtype dtype, int H, int c, int c_z) {
  if (kernel == DCP_KERNEL_GENERIC) return fused_generic_supports(dtype, H, c, c_z) ? 1 : 0;
  if (kernel == DCP_KERNEL_MMA) return fused_mma_supports(dtype, H, c, c_z) ? 1 : 0;
  return 0;
}

dcp_status dcp_event_create(void** ev) {
  if (!ev) return DCP_ERR_INVALID_ARG;
  cudaEvent_t e;
  if (cudaEventCreate(&e) != cudaSuccess) return DCP_ERR_CUDA;
  *ev = (void*)e;
  return DCP_OK;
}
dcp_status dcp_event_record(void* ev, void* stream) {
  if (!ev) return DCP_ERR_INVALID_ARG;
  return cudaEventRecord((cudaEvent_t)ev, (cudaStream_t)stream) == cudaSuccess ? DCP_OK : DCP_ERR_CUDA;
}
dcp_status dcp_event_elapsed_ms(void* ev_begin, void* ev_end, float* ms) {
  if (!ev_begin || !ev_end || !ms) return DCP_ERR_INVALID_ARG;
  if (cudaEventSynchronize((cudaEvent_t)ev_end) != cudaSuccess) return DCP_ERR_CUDA;
  return cudaEventElapsedTime(ms, (cudaEvent_t)ev_begin, (cudaEvent_t)ev_end) == cudaSuccess ? DCP_OK : DCP_ERR_CUDA;
}
dcp_status dcp_event_destroy(void* ev) {
  if (!ev) return DCP_ERR_INVALID_ARG;
  return cudaEventDestroy((cudaEvent_t)ev) == cudaSuccess ? DCP_OK : DCP_ERR_CUDA;
}

int dcp_last_launch_count(void) { return g_launches; }

const char* dcp_status_string(dcp_status st) {
  switch (st) {
    case DCP_OK: return "DCP_OK";
    case DCP_ERR_INVALID_ARG: return "DCP_ERR_INVALID_ARG";
    case DCP_ERR_UNSUPPORTED: return "DCP_ERR_UNSUPPORTED";
    case DCP_ERR_WORKSPACE: return "DCP_ERR_WORKSPACE";
    case DCP_ERR_CUDA: return "DCP_ERR_CUDA";
    case DCP_ERR_SCRATCH_LIMIT: return "DCP_ERR_SCRATCH_LIMIT (needs more than dcp_no_alloc_scratch_bytes() of workspace)";
    default: return "DCP_ERR_UNKNOWN";
  }
}

int dcp_version(void) { return 200; }

}  // extern "C"
