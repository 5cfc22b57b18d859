// libdesigncp internal: host-side launchers of every kernel (one translation unit each).
#pragma once
#include "common.cuh"

namespace dcp {

enum GemmEpilogue { EPI_NONE = 0, EPI_SIGMOID = 1 };

// C[M,N] = epi(A[M,K] * W[K,N] + bias[N])  row-major, fp32 accumulate (SIMT; exact-order per element).
// a_is_f32: A is float (LayerNorm'ed s) instead of the storage dtype.  Step a1 / a9 of SURVEY.md section 8(a).
cudaError_t launch_gemm(dcp_dtype dt, bool a_is_f32, const void* A, int64_t lda, const void* W, const void* bias,
                        void* C, int64_t ldc, int64_t M, int N, int K, GemmEpilogue epi, cudaStream_t st);

// s~ = LayerNorm(s; gamma, beta) -> float [rows, width]      (optional LN_s, reading #3 in DESIGN.md)
cudaError_t launch_layernorm_rows(dcp_dtype dt, const void* x, const void* gamma, const void* beta, float* y,
                                  int64_t rows, int width, float eps, cudaStream_t st);

// wg[k,h] = gamma_k * W_b[k,h] (fp32), c0[h] = sum_k beta_k W_b[k,h]
cudaError_t launch_fold_ln_z(dcp_dtype dt, const void* w_b, const void* gamma, const void* beta, float* wg, float* c0,
                             int c_z, int H, cudaStream_t st);

// Generic fp32 CUDA-core fused kernel (steps a2-a7).  Returns cudaErrorInvalidValue for unsupported shapes.
cudaError_t launch_fused_generic(dcp_dtype dt, const FusedParams& p, cudaStream_t st);
bool fused_generic_supports(dcp_dtype dt, int H, int c, int c_z);

// ---- bf16 tensor-core path (fused_mma.cu, gemm_mma.cu)
enum GemmOutMode { GEMM_OUT_PLAIN = 0, GEMM_OUT_SIGMOID = 1, GEMM_OUT_HEADPAD = 2, GEMM_OUT_TRANSPOSED = 3,
                   GEMM_OUT_KFRAG = 4, GEMM_OUT_VFRAG = 5 };

// C_seg = epi(A[M,K] * W_seg[K,N] + bias_seg) for seg < nseg, all bf16 with fp32 accumulation (one launch).
struct GemmMmaParams {
  const void* A;        // [M, K] bf16, row pitch lda
  int64_t lda, M;
  int N, K, nseg;
  const void* W[4];     // [K, N] bf16 row-major
  const void* bias[4];  // [N] bf16 or nullptr
  void* C[4];
  int mode[4];          // GemmOutMode
  float scale[4];       // HEADPAD only
  int64_t ldc[4];       // PLAIN / SIGMOID: row pitch; TRANSPOSED: pitch of the transposed rows
  int H, c, cp;         // HEADPAD: C[(row*H + h)*cp + d] for column h*c + d; KFRAG / VFRAG: MMA-fragment order (fused_mma.cu)
  // optional: the LayerNorm(z) fold (fold_ln_z_mma) rides along as one extra CTA of the tcgen05 GEMM launch
  // (fold_w_b == nullptr: not requested; launch_gemm_mma reports through `fold_done` whether it was done)
  const void *fold_w_b, *fold_gamma, *fold_beta;
  void* fold_wfold;
  float *fold_c1, *fold_c0;
  int fold_c_z, fold_H, fold_H_pad;
  // optional, GEMM_OUT_PLAIN segments of the tcgen05 GEMM only: C = bf16(acc + residual[row][col]) (fp32 add, one rounding);
  // residual may be C itself (in place: a CTA reads its tile's residual before the barrier that precedes its stores)
  const void* residual;
  int64_t ldr;
  bool pdl;             // host only: launch as a programmatic dependent of the previous kernel in the stream (common.cuh)
};
cudaError_t launch_gemm_mma(const GemmMmaParams& p, cudaStream_t st, bool* fold_done = nullptr);   // dispatches to launch_gemm_tc when it applies
// tcgen05 / TMA GEMM (gemm_tc.cu): N % 128 == 0, K % 64 == 0, 16-byte aligned operands
bool gemm_tc_supports(const GemmMmaParams& p);
cudaError_t launch_gemm_tc(const GemmMmaParams& p, cudaStream_t st);   // also runs the requested LayerNorm(z) fold
cudaError_t launch_layernorm_rows_bf16(const void* x, const void* gamma, const void* beta, void* y, int64_t rows,
                                       int width, float eps, cudaStream_t st);
// wfold [H_pad][c_z] bf16 = (gamma (.) W_b * log2 e)^T, c1[h] = sum_k wfold[h][k], c0[h] = log2 e * sum_k beta_k W_b[k,h]
cudaError_t launch_fold_ln_z_mma(const void* w_b, const void* gamma, const void* beta, void* wfold, float* c1,
                                 float* c0, int c_z, int H, int H_pad, cudaStream_t st);

// One launch of the persistent fused kernel over every (query part, 32-query tile, key chunk, key segment) unit:
// query rows [q_begin, q_end) cut into n_qparts Eq.-5 parts (row stripes / grid row blocks), keys [k_begin, k_end)
// into n_kparts Eq.-5 chunks (key_split / grid key blocks), each chunk into nseg Eq.-5 segments; unit
// (chunk cb, segment sg) writes partial-state slot slot0 + cb*nseg + sg.
struct MmaParams {
  const void* qp;       // [I][H][cp] bf16, scaled by log2(e)/sqrt(c)
  const void* kfr;      // K in QK^T B-fragment order: [key tile of 16][H][cp/16][32 lanes][8] bf16 (zero padded)
  const void* vfr;      // V in PV B-fragment order:   [key tile of 16][H][cp/16][32 lanes][8] bf16 (zero padded)
  const void* wfold;    // [16][c_z] bf16
  const float* c1;      // [16]
  const float* c0;      // [16]
  float* st_m;          // [slots, state_rows, H]   (natural-log units)
  float* st_l;          // [slots, state_rows, H]
  float* st_acc;        // [slots, state_rows, H*c]
  int64_t state_rows, state_row0;
  int I;
  int q_begin, q_end, n_qparts;
  int k_begin, k_end, n_kparts;
  int nseg, slot0;
  int tile_h;           // fused_mma_kernel: query rows per work unit (25..32; the atom kernel's tile is fixed)
  int H, c, c_z;
  float eps;
  // optional: the bias of this call comes from a cache (bias_tiles.cu) instead of z; launch_fused_mma then forwards to
  // cached_attn_kernel (cached_attn.cu), which reads no z at all.  Whole-tensor rows, one row part, tile height 32.
  const uint32_t* bias_cache;
  bool pdl;             // host only: launch as a programmatic dependent of the previous kernel in the stream
};
cudaError_t launch_fused_mma(const MmaParams& p, const void* z, int64_t ldz, cudaStream_t st);
// attention of one block over a bias cache (cached_attn.cu): p as for launch_fused_mma with p.bias_cache set
cudaError_t launch_cached_attn(const MmaParams& p, cudaStream_t st);
bool fused_mma_supports(dcp_dtype dt, int H, int c, int c_z);
int mma_head_pad(int c);
int64_t mma_frag_elems(int64_t I, int H, int c);   // bf16 elements of kfr (= of vfr)
// Units of the tensor-core kernels: *nseg = Eq.-5 segments per key chunk, *tile_h = query rows per unit (fused_mma_kernel:
// 25..32, chosen so that the unit count fills whole waves of 148 SMs; fused_atom_kernel: fixed).  Pure functions of
// (I, H, n_qparts, n_kparts): every call with the same decomposition cuts its rows and keys alike.
void mma_pick_units(int64_t I, int H, int n_qparts, int n_kparts, int force_nseg, int force_tile_h, int* nseg, int* tile_h);
// atom-level shape (c_atompair = 16, H = 4, c = 32): fused_atom.cu, dispatched to by launch_fused_mma
cudaError_t launch_fused_atom(const MmaParams& p, const void* z, int64_t ldz, cudaStream_t st);
bool fused_atom_supports(dcp_dtype dt, int H, int c, int c_z);
int fused_atom_tile_q();

// Sparse k-neighbour atom attention (sparse_atom.cu): q, k, v, g [L][H*32] bf16 from the prologue
// GEMM, p_slice [L][kn][16], idx [L][kn] (negative = unused slot) -> gated [L][H*32]
bool sparse_atom_supports(dcp_dtype dt, int H, int c, int c_z, int kn);
cudaError_t launch_sparse_atom(const void* q, const void* k, const void* v, const void* g, const void* p_slice,
                               const int32_t* idx, const void* wfold, const float* c1, const float* c0, void* gated,
                               int64_t L, int kn, int H, float eps, cudaStream_t st);

// p_slice[l, j, :] = P[l, idx[l, j], :] (row_bytes = c_atompair * element size, a multiple of 16; zeros for idx < 0)
cudaError_t launch_gather_pair_slice(const void* P, int64_t ldp_bytes, const int32_t* idx, void* out, int64_t L, int kn,
                                     int row_bytes, cudaStream_t st);

// k nearest neighbours of every atom (knn.cu): x [L][3] fp32 -> idx [L][k], ordered by (d2, index)
bool knn_supports(int64_t L, int k);
cudaError_t launch_knn(const float* x, int32_t* idx, int64_t L, int k, cudaStream_t st);
// the structured budget: sequence-local atoms first, inter-chain quota when n_chains > 3
cudaError_t launch_knn_budget(const float* x, const int32_t* residue_id, const int32_t* chain_id, int32_t* idx, int64_t L, int k,
                              int n_seq, int n_chains, cudaStream_t st);

// Pairwise SwiGLU transition z <- z + W3 (SiLU(W1 LN z) (.) W2 LN z) (pair_transition.cu)
bool pair_transition_supports(dcp_dtype dt, int c_z);
size_t pair_transition_workspace_bytes();
cudaError_t launch_pair_transition(const void* z_in, void* z_out, int64_t n_pairs, const void* w1, const void* w2,
                                   const void* w3, const void* gamma, const void* beta, float eps, void* workspace,
                                   cudaStream_t st);

// Bias cache of the attention stack (bias_tiles.cu): the biases LN_b(z) W_b^b of up to bias_tiles_max_blocks() blocks in one
// pass over z, as fp16 tiles in the layout cached_attn_kernel consumes (MmaParams.bias_cache)
int bias_tiles_max_blocks();
int64_t bias_tiles_block_words(int64_t I);          // 32-bit words of one block's cache
size_t bias_tiles_fold_bytes(int n_blocks);         // scratch for the folded weights of a pass
cudaError_t launch_bias_tiles(const void* z, int64_t ldz, int64_t I, const dcp_weights* blocks, int n_blocks, float eps,
                              void* fold_ws, void* cache, cudaStream_t st);

// Merge (step a8) + normalise + gate (first half of a9); or raw merged state out.
cudaError_t launch_merge(dcp_dtype dt, const MergeParams& p, cudaStream_t st);

}  // namespace dcp
