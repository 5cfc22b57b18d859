/* libdesigncp -- attention with pair bias on one B200 (sm_100a): the one-GPU core that Design-CP
 * (arxiv/paper_2607_05439) distributes.  Plain C ABI: pointers and sizes only, no torch types.
 *
 * The layer (citations are lines of /root/reference/PAPER.md; readings in DESIGN.md):
 *   PAPER.md:58  (sec 3.1)  "a learned projection of Z produces a per-head pair bias B in R^{IxIxH} that is
 *                            added to the attention logits before the softmax, softmax(QK^T/sqrt(d) + B)"
 *   PAPER.md:83  (Eq. 2)    Attn^(p) = softmax(Q^(p) K^T / sqrt(d) + B^(p)) V,  B^(p) = f_B(Z^(p)) in R^{I_p x I x H}
 *   BASELINE.json config 0  out = W_o ( sigmoid(s W_g) (.) softmax(Q K^T/sqrt(c) + LN(z) W_b) V )
 *   PAPER.md:72 (Eq. 1), :337 (Eq. 5)  row shards  I_p = floor(I/P)+[p < I mod P], start_p = p floor(I/P)+min(p, I mod P)
 *   PAPER.md:90 (sec 3.3), :446 (C.2)  sqrt(P) x sqrt(P) grid; partial outputs merged by an online softmax
 *
 * Layout: every tensor is row-major, last index fastest.
 *   s   [I, c_s]        single track                        z   [I, I, c_z]   z[i, j, :] biases query i <- key j
 *   W_q, W_k, W_v, W_g [c_s, H*c] (column h*c+d = head h, channel d)   W_b [c_z, H]   W_o [H*c, c_s]
 *   out [I, c_s]
 * dtype is the STORAGE type of s, z, the weights and out (DCP_F32 or DCP_BF16); all accumulation is fp32.
 *
 * Ownership: the caller owns every buffer.  The library allocates nothing persistent, keeps no global state
 * (except a one-time cudaFuncSetAttribute per kernel) and is re-entrant.  Inputs are read-only and must not
 * alias out/workspace.  Unless a function says HOST, pointers are DEVICE pointers on the current device.
 * Asynchrony: work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = default stream) and the
 * call returns after the launches.  DCP_ERR_CUDA reports launch-time errors; execution errors surface at the
 * caller's next synchronisation.  No function aborts or throws.
 */
#ifndef DESIGNCP_H
#define DESIGNCP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  DCP_OK = 0,
  DCP_ERR_INVALID_ARG = 1, /* null pointer, non-positive size, parts > I, GRID with non-square parts,
                              misaligned pointer / pitch (16 B), c_z*sizeof(elt) % 16 != 0                         */
  DCP_ERR_UNSUPPORTED = 2, /* a (dtype, H, c, c_z) the kernels are not instantiated for; a tensor-core shape with
                              c_s % 8 != 0 (its GEMMs move 16-byte row pieces); a tile the kernel does not have   */
  DCP_ERR_WORKSPACE = 3,   /* workspace too small (see dcp_workspace_bytes)                                       */
  DCP_ERR_CUDA = 4,        /* a CUDA runtime / driver call failed at launch time                                  */
  DCP_ERR_SCRATCH_LIMIT = 5 /* dcp_pair_bias_attention_no_alloc: the problem needs more workspace than the library's
                              static scratch array holds (dcp_no_alloc_scratch_bytes); use the caller-workspace entry */
} dcp_status;

typedef enum { DCP_F32 = 0, DCP_BF16 = 1 } dcp_dtype;

/* How the layer is cut (the on-device emulation of Design-CP's schemes):
 *   MONOLITHIC  one problem; keys processed as `key_split` Eq.-5 chunks merged left to right
 *   ROW         PAPER.md:72-86: `parts` query stripes (Eq. 5), each against ALL keys
 *   GRID        PAPER.md:90: G x G quadrants, G = sqrt(parts) (parts must be a perfect square), each producing a
 *               partial (m, l, acc) from its own block of z; the G key blocks of a row are merged left to right
 * On the tensor-core kernels all stripes / quadrants of a call are work units of ONE persistent launch (each unit
 * reads only its own block of z, through a strided view); the generic kernel launches once per stripe / quadrant. */
typedef enum { DCP_MONOLITHIC = 0, DCP_ROW = 1, DCP_GRID = 2 } dcp_decomp;

/* Which fused kernel runs the (query-tile, key-tile) loop. */
typedef enum {
  DCP_KERNEL_AUTO = 0,   /* fastest kernel instantiated for the shape                                            */
  DCP_KERNEL_GENERIC = 1,/* fp32 CUDA-core kernel: any shape with H <= 16, H*c % 32 == 0, H*c <= 768             */
  DCP_KERNEL_MMA = 2     /* bf16 tensor-core kernel (TMA-streamed z): DCP_BF16 only, shapes of configs 1-4       */
} dcp_kernel;

typedef struct {
  const void *w_q, *w_k, *w_v, *w_g; /* [c_s, H*c]                                                */
  const void *w_b;                   /* [c_z, H]                                                  */
  const void *w_o;                   /* [H*c, c_s]                                                */
  const void *ln_z_gamma, *ln_z_beta;/* [c_z]    LayerNorm over the channel axis of z             */
  const void *ln_s_gamma, *ln_s_beta;/* [c_s] or both NULL = no LayerNorm on s (BASELINE formula) */
  const void *b_q;                   /* [H*c] or NULL                                             */
  float ln_eps;                      /* <= 0 means 1e-5                                           */
} dcp_weights;

typedef struct {
  int parts;     /* ROW: number of stripes, 1 <= parts <= I.  GRID: P, a perfect square with sqrt(P) <= I.
                    MONOLITHIC: ignored.                                                                 */
  int key_split; /* MONOLITHIC / ROW: key chunks (Eq. 5) merged left to right; <= 0 means 1.  GRID: ignored
                    (the key axis is cut into sqrt(parts) blocks).                                       */
  int kernel;    /* a dcp_kernel                                                                         */
  int tile_q, tile_k; /* query / key tile of the fused kernel (north_star's `tile`): 0 = automatic.  fused_mma_kernel
                    (tokens) takes any query-tile height 25..32 (its last TMA box is trimmed to the tile) and picks
                    the one whose unit count fills whole waves of SMs; key tile 16.  fused_atom_kernel: 64 x 32,
                    fused_generic_kernel: 8 x 32, fixed.  Any other non-zero value is DCP_ERR_UNSUPPORTED.  The
                    tiling changes no row's arithmetic: results are bitwise independent of tile_q.           */
  int key_segments; /* tensor-core kernels: Eq.-5 segments each key chunk is cut into (the units that fill the 148
                    SMs; one partial state per segment, merged left to right like the chunks).  0 = automatic, a
                    pure function of (I, number of chunks), so that every decomposition cuts a row's keys alike
                    and the bitwise decomposition contract holds; 1..64 = forced (the contract then holds between
                    calls that force the same value).                                                      */
  void *ev_fused_begin, *ev_fused_end; /* optional cudaEvent_t (from dcp_event_create): recorded on `stream` just
                    before the first and just after the last fused-kernel launch of the call (bench.py times the
                    dominant kernel with them); NULL = not recorded                                       */
} dcp_plan;

/* Bytes of device workspace dcp_pair_bias_attention needs for this problem (q,k,v,g, the partial states
 * [chunks][I][H] x2 and [chunks][I][H*c] fp32, the gated activations, folded weights).  `plan` may be NULL
 * (MONOLITHIC defaults). */
dcp_status dcp_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype,
                               dcp_decomp decomp, const dcp_plan *plan, size_t *bytes);

/* The layer.  z is read exactly once; the I*I*H logits never reach memory.
 * ldz = elements between z[i,0,0] and z[i+1,0,0] (0 means I*c_z); lets z be a view of a larger tensor.
 * workspace: device, 256-byte aligned, >= dcp_workspace_bytes(...).  The result does not depend on `decomp`
 * beyond rounding. */
dcp_status dcp_pair_bias_attention(const void *s, const void *z, int64_t ldz, const dcp_weights *w, void *out,
                                   int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype,
                                   dcp_decomp decomp, const dcp_plan *plan,
                                   void *workspace, size_t workspace_bytes, void *stream);

/* Atom-level dense variant ("an analogous pair representation P in R^{LxLxc_atompair}";
 * BASELINE.json config 4): the same computation with (L, c_atom, c_atompair) for (I, c_s, c_z). */
dcp_status dcp_atom_pair_bias_attention(const void *a, const void *p, int64_t ldp, const dcp_weights *w,
                                        void *out, int64_t L, int c_atom, int H, int c, int c_atompair,
                                        dcp_dtype dtype, dcp_decomp decomp, const dcp_plan *plan,
                                        void *workspace, size_t workspace_bytes, void *stream);

/* Sparse k-neighbour atom-level attention ("each query atom attends to a budget of k neighbours ... The
 * relevant slice of P is gathered at those k indices and then projected to the per-head bias"; :303 the block
 * consumes a [L, k, c_atompair] slice, k = n_attn-keys, default 128; :456 K/V/B entries gathered at the indices).
 * For query atom l: keys m = idx[l, j] (j < k), logit_j^h = q_l^h.k_m^h/sqrt(c) + LN(p_slice[l, j, :]).W_b[:, h],
 * softmax over the VALID slots, out_l = (sigmoid(a_l W_g) (.) sum_j a_j v_m) W_o.
 *   a [L, c_atom], p_slice [L, k, c_atompair], out [L, c_atom]: device, storage dtype, row-major, 16-byte aligned;
 *   idx [L, k]: device int32; idx < 0 marks an unused slot (an atom without valid slots gets out = 0); a neighbour
 *   listed twice counts twice; an index >= L is treated like a negative one (unused slot).
 * Instantiated for DCP_BF16, c = 32, c_atompair = 16, H <= 16, k <= 512, c_atom % 8 == 0 (DCP_ERR_UNSUPPORTED
 * otherwise).  workspace >= dcp_sparse_atom_workspace_bytes(...), 256-byte aligned.  Enqueues on `stream`.
 * `plan` may be NULL; only its ev_fused_begin / ev_fused_end (recorded around the gather kernel) are used. */
dcp_status dcp_sparse_atom_workspace_bytes(int64_t L, int c_atom, int H, int c, dcp_dtype dtype, size_t *bytes);
dcp_status dcp_sparse_atom_attention(const void *a, const void *p_slice, const int32_t *idx, const dcp_weights *w,
                                     void *out, int64_t L, int k, int c_atom, int H, int c, int c_atompair,
                                     dcp_dtype dtype, const dcp_plan *plan, void *workspace, size_t workspace_bytes,
                                     void *stream);

/* Pairwise SwiGLU transition (PAPER.md:381-385 Eq. 6, :387-409 Algorithm 1):
 *     z_out = z + ( SiLU(LN(z) W_1) (.) LN(z) W_2 ) W_3        for every pair (row of z) independently,
 * LN = LayerNorm over the channel axis with affine ln_gamma, ln_beta (population variance, eps; <= 0 means 1e-5).
 *   z, z_out [n_pairs, c_z] row-major device (n_pairs = I * I for the token-pair tensor); z_out may be z (in place);
 *   w1, w2 [c_z, 4 c_z], w3 [4 c_z, c_z] row-major device, ln_gamma, ln_beta [c_z]; all in the storage dtype, 16-byte
 *   aligned.  Instantiated for DCP_BF16, c_z = 128 (DCP_ERR_UNSUPPORTED otherwise); n_pairs < 2^31.
 * workspace >= dcp_pair_transition_workspace_bytes (folded weights), 256-byte aligned.  Enqueues on `stream`. */
dcp_status dcp_pair_transition_workspace_bytes(int c_z, dcp_dtype dtype, size_t *bytes);
dcp_status dcp_pair_transition(const void *z, void *z_out, int64_t n_pairs, int c_z, const void *w1, const void *w2,
                               const void *w3, const void *ln_gamma, const void *ln_beta, float ln_eps, dcp_dtype dtype,
                               void *workspace, size_t workspace_bytes, void *stream);

/* A stack of non-triangular Pairformer blocks on a resident pair tensor (first step).
 * PAPER.md:289 "The Pairformer block ... is ... an AttentionPairBias (16 heads, optional QK-norm) followed by a Transition
 * module; both stock configurations explicitly disable the ... triangle multiplication and triangle attention paths";
 * :293 "Two non-triangular Pairformer blocks (each 16-head AttentionPairBias + Transition) then refine (S, Z)".
 * Block b (reading 23):   S <- S + AttentionPairBias_b(S, Z)   (dcp_pair_bias_attention, MONOLITHIC)
 *                                   Z <- Z + Transition_b(Z)             (dcp_pair_transition, Eq. 6)
 * and block b + 1 sees the updated (S, Z).  s [I, c_s] and z [I, I, c_z] are device tensors updated IN PLACE, stored in
 * the storage dtype after every block.  blocks: HOST array of n_blocks entries whose pointers are device pointers
 * (attn as in dcp_pair_bias_attention; w1, w2 [c_z, 4 c_z], w3 [4 c_z, c_z], ln_gamma, ln_beta [c_z] as in
 * dcp_pair_transition); it is read during the call only.  DCP_BF16 with c_z = 128 and an (H, c) the fused kernel is
 * instantiated for (DCP_ERR_UNSUPPORTED otherwise); I * I < 2^31.  workspace >= dcp_pairformer_stack_workspace_bytes,
 * 256-byte aligned.  Enqueues 7 launches per block on `stream` and returns. */
typedef struct {
  dcp_weights attn;
  const void *w1, *w2, *w3, *ln_gamma, *ln_beta;
  float ln_eps; /* <= 0 means 1e-5 */
} dcp_block_weights;
dcp_status dcp_pairformer_stack_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t *bytes);
dcp_status dcp_pairformer_stack(void *s, void *z, const dcp_block_weights *blocks, int n_blocks, int64_t I, int c_s,
                                int H, int c, int c_z, dcp_dtype dtype, void *workspace, size_t workspace_bytes,
                                void *stream);

/* The diffusion transformer's attention stack on a resident, READ-ONLY pair tensor.
 * PAPER.md:294 "Eighteen sequential AttentionPairBiasDiffusion + ConditionedTransitionBlock blocks (16 heads each ...)
 * update the token-level latent A_I in R^{B x I x c_token} using the local pair bias derived from Z.  This is the stage
 * that dominates per-step compute"; :285 c_token = 768.  Block b = 0 .. n_blocks-1 (reading 25):
 *       A <- A + AttentionPairBias_b(A, Z)        (the layer of dcp_pair_bias_attention with blocks[b], MONOLITHIC)
 * a [I, c_s] (c_s = c_token) is updated IN PLACE and stored in the storage dtype once per block (the residual is added
 * in fp32 inside the output projection); z [I, I, c_z] (row pitch ldz elements, 0 = I * c_z) is only read: every block
 * re-streams it and derives its own bias LN_b(z) W_b^b.  The conditional (AdaLN) normalisation and the
 * ConditionedTransitionBlock have no formulas in the paper and are not part of the call.
 * blocks: HOST array of n_blocks dcp_weights whose pointers are device pointers, read during the call only.
 * DCP_BF16 and a (H, c, c_z) the tensor-core kernel is instantiated for (DCP_ERR_UNSUPPORTED otherwise).
 * workspace >= dcp_attention_stack_workspace_bytes, 256-byte aligned.  Enqueues 4 launches per block on `stream`
 * (chained by programmatic dependent launch), no host synchronisation: capturable into a CUDA graph. */
dcp_status dcp_attention_stack_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t *bytes);
dcp_status dcp_attention_stack(void *a, const void *z, int64_t ldz, const dcp_weights *blocks, int n_blocks, int64_t I,
                               int c_s, int H, int c, int c_z, dcp_dtype dtype, void *workspace, size_t workspace_bytes,
                               void *stream);

/* The same stack with a BIAS CACHE: every block derives its bias LN_b(z) W_b^b from the same read-only
 * pair tensor, so one pass over z per 23 blocks computes the LayerNorm statistics once per pair and writes every block's
 * bias as fp16 tiles (H * 2 = 32 bytes per pair and block; PAPER.md:81 materialises B in R^{I x I x H} per block too);
 * each block then streams its 32 bytes per pair instead of the 256 bytes of z.  Same result as dcp_attention_stack up
 * to the fp16 rounding of the bias (2^-11 relative, below the bf16 rounding of P that follows).
 * bias_cache: device, 16-byte aligned, >= dcp_attention_stack_cache_bytes(I, n_blocks) (I = 3000, 18 blocks: 5.2 GB);
 * it is scratch, valid only during the call.  H = 16, c_z = 128, DCP_BF16, all blocks with the same ln_eps
 * (DCP_ERR_UNSUPPORTED otherwise).  workspace >= dcp_attention_stack_cached_workspace_bytes.  Launches only, no host
 * synchronisation: capturable into a CUDA graph like dcp_attention_stack (tests/test_gpu_graph.py). */
dcp_status dcp_attention_stack_cache_bytes(int64_t I, int n_blocks, size_t *bytes);
dcp_status dcp_attention_stack_cached_workspace_bytes(int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, size_t *bytes);
dcp_status dcp_attention_stack_cached(void *a, const void *z, int64_t ldz, const dcp_weights *blocks, int n_blocks, int64_t I,
                                      int c_s, int H, int c, int c_z, dcp_dtype dtype, void *bias_cache,
                                      size_t bias_cache_bytes, void *workspace, size_t workspace_bytes, void *stream);

/* p_slice[l, j, :] = p[l, idx[l, j], :] ("The relevant slice of P is gathered at those k indices"): the
 * dense atom-pair tensor p [L, L, c_atompair] (row pitch ldp elements, 0 = L * c_atompair) -> the slice
 * [L, k, c_atompair] that dcp_sparse_atom_attention consumes; slots with idx < 0 are filled with zeros.  Device
 * pointers, dtype DCP_F32 or DCP_BF16, c_atompair * element size a multiple of 16 bytes, 16-byte aligned
 * (DCP_ERR_INVALID_ARG otherwise); an index >= L is treated like a negative one. */
dcp_status dcp_gather_pair_slice(const void *p, int64_t ldp, const int32_t *idx, void *p_slice, int64_t L, int k,
                                 int c_atompair, dcp_dtype dtype, void *stream);

/* Neighbour lists for dcp_sparse_atom_attention ("The kNN indices are computed once per denoising step
 * from the current noised coordinates X^(t) via a single cdist call"; :454 distance matrix + top-k per row, here
 * without the [L, L] matrix).  x [L, 3] fp32 device; idx [L, k] int32 device: the k atoms with the smallest squared
 * Euclidean distance to atom l (itself included), ordered by (distance, atom index) ascending -- unique, and
 * bit-exact against the oracle: distances in binary32, t = x_m - x_l, d2 = (t0 t0 + t1 t1) + t2 t2, no FMA.
 * 1 <= k <= min(L, 512) (DCP_ERR_INVALID_ARG / DCP_ERR_UNSUPPORTED otherwise).  Pure spatial top-k: the paper's
 * sequence-local and inter-chain quotas are dcp_knn_budget below. */
dcp_status dcp_knn(const float *x, int32_t *idx, int64_t L, int k, void *stream);

/* The STRUCTURED neighbour budget: "a fixed number n_seq of per-residue sequence-local neighbours
 * (default n_seq = 2, namely the query atom plus its immediate flanking residues' atoms), and the spatially closest
 * atoms beyond those, until the per-query budget k ... is filled ... When the input is a multi-chain assembly with more
 * than three chains, the budget is split into an intra-chain quota of k - max(32, k/4) neighbours and an inter-chain
 * quota of at least 32 neighbours".  Inputs as PAPER.md:454 names them: x [L, 3] fp32, residue_id [L] and chain_id [L]
 * int32 (device).  Readings (#26): closest = smallest (binary32 squared distance as in dcp_knn, atom index);
 * sequence-local = same chain and |residue_id difference| <= n_seq - 1 (n_seq = 0: none), taken first; with
 * n_chains > 3 the min(max(32, k/4), k - 1) closest atoms of OTHER chains are served first, the own chain gets the
 * rest (sequence-local atoms first), and whatever one side cannot fill goes to the other.  n_chains = the number of
 * distinct values in chain_id (the caller knows it; only "> 3" matters).  idx [L, k]: the selected atoms by
 * (distance, index) ascending, the query itself included; bit-exact against oracle/knn_budget.py.
 * 1 <= k <= min(L, 512), n_seq >= 0 (DCP_ERR_INVALID_ARG / DCP_ERR_UNSUPPORTED otherwise). */
dcp_status dcp_knn_budget(const float *x, const int32_t *residue_id, const int32_t *chain_id, int32_t *idx, int64_t L,
                          int k, int n_seq, int n_chains, void *stream);

/* The layer for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): dcp_pair_bias_attention (PAPER.md:58, :83 Eq. 2, :90) with its workspace in a
 * static device array of DCP_NO_ALLOC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds
 * until exit.  Arguments, layouts, result and errors as dcp_pair_bias_attention (s, z, w, out: device, caller-owned);
 * the call and everything under it calls no cudaMalloc, cudaFree or allocating library routine.
 * Limit: dcp_workspace_bytes(...) for the problem and plan must be <= dcp_no_alloc_scratch_bytes() (32 MiB: the
 * monolithic token-level layer up to I = 2048 at c_s = 384, H = 16, c = 48), else DCP_ERR_SCRATCH_LIMIT and nothing is
 * launched.  All calls on a device share the one array, which keeps the previous call's contents (the layer writes
 * every region before reading it, nothing needs clearing): calls ordered on one stream are safe, calls that overlap on
 * the GPU (other streams, other host threads on the same device) RACE -- serialise them or use the workspace entry. */
#define DCP_NO_ALLOC_SCRATCH_BYTES ((size_t)32 << 20)
size_t dcp_no_alloc_scratch_bytes(void);
dcp_status dcp_pair_bias_attention_no_alloc(const void *s, const void *z, int64_t ldz, const dcp_weights *w, void *out,
                                            int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype,
                                            dcp_decomp decomp, const dcp_plan *plan, void *stream);

/* End-to-end entry with HOST inputs/outputs: s_host, z_host, out_host are HOST pointers (pinned memory gives
 * full PCIe rate); weights stay device-resident (they are parameters, not per-step inputs).  Copies s and z
 * to the device staging buffers s_dev [I,c_s], z_dev [I,I,c_z], runs the layer, copies out back, all on
 * `stream`.  Returns after enqueueing; synchronise the stream before reading out_host. */
dcp_status dcp_pair_bias_attention_host(const void *s_host, const void *z_host, const dcp_weights *w,
                                        void *out_host, void *s_dev, void *z_dev, void *out_dev,
                                        int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype,
                                        dcp_decomp decomp, const dcp_plan *plan,
                                        void *workspace, size_t workspace_bytes, void *stream);

/* Diagnostic: the partial online-softmax state of query rows [q0,q1) against keys [k0,k1) only:
 * m [q1-q0, H] = the state's reference, l [q1-q0, H] = sum_j e^{logit-m}, acc [q1-q0, H*c] = sum_j e^{logit-m} v_j
 * (fp32, natural-log units).  A state is defined up to its reference: (m, l, acc) and (m', l e^{m-m'}, acc e^{m-m'})
 * are the same state, and dcp_merge_states treats them alike.  DCP_KERNEL_GENERIC returns m = max_j logit; the
 * tensor-core kernels move a row's reference lazily (only when a key tile's maximum exceeds it by more than 8 in
 * log2 units), so their m satisfies  max_j logit - 8 ln 2 <= m <= max_j logit  (reading 19).
 * Pointers, ldz and the workspace obey the same alignment rules as dcp_pair_bias_attention (16 bytes; workspace
 * 256; >= dcp_workspace_bytes of the MONOLITHIC plan); m, l, acc 16-byte aligned. */
dcp_status dcp_partial_states(const void *s, const void *z, int64_t ldz, const dcp_weights *w,
                              int64_t I, int c_s, int H, int c, int c_z, dcp_dtype dtype, int kernel,
                              int64_t q0, int64_t q1, int64_t k0, int64_t k1,
                              float *m, float *l, float *acc,
                              void *workspace, size_t workspace_bytes, void *stream);

/* The merge kernel alone: left fold over `n_parts` partial states of `rows` rows:
 * m' = max(m_a, m_b), l' = l_a e^{m_a-m'} + l_b e^{m_b-m'}, acc' likewise.  m, l: [n_parts, rows, H];
 * acc: [n_parts, rows, H*c]; outputs m_out, l_out [rows, H], acc_out [rows, H*c].  All fp32, device.  An empty
 * state (m = -inf, l = 0, acc = 0) is the identity of the fold, also when both operands are empty. */
dcp_status dcp_merge_states(int n_parts, int64_t rows, int H, int c, const float *m, const float *l,
                            const float *acc, float *m_out, float *l_out, float *acc_out, void *stream);

/* Eq. 5, host only: shard p of n items over `parts` shards. */
dcp_status dcp_shard_range(int64_t n, int parts, int p, int64_t *start, int64_t *len);

/* Host only: how a call with this plan is cut into work units on the tensor-core kernels -- key_segments (Eq.-5 segments
 * per key chunk), tile_q (query rows per unit) and slots (partial states per row = key chunks x segments); 1 / 0 / chunks
 * for the generic kernel.  key_segments depends on (I, key chunks) only, never on the row partition: that is what makes
 * row(P) == monolithic and grid(G x G) == monolithic(key_split = G) bitwise.  `plan` may be NULL. */
dcp_status dcp_plan_units(int64_t I, int H, int c, int c_z, dcp_dtype dtype, dcp_decomp decomp, const dcp_plan *plan,
                          int *key_segments, int *tile_q, int *slots);

/* 1 if fused kernel `kernel` (a dcp_kernel, not AUTO) is instantiated for this (dtype, H, c, c_z), else 0. Host only. */
int dcp_kernel_supported(int kernel, dcp_dtype dtype, int H, int c, int c_z);

/* Measurement probes (bench.py): kernels that compute nothing the method needs and exist to MEASURE the ceilings of the
 * two rows whose bound is neither HBM nor the tensor pipe.  dcp_probe_l2_gather: n_warps warps each make
 * gathers_per_warp (a multiple of 8) warp-level 128-bit loads covering two random 256-byte rows of `table`
 * [n_rows][256 bytes] (device, 16-byte aligned; keep it L2-resident): bytes moved = n_warps * gathers_per_warp * 512 --
 * the access pattern of the sparse atom attention's K / V gather.  dcp_probe_scan: one warp per query atom of x [L, 3]
 * scans all L candidates exactly like dcp_knn (binary32 distance in the pinned order, one compare + ballot per 32
 * candidates from shared-memory tiles) without selecting anything: L * L distance pairs.  `sink`: one device word,
 * never written in practice.  Both enqueue on `stream`. */
dcp_status dcp_probe_l2_gather(const void *table, int64_t n_rows, int64_t n_warps, int gathers_per_warp, uint32_t *sink,
                               void *stream);
dcp_status dcp_probe_scan(const float *x, int64_t L, uint32_t *sink, void *stream);

/* CUDA-event helpers for callers without a CUDA runtime binding (bench.py): timing-enabled events. */
dcp_status dcp_event_create(void **ev);
dcp_status dcp_event_record(void *ev, void *stream);
dcp_status dcp_event_elapsed_ms(void *ev_begin, void *ev_end, float *ms); /* synchronises on ev_end */
dcp_status dcp_event_destroy(void *ev);

/* Number of kernels the last dcp_pair_bias_attention* call on this thread launched (bench.py's gpu_launches). */
int dcp_last_launch_count(void);

const char *dcp_status_string(dcp_status st);
int dcp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DESIGNCP_H */
