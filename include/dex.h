/* dex.h — C ABI of the B200-native Depth Exploration Decoding (DEX) step library.
 *
 * One thing lives behind this boundary: the expand -> exit -> commit -> collapse step of
 * DEX (arxiv/paper_2606_29223), PAPER.md:143-190 (Alg. 1) and PAPER.md:196-208 (Sec. 3.2),
 * with greedy DECS decoding, PAPER.md:454-482 (Alg. 2).  Every call below is hand-written
 * CUDA for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - plain C, opaque handle, every call returns int32_t: DEX_OK or a negative DEX_E* code;
 *     dex_last_error() returns a static/ctx-owned string.  Nothing throws or aborts.
 *   - Ownership: ALL device memory (weights, workspace) is allocated by the caller and only
 *     borrowed; it must outlive the context.  The library never calls cudaMalloc.  It owns
 *     host-side bookkeeping and one small pinned host buffer for step results.
 *   - "device" / "host" is stated for every pointer.  All device pointers must be 16-byte
 *     aligned; the workspace 1024-byte aligned.
 *   - The CUDA stream is the caller's (cudaStream_t passed as void*); all work of a call is
 *     enqueued on it; calls that return results synchronise that stream before returning.
 *   - Not thread-safe per context.
 */
#ifndef DEX_B200_H
#define DEX_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DEX_OK          0
#define DEX_EINVAL     -1   /* bad argument / config (e.g. depth set violates Def. 4)   */
#define DEX_ECAPACITY  -2   /* workspace, max_ctx, max_seqs or row capacity exceeded     */
#define DEX_ESTATE     -3   /* call not legal in the current FSM state                   */
#define DEX_ECUDA      -4   /* a CUDA runtime / driver call failed (see dex_last_error)  */

#define DEX_MAX_DEPTHS  8   /* |X| <= 8: the range the paper evaluates    */

/* dex_step flags */
#define DEX_STEP_AUTOCOLLAPSE 1u  /* commit + collapse inside the step (Alg. 1 lines 9-13) */

typedef struct dex_ctx dex_ctx;

/* Model + runtime shape.  Llama-style pre-norm decoder (BASELINE.json:configs; reading R13
 * in DESIGN.md): RMSNorm, rotate-half RoPE, GQA, SwiGLU, untied embed / LM head, no biases;
 * every exit depth is decoded by the shared final RMSNorm + LM head. */
typedef struct dex_config {
  int32_t n_layers;      /* L                                                             */
  int32_t d_model;       /* d, multiple of 8                                              */
  int32_t n_heads;
  int32_t n_kv_heads;    /* divides n_heads                                               */
  int32_t head_dim;      /* 64 or 128                                                     */
  int32_t d_ffn;         /* multiple of 8                                                 */
  int32_t vocab;
  float   rms_eps;
  float   rope_theta;
  int32_t max_seqs;      /* independent sequences (lattices) batched into the same launches */
  int32_t max_ctx;       /* max committed positions per sequence (prompt + generated)     */
  int32_t page_size;     /* committed-KV page, positions; multiple of 64                  */
  int32_t decs;          /* 1: Alg. 2 masking of shallower slot-chain proposals; 0: plain argmax */
  int32_t eos_id;        /* -1: none (stop rule = max length only)      */
  int32_t debug_taps;    /* 1: keep per-layer hidden rows / anchor logits for dex_debug_read */
  int32_t act_planes;    /* 1: activations enter the MMAs as bf16; 2: as bf16 hi+lo pair  */
  int32_t use_graph;     /* 1: replay the step as a CUDA graph                            */
  int32_t round_kernel;  /* 1: one persistent kernel per round (k_round: phases separated by grid barriers; the
                            measured path); 0: one launch per op; 2: k_flow, the round as a barrier-free dataflow
                            program (experimental: bit-identical results, slower; falls back to k_round for shapes
                            its tables do not cover) */
  int32_t sample;        /* 0: greedy (Alg. 2 line 9); 1: sampling-mode DECS (Alg. 2 lines 10-15):
                            y = argmax_v (l_v / temperature + G_v) with a Gumbel(0,1) row shared by every depth of a
                            slot chain, drawn by a counter-based generator from (sample_seed, sequence, absolute
                            position of the decoded token) - reading R24 in DESIGN.md.  Needs round_kernel = 1 */
  float   temperature;   /* tau > 0 (sample = 1)                                           */
  int32_t sample_seed;
  int32_t adapter_dim;   /* m > 0: inducing-adapter exits (App. C.2): a row leaving the NON-final
                            depth d_k (k < N-1) is decoded from h~ = h + alpha_k (W2_k SiLU(W1_k RMSNorm(h; norm_k) + b1_k)
                            + b2_k) by the shared final norm + LM head; the hidden handed to deeper stages stays h
                            (lossless).  m is the adapter width (paper: 2 d_model), a multiple of 64,
                            <= d_ffn.  Needs round_kernel = 1, N >= 2 and the ad_* tensors of dex_weights.  0: off */
  int32_t lookahead;     /* P > 0: sparse exploration lattice (reading R26 in DESIGN.md): a node is expanded
                            only if it lies at most P token positions ahead of the commit position and its parent was
                            expanded; the commit takes the shallowest matching anchor whose continuation was explored.
                            Lossless for every P; P >= N-1 or 0: the full lattice of Sec. 3.2 */
} dex_config;

/* Device pointers to the packed tensors (row-major, "out x in"; layout = dex_synth/gen.py):
 *   embed [V,d] bf16, lm_head [V,d] bf16, wqkv [L,(nh+2nkv)*hd,d] bf16 (q heads, k heads, v heads),
 *   wo [L,d,nh*hd] bf16, wgu [L,2,ffn,d] bf16 (gate, up), wdn [L,d,ffn] bf16,
 *   norm_attn [L,d] f32, norm_ffn [L,d] f32, norm_final [d] f32;
 *   adapters (adapter_dim = m > 0 only, else ignored; one per non-final depth, k = 0..N-2):
 *   ad_w1 [N-1,m,d] bf16, ad_w2 [N-1,d,m] bf16, ad_b1 [N-1,m] f32, ad_b2 [N-1,d] f32, ad_norm [N-1,d] f32,
 *   ad_alpha [N-1] f32. */
typedef struct dex_weights {
  const void*  embed;
  const void*  lm_head;
  const void*  wqkv;
  const void*  wo;
  const void*  wgu;
  const void*  wdn;
  const float* norm_attn;
  const float* norm_ffn;
  const float* norm_final;
  const void*  ad_w1;
  const void*  ad_w2;
  const float* ad_b1;
  const float* ad_b2;
  const float* ad_norm;
  const float* ad_alpha;
} dex_weights;

/* Per-sequence record of one round of Alg. 1 (host memory). */
typedef struct dex_step_result {
  int32_t active;            /* sequence took part in this round                           */
  int32_t committed;         /* 1 if the anchor reached final depth and a token was committed */
  int32_t token;             /* y = u_{N-1}; -1 if none                     */
  int32_t match_k;           /* selected anchor branch b_k (N-1 = fallback); -1 if none    */
  int32_t q_before;          /* FSM state entering the round                               */
  int32_t q_after;           /* FSM state leaving it (after collapse / advance)            */
  int32_t exit_rows;         /* new lattice nodes decoded this round (2^q)                 */
  int32_t critical_layers;   /* max |Pi_m| over live stages (paper's charged depth)        */
  int64_t layer_evals;       /* sum_m rows_m * |Pi_m| executed this round                  */
  int32_t rows_per_stage[DEX_MAX_DEPTHS];
  int32_t anchor_tokens[DEX_MAX_DEPTHS]; /* u_0..u_{N-1} when the anchor is at final depth */
  float   ref_top1;          /* final-depth anchor's best and second-best logit            */
  float   ref_top2;
  int32_t n_tokens;          /* committed tokens incl. prompt after the round              */
  int32_t done;              /* eos hit or max_ctx reached                                 */
  int32_t branch_mask;       /* bit k: the continuation of anchor branch b_k (the position child of anchor k) was
                                explored, so a commit may collapse onto it; all ones on the full lattice */
  int32_t reserved;
} dex_step_result;

/* Bytes of device workspace dex_init needs (committed KV pages, slot KV, hidden rows,
 * activation planes, split-K partials, row tables, FSM, exit scratch).  host: cfg, depths, out. */
int32_t dex_workspace_bytes(const dex_config* cfg, const int32_t* depths, int32_t n_depths,
                            size_t* out_bytes);

/* Create a context.  depths (host): the exploration set X = {d_0 < ... < d_{N-1} = L}
 * (Def. 4), strictly increasing, in [1,L], last == L, N <= DEX_MAX_DEPTHS;
 * DEX_EINVAL otherwise.  depths = {L} IS the autoregressive baseline.  w (host struct of
 * device pointers), workspace (device, >= dex_workspace_bytes, 1024-aligned), stream
 * (cudaStream_t).  Builds TMA descriptors, RoPE tables, zeroes the FSM. */
int32_t dex_init(dex_ctx** out, const dex_config* cfg, const dex_weights* w,
                 const int32_t* depths, int32_t n_depths,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* S <- init(x, {E_k})  (Alg. 1 line 2; reading R3): resets sequence `seq`,
 * fills the committed K/V of prompt[0..n-2] at all layers (chunks of <=128 causal rows
 * through the same segment kernels), makes prompt[n-1] the first root-slot input, q <- 0.
 * prompt: host int32[n], 1 <= n <= max_ctx.  Returns after the work is enqueued. */
int32_t dex_prefill(dex_ctx* ctx, int32_t seq, const int32_t* prompt, int32_t n);

/* One round of Alg. 1 (lines 5-16) for every active sequence: expand all frontier nodes
 * through their next stage (one grouped launch per layer op), DECS-decode all new nodes,
 * insert into B; if the anchor reached final depth: validate_and_commit and, with
 * DEX_STEP_AUTOCOLLAPSE, collapse; else advance.  Without the flag a sequence whose anchor
 * reached final depth is left pending and must be finished with dex_collapse before the
 * next dex_step (DEX_ESTATE otherwise).  out: host dex_step_result[max_seqs].  Returns
 * after the results are visible on the host. */
int32_t dex_step(dex_ctx* ctx, uint32_t flags, dex_step_result* out);

/* collapse(B, S, q, b) as a primitive (Alg. 1 line 13): commit `token`
 * for sequence `seq`, append the root slot's K/V of all L layers to the committed pages,
 * keep the sub-tree consistent with anchor branch `branch_k` (N-1 = fallback: nothing
 * survives) and compact B, frontier hidden rows and slot K/V in place.  DEX_ESTATE unless a
 * commit is pending; DEX_EINVAL if branch_k < N-1 and B[anchor(branch_k)] != token or the branch's continuation
 * was not explored (sparse lattice, dex_step_result.branch_mask).
 * Used by tests and by the parity harness to teacher-force the oracle's token (R17). */
int32_t dex_collapse(dex_ctx* ctx, int32_t seq, int32_t branch_k, int32_t token);

/* Roll sequence `seq` back to its first n committed tokens (1 <= n <= committed count): the
 * lattice is emptied (q <- 0), committed K/V of positions >= n-1 is dropped (its pages return
 * to the pool), token n-1 becomes the next root-slot input, a pending commit is cancelled and
 * `done` is cleared.  K/V of positions < n-1 is untouched, so rewinding to the prompt length
 * restores exactly the state dex_prefill left (used by bench.py to repeat a run without
 * re-prefilling).  DEX_ESTATE if the sequence was never prefilled.  Enqueued, not synchronised. */
int32_t dex_rewind(dex_ctx* ctx, int32_t seq, int32_t n);

/* Committed tokens of a sequence (prompt included) -> host int32[cap]; *n_out = count. */
int32_t dex_get_tokens(dex_ctx* ctx, int32_t seq, int32_t* out, int32_t cap, int32_t* n_out);

/* Debug taps (cfg.debug_taps = 1 only; DEX_ESTATE otherwise).  dst: HOST buffers.
 *   DEX_TAP_HIDDEN : a = node id of the last round (level q_before) -> float[len_m * d],
 *                    residual stream after each layer of that node's stage
 *   DEX_TAP_LOGITS : final-depth anchor logits of the last round -> float[vocab]
 *                    (recomputed by a plain CUDA-core kernel from the anchor's exit row)
 *   DEX_TAP_REF_BLOCKS : what the FUSED exit itself reduced for the final-depth anchor of the last round (tcgen05
 *                    accumulators, no recompute): float[2 * 4 * ceil(vocab / 128)] = (top-1, top-2) logit of every block
 *                    of 32 consecutive vocabulary ids (-inf where a block has fewer than 1 / 2 live ids)
 *   DEX_TAP_B      : explore buffer B of `seq` -> int32[2^N - 1] (-1 = empty)
 *   DEX_TAP_FSM    : int32[4] = {q, ctx_len, n_tokens, pending}
 *   DEX_TAP_ROUND_TIMES : uint64[20 * max_m|Pi_m| + 4] SM clock-cycle stamps taken by CTA 0 of
 *                    the last round kernel: start, then after every item phase and grid barrier */
#define DEX_TAP_HIDDEN 1
#define DEX_TAP_LOGITS 2
#define DEX_TAP_B      3
#define DEX_TAP_FSM    4
#define DEX_TAP_ROUND_TIMES 5
#define DEX_TAP_REF_BLOCKS 6
int32_t dex_debug_read(dex_ctx* ctx, int32_t what, int32_t seq, int32_t a, void* dst, size_t dst_bytes);

/* Kernel-level tap for parity tests of the weight-streaming GEMM:
 * y[rows,out] (host f32) = x[rows,k] (host f32, split to bf16 planes on device) . W[out,k]^T
 * with W = weight kind `which` (0 qkv, 1 o, 2 gate/up, 3 down, 4 lm_head) of layer `layer`,
 * through exactly the launch configuration dex_step uses.  rows <= 128. */
int32_t dex_debug_gemm(dex_ctx* ctx, int32_t which, int32_t layer, const float* x, int32_t rows, float* y);

/* Per-kernel-class device time of the last dex_step in microseconds (CUDA events around each
 * launch on the context's stream; only while profiling is on (dex_profile), which bypasses graph
 * replay): host float[8] = {bookkeeping, segment GEMMs (or the whole round kernel), glue
 * (norm/rope/silu), attention, exit GEMM, commit+collapse, 0, total}. */
int32_t dex_debug_phase_us(dex_ctx* ctx, float* out8);

/* Measurement hook used by bench.py.  Copies out (host double[8] each, may be NULL) the
 * per-class device microseconds accumulated over the dex_step calls since the last reset
 * (same classes as dex_debug_phase_us; zeros unless profiling was on) and the counters
 * {rounds, kernel launches, segment-GEMM launches, segment-GEMM algorithmic weight bytes,
 *  exit-GEMM LM-head bytes (algorithmic: once per round), committed-KV bytes attended, LM-head bytes re-streamed for
 *  further live exit chunks (traffic, not algorithmic), 0}; then, if on >= 0, resets both
 * and switches profiling off (0), on (1: the configured launch structure, graph replay off) or on
 * through the per-op kernels (2: phase breakdown even when round_kernel = 1).  on < 0: read only. */
int32_t dex_profile(dex_ctx* ctx, int32_t on, double* phase_us_acc8, double* counters8);

/* The weight-streaming GEMM of the layer segment (north_star (a); the k_gemm kernel of dex_step's per-op path) through an
 * entry point that ALLOCATES NOTHING and needs no context - for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it):
 *     y[rows, out] (f32) = x[rows, k] (f32) . W[out, k]^T (bf16),  the same tiles and fixed K split as the context path.
 * w_dev: device, bf16 [out_dim, k_dim] row-major, 16-byte aligned; x_dev: device f32 [rows, k_dim]; y_dev: device f32
 * [rows, out_dim] (written); act_planes: 1 (x enters the MMA as bf16) or 2 (bf16 hi + lo pair, reading R23); stream:
 * cudaStream_t.  The work is enqueued on the stream, not synchronised.  The kernel's scratch (operand planes, row table,
 * split-K partials) is ONE static device array of 10 MiB + 8 KiB that every GPU loading the library holds until exit.
 * Limits: rows <= 32, k_dim <= 16384 (a multiple of 8), out_dim <= 262144 and
 * ceil(k_dim / 512) * round16(rows) * round4(out_dim) <= 2 Mi floats; DEX_ECAPACITY beyond them, DEX_EINVAL for null /
 * misaligned pointers or bad sizes, DEX_ECUDA if a CUDA call fails (message: dex_last_error(NULL)).  Every call shares the
 * array: calls on one stream are ordered, calls that OVERLAP on the GPU (several streams or threads) race on it.  Calls
 * no cudaMalloc / cudaFree or allocating library routine. */
int32_t dex_gemm_noalloc(const void* w_dev, const float* x_dev, int32_t rows, int32_t out_dim, int32_t k_dim,
                         int32_t act_planes, float* y_dev, void* cuda_stream);

int32_t dex_destroy(dex_ctx* ctx);
const char* dex_last_error(const dex_ctx* ctx);   /* ctx may be NULL: last global error */

#ifdef __cplusplus
}
#endif
#endif /* DEX_B200_H */
