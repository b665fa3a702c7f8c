// common.cuh — device-side state layout shared by the DEX kernels (HBM layout: DESIGN.md "Data layout").
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "../../include/dex.h"

namespace dexk {

constexpr int kMaxGrp = DEX_MAX_DEPTHS;
constexpr int kMaxAnc = DEX_MAX_DEPTHS;
constexpr int kChunk = 64;          // attention reduces over absolute positions in chunks of 64 (H3)
constexpr int kTileM = 128;         // GEMM: weight rows (out features) per MMA tile
constexpr int kTileK = 64;          // GEMM: bf16 K elements per pipeline stage (128 B rows, SW128)
constexpr int kBoxRows = 16;        // activation rows per TMA box
constexpr int kPrefillRows = 128;   // rows per prefill chunk
constexpr int kSsSeg = 64;          // sum-of-squares segments per row (128 elements each, d <= 8192)

// A "plan" = groups of stacked rows, each streaming its own layer segment.  Decode: group m =
// explorer E_m with stage Pi_m = Layers(d_{m-1}, d_m].  Prefill: one group
// over all L layers.  Exit: groups are <=256-row chunks of all rows, "layer" 0 of the LM head.
struct Plan {
  int n_grp;
  int row_base[kMaxGrp];   // first row of the group (multiple of 16)
  int rows_cap[kMaxGrp];   // row capacity (multiple of 16, <= 256)
  int layer_lo[kMaxGrp];   // d_{m-1}
  int layer_len[kMaxGrp];  // |Pi_m|
};

// One lattice row of the current round (an exploration token).
struct RowInfo {
  int valid;               // 0: dead row
  int seq;
  int node;                // heap id in the binary expansion tree (reading R2); prefill: -1
  int pos;                 // absolute token position (RoPE, causal limit)
  int grp;                 // plan group (= stage m for decode rows)
  int slot;                // compact slot id whose K/V this row writes; -1: write committed pages
  int n_paged;             // positions [0, n_paged) are read from committed pages
  int n_anc;               // positions n_paged + i, i < n_anc, are read from slot anc[i]; then own slot
  int anc[kMaxAnc];
  int parent_row;          // >= 0: h_in = frontier hidden of that row; -1: h_in = Embed[tok_in]
  int tok_in;
  int is_ref;              // final-depth anchor node 2^{N-1}-1: never masked (Alg. 2 lines 1-4)
  int n_mask;              // DECS: tokens proposed by shallower nodes of the same slot chain
  int mask_tok[kMaxAnc];
  int exit_row;            // dense index of this row among the round's valid rows: its row of the exit operand act_e
  int pad[3];
};
static_assert(sizeof(RowInfo) == 32 * 4, "RowInfo is 128 bytes");

// Per-sequence FSM and committed-prefix bookkeeping.
struct SeqState {
  int active;
  int q;                   // rounds completed since the last commit
  int ctx_len;             // committed K/V positions (= n_tok - 1)
  int n_tok;               // committed tokens incl. prompt
  int last_tok;            // x[n-1]: the next root-slot input
  int pending;             // anchor at final depth, commit not yet applied
  int done;
  int pad;
};

// What the apply/collapse kernels do for a sequence after a round.
struct CollapseCmd {
  int op;                  // 0 none, 1 advance (q+1), 2 commit+collapse, 3 hold (pending)
  int k_sel;
  int token;
  int q_old;
};

// All device pointers + shape; passed by value to kernels.
struct Dev {
  // shape
  int L, d, nh, nkv, hd, ffn, vocab, qkv_out;
  float eps;
  int N;                   // |X|
  int depths[kMaxGrp];     // X
  int max_seqs, max_ctx, page_size, pages_per_seq, n_slots;  // n_slots = 2^{N-1} compact slots / seq
  int n_nodes;             // 2^N - 1
  int R_cap;               // rows of every row-indexed buffer
  int R_dec;               // rows used by the decode plan
  int exit_chunk;          // rows per exit-head group (= largest decode group, rounded to 16: the exit shares the ring)
  int decs, planes, taps;
  int sample;              // sampling-mode DECS (Alg. 2 lines 10-15)
  float inv_tau;           // 1 / temperature
  unsigned sample_seed;
  int max_len;             // max_m |Pi_m|
  int lookahead;           // P > 0: position look-ahead cap of the sparse lattice (R26); 0: full lattice
  int ad_m;                // inducing-adapter width m (0: exits decode h directly); adapter k serves stage k < N-1
  const float *ad_b1, *ad_b2, *ad_norm, *ad_alpha;   // [N-1][m], [N-1][d], [N-1][d], [N-1]
  // weights
  const __nv_bfloat16 *embed, *lm_head;
  const float *norm_attn, *norm_ffn, *norm_final;
  // state
  SeqState* seqs;          // [max_seqs]
  int* tokens;             // [max_seqs][max_ctx + 1]
  int* B;                  // [max_seqs][n_nodes] explore buffer
  int* page_table;         // [max_seqs][pages_per_seq]
  __nv_bfloat16 *kpool, *vpool;   // [L][n_pages][page_size][nkv][hd]
  __nv_bfloat16 *kslot, *vslot;   // [max_seqs][n_slots][L][nkv][hd]
  float* x_cur;            // [R_cap][d] residual stream of this round's rows
  float* x_front;          // [R_cap][d] frontier hidden (h_out of the previous level)
  float* ss_part;          // [R_cap][kSsSeg] sum of squares of the row the last norm was taken of, per 128-element
                           // segment.  The RMSNorm scale is DEFERRED: operand planes hold x*w, consumers of the GEMM
                           // output multiply by inv_rms(row) = rsqrt(sum_seg ss / d + eps) (exact: the scale is per row)
  int* attn_cnt;           // [R_cap][nh] chunk partials written (last writer merges them)
  RowInfo* rows;           // [R_cap]
  int* grp_nb;             // [kMaxGrp] live row extent per decode/prefill group (multiple of 16)
  int* exit_nb;            // [kMaxGrp] live row extent per exit chunk (of the DENSE exit rows)
  int* exit_map;           // [R_cap] dense exit row -> lattice row (-1 beyond the round's valid rows).  The exit head works on
                           // dense rows, so a round streams the LM head once per exit_chunk VALID rows, not per row slot
  __nv_bfloat16 *act_a, *act_o, *act_f, *act_e;   // [planes][R_cap][K] MMA operands
  float* part;             // split-K partial sums, per op [S_op][R_cap][ld_op] (OpDesc)
  unsigned int* gbar;      // grid-barrier arrival counter of the round kernel (reset every round)
  void* item_recs;         // [grid][item_cap] 32-byte item records of k_flow (written by each CTA in its prologue)
  int item_cap;
  int* flow_ctr;           // [kFcTotal] arrival counters / ready flags of the dataflow round kernel (k_flow), zeroed every round
  float* qbuf;             // [R_cap][nh*hd]
  float* attn_part;        // [R_cap][nh][4 * max_chunks][hd + 2]: (o, max, sum) per 16 positions (k_round) / per chunk (k_attn)
  int max_chunks;
  float2* rope;            // [max_ctx + kMaxAnc + 1][hd/2] (cos, sin)
  unsigned long long* best_key;   // [R_cap]
  float2* ref_tile;        // [max_seqs][ref_tiles] per (tile, lane-quarter) top-2 of the anchor row
  int ref_tiles;
  CollapseCmd* cmd;        // [max_seqs]
  dex_step_result* result_dev;    // [max_seqs] (mapped pinned host memory)
  int* dbg_host;           // [16] mapped pinned host words behind the results: written by a kernel before it traps on a protocol timeout
  float* tap_hidden;       // [R_cap][max_len][d] (taps only)
  unsigned long long* tap_times;  // [20 * max_len + 4] globaltimer stamps of CTA 0 in k_round (taps only)
  int n_pages;
};

__host__ __device__ inline size_t kv_page_elems(const Dev& D) { return (size_t)D.page_size * D.nkv * D.hd; }
__host__ __device__ inline size_t kv_layer_elems(const Dev& D) { return (size_t)D.n_pages * kv_page_elems(D); }

// Address of K (or V) of committed position p of sequence s at layer l: [nkv][hd].
__device__ __forceinline__ size_t page_off(const Dev& D, int s, int l, int p) {
  int pg = D.page_table[s * D.pages_per_seq + p / D.page_size];
  return (size_t)l * kv_layer_elems(D) + (size_t)pg * kv_page_elems(D) + (size_t)(p % D.page_size) * D.nkv * D.hd;
}
__device__ __forceinline__ size_t slot_off(const Dev& D, int s, int slot, int l) {
  return (((size_t)s * D.n_slots + slot) * D.L + l) * D.nkv * D.hd;
}

// Order-preserving float -> uint32 (larger float <=> larger key).
__device__ __forceinline__ uint32_t f2key(float f) {
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
  uint32_t u = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
  return __uint_as_float(u);
}

// Sum of squares of four values in ONE fixed instruction sequence: every producer of ss_part (k_gather_norm, k_add_norm,
// the glue units of the round kernels) must give the same bits for the same x, whichever kernel computes it - a row's
// first norm of a stage is taken by k_gather_norm in a DEX round and by the previous layer's add+norm in the AR pass (H3).
__device__ __forceinline__ float sumsq4(float4 v) {
  return __fmaf_rn(v.w, v.w, __fmaf_rn(v.z, v.z, __fmaf_rn(v.y, v.y, __fmul_rn(v.x, v.x))));
}

__device__ __forceinline__ float inv_rms(const Dev& D, int r) {
  const float4* p = reinterpret_cast<const float4*>(D.ss_part + (size_t)r * kSsSeg);
  const int n4 = ((D.d + 127) / 128 + 3) / 4;            // float4 groups that hold segments (unused segments hold 0)
  float4 v[kSsSeg / 4];
#pragma unroll
  for (int i = 0; i < kSsSeg / 4; ++i) v[i] = (i < n4) ? p[i] : make_float4(0.f, 0.f, 0.f, 0.f);   // one batch of loads
  float ss = 0.f;
#pragma unroll
  for (int i = 0; i < kSsSeg / 4; ++i) ss += (v[i].x + v[i].y) + (v[i].z + v[i].w);   // fixed order
  return 1.0f / sqrtf(ss / (float)D.d + D.eps);
}

// Gumbel(0,1) noise of (seed, sequence, absolute position of the decoded token, vocabulary id): splitmix64 finaliser
// of a counter, 24-bit uniform, G = -log(-log u).  The CPU checker implements the same generator on its own (R24).
__device__ __forceinline__ float gumbel_noise(unsigned seed, int seq, int pos, int v) {
  const unsigned long long key = (unsigned long long)seed ^ ((unsigned long long)seq << 56);
  const unsigned long long ctr = ((unsigned long long)(unsigned)pos << 32) + (unsigned long long)(unsigned)v + 1ull;
  unsigned long long z = key + 0x9E3779B97F4A7C15ull * ctr;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  const float u = ((float)(unsigned)(z >> 41) + 0.5f) * 1.1920928955078125e-07f;   // 2^-23: exact in fp32
  return -logf(-logf(u));
}

// fp32 -> bf16 hi (+ lo residual) planes.
__device__ __forceinline__ void split_store(__nv_bfloat16* base, size_t plane_stride, size_t idx, float v, int planes) {
  __nv_bfloat16 hi = __float2bfloat16_rn(v);
  base[idx] = hi;
  if (planes > 1) base[plane_stride + idx] = __float2bfloat16_rn(v - __bfloat162float(hi));
}

// ---------------------------------------------------------------------------------------
// Tree arithmetic (heap reading R2: depth child 2i+1, position child 2i+2).  A node of
// level q is (q, o) with o in [0, 2^q): the bits of o, MSB first, are the moves from the
// root (0 = depth move, 1 = position move).
__host__ __device__ inline int node_id(int level, int o) { return (1 << level) - 1 + o; }
__host__ __device__ inline int node_level(int node) {
  int l = 0;
  while ((2 << l) - 1 <= node) ++l;
  return l;
}
__host__ __device__ inline int stage_of(int level, int o) {  // trailing depth moves
  if (o == 0) return level;
  int m = 0;
  while (((o >> m) & 1) == 0) ++m;
  return m;
}
__host__ __device__ inline int cap_of(int N, int m) {  // max rows of stage m per sequence
  int e = N - 2 - m;
  return e > 0 ? (1 << e) : 1;
}
// index of (level q, offset o) among the level's rows of its stage, ascending o
__host__ __device__ inline int idx_in_stage(int level, int o, int m) { return (m == level) ? 0 : (o >> (m + 1)); }
__host__ __device__ inline int compact_slot(int root_node) { return (root_node + 1) >> 1; }

struct GemmArgs {
  Plan plan;
  int step;                // layer-step j (layer = layer_lo[g] + j); groups with j >= layer_len are idle
  int out_dim, k_dim;
  int n_tiles;             // ceil(out / 128)
  int ksplit, kb_per_split, kb_total;
  int planes;
  int mode;                // 0: store split-K partials, 1: fused argmax (exit head)
  int x_cap;               // activation rows per ring stage (multiple of 16)
  int n_stages;            // ring depth
  int acc_cols;            // TMEM columns per accumulator stage (power of two >= 32)
  int n_acc;               // accumulator stages (2; 1 when two planes of 256 rows fill the 512 TMEM columns)
  int stacked;             // 1: both activation planes are one B operand of N = x_cap + nb (gemm_dev.cuh)
  const int* grp_nb;
  const RowInfo* rows;
  int n_rows;              // R_cap
  float* part;
  int part_ld;
  size_t part_split_stride;
  unsigned long long* best_key;
  float2* ref_tile;
  int ref_tiles;
  int vocab;
  const int* exit_map;     // mode 1: dense exit row -> lattice row
};

// One projection kind (Y = X . W^T) and its fixed split of K: the split depends on the operator
// shape only, never on how many rows or stages share a launch (H3: DEX stream == AR stream).
struct OpDesc {
  int out_dim, k_dim;
  int n_tiles;             // ceil(out / 128)
  int ksplit, kbps, kb_total;
  int part_ld;             // row stride of this op's partials (out rounded up to 4)
  size_t split_stride;     // R_cap * part_ld
};

struct TmSet {             // TMA descriptors of the round kernel: weights qkv,o,gu,dn,lm_head,ad_w1,ad_w2; operands a,o,f,e
  CUtensorMap w[7];
  CUtensorMap x[4];
  CUtensorMap wgu2;        // k_flow: gate/up viewed as [2L][ffn][d], so gate tile b and up tile b are both 128-row boxes
};

// k_flow (flow.cu): counters in Dev::flow_ctr.  All are monotonic within a round (targets scale with the layer-step).
constexpr int kFlowTiles = 256;                       // max 128-row tiles of one projection (per stage)
constexpr int kFlowSlices = 64;                       // max K slices (one item's K range) / KV heads
constexpr int kFcTile = 0;                            // [4 ops][8 stages][kFlowTiles] split arrivals of an out tile
constexpr int kFcXa = 4 * kMaxGrp * kFlowTiles;       // [8][64] down-proj tiles finalized per K slice of act_a (QKV operand)
constexpr int kFcAo = kFcXa + kMaxGrp * kFlowSlices;  // [8][64] (row, head) attention outputs merged per K slice of act_o
constexpr int kFcXf = kFcAo + kMaxGrp * kFlowSlices;  // [8][64] o-proj tiles finalized per K slice of act_a (gate/up operand)
constexpr int kFcF = kFcXf + kMaxGrp * kFlowSlices;   // [8][64] gate/up pairs finalized per K slice of act_f (down operand)
constexpr int kFcQkv = kFcF + kMaxGrp * kFlowSlices;  // [8][64] QKV tiles finalized per KV head group
constexpr int kFcTotal = kFcQkv + kMaxGrp * kFlowSlices;
// Dev-independent tables of k_flow (host-built, RoundArgs::flow_tab): QKV tile order + the KV groups a tile touches
constexpr int kFtPerm = 0, kFtGlo = kFlowTiles, kFtGhi = 2 * kFlowTiles, kFtTarget = 3 * kFlowTiles, kFtTotal = 3 * kFlowTiles + kFlowSlices;

struct RoundArgs {
  Dev D;
  Plan dec, ext;
  OpDesc op[7];                    // qkv, o, gate/up, down, lm_head, adapter W1, adapter W2
  int x_cap, n_stages, acc_cols, stacked;   // shared-memory ring / TMEM geometry
  int n_chunks;                    // attention chunks that can hold a live position (host upper bound)
  int attn_smem_off;               // byte offset of the attention scratch (AttnSmem) in dynamic shared memory
  const int* flow_tab;             // k_flow: [kFtTotal] QKV tile order, KV groups touched by a tile, tiles per group
  size_t part_off[4];              // k_flow: float offset of each layer op's own split-K partial region in Dev::part
};

}  // namespace dexk
