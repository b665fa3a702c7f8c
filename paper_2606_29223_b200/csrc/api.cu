// api.cu — the C ABI of include/dex.h: context, workspace carving, TMA descriptors, page
// allocator, launch sequence of one DEX round (Alg. 1 lines 5-16), prefill,
// collapse primitive, debug taps.  Host logic only; every step of the path runs in the kernels.
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <vector>

#include "common.cuh"

namespace dexk {
cudaError_t gemm_init();
cudaError_t launch_gemm(const CUtensorMap&, const CUtensorMap&, const GemmArgs&, int, size_t, cudaStream_t);
cudaError_t launch_rows_decode(const Dev&, const Plan&, cudaStream_t);
cudaError_t launch_rows_prefill(const Dev&, int, int, int, cudaStream_t);
cudaError_t launch_seq_init(const Dev&, int, int, cudaStream_t);
cudaError_t launch_rope_table(const Dev&, double, int, cudaStream_t);
cudaError_t launch_gather_norm(const Dev&, const Plan&, int, cudaStream_t);
cudaError_t launch_add_norm(const Dev&, const Plan&, int, int, int, const OpDesc&, cudaStream_t);
cudaError_t launch_rope_kv(const Dev&, const Plan&, int, int, const OpDesc&, cudaStream_t);
cudaError_t launch_silu_mul(const Dev&, const Plan&, int, int, const OpDesc&, cudaStream_t);
cudaError_t round_init();
size_t round_attn_smem(int);
cudaError_t launch_round(const TmSet&, const RoundArgs&, int, size_t, cudaStream_t);
cudaError_t flow_init();
cudaError_t launch_flow(const TmSet&, const RoundArgs&, int, size_t, cudaStream_t);
cudaError_t launch_attn(const Dev&, const Plan&, int, int, int, int, cudaStream_t);
cudaError_t launch_decide(const Dev&, const Plan&, int, cudaStream_t);
cudaError_t launch_set_cmd(const Dev&, int, int, int, cudaStream_t);
cudaError_t launch_collapse(const Dev&, const Plan&, int, cudaStream_t);
cudaError_t launch_tap_logits(const Dev&, int, float*, cudaStream_t);
cudaError_t launch_tap_ref_tiles(const Dev&, int, int, float2*, cudaStream_t);
cudaError_t launch_debug_rows(const Dev&, int, cudaStream_t);
cudaError_t launch_debug_split(const float*, __nv_bfloat16*, int, int, size_t, int, cudaStream_t);
cudaError_t launch_debug_sum(const float*, float*, int, int, int, int, size_t, cudaStream_t);
}  // namespace dexk

using namespace dexk;

namespace {

std::string g_last_error;

struct OpCfg {          // one projection: Y = X . W^T
  CUtensorMap tmW;
  OpDesc dec;           // decode rounds: fine fixed K split (items of <= kDecodeKb K-blocks)
  OpDesc pre;           // prefill chunks (128 rows): coarse split, fewer partials
};
constexpr int kDecodeKb = 8;
struct RingCfg {        // shared-memory ring of the GEMM for a plan
  int x_cap, n_stages, acc_cols, n_acc, stacked;
  size_t smem;
};
struct HostSeq {
  int active = 0, q = 0, ctx_len = 0, n_tok = 0, pending = 0, done = 0;
  int anchor_tokens[DEX_MAX_DEPTHS];
  int branch_mask = 0;
  int last_q_before = 0;
  std::vector<int> pages;
};
enum Phase { PH_BOOK = 0, PH_GEMM, PH_GLUE, PH_ATTN, PH_EXIT, PH_COMMIT, PH_N };

}  // namespace

struct dex_ctx {
  dex_config cfg;
  Dev D;
  Plan dec_plan, pre_plan, exit_plan;
  RingCfg dec_ring, pre_ring, exit_ring;
  OpCfg op[7];                        // qkv, o, gate/up, down, lm_head, adapter W1, adapter W2
  CUtensorMap tmX[4];                 // act_a, act_o, act_f, act_e
  cudaStream_t stream;
  int n_sms;
  std::vector<HostSeq> seqs;
  std::vector<int> free_pages;
  std::vector<int> page_table_host;
  dex_step_result* result_host;       // pinned, mapped
  float* dbg_stage;                   // device staging for debug taps (taps only)
  size_t dbg_floats;
  TmSet tms;
  RingCfg round_ring;
  int round_attn_off;
  bool round_ok;                      // the round kernel's ring + attention scratch fit shared memory
  bool flow_ok;                       // the shape fits the dataflow round kernel's tables (else round_kernel = 2 runs k_round)
  const int* flow_tab;                // device copy of the k_flow tables (QKV tile order, KV groups per tile)
  size_t part_off[4];                 // k_flow: float offsets of the per-op split-K partial regions
  bool has_ad;                        // inducing-adapter exits (cfg.adapter_dim > 0, N >= 2): round kernel only
  std::map<long long, cudaGraphExec_t> graphs;
  std::string err;
  // phase timing (taps only)
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev[PH_N];
  size_t ev_used[PH_N];
  float phase_us[8];
  double phase_us_acc[8];
  int profiling;
  int phase_split;                    // profiling through the per-op kernels (phase breakdown) instead of k_round
  double counters[8];                 // rounds, kernel launches, gemm launches, gemm weight bytes, exit bytes, kv bytes
};

namespace {

int fail(dex_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_last_error = buf;
  if (c) c->err = buf;
  return code;
}
#define CU(c, call)                                                                      \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess) return fail(c, DEX_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
int cu_or_fail0(dex_ctx* c, cudaError_t e, const char* what) {
  if (e != cudaSuccess) return fail(c, DEX_ECUDA, "%s: %s", what, cudaGetErrorString(e));
  return DEX_OK;
}
int round16i(int v) { return (v + 15) & ~15; }

int validate(const dex_config* cfg, const int32_t* depths, int32_t n) {
  if (!cfg || !depths) return fail(nullptr, DEX_EINVAL, "null config / depths");
  if (n < 1 || n > DEX_MAX_DEPTHS) return fail(nullptr, DEX_EINVAL, "n_depths must be in [1,%d]", DEX_MAX_DEPTHS);
  for (int i = 0; i < n; ++i) {
    if (depths[i] < 1 || depths[i] > cfg->n_layers || (i && depths[i] <= depths[i - 1]))
      return fail(nullptr, DEX_EINVAL, "exploration set must be strictly increasing in [1,L] (Def. 4)");
  }
  if (depths[n - 1] != cfg->n_layers) return fail(nullptr, DEX_EINVAL, "exploration set must end at L (Def. 4)");
  if (cfg->head_dim != 64 && cfg->head_dim != 128) return fail(nullptr, DEX_EINVAL, "head_dim must be 64 or 128");
  if (cfg->n_kv_heads < 1 || cfg->n_heads % cfg->n_kv_heads) return fail(nullptr, DEX_EINVAL, "n_kv_heads must divide n_heads");
  if (cfg->d_model % 8 || cfg->d_ffn % 8) return fail(nullptr, DEX_EINVAL, "d_model and d_ffn must be multiples of 8");
  if (cfg->page_size < 64 || cfg->page_size % 64) return fail(nullptr, DEX_EINVAL, "page_size must be a multiple of 64");
  if (cfg->max_seqs < 1 || cfg->max_seqs > 8) return fail(nullptr, DEX_EINVAL, "max_seqs must be in [1,8]");
  if (cfg->max_ctx < 2) return fail(nullptr, DEX_EINVAL, "max_ctx too small");
  if (cfg->round_kernel < 0 || cfg->round_kernel > 2) return fail(nullptr, DEX_EINVAL, "round_kernel must be 0, 1 or 2");
  if (cfg->sample != 0 && cfg->sample != 1) return fail(nullptr, DEX_EINVAL, "sample must be 0 or 1");
  if (cfg->sample && !(cfg->temperature > 0.f)) return fail(nullptr, DEX_EINVAL, "temperature must be > 0");
  if (cfg->sample && !cfg->round_kernel) return fail(nullptr, DEX_EINVAL, "sampling mode needs round_kernel >= 1");
  if (cfg->act_planes != 1 && cfg->act_planes != 2) return fail(nullptr, DEX_EINVAL, "act_planes must be 1 or 2");
  if (cfg->vocab < 2) return fail(nullptr, DEX_EINVAL, "vocab too small");
  if (cfg->lookahead < 0) return fail(nullptr, DEX_EINVAL, "lookahead must be >= 0");
  if (cfg->adapter_dim < 0 || cfg->adapter_dim % 64 || cfg->adapter_dim > cfg->d_ffn)
    return fail(nullptr, DEX_EINVAL, "adapter_dim must be a multiple of 64 in [0, d_ffn]");
  if (cfg->adapter_dim && !cfg->round_kernel) return fail(nullptr, DEX_EINVAL, "inducing adapters need round_kernel >= 1");
  if (cfg->adapter_dim && n < 2) return fail(nullptr, DEX_EINVAL, "inducing adapters need a non-final depth (N >= 2)");
  if (cfg->d_model > 8192) return fail(nullptr, DEX_ECAPACITY, "d_model > 8192 not supported");
  if (cfg->max_seqs * cap_of(n, 0) > 256) return fail(nullptr, DEX_ECAPACITY, "max_seqs * 2^(N-2) rows exceed 256 per stage");
  return DEX_OK;
}

void fill_desc(OpDesc& o, int out, int k, int R_cap) {
  o.out_dim = out;
  o.k_dim = k;
  o.n_tiles = (out + kTileM - 1) / kTileM;
  o.kb_total = (k + kTileK - 1) / kTileK;
  o.part_ld = (int)align_up((size_t)out, 4);
  o.split_stride = (size_t)R_cap * o.part_ld;
}
// prefill: split K only as far as needed to give every SM work
void split_coarse(OpDesc& o, bool allow_split) {
  int S = 1;
  if (allow_split)
    while (S < 8 && o.n_tiles * S < 256 && S * 2 <= o.kb_total) S *= 2;
  o.kbps = (o.kb_total + S - 1) / S;
  o.ksplit = (o.kb_total + o.kbps - 1) / o.kbps;
}
// decode: items of <= kDecodeKb K-blocks (128 KiB of weights): many small items, dealt round-robin
// across the ops of a round, keep every SM's byte count equal and fit the prefetch ring
void split_fine(OpDesc& o, bool allow_split) {
  o.kbps = allow_split ? std::min(kDecodeKb, o.kb_total) : o.kb_total;
  o.ksplit = (o.kb_total + o.kbps - 1) / o.kbps;
}

// Shape-only quantities shared by dex_workspace_bytes and dex_init.
struct Layout {
  int N, R_dec, R_cap, exit_chunk, max_chunks, n_slots, n_nodes, pages_per_seq, n_pages, max_len, ref_tiles;
  Plan dec, pre, ext;
  OpCfg op[7];
  size_t part_floats;
  size_t part_off[4];
  int item_cap;
  size_t off[40];
  size_t total;
  size_t dbg_floats;
};
enum Buf {
  B_SEQS, B_TOKENS, B_B, B_PT, B_ROWS, B_GNB, B_ENB, B_KEY, B_REFT, B_CMD, B_SS, B_ACNT, B_KPOOL, B_VPOOL, B_KSLOT, B_VSLOT,
  B_XCUR, B_XFRONT, B_ACTA, B_ACTO, B_ACTF, B_ACTE, B_PART, B_QBUF, B_APART, B_ROPE, B_TAPH, B_DBG, B_GBAR, B_TAPT, B_FCTR, B_FTAB, B_ITEMS, B_EMAP, B_COUNT
};

void make_layout(const dex_config& c, const int32_t* depths, int n, Layout& L) {
  memset(&L, 0, sizeof(Layout));
  L.N = n;
  L.n_nodes = (1 << n) - 1;
  L.n_slots = 1 << (n - 1);
  int base = 0;
  L.dec.n_grp = n;
  L.max_len = 0;
  for (int m = 0; m < n; ++m) {
    L.dec.row_base[m] = base;
    L.dec.rows_cap[m] = c.max_seqs * cap_of(n, m);      // compact: a 16-row TMA box may run into the next group
    L.dec.layer_lo[m] = m ? depths[m - 1] : 0;
    L.dec.layer_len[m] = depths[m] - L.dec.layer_lo[m];
    L.max_len = std::max(L.max_len, L.dec.layer_len[m]);
    base += L.dec.rows_cap[m];
  }
  L.R_dec = base;
  L.R_cap = round16i(std::max(L.R_dec, kPrefillRows)) + 16;
  L.pre.n_grp = 1;
  L.pre.row_base[0] = 0;
  L.pre.rows_cap[0] = kPrefillRows;
  L.pre.layer_lo[0] = 0;
  L.pre.layer_len[0] = c.n_layers;
  // exit-head groups: chunks of the largest decode group's size, so the exit op fits the decode ring geometry
  // (the LM head is streamed once per chunk: 2 chunks at N = 8, where all rows = 2 x the stage-0 rows)
  L.exit_chunk = std::min(256, round16i(L.dec.rows_cap[0]));
  L.ext.n_grp = (L.R_dec + L.exit_chunk - 1) / L.exit_chunk;
  for (int g = 0; g < L.ext.n_grp; ++g) {
    L.ext.row_base[g] = L.exit_chunk * g;
    L.ext.rows_cap[g] = std::min(L.exit_chunk, L.R_dec - L.exit_chunk * g);
    L.ext.layer_lo[g] = 0;
    L.ext.layer_len[g] = 1;
  }
  const int qkv_out = (c.n_heads + 2 * c.n_kv_heads) * c.head_dim;
  const int outs[5] = {qkv_out, c.d_model, 2 * c.d_ffn, c.d_model, c.vocab};
  const int ks[5] = {c.d_model, c.n_heads * c.head_dim, c.d_model, c.d_ffn, c.d_model};
  L.part_floats = 0;
  for (int i = 0; i < 5; ++i) {
    fill_desc(L.op[i].dec, outs[i], ks[i], L.R_cap);
    fill_desc(L.op[i].pre, outs[i], ks[i], L.R_cap);
    split_fine(L.op[i].dec, i != 4);
    split_coarse(L.op[i].pre, i != 4);
    if (i != 4) {
      L.part_floats = std::max(L.part_floats, (size_t)L.op[i].dec.ksplit * L.op[i].dec.split_stride);
      L.part_floats = std::max(L.part_floats, (size_t)L.op[i].pre.ksplit * L.op[i].pre.split_stride);
    }
  }
  if (c.adapter_dim > 0) {   // adapter projections: decode rounds only
    const int ao[2] = {c.adapter_dim, c.d_model}, ak[2] = {c.d_model, c.adapter_dim};
    for (int i = 0; i < 2; ++i) {
      fill_desc(L.op[5 + i].dec, ao[i], ak[i], L.R_cap);
      split_fine(L.op[5 + i].dec, true);
      L.op[5 + i].pre = L.op[5 + i].dec;
      L.part_floats = std::max(L.part_floats, (size_t)L.op[5 + i].dec.ksplit * L.op[5 + i].dec.split_stride);
    }
  }
  {   // k_flow keeps the partials of the four layer ops in regions of their own (ops of a layer-step overlap there)
    size_t off = 0;
    for (int i = 0; i < 4; ++i) {
      L.part_off[i] = off;
      off += align_up((size_t)L.op[i].dec.ksplit * L.op[i].dec.split_stride, 256);
    }
    L.part_floats = std::max(L.part_floats, off);
  }
  L.max_chunks = (c.max_ctx + n) / kChunk + 1;
  L.pages_per_seq = (c.max_ctx + c.page_size - 1) / c.page_size;
  L.n_pages = L.pages_per_seq * c.max_seqs;
  L.ref_tiles = L.op[4].dec.n_tiles * 4;
  L.dbg_floats = c.debug_taps ? (size_t)kPrefillRows * (std::max(c.d_ffn, c.d_model) + std::max(std::max(qkv_out, 2 * c.d_ffn), c.d_model) + 4) + c.vocab : 0;

  const size_t kv_pool = (size_t)c.n_layers * L.n_pages * c.page_size * c.n_kv_heads * c.head_dim * 2;
  const size_t kv_slot = (size_t)c.max_seqs * L.n_slots * c.n_layers * c.n_kv_heads * c.head_dim * 2;
  const size_t P = c.act_planes, R = L.R_cap;
  size_t sz[B_COUNT];
  sz[B_SEQS] = sizeof(SeqState) * c.max_seqs;
  sz[B_TOKENS] = sizeof(int) * (size_t)c.max_seqs * (c.max_ctx + 1);
  sz[B_B] = sizeof(int) * (size_t)c.max_seqs * L.n_nodes;
  sz[B_PT] = sizeof(int) * (size_t)L.n_pages;
  sz[B_ROWS] = sizeof(RowInfo) * R;
  sz[B_GNB] = sizeof(int) * kMaxGrp;
  sz[B_ENB] = sizeof(int) * kMaxGrp;
  sz[B_KEY] = sizeof(unsigned long long) * R;
  sz[B_REFT] = sizeof(float2) * (size_t)c.max_seqs * L.ref_tiles;
  sz[B_CMD] = sizeof(CollapseCmd) * c.max_seqs;
  sz[B_SS] = sizeof(float) * R * kSsSeg;
  sz[B_ACNT] = sizeof(int) * R * c.n_heads;
  sz[B_KPOOL] = kv_pool;
  sz[B_VPOOL] = kv_pool;
  sz[B_KSLOT] = kv_slot;
  sz[B_VSLOT] = kv_slot;
  sz[B_XCUR] = sizeof(float) * R * c.d_model;
  sz[B_XFRONT] = sizeof(float) * R * c.d_model;
  sz[B_ACTA] = 2 * P * R * c.d_model;
  sz[B_ACTO] = 2 * P * R * c.n_heads * c.head_dim;
  sz[B_ACTF] = 2 * P * R * c.d_ffn;
  sz[B_ACTE] = 2 * P * R * c.d_model;
  sz[B_PART] = sizeof(float) * L.part_floats;
  sz[B_QBUF] = sizeof(float) * R * c.n_heads * c.head_dim;
  sz[B_APART] = sizeof(float) * R * c.n_heads * (size_t)L.max_chunks * 4 * (c.head_dim + 2);   // k_round: 4 sub-partials per chunk
  sz[B_ROPE] = sizeof(float2) * (size_t)(c.max_ctx + kMaxAnc + 1) * (c.head_dim / 2);
  sz[B_TAPH] = c.debug_taps ? sizeof(float) * R * (size_t)L.max_len * c.d_model : 0;
  sz[B_DBG] = sizeof(float) * L.dbg_floats;
  sz[B_GBAR] = 256;
  sz[B_TAPT] = c.debug_taps ? sizeof(unsigned long long) * (20 * (size_t)L.max_len + 68) : 0;
  {   // k_flow item records: all items of a round / 128 CTAs (the launch needs >= 128 SMs) + one per op + slack
    size_t items = 0;
    for (int i = 0; i < 4; ++i) items += (size_t)L.op[i].dec.n_tiles * L.op[i].dec.ksplit;
    items *= (size_t)n * L.max_len;
    if (c.adapter_dim > 0) items += (size_t)(n - 1) * ((size_t)L.op[5].dec.n_tiles * L.op[5].dec.ksplit + (size_t)L.op[6].dec.n_tiles * L.op[6].dec.ksplit);
    items += (size_t)L.ext.n_grp * L.op[4].dec.n_tiles;
    L.item_cap = (int)(items / 128 + 4 * L.max_len * n + 3 + 16);   // + one per (op, stage) for the round-robin remainders
  }
  sz[B_ITEMS] = (size_t)32 * L.item_cap * 160;              // up to 160 CTAs
  sz[B_EMAP] = sizeof(int) * R;
  sz[B_FCTR] = sizeof(int) * kFcTotal;
  sz[B_FTAB] = sizeof(int) * kFtTotal;
  size_t off = 0;
  for (int i = 0; i < B_COUNT; ++i) {
    L.off[i] = off;
    off += align_up(sz[i], 1024);
  }
  L.total = off;
}

RingCfg make_ring(const Plan& p, int planes) {
  RingCfg r;
  r.x_cap = 16;
  for (int g = 0; g < p.n_grp; ++g) r.x_cap = std::max(r.x_cap, round16i(p.rows_cap[g]));
  const size_t stage = 16384 + (size_t)planes * r.x_cap * 128;
  const size_t budget = 200 * 1024;
  r.n_stages = (int)std::max<size_t>(2, std::min<size_t>(12, budget / stage));
  r.stacked = (planes == 2 && 2 * r.x_cap <= 256) ? 1 : 0;   // one {64, 16, 2} box per 16 rows, N = 2*nb
  r.acc_cols = 32;                                           // hi and lo sums in columns of their own in either layout
  while (r.acc_cols < planes * r.x_cap) r.acc_cols *= 2;
  r.n_acc = 2 * r.acc_cols <= 512 ? 2 : 1;
  r.smem = r.n_stages * stage + 1024 + 512;
  return r;
}

typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int encode_3d(dex_ctx* c, EncodeFn fn, CUtensorMap* tm, const void* base, uint64_t d0, uint64_t d1, uint64_t d2,
              uint32_t box1, uint32_t box2 = 1) {
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
  cuuint32_t box[3] = {(cuuint32_t)kTileK, box1, box2};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(c, DEX_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return DEX_OK;
}

// ---- phase timing (taps only) ----
void ph_begin(dex_ctx* c, Phase p) {
  if (!c->profiling) return;
  if (c->ev_used[p] == c->ev[p].size()) {
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    c->ev[p].push_back({a, b});
  }
  cudaEventRecord(c->ev[p][c->ev_used[p]].first, c->stream);
}
void ph_end(dex_ctx* c, Phase p) {
  if (!c->profiling) return;
  cudaEventRecord(c->ev[p][c->ev_used[p]].second, c->stream);
  c->ev_used[p]++;
}

int run_gemm(dex_ctx* c, int which, const OpDesc& o, const CUtensorMap& tmX, const Plan& plan, const RingCfg& ring, int step,
             int mode, const int* grp_nb) {
  GemmArgs a;
  memset(&a, 0, sizeof a);
  a.plan = plan;
  a.step = step;
  a.out_dim = o.out_dim;
  a.k_dim = o.k_dim;
  a.n_tiles = o.n_tiles;
  a.ksplit = o.ksplit;
  a.kb_per_split = o.kbps;
  a.kb_total = o.kb_total;
  a.planes = c->cfg.act_planes;
  a.mode = mode;
  a.x_cap = ring.x_cap;
  a.n_stages = ring.n_stages;
  a.acc_cols = ring.acc_cols;
  a.n_acc = ring.n_acc;
  a.stacked = ring.stacked;
  a.grp_nb = grp_nb;
  a.rows = c->D.rows;
  a.n_rows = c->D.R_cap;
  a.part = c->D.part;
  a.part_ld = o.part_ld;
  a.part_split_stride = o.split_stride;
  a.best_key = c->D.best_key;
  a.ref_tile = c->D.ref_tile;
  a.ref_tiles = c->D.ref_tiles;
  a.vocab = c->D.vocab;
  a.exit_map = c->D.exit_map;
  if (which == 4) {   // the LM head is one [V, d] matrix: every exit chunk streams "layer" 0
    for (int g = 0; g < kMaxGrp; ++g) a.plan.layer_lo[g] = 0;
  }
  CU(c, launch_gemm(c->op[which].tmW, tmX, a, c->n_sms, ring.smem, c->stream));
  return DEX_OK;
}

// Layers of one plan: for j = 0 .. max_len-1, every live group runs its layer lo+j (a2 + a3).
int enqueue_layers(dex_ctx* c, const Plan& plan, const RingCfg& ring, int rows, int n_chunks, int max_len, bool prefill) {
  const Dev& D = c->D;
  const OpDesc* o[4];
  for (int i = 0; i < 4; ++i) o[i] = prefill ? &c->op[i].pre : &c->op[i].dec;
  for (int j = 0; j < max_len; ++j) {
    int rc;
    ph_begin(c, PH_GEMM);
    rc = run_gemm(c, 0, *o[0], c->tmX[0], plan, ring, j, 0, D.grp_nb);
    ph_end(c, PH_GEMM);
    if (rc) return rc;
    ph_begin(c, PH_GLUE);
    CU(c, launch_rope_kv(D, plan, rows, j, *o[0], c->stream));
    ph_end(c, PH_GLUE);
    ph_begin(c, PH_ATTN);
    CU(c, launch_attn(D, plan, rows, j, n_chunks, prefill ? 0 : 1, c->stream));
    ph_end(c, PH_ATTN);
    ph_begin(c, PH_GEMM);
    rc = run_gemm(c, 1, *o[1], c->tmX[1], plan, ring, j, 0, D.grp_nb);
    ph_end(c, PH_GEMM);
    if (rc) return rc;
    ph_begin(c, PH_GLUE);
    CU(c, launch_add_norm(D, plan, rows, j, 0, *o[1], c->stream));
    ph_end(c, PH_GLUE);
    ph_begin(c, PH_GEMM);
    rc = run_gemm(c, 2, *o[2], c->tmX[0], plan, ring, j, 0, D.grp_nb);
    ph_end(c, PH_GEMM);
    if (rc) return rc;
    ph_begin(c, PH_GLUE);
    CU(c, launch_silu_mul(D, plan, rows, j, *o[2], c->stream));
    ph_end(c, PH_GLUE);
    ph_begin(c, PH_GEMM);
    rc = run_gemm(c, 3, *o[3], c->tmX[2], plan, ring, j, 0, D.grp_nb);
    ph_end(c, PH_GEMM);
    if (rc) return rc;
    ph_begin(c, PH_GLUE);
    CU(c, launch_add_norm(D, plan, rows, j, 1, *o[3], c->stream));
    ph_end(c, PH_GLUE);
  }
  return DEX_OK;
}

// The persistent round kernel: all layer-steps of all live stages + the exit head in one launch.
int enqueue_round(dex_ctx* c, int n_chunks) {
  RoundArgs a;
  memset(&a, 0, sizeof a);
  a.D = c->D;
  a.dec = c->dec_plan;
  a.ext = c->exit_plan;
  for (int i = 0; i < 7; ++i) a.op[i] = c->op[i].dec;
  a.x_cap = c->round_ring.x_cap;
  a.n_stages = c->round_ring.n_stages;
  a.acc_cols = c->round_ring.acc_cols;
  a.stacked = c->round_ring.stacked;
  a.n_chunks = n_chunks;
  a.attn_smem_off = c->round_attn_off;
  a.flow_tab = c->flow_tab;
  for (int i = 0; i < 4; ++i) a.part_off[i] = c->part_off[i];
  ph_begin(c, PH_GEMM);
  if (c->cfg.round_kernel == 2 && c->flow_ok) CU(c, launch_flow(c->tms, a, c->n_sms, c->round_ring.smem, c->stream));
  else CU(c, launch_round(c->tms, a, c->n_sms, c->round_ring.smem, c->stream));
  ph_end(c, PH_GEMM);
  return DEX_OK;
}

int enqueue_collapse(dex_ctx* c) {
  ph_begin(c, PH_COMMIT);
  CU(c, launch_collapse(c->D, c->dec_plan, c->cfg.eos_id, c->stream));
  ph_end(c, PH_COMMIT);
  return DEX_OK;
}

int enqueue_step(dex_ctx* c, uint32_t flags, int n_chunks) {
  const Dev& D = c->D;
  ph_begin(c, PH_BOOK);
  CU(c, launch_rows_decode(D, c->dec_plan, c->stream));
  CU(c, launch_gather_norm(D, c->dec_plan, D.R_dec, c->stream));
  ph_end(c, PH_BOOK);
  int rc;
  if (c->cfg.round_kernel && c->round_ok && (!c->phase_split || c->cfg.sample || c->has_ad)) {
    rc = enqueue_round(c, n_chunks);
    if (rc) return rc;
  } else {
    rc = enqueue_layers(c, c->dec_plan, c->dec_ring, D.R_dec, n_chunks, D.max_len, false);
    if (rc) return rc;
    ph_begin(c, PH_EXIT);
    rc = run_gemm(c, 4, c->op[4].dec, c->tmX[3], c->exit_plan, c->exit_ring, 0, 1, D.exit_nb);
    ph_end(c, PH_EXIT);
    if (rc) return rc;
  }
  ph_begin(c, PH_COMMIT);
  CU(c, launch_decide(D, c->dec_plan, (flags & DEX_STEP_AUTOCOLLAPSE) ? 1 : 0, c->stream));
  ph_end(c, PH_COMMIT);
  return enqueue_collapse(c);
}

int ensure_pages(dex_ctx* c, int s, int n_positions) {
  HostSeq& hs = c->seqs[s];
  const int need = (n_positions + c->cfg.page_size - 1) / c->cfg.page_size;
  if (need > c->D.pages_per_seq) return fail(c, DEX_ECAPACITY, "sequence %d exceeds max_ctx", s);
  bool changed = false;
  while ((int)hs.pages.size() < need) {
    if (c->free_pages.empty()) return fail(c, DEX_ECAPACITY, "out of KV pages");
    int pg = c->free_pages.back();
    c->free_pages.pop_back();
    c->page_table_host[s * c->D.pages_per_seq + hs.pages.size()] = pg;
    hs.pages.push_back(pg);
    changed = true;
  }
  if (changed)
    CU(c, cudaMemcpyAsync(c->D.page_table + s * c->D.pages_per_seq, &c->page_table_host[s * c->D.pages_per_seq],
                          sizeof(int) * c->D.pages_per_seq, cudaMemcpyHostToDevice, c->stream));
  return DEX_OK;
}

// Algorithmic bytes and launch counts of one round, from the host mirror of the FSM
// (DESIGN.md "Roofline accounting"): a live stage streams its layer's weights once per layer-step.
void account_round(dex_ctx* c) {
  const Dev& D = c->D;
  bool live[kMaxGrp] = {false};
  double kv = 0;
  for (int s = 0; s < c->cfg.max_seqs; ++s) {
    const HostSeq& hs = c->seqs[s];
    if (!hs.active || hs.done) continue;
    for (int m = 0; m <= hs.q && m < D.N; ++m) {
      live[m] = true;
      kv += (double)c->dec_plan.layer_len[m] * hs.ctx_len * 2.0 * D.nkv * D.hd * 2.0;   // committed K+V read once per stage layer
    }
  }
  double wbytes = 0;
  int gemm_launches = 0;
  for (int j = 0; j < D.max_len; ++j) {
    for (int m = 0; m < D.N; ++m)
      if (live[m] && j < c->dec_plan.layer_len[m]) {
        for (int i = 0; i < 4; ++i) wbytes += 2.0 * c->op[i].dec.out_dim * c->op[i].dec.k_dim;
      }
    gemm_launches += 4;
  }
  if (c->has_ad)   // every live non-final stage streams its adapter once per round
    for (int m = 0; m + 1 < D.N; ++m)
      if (live[m]) wbytes += 2.0 * (c->op[5].dec.out_dim * (double)c->op[5].dec.k_dim + c->op[6].dec.out_dim * (double)c->op[6].dec.k_dim);
  const bool mega = c->cfg.round_kernel && c->round_ok && (!c->phase_split || c->cfg.sample || c->has_ad);
  c->counters[0] += 1;
  c->counters[1] += mega ? 7.0 : 2 + 10.0 * D.max_len + 1 + 1 + 3;
  c->counters[2] += mega ? 1 : gemm_launches;
  c->counters[3] += wbytes;
  // algorithmic: the LM head once per round; the kernel re-streams it once per further exit chunk of
  // exit_chunk VALID rows (2 chunks only at N = 8, q = 7: 128 rows) - that re-stream is traffic, reported separately
  long long n_valid = 0;                              // rows decoded this round = 2^q per live sequence (sparse lattice: an upper bound)
  for (int s = 0; s < c->cfg.max_seqs; ++s) {
    const HostSeq& hs = c->seqs[s];
    if (hs.active && !hs.done) n_valid += 1ll << std::min(hs.q, D.N - 1);
  }
  const int live_chunks = (int)((n_valid + D.exit_chunk - 1) / D.exit_chunk);   // the exit head works on DENSE rows (Dev::exit_map)
  c->counters[4] += 2.0 * c->op[4].dec.out_dim * c->op[4].dec.k_dim;
  c->counters[6] += 2.0 * c->op[4].dec.out_dim * c->op[4].dec.k_dim * std::max(0, live_chunks - 1);
  c->counters[5] += kv;
}

void collect_phase_times(dex_ctx* c) {
  if (!c->profiling) return;
  float total = 0.f;
  for (int p = 0; p < PH_N; ++p) {
    float us = 0.f;
    for (size_t i = 0; i < c->ev_used[p]; ++i) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, c->ev[p][i].first, c->ev[p][i].second);
      us += ms * 1000.f;
    }
    // bookkeeping, gemm, glue, attention, exit, commit+collapse
    c->phase_us[p] = us;
    c->phase_us_acc[p] += us;
    total += us;
    c->ev_used[p] = 0;
  }
  c->phase_us[6] = 0.f;
  c->phase_us[7] = total;
}

}  // namespace

namespace dexk {
// for entry points outside this file (noalloc.cu): the string dex_last_error(NULL) returns
void set_global_error(const char* msg) { g_last_error = msg ? msg : ""; }
}  // namespace dexk

// =============================================================================================
extern "C" {

const char* dex_last_error(const dex_ctx* ctx) { return ctx ? ctx->err.c_str() : g_last_error.c_str(); }

int32_t dex_workspace_bytes(const dex_config* cfg, const int32_t* depths, int32_t n_depths, size_t* out_bytes) {
  int rc = validate(cfg, depths, n_depths);
  if (rc) return rc;
  if (!out_bytes) return fail(nullptr, DEX_EINVAL, "null out_bytes");
  Layout* L = new Layout;
  make_layout(*cfg, depths, n_depths, *L);
  *out_bytes = L->total;
  delete L;
  return DEX_OK;
}

int32_t dex_init(dex_ctx** out, const dex_config* cfg, const dex_weights* w, const int32_t* depths, int32_t n_depths,
                 void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return fail(nullptr, DEX_EINVAL, "null out");
  *out = nullptr;
  int rc = validate(cfg, depths, n_depths);
  if (rc) return rc;
  if (!w || !w->embed || !w->lm_head || !w->wqkv || !w->wo || !w->wgu || !w->wdn || !w->norm_attn || !w->norm_ffn ||
      !w->norm_final)
    return fail(nullptr, DEX_EINVAL, "null weight pointer");
  if (cfg->adapter_dim && (!w->ad_w1 || !w->ad_w2 || !w->ad_b1 || !w->ad_b2 || !w->ad_norm || !w->ad_alpha))
    return fail(nullptr, DEX_EINVAL, "adapter_dim > 0 but an adapter tensor is null");
  if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 1023)) return fail(nullptr, DEX_EINVAL, "workspace must be 1024-byte aligned");
  std::unique_ptr<Layout> Lp(new Layout);
  Layout& L = *Lp;
  make_layout(*cfg, depths, n_depths, L);
  if (workspace_bytes < L.total) return fail(nullptr, DEX_ECAPACITY, "workspace too small: need %zu bytes", L.total);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(nullptr, DEX_ECUDA, "no CUDA device: this library has no CPU fallback");
  dex_ctx* c = new dex_ctx;
  c->cfg = *cfg;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->dec_plan = L.dec;
  c->pre_plan = L.pre;
  c->exit_plan = L.ext;
  c->result_host = nullptr;
  memset(c->ev_used, 0, sizeof c->ev_used);
  memset(c->phase_us, 0, sizeof c->phase_us);
  memset(c->phase_us_acc, 0, sizeof c->phase_us_acc);
  memset(c->counters, 0, sizeof c->counters);
  c->profiling = 0;
  c->phase_split = 0;
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&c->n_sms, cudaDevAttrMultiProcessorCount, dev);

  Dev& D = c->D;
  memset(&D, 0, sizeof D);
  D.L = cfg->n_layers; D.d = cfg->d_model; D.nh = cfg->n_heads; D.nkv = cfg->n_kv_heads; D.hd = cfg->head_dim;
  D.ffn = cfg->d_ffn; D.vocab = cfg->vocab; D.qkv_out = (cfg->n_heads + 2 * cfg->n_kv_heads) * cfg->head_dim;
  D.eps = cfg->rms_eps; D.N = n_depths;
  for (int i = 0; i < n_depths; ++i) D.depths[i] = depths[i];
  D.max_seqs = cfg->max_seqs; D.max_ctx = cfg->max_ctx; D.page_size = cfg->page_size;
  D.pages_per_seq = L.pages_per_seq; D.n_pages = L.n_pages; D.n_slots = L.n_slots; D.n_nodes = L.n_nodes;
  D.R_cap = L.R_cap; D.R_dec = L.R_dec; D.exit_chunk = L.exit_chunk; D.decs = cfg->decs; D.planes = cfg->act_planes; D.taps = cfg->debug_taps;
  D.sample = cfg->sample; D.inv_tau = cfg->sample ? 1.0f / cfg->temperature : 1.0f; D.sample_seed = (unsigned)cfg->sample_seed;
  D.max_len = L.max_len; D.max_chunks = L.max_chunks; D.ref_tiles = L.ref_tiles;
  D.lookahead = (cfg->lookahead >= n_depths - 1) ? 0 : cfg->lookahead;   // P >= N-1 is the full lattice
  c->has_ad = cfg->adapter_dim > 0;
  D.ad_m = cfg->adapter_dim;
  if (c->has_ad) { D.ad_b1 = w->ad_b1; D.ad_b2 = w->ad_b2; D.ad_norm = w->ad_norm; D.ad_alpha = w->ad_alpha; }
  D.embed = static_cast<const __nv_bfloat16*>(w->embed);
  D.lm_head = static_cast<const __nv_bfloat16*>(w->lm_head);
  D.norm_attn = w->norm_attn; D.norm_ffn = w->norm_ffn; D.norm_final = w->norm_final;
  uint8_t* ws = static_cast<uint8_t*>(workspace);
#define WSP(T, b) reinterpret_cast<T*>(ws + L.off[b])
  D.seqs = WSP(SeqState, B_SEQS); D.tokens = WSP(int, B_TOKENS); D.B = WSP(int, B_B); D.page_table = WSP(int, B_PT);
  D.rows = WSP(RowInfo, B_ROWS); D.grp_nb = WSP(int, B_GNB); D.exit_nb = WSP(int, B_ENB);
  D.best_key = WSP(unsigned long long, B_KEY); D.ref_tile = WSP(float2, B_REFT); D.cmd = WSP(CollapseCmd, B_CMD);
  D.ss_part = WSP(float, B_SS); D.attn_cnt = WSP(int, B_ACNT);
  D.kpool = WSP(__nv_bfloat16, B_KPOOL); D.vpool = WSP(__nv_bfloat16, B_VPOOL);
  D.kslot = WSP(__nv_bfloat16, B_KSLOT); D.vslot = WSP(__nv_bfloat16, B_VSLOT);
  D.x_cur = WSP(float, B_XCUR); D.x_front = WSP(float, B_XFRONT);
  D.act_a = WSP(__nv_bfloat16, B_ACTA); D.act_o = WSP(__nv_bfloat16, B_ACTO);
  D.act_f = WSP(__nv_bfloat16, B_ACTF); D.act_e = WSP(__nv_bfloat16, B_ACTE);
  D.part = WSP(float, B_PART); D.qbuf = WSP(float, B_QBUF); D.attn_part = WSP(float, B_APART);
  D.rope = WSP(float2, B_ROPE); D.tap_hidden = cfg->debug_taps ? WSP(float, B_TAPH) : nullptr;
  D.gbar = WSP(unsigned int, B_GBAR);
  D.exit_map = WSP(int, B_EMAP);
  D.flow_ctr = WSP(int, B_FCTR);
  D.item_recs = WSP(void, B_ITEMS);
  D.item_cap = L.item_cap;
  c->flow_tab = WSP(int, B_FTAB);
  for (int i = 0; i < 4; ++i) c->part_off[i] = L.part_off[i];
  D.tap_times = cfg->debug_taps ? WSP(unsigned long long, B_TAPT) : nullptr;
  c->dbg_stage = cfg->debug_taps ? WSP(float, B_DBG) : nullptr;
  c->dbg_floats = L.dbg_floats;
#undef WSP
  for (int i = 0; i < 7; ++i) c->op[i] = L.op[i];
  c->dec_ring = make_ring(c->dec_plan, cfg->act_planes);
  c->pre_ring = make_ring(c->pre_plan, cfg->act_planes);
  c->exit_ring = make_ring(c->exit_plan, cfg->act_planes);
  {   // the round kernel streams the decode stages and the exit chunks through one ring
    Plan both = c->dec_plan;
    both.n_grp = 1;
    both.rows_cap[0] = std::max(c->dec_ring.x_cap, c->exit_ring.x_cap);
    c->round_ring = make_ring(both, cfg->act_planes);
    // the round kernel also carves its attention scratch out of dynamic shared memory: fewer ring stages
    const size_t stage = 16384 + (size_t)cfg->act_planes * c->round_ring.x_cap * 128;
    const size_t attn = (round_attn_smem(cfg->head_dim) + 1023) / 1024 * 1024;
    // 227 KB per block (232448 B) minus the kernels' static shared memory (k_round: row cache, 4.8 KB; k_flow: 3.8 KB)
    // and alignment slack: the dynamic request is at most budget constant + 511 B, the kernels' limits are 222 / 223 KB.
    // (219 KB, as this stood for part of round 2, left a 256-row single-plane stage short of 3 ring stages: c5 fell
    // back to the per-op path; at 221 KB it has 148480 B for 3 x 49152.)
    const size_t budget = 221 * 1024 - attn - 2048;
    c->round_ok = budget / stage >= 3 && c->round_ring.n_acc == 2;   // too few ring stages (very wide stages): per-op path   // too few ring stages (very wide stages): per-op path
    if ((cfg->sample || c->has_ad) && !c->round_ok) {
      delete c;
      return fail(nullptr, DEX_ECAPACITY, "sampling mode / inducing adapters need the round kernel, whose ring does not fit this stage width");
    }
    c->round_ring.n_stages = (int)std::max<size_t>(2, std::min<size_t>(12, budget / stage));
    c->round_attn_off = (int)((c->round_ring.n_stages * stage + 1023 + 512) / 1024 * 1024);
    c->round_ring.smem = c->round_attn_off + attn + 1024;
  }

#define INIT_FAIL(expr)          \
  do {                           \
    int rc_ = (expr);            \
    if (rc_) {                   \
      g_last_error = c->err;     \
      delete c;                  \
      return rc_;                \
    }                            \
  } while (0)

  // TMA descriptors (driver entry point fetched at run time: no link-time libcuda dependency)
  void* fnp = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fnp, cudaEnableDefault, &qres) != cudaSuccess || !fnp) {
    delete c;
    return fail(nullptr, DEX_ECUDA, "cuTensorMapEncodeTiled entry point not found");
  }
  EncodeFn enc = reinterpret_cast<EncodeFn>(fnp);
  if (round_init() != cudaSuccess) {
    delete c;
    return fail(nullptr, DEX_ECUDA, "cannot raise the round kernel's dynamic shared memory limit");
  }
  if (flow_init() != cudaSuccess) {
    delete c;
    return fail(nullptr, DEX_ECUDA, "cannot raise the dataflow round kernel's dynamic shared memory limit");
  }
  if (gemm_init() != cudaSuccess) {
    delete c;
    return fail(nullptr, DEX_ECUDA, "cannot raise the GEMM kernel's dynamic shared memory limit");
  }
  const void* wptr[5] = {w->wqkv, w->wo, w->wgu, w->wdn, w->lm_head};
  for (int i = 0; i < 5; ++i)
    INIT_FAIL(encode_3d(c, enc, &c->op[i].tmW, wptr[i], c->op[i].dec.k_dim, c->op[i].dec.out_dim, i == 4 ? 1 : D.L, kTileM));
  // every ring of this context must agree on the activation box (one tensor map per operand)
  const bool all_stacked = c->dec_ring.stacked && c->pre_ring.stacked && c->exit_ring.stacked && c->round_ring.stacked;
  c->dec_ring.stacked = c->pre_ring.stacked = c->exit_ring.stacked = c->round_ring.stacked = all_stacked ? 1 : 0;
  const void* xptr[4] = {D.act_a, D.act_o, D.act_f, D.act_e};
  const int xk[4] = {D.d, D.nh * D.hd, D.ffn, D.d};
  for (int i = 0; i < 4; ++i)
    INIT_FAIL(encode_3d(c, enc, &c->tmX[i], xptr[i], xk[i], D.R_cap, cfg->act_planes, kBoxRows, all_stacked ? 2 : 1));
  memset(&c->tms, 0, sizeof c->tms);
  if (c->has_ad) {
    const void* aptr[2] = {w->ad_w1, w->ad_w2};
    for (int i = 0; i < 2; ++i)
      INIT_FAIL(encode_3d(c, enc, &c->op[5 + i].tmW, aptr[i], c->op[5 + i].dec.k_dim, c->op[5 + i].dec.out_dim, n_depths - 1, kTileM));
  }
  // k_flow: gate/up as [2L][ffn][d] (gate tile b and up tile b of a layer are both 128-row boxes, whatever ffn % 128 is)
  INIT_FAIL(encode_3d(c, enc, &c->tms.wgu2, w->wgu, D.d, D.ffn, 2 * (uint64_t)D.L, kTileM));
  {
    // QKV tile order by KV head group (q tiles of the group, then its k and v tile) and the groups a tile touches
    const int hd = D.hd, Gq = D.nh / D.nkv, n_t = c->op[0].dec.n_tiles;
    c->flow_ok = (D.nh * hd) % kTileM == 0 && (D.nkv * hd) % kTileM == 0 && n_t <= kFlowTiles &&
                 2 * ((D.ffn + kTileM - 1) / kTileM) <= kFlowTiles && (D.d + kTileM - 1) / kTileM <= kFlowTiles && D.nkv <= kFlowSlices;
    for (int i = 0; i < 4; ++i) c->flow_ok = c->flow_ok && c->op[i].dec.ksplit <= kFlowSlices;
    c->flow_ok = c->flow_ok && 4 * L.max_len * n_depths + 3 <= 400 && c->n_sms >= 128 && c->n_sms <= 160;   // item records, op table
    std::vector<int> tab(kFtTotal, 0);
    if (c->flow_ok) {
      auto grp_of = [&](int hh) { return hh < D.nh ? hh / Gq : (hh < D.nh + D.nkv ? hh - D.nh : hh - D.nh - D.nkv); };
      for (int t = 0; t < n_t; ++t) {
        const int h_lo = t * kTileM / hd, h_hi = std::min((t * kTileM + kTileM - 1) / hd, D.nh + 2 * D.nkv - 1);
        int lo = 1 << 30, hi = -1;
        for (int hh = h_lo; hh <= h_hi; ++hh) { lo = std::min(lo, grp_of(hh)); hi = std::max(hi, grp_of(hh)); }
        tab[kFtGlo + t] = lo; tab[kFtGhi + t] = hi;
        for (int g = lo; g <= hi; ++g) tab[kFtTarget + g] += 1;
      }
      int n = 0;
      for (int g = 0; g < D.nkv; ++g)
        for (int t = 0; t < n_t; ++t)
          if (tab[kFtGlo + t] == g) tab[kFtPerm + n++] = t;
    }
    INIT_FAIL(cu_or_fail0(c, cudaMemcpy(const_cast<int*>(c->flow_tab), tab.data(), sizeof(int) * kFtTotal, cudaMemcpyHostToDevice), "flow tables"));
  }
  for (int i = 0; i < (c->has_ad ? 7 : 5); ++i) c->tms.w[i] = c->op[i].tmW;
  for (int i = 0; i < 4; ++i) c->tms.x[i] = c->tmX[i];

  // state: FSM zeroed, free pages, result buffer, RoPE table
  auto cu_or_fail = [&](cudaError_t e, const char* what) -> int {
    if (e != cudaSuccess) return fail(c, DEX_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    return DEX_OK;
  };
  INIT_FAIL(cu_or_fail(cudaMemsetAsync(ws, 0, L.off[B_KPOOL], c->stream), "memset state"));
  INIT_FAIL(cu_or_fail(cudaMemsetAsync(D.rows, 0, sizeof(RowInfo) * D.R_cap, c->stream), "memset rows"));
  INIT_FAIL(cu_or_fail(cudaHostAlloc(reinterpret_cast<void**>(&c->result_host), sizeof(dex_step_result) * cfg->max_seqs + 64,
                                     cudaHostAllocMapped),
                       "cudaHostAlloc"));
  memset(c->result_host, 0, sizeof(dex_step_result) * cfg->max_seqs + 64);
  INIT_FAIL(cu_or_fail(cudaHostGetDevicePointer(reinterpret_cast<void**>(&D.result_dev), c->result_host, 0),
                       "cudaHostGetDevicePointer"));
  D.dbg_host = reinterpret_cast<int*>(D.result_dev + cfg->max_seqs);
  c->seqs.resize(cfg->max_seqs);
  c->page_table_host.assign((size_t)D.n_pages, 0);
  for (int p = D.n_pages - 1; p >= 0; --p) c->free_pages.push_back(p);
  INIT_FAIL(cu_or_fail(launch_rope_table(D, (double)cfg->rope_theta, cfg->max_ctx + kMaxAnc + 1, c->stream), "rope table"));
  INIT_FAIL(cu_or_fail(cudaStreamSynchronize(c->stream), "init sync"));
#undef INIT_FAIL
  *out = c;
  return DEX_OK;
}

int32_t dex_destroy(dex_ctx* c) {
  if (!c) return DEX_OK;
  cudaStreamSynchronize(c->stream);
  for (auto& kv : c->graphs) cudaGraphExecDestroy(kv.second);
  for (int p = 0; p < PH_N; ++p)
    for (auto& e : c->ev[p]) {
      cudaEventDestroy(e.first);
      cudaEventDestroy(e.second);
    }
  if (c->result_host) cudaFreeHost(c->result_host);
  delete c;
  return DEX_OK;
}

int32_t dex_prefill(dex_ctx* c, int32_t seq, const int32_t* prompt, int32_t n) {
  if (!c) return fail(nullptr, DEX_EINVAL, "null ctx");
  if (seq < 0 || seq >= c->cfg.max_seqs) return fail(c, DEX_EINVAL, "seq out of range");
  if (!prompt || n < 1) return fail(c, DEX_EINVAL, "empty prompt");
  if (n > c->cfg.max_ctx) return fail(c, DEX_ECAPACITY, "prompt longer than max_ctx");
  for (int i = 0; i < n; ++i)
    if (prompt[i] < 0 || prompt[i] >= c->cfg.vocab) return fail(c, DEX_EINVAL, "prompt token out of range");
  HostSeq& hs = c->seqs[seq];
  for (int pg : hs.pages) c->free_pages.push_back(pg);   // reset the sequence
  hs = HostSeq();
  const Dev& D = c->D;
  int rc = ensure_pages(c, seq, n);
  if (rc) return rc;
  CU(c, cudaMemcpyAsync(D.tokens + (size_t)seq * (D.max_ctx + 1), prompt, sizeof(int) * n, cudaMemcpyHostToDevice, c->stream));
  for (int p0 = 0; p0 < n - 1; p0 += kPrefillRows) {
    const int R = std::min(kPrefillRows, n - 1 - p0);
    CU(c, launch_rows_prefill(D, seq, p0, R, c->stream));
    CU(c, launch_gather_norm(D, c->pre_plan, R, c->stream));
    const int n_chunks = (p0 + R - 1) / kChunk + 1;
    rc = enqueue_layers(c, c->pre_plan, c->pre_ring, R, n_chunks, D.L, true);
    if (rc) return rc;
  }
  CU(c, launch_seq_init(D, seq, n, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));   // prompt is a caller buffer: copies must have completed
  for (int p = 0; p < PH_N; ++p) c->ev_used[p] = 0;
  hs.active = 1; hs.q = 0; hs.ctx_len = n - 1; hs.n_tok = n; hs.pending = 0; hs.done = (n >= c->cfg.max_ctx);
  return DEX_OK;
}

int32_t dex_step(dex_ctx* c, uint32_t flags, dex_step_result* out) {
  if (!c || !out) return fail(c, DEX_EINVAL, "null argument");
  const Dev& D = c->D;
  int n_live = 0, max_pos = 0;
  for (int s = 0; s < c->cfg.max_seqs; ++s) {
    HostSeq& hs = c->seqs[s];
    if (hs.active && hs.pending) return fail(c, DEX_ESTATE, "sequence %d has a pending commit: call dex_collapse", s);
    if (!hs.active || hs.done) continue;
    int rc = ensure_pages(c, s, hs.ctx_len + 1);
    if (rc) return rc;
    ++n_live;
    max_pos = std::max(max_pos, hs.ctx_len + D.N - 1);
  }
  if (n_live > 0) {
    const int n_chunks = max_pos / kChunk + 1;
    account_round(c);
    if (c->cfg.use_graph && !c->profiling) {
      const long long key = ((long long)n_chunks << 8) | (flags & 0xff);
      auto it = c->graphs.find(key);
      if (it == c->graphs.end()) {
        cudaGraph_t g;
        CU(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        int rc = enqueue_step(c, flags, n_chunks);
        cudaError_t e = cudaStreamEndCapture(c->stream, &g);
        if (rc) {
          if (e == cudaSuccess && g) cudaGraphDestroy(g);
          return rc;
        }
        CU(c, e);
        cudaGraphExec_t ge;
        CU(c, cudaGraphInstantiate(&ge, g, 0));
        cudaGraphDestroy(g);
        it = c->graphs.emplace(key, ge).first;
      }
      CU(c, cudaGraphLaunch(it->second, c->stream));
    } else {
      int rc = enqueue_step(c, flags, n_chunks);
      if (rc) return rc;
    }
    {
      cudaError_t e_ = cudaStreamSynchronize(c->stream);
      if (e_ != cudaSuccess) {
        const int* dbg = reinterpret_cast<const int*>(c->result_host + c->cfg.max_seqs);
        return fail(c, DEX_ECUDA, "dex_step: %s (kernel timeout record: code %d cta %d args %d %d %d %d | %d %d %d %d %d %d %d %d %d %d)",
                    cudaGetErrorString(e_), dbg[0], dbg[1], dbg[2], dbg[3], dbg[4], dbg[5], dbg[6], dbg[7], dbg[8], dbg[9], dbg[10],
                    dbg[11], dbg[12], dbg[13], dbg[14], dbg[15]);
      }
    }
    collect_phase_times(c);
  }
  for (int s = 0; s < c->cfg.max_seqs; ++s) {
    HostSeq& hs = c->seqs[s];
    if (n_live == 0 || !hs.active || hs.done) {
      memset(&out[s], 0, sizeof(dex_step_result));
      out[s].token = -1; out[s].match_k = -1;
      out[s].q_before = out[s].q_after = hs.q; out[s].n_tokens = hs.n_tok; out[s].done = hs.done;
      for (int i = 0; i < DEX_MAX_DEPTHS; ++i) out[s].anchor_tokens[i] = -1;
      continue;
    }
    out[s] = c->result_host[s];
    hs.last_q_before = out[s].q_before;
    hs.q = out[s].q_after;
    hs.n_tok = out[s].n_tokens;
    hs.ctx_len = hs.n_tok - 1;
    hs.done = out[s].done;
    hs.pending = (!out[s].committed && out[s].q_before == D.N - 1) ? 1 : 0;
    memcpy(hs.anchor_tokens, out[s].anchor_tokens, sizeof hs.anchor_tokens);
    hs.branch_mask = out[s].branch_mask;
  }
  return DEX_OK;
}

int32_t dex_collapse(dex_ctx* c, int32_t seq, int32_t branch_k, int32_t token) {
  if (!c) return fail(nullptr, DEX_EINVAL, "null ctx");
  if (seq < 0 || seq >= c->cfg.max_seqs) return fail(c, DEX_EINVAL, "seq out of range");
  HostSeq& hs = c->seqs[seq];
  const int N = c->D.N;
  if (!hs.active || !hs.pending) return fail(c, DEX_ESTATE, "no pending commit: the anchor is not at final depth");
  if (branch_k < 0 || branch_k > N - 1) return fail(c, DEX_EINVAL, "branch_k out of range");
  if (token < 0 || token >= c->cfg.vocab) return fail(c, DEX_EINVAL, "token out of range");
  if (branch_k < N - 1 && hs.anchor_tokens[branch_k] != token)
    return fail(c, DEX_EINVAL, "B[anchor(%d)] = %d != token %d", branch_k, hs.anchor_tokens[branch_k], token);
  if (branch_k < N - 1 && !((hs.branch_mask >> branch_k) & 1))
    return fail(c, DEX_EINVAL, "the continuation of branch %d was not explored (sparse lattice)", branch_k);
  CU(c, launch_set_cmd(c->D, seq, branch_k, token, c->stream));
  int rc = enqueue_collapse(c);
  if (rc) return rc;
  CU(c, cudaStreamSynchronize(c->stream));
  for (int p = 0; p < PH_N; ++p) c->ev_used[p] = 0;
  hs.pending = 0;
  hs.q = (branch_k < N - 1) ? (N - 1 - branch_k) : 0;
  hs.n_tok += 1;
  hs.ctx_len += 1;
  hs.done = (hs.n_tok >= c->cfg.max_ctx || token == c->cfg.eos_id) ? 1 : 0;
  return DEX_OK;
}

int32_t dex_rewind(dex_ctx* c, int32_t seq, int32_t n) {
  if (!c) return fail(nullptr, DEX_EINVAL, "null ctx");
  if (seq < 0 || seq >= c->cfg.max_seqs) return fail(c, DEX_EINVAL, "seq out of range");
  HostSeq& hs = c->seqs[seq];
  if (!hs.active) return fail(c, DEX_ESTATE, "sequence %d was never prefilled", seq);
  if (n < 1 || n > hs.n_tok) return fail(c, DEX_EINVAL, "n must be in [1, %d]", hs.n_tok);
  const int keep = (n + c->cfg.page_size - 1) / c->cfg.page_size;   // pages holding positions < n
  while ((int)hs.pages.size() > keep) {
    c->free_pages.push_back(hs.pages.back());
    hs.pages.pop_back();
  }
  CU(c, launch_seq_init(c->D, seq, n, c->stream));
  hs.q = 0; hs.ctx_len = n - 1; hs.n_tok = n; hs.pending = 0; hs.done = (n >= c->cfg.max_ctx);
  hs.last_q_before = 0;
  return DEX_OK;
}

int32_t dex_get_tokens(dex_ctx* c, int32_t seq, int32_t* out, int32_t cap, int32_t* n_out) {
  if (!c || !out || !n_out) return fail(c, DEX_EINVAL, "null argument");
  if (seq < 0 || seq >= c->cfg.max_seqs) return fail(c, DEX_EINVAL, "seq out of range");
  const int n = std::min(cap, c->seqs[seq].n_tok);
  *n_out = c->seqs[seq].n_tok;
  if (n > 0) {
    CU(c, cudaMemcpyAsync(out, c->D.tokens + (size_t)seq * (c->D.max_ctx + 1), sizeof(int) * n, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
  }
  return DEX_OK;
}

int32_t dex_debug_read(dex_ctx* c, int32_t what, int32_t seq, int32_t a, void* dst, size_t dst_bytes) {
  if (!c || !dst) return fail(c, DEX_EINVAL, "null argument");
  if (seq < 0 || seq >= c->cfg.max_seqs) return fail(c, DEX_EINVAL, "seq out of range");
  const Dev& D = c->D;
  const HostSeq& hs = c->seqs[seq];
  if (what == DEX_TAP_FSM) {
    if (dst_bytes < 4 * sizeof(int)) return fail(c, DEX_EINVAL, "dst too small");
    SeqState st;
    CU(c, cudaMemcpyAsync(&st, D.seqs + seq, sizeof st, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    int* o = static_cast<int*>(dst);
    o[0] = st.q; o[1] = st.ctx_len; o[2] = st.n_tok; o[3] = st.pending;
    return DEX_OK;
  }
  if (what == DEX_TAP_B) {
    if (dst_bytes < sizeof(int) * D.n_nodes) return fail(c, DEX_EINVAL, "dst too small");
    CU(c, cudaMemcpyAsync(dst, D.B + (size_t)seq * D.n_nodes, sizeof(int) * D.n_nodes, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DEX_OK;
  }
  if (!c->cfg.debug_taps) return fail(c, DEX_ESTATE, "debug_taps is off");
  if (what == DEX_TAP_HIDDEN) {
    const int q = hs.last_q_before;
    const int o = a - ((1 << q) - 1);
    if (o < 0 || o >= (1 << q)) return fail(c, DEX_EINVAL, "node %d is not on the last round's level %d", a, q);
    const int m = stage_of(q, o);
    const int row = c->dec_plan.row_base[m] + seq * cap_of(D.N, m) + idx_in_stage(q, o, m);
    const size_t bytes = sizeof(float) * (size_t)c->dec_plan.layer_len[m] * D.d;
    if (dst_bytes < bytes) return fail(c, DEX_EINVAL, "dst too small");
    CU(c, cudaMemcpyAsync(dst, D.tap_hidden + (size_t)row * D.max_len * D.d, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DEX_OK;
  }
  if (what == DEX_TAP_ROUND_TIMES) {
    const size_t bytes = sizeof(unsigned long long) * (20 * (size_t)D.max_len + 68);
    if (dst_bytes < bytes) return fail(c, DEX_EINVAL, "dst too small");
    CU(c, cudaMemcpyAsync(dst, D.tap_times, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DEX_OK;
  }
  if (what == DEX_TAP_LOGITS) {
    if (hs.last_q_before != D.N - 1) return fail(c, DEX_ESTATE, "the last round did not reach final depth");
    if (dst_bytes < sizeof(float) * D.vocab) return fail(c, DEX_EINVAL, "dst too small");
    const int row = c->dec_plan.row_base[D.N - 1] + seq * cap_of(D.N, D.N - 1);
    float* tmp = c->dbg_stage + (c->dbg_floats - D.vocab);
    CU(c, launch_tap_logits(D, row, tmp, c->stream));
    CU(c, cudaMemcpyAsync(dst, tmp, sizeof(float) * D.vocab, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DEX_OK;
  }
  if (what == DEX_TAP_REF_BLOCKS) {
    if (hs.last_q_before != D.N - 1) return fail(c, DEX_ESTATE, "the last round did not reach final depth");
    const size_t bytes = sizeof(float2) * D.ref_tiles;
    if (dst_bytes < bytes || c->dbg_floats < 2 * (size_t)D.ref_tiles) return fail(c, DEX_EINVAL, "dst too small");
    const int row = c->dec_plan.row_base[D.N - 1] + seq * cap_of(D.N, D.N - 1);
    float2* tmp = reinterpret_cast<float2*>(c->dbg_stage);
    CU(c, launch_tap_ref_tiles(D, row, seq, tmp, c->stream));
    CU(c, cudaMemcpyAsync(dst, tmp, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DEX_OK;
  }
  return fail(c, DEX_EINVAL, "unknown tap %d", what);
}

int32_t dex_debug_gemm(dex_ctx* c, int32_t which, int32_t layer, const float* x, int32_t rows, float* y) {
  if (!c || !x || !y) return fail(c, DEX_EINVAL, "null argument");
  if (!c->cfg.debug_taps) return fail(c, DEX_ESTATE, "debug_taps is off");
  if (which < 0 || which > 3) return fail(c, DEX_EINVAL, "which must be 0..3");
  if (layer < 0 || layer >= c->D.L) return fail(c, DEX_EINVAL, "layer out of range");
  if (rows < 1 || rows > kPrefillRows) return fail(c, DEX_EINVAL, "rows must be in [1,128]");
  const Dev& D = c->D;
  const OpDesc& o = c->op[which].dec;
  __nv_bfloat16* act[4] = {D.act_a, D.act_o, D.act_a, D.act_f};
  const int xm[4] = {0, 1, 0, 2};
  float* xs = c->dbg_stage;
  float* ys = c->dbg_stage + (size_t)kPrefillRows * std::max(D.ffn, D.d);
  CU(c, cudaMemcpyAsync(xs, x, sizeof(float) * (size_t)rows * o.k_dim, cudaMemcpyHostToDevice, c->stream));
  CU(c, launch_debug_rows(D, rows, c->stream));
  CU(c, launch_debug_split(xs, act[which], rows, o.k_dim, (size_t)D.R_cap * o.k_dim, D.planes, c->stream));
  Plan p = c->pre_plan;
  p.layer_lo[0] = layer;
  p.layer_len[0] = 1;
  int rc = run_gemm(c, which, o, c->tmX[xm[which]], p, c->pre_ring, 0, 0, D.grp_nb);
  if (rc) return rc;
  CU(c, launch_debug_sum(D.part, ys, rows, o.out_dim, o.part_ld, o.ksplit, o.split_stride, c->stream));
  CU(c, cudaMemcpyAsync(y, ys, sizeof(float) * (size_t)rows * o.out_dim, cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
  for (int ph = 0; ph < PH_N; ++ph) c->ev_used[ph] = 0;
  return DEX_OK;
}

int32_t dex_debug_phase_us(dex_ctx* c, float* out8) {
  if (!c || !out8) return fail(c, DEX_EINVAL, "null argument");
  if (!c->profiling) return fail(c, DEX_ESTATE, "profiling is off");
  memcpy(out8, c->phase_us, sizeof(float) * 8);
  return DEX_OK;
}

int32_t dex_profile(dex_ctx* c, int32_t on, double* phase_us_acc8, double* counters8) {
  if (!c) return fail(c, DEX_EINVAL, "null ctx");
  if (phase_us_acc8) memcpy(phase_us_acc8, c->phase_us_acc, sizeof(double) * 8);
  if (counters8) memcpy(counters8, c->counters, sizeof(double) * 8);
  if (on >= 0) {
    c->profiling = on ? 1 : 0;
    c->phase_split = (on == 2) ? 1 : 0;
    memset(c->phase_us_acc, 0, sizeof c->phase_us_acc);
    memset(c->counters, 0, sizeof c->counters);
  }
  return DEX_OK;
}

}  // extern "C"
