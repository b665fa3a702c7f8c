// flow.cu — k_flow: the persistent round kernel as a DATAFLOW program (Alg. 1 lines 5-6).
//
// Same work as k_round (round.cu): for every layer-step all live stages run QKV -> attention -> O -> gate/up -> down,
// then the fused exit.  k_round separates the nine activities of a layer-step by grid barriers; every barrier and
// glue phase leaves HBM idle once the shared-memory ring is full (2.5 us of stream).  Here the layer-steps have NO
// grid barrier: every dependency is a counter in global memory.
//
//   * split-K partials are reduced by the LAST ARRIVER: the CTA whose item completes an out tile (all K splits
//     written, counted with one acq_rel atomic per item) sums the partials in split order (H3: the bits do not depend
//     on who arrives last) and finalizes the tile on its finalizer warps - QKV: deferred-norm scale + RoPE + slot K/V;
//     O / down: residual add + next operand planes + sum of squares of the 128-column segment; gate/up: SwiGLU (gate
//     tile b and up tile b are counted together; the weights stay in their [2][ffn][d] layout, the tensor map views
//     them as [2L][ffn][d]);
//   * a finished tile bumps the READY counter of the consumer's K slice (an item's K range: 8 K-blocks = 512
//     columns); the activation producer of a consuming item polls exactly the slice it needs (relaxed loads, requested
//     one item ahead), so consumers start while the producing op is still streaming.  Item orders are chosen for that: QKV by KV head
//     (q, k, v tiles of a head adjacent) -> attention of the first heads overlaps the rest of the QKV stream; O and
//     down split-major (early splits need early heads / early gate-up pairs); gate/up pair-major;
//   * attention tasks wait for the QKV counter of their KV head group, the last merger of a (row, head) bumps the
//     ready counter of the O operand slice;
//   * with several live stages (DEX rounds) an op is one projection of ONE stage and the ops are SKEWED across stages
//     (see the micro-op schedule in the kernel), so between two dependent projections of a stage lie the streams of the
//     other stages: depth-parallel stages hide each other's latency.
// Only the tail of the round (inducing adapters, exit head) keeps grid barriers.
//
//   warp 0      weight producer (TMA, always ahead)         warp 1      activation producer (waits on slice counters)
//   warp 8      tcgen05.mma issuer, owns TMEM               warps 2, 3, 10, 11  finalizer group: finalizes completed
//   warps 4-7   epilogue: TMEM -> split-K partials / arg-max            tiles, runs attention tasks
//   warp 9      counter: counts this CTA's finished items into the tile counters (one atomic per item, a batch of up
//               to 32 in flight), queues the tiles it completed for the finalizer group
//   (which warp takes which role follows the SM's four schedulers: see kWarp* below)
#include "round_dev.cuh"

namespace dexk {

constexpr int kFlowThreads = 384;
constexpr int kFT = 128;             // finalizer group threads
// Warp roles.  Warps are dealt to the SM's four schedulers by warp % 4.  The finalizer warps run attention MMAs and
// split-K sums WHILE the pipeline streams, so they must not share a scheduler with the single-issuer pipeline warps:
//   scheduler 0: weight producer (0), epilogue (4), MMA issuer (8)      scheduler 2: finalizer (2), epilogue (6), finalizer (10)
//   scheduler 1: activation producer (1), epilogue (5), counter (9)     scheduler 3: finalizer (3), epilogue (7), finalizer (11)
// (epilogue warp w reads TMEM lanes 32 (w % 4) .. +31: one per scheduler in any case).
constexpr int kWarpW = 0, kWarpA = 1, kWarpM = 8, kWarpC = 9, kWarpE0 = 4;
__device__ __forceinline__ int flow_fin_index(int warp) { return warp == 2 ? 0 : (warp == 3 ? 1 : (warp == 10 ? 2 : (warp == 11 ? 3 : -1))); }

// ---------------------------------------------------------------- small helpers
__device__ __forceinline__ int ld_acquire_s32(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int ld_relaxed_s32(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_s32(int* p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int atom_acq_rel_add_s32(int* p, int v) {
  int old;
  asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], %2;\n" : "=r"(old) : "l"(p), "r"(v) : "memory");
  return old;
}
__device__ __forceinline__ unsigned ld_acquire_cta_shared(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.cta.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_cta_shared_add(unsigned* p, unsigned v) {
  asm volatile("red.release.cta.shared.add.u32 [%0], %1;\n" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
// A bounded wait ran out: leave a record in mapped host memory (dex_step reports it), then trap instead of hanging.
__device__ __noinline__ void flow_die(const Dev& D, int code, int v0, int v1, int v2, int v3) {
  if ((threadIdx.x & 31) == 0 || code < 0) {
    volatile int* h = D.dbg_host;
    h[1] = blockIdx.x; h[2] = v0; h[3] = v1; h[4] = v2; h[5] = v3;
    if (code == 1) {                                         // the waiting item's stage: what has arrived so far
      const int m = v1 >> 16;
      const volatile int* c = D.flow_ctr;
      h[6] = c[kFcTile + (0 * kMaxGrp + m) * kFlowTiles + 0]; h[7] = c[kFcTile + (0 * kMaxGrp + m) * kFlowTiles + 1];
      h[8] = c[kFcTile + (1 * kMaxGrp + m) * kFlowTiles + 0]; h[9] = c[kFcTile + (1 * kMaxGrp + m) * kFlowTiles + 1];
      h[10] = c[kFcQkv + m * kFlowSlices + 0]; h[11] = c[kFcQkv + m * kFlowSlices + 1];
      h[12] = c[kFcAo + m * kFlowSlices + 0]; h[13] = c[kFcXf + m * kFlowSlices + 0];
      h[14] = c[kFcXa + m * kFlowSlices + 0]; h[15] = c[kFcF + m * kFlowSlices + 0];
    }
    h[0] = code;
    __threadfence_system();
  }
  __nanosleep(1000000);
  __trap();
}
__device__ __forceinline__ int tiles_in_slice(int dim, int slice_cols, int s) {   // 128-column tiles overlapping K slice s
  const int c0 = s * slice_cols, c1 = min(c0 + slice_cols, dim);
  return (c1 + 127) / 128 - c0 / 128;
}

// ---------------------------------------------------------------- the round's op / item sequence
struct FOp {
  int which, j, ext;
  unsigned mask;
  int n_tiles, ksplit, kbps, kb_total, per_grp, n_items;
};
struct FItem {
  int g, nb, tile, split, kb0, kb1, row0, row_end;
  int c1, c2;              // TMA coordinates: weight row, "layer"
  int col0, col_end;       // partial column of TMEM lane 0; columns >= col_end are not stored
  int cnt_idx, cnt_target; // finalization counter of the tile (gate/up: of the pair) and its arrivals per layer-step
};

struct FSeq {
  const RoundArgs* a;
  const int* s_nb;         // [16]
  const short* s_perm;     // QKV tile order
  int n_steps, n_ops, n_ad_ops, G, cta, gu_half;   // gu_half = ceil(ffn / 128)
  const struct FRec* recs;   // this CTA's decoded items and their count (prologue of k_flow)
  int n_my;
  const int* mops;           // layer micro-ops in schedule order: (step j) << 8 | (kind) << 4 | stage
  int n_layer;               // their count

  __device__ __forceinline__ void op_info(int t, FOp& o) const {
    unsigned mask = 0;
    if (t < n_layer) {                                     // one projection of ONE stage at one layer-step
      const int e = mops[t];
      o.j = e >> 8; o.which = (e >> 4) & 15; o.ext = 0;
      mask = 1u << (e & 15);
    } else if (t < n_layer + n_ad_ops) {
      o.j = 0; o.which = 5 + t - n_layer; o.ext = 0;
      for (int g = 0; g + 1 < a->dec.n_grp; ++g)
        if (s_nb[g] > 0) mask |= 1u << g;
    } else {
      o.j = 0; o.which = 4; o.ext = 1;
      for (int g = 0; g < a->ext.n_grp; ++g)
        if (s_nb[8 + g] > 0) mask |= 1u << g;
    }
    o.mask = mask;
    const OpDesc& d = a->op[o.which];
    o.n_tiles = (t < n_layer && o.which == 2) ? 2 * gu_half : d.n_tiles;
    o.ksplit = d.ksplit; o.kbps = d.kbps; o.kb_total = d.kb_total;
    o.per_grp = o.n_tiles * d.ksplit;
    o.n_items = __popc(mask) * o.per_grp;
  }
  __device__ __forceinline__ void decode(const FOp& o, int i, FItem& it) const {
    const int gi = i / o.per_grp, rem = i - gi * o.per_grp;
    it.g = __fns(o.mask, 0, gi + 1);
    const Plan& p = o.ext ? a->ext : a->dec;
    it.nb = s_nb[(o.ext ? 8 : 0) + it.g];
    it.row0 = p.row_base[it.g];
    it.row_end = it.row0 + p.rows_cap[it.g];
    const OpDesc& d = a->op[o.which];
    if (!o.ext && o.which < 4) {
      const int layer = p.layer_lo[it.g] + o.j;
      if (o.which == 0) {                           // by KV head group, splits fastest
        const int ti = rem / o.ksplit;
        it.split = rem - ti * o.ksplit;
        it.tile = s_perm[ti];
        it.c1 = it.tile * kTileM; it.c2 = layer;
        it.col0 = it.tile * kTileM; it.col_end = d.out_dim;
        it.cnt_idx = it.tile; it.cnt_target = o.ksplit;
      } else if (o.which == 2) {                           // pair-major: gate tile b, up tile b, splits fastest
        const int ti = rem / o.ksplit;
        it.split = rem - ti * o.ksplit;
        const int half = ti & 1, b = ti >> 1;
        it.tile = ti;
        it.c1 = b * kTileM; it.c2 = 2 * layer + half;
        it.col0 = half * a->D.ffn + b * kTileM; it.col_end = half * a->D.ffn + a->D.ffn;
        it.cnt_idx = b; it.cnt_target = 2 * o.ksplit;
      } else {                                             // O, down: split-major
        it.split = rem / o.n_tiles;
        it.tile = rem - it.split * o.n_tiles;
        it.c1 = it.tile * kTileM; it.c2 = layer;
        it.col0 = it.tile * kTileM; it.col_end = d.out_dim;
        it.cnt_idx = it.tile; it.cnt_target = o.ksplit;
      }
    } else {
      it.tile = rem / o.ksplit;
      it.split = rem - it.tile * o.ksplit;
      it.c1 = it.tile * kTileM; it.c2 = o.ext ? 0 : it.g;  // adapter k serves stage k
      it.col0 = it.tile * kTileM; it.col_end = d.out_dim;
      it.cnt_idx = it.tile; it.cnt_target = o.ksplit;
    }
    it.kb0 = it.split * o.kbps;
    it.kb1 = min(it.kb0 + o.kbps, o.kb_total);
  }
};

struct FWalker {           // this CTA's items, in order (dealt round-robin, continuing across ops)
  int t, i, rr;
  bool valid;
  FOp o;
  FItem it;
  __device__ __forceinline__ void start(const FSeq& q) {
    t = 0; rr = 0;
    q.op_info(0, o);
    i = q.cta;
    settle(q);
  }
  __device__ __forceinline__ void settle(const FSeq& q) {
    while (t < q.n_ops && i >= o.n_items) {
      rr = (rr + o.n_items) % q.G;
      ++t;
      if (t < q.n_ops) {
        q.op_info(t, o);
        i = (q.cta + q.G - rr) % q.G;
      }
    }
    valid = t < q.n_ops;
    if (valid) q.decode(o, i, it);
  }
  __device__ __forceinline__ void next(const FSeq& q) {
    i += q.G;
    settle(q);
  }
};

// Precomputed item records: the CTA decodes its items ONCE in the prologue (all threads in parallel) into 32-byte records
// in global memory and the roles read them (two 16-byte loads per item, the next record requested one item ahead)
// instead of each walking the list themselves (op_info / decode: integer divisions, ~300 instructions per item, inlined
// into six warp roles).  ncu's source page put most of k_flow's instruction-fetch stalls in those walkers; with the
// records c2 went from 172 to 227 tokens/s.  (k_round gains nothing from it: its glue warps sleep while the GEMM phases
// stream, and the prologue costs as much as the walkers.)
constexpr int kMaxOps = 400;            // ops of a round
struct __align__(16) FRec {
  int c1, col0;
  short c2, t, kb0, kb1, nb, row0, row_end, cnt_idx;
  unsigned char g, split, which, cnt_target;
  int j;
};
static_assert(sizeof(FRec) == 32, "FRec is 32 bytes");

struct FRecWalker {        // same interface as FWalker
  const FRec* recs;
  int k, n, t, i;
  bool valid;
  struct { int which, j; } o;
  FItem it;
  uint4 na, nb_;
  int ffn, n_layer_ops;
  const RoundArgs* a;
  __device__ __forceinline__ void fetch(int idx) {
    if (idx < n) {
      const uint4* p = reinterpret_cast<const uint4*>(recs + idx);
      na = p[0];
      nb_ = p[1];
    }
  }
  __device__ __forceinline__ void take() {
    valid = k < n;
    i = k;
    if (!valid) return;
    it.c1 = (int)na.x; it.col0 = (int)na.y;
    it.c2 = (short)(na.z & 0xffffu); t = (short)(na.z >> 16);
    it.kb0 = (short)(na.w & 0xffffu); it.kb1 = (short)(na.w >> 16);
    it.nb = (short)(nb_.x & 0xffffu); it.row0 = (short)(nb_.x >> 16);
    it.row_end = (short)(nb_.y & 0xffffu); it.cnt_idx = (short)(nb_.y >> 16);
    it.g = (int)(nb_.z & 0xffu); it.split = (int)((nb_.z >> 8) & 0xffu);
    o.which = (int)((nb_.z >> 16) & 0xffu); it.cnt_target = (int)(nb_.z >> 24);
    o.j = (int)nb_.w;
    it.tile = it.col0 / kTileM;
    it.col_end = (t < n_layer_ops && o.which == 2) ? (it.col0 >= ffn ? 2 * ffn : ffn) : a->op[o.which].out_dim;
    fetch(k + 1);
  }
  __device__ __forceinline__ void start(const FSeq& q) {
    recs = q.recs; n = q.n_my; k = 0; a = q.a; ffn = q.a->D.ffn; n_layer_ops = q.n_layer;
    fetch(0);
    take();
  }
  __device__ __forceinline__ void next(const FSeq&) {
    ++k;
    take();
  }
};

template <int GT>
__device__ __forceinline__ void bar_f() { asm volatile("bar.sync 1, %0;\n" ::"n"(GT) : "memory"); }

// Decision record handed from finalizer warp 0 to the group (double-buffered by loop iteration).
struct FJob {              // a completed out tile (gate/up: pair) waiting for its finalization
  int which, m, idx, j, row0, row_hi;
};
constexpr int kFlowQueue = 64;
struct FDec {
  int kind;                // 0 idle, 1 finalize a tile, 2 attention task, 3 layer-steps done
  int j;
  FJob job;
  AttnTask tk;
};

// ---------------------------------------------------------------- the kernel
template <bool PT>
__global__ void __launch_bounds__(kFlowThreads, 1) k_flow(const __grid_constant__ TmSet tm, const __grid_constant__ RoundArgs a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const Dev& D = a.D;
  const uint32_t plane_bytes = a.x_cap * 128;
  const uint32_t stage_bytes = kABytes + D.planes * plane_bytes;
  const int NS = a.n_stages;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)NS * stage_bytes);
  uint64_t* full = bars;
  uint64_t* empty = bars + NS;
  uint64_t* tfull = bars + 2 * NS;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  __shared__ int s_nb[16];
  __shared__ uint32_t s_valid[32];
  __shared__ int s_nvalid[kMaxGrp];
  __shared__ int s_live_ms;
  __shared__ int s_cum[kMaxGrp + 1];
  __shared__ int s_steps;
  __shared__ unsigned s_seen;            // grid barriers completed (tail of the round)
  __shared__ unsigned s_edone[4];        // items completed by each epilogue warp (an item is written when all four have)
  __shared__ short s_perm[kFlowTiles];
  __shared__ unsigned char s_glo[kFlowTiles], s_ghi[kFlowTiles];
  __shared__ int s_qtarget[kFlowSlices];
  __shared__ int s_ao_cnt[kFlowSlices];
  __shared__ FDec s_dec[2];
  __shared__ SeqState s_seq[8];          // the round's FSM snapshot
  __shared__ FJob s_queue[kFlowQueue];
  __shared__ unsigned s_qhead, s_qtail;  // jobs pushed by the counter warp / taken by the finalizer group
  __shared__ unsigned s_cdone;           // the counter warp has counted every layer-step item of this CTA
  __shared__ unsigned s_tail_items[3];   // this CTA's items up to and including tail op k (adapters W1, W2)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x < 32) s_valid[threadIdx.x] = 0;
  if (threadIdx.x >= 32 && threadIdx.x < 40) {
    const int s_ = threadIdx.x - 32;
    SeqState z;
    z.active = 0; z.q = 0; z.ctx_len = 0; z.n_tok = 0; z.last_tok = 0; z.pending = 0; z.done = 1; z.pad = 0;
    s_seq[s_] = s_ < D.max_seqs ? D.seqs[s_] : z;
  }
  if (threadIdx.x < kMaxGrp) s_nvalid[threadIdx.x] = 0;
  __syncthreads();
  for (int r = threadIdx.x; r < D.R_cap; r += blockDim.x)
    if (D.rows[r].valid) {
      atomicOr(&s_valid[r >> 5], 1u << (r & 31));
      if (r < D.R_dec) atomicAdd(&s_nvalid[D.rows[r].grp], 1);
    }
  for (int i = threadIdx.x; i < kFlowTiles; i += blockDim.x) {
    s_perm[i] = (short)a.flow_tab[kFtPerm + i];
    s_glo[i] = (unsigned char)a.flow_tab[kFtGlo + i];
    s_ghi[i] = (unsigned char)a.flow_tab[kFtGhi + i];
  }
  for (int i = threadIdx.x; i < kFlowSlices; i += blockDim.x) s_qtarget[i] = a.flow_tab[kFtTarget + i];
  __syncthreads();
  if (threadIdx.x == 0) {
    int steps = 0;
    for (int g = 0; g < 8; ++g) {
      // a stage without an expanded row (sparse lattice: only holes) is not live here: the counters order the ops of
      // a stage through waits that its rows satisfy, and it has nothing to compute anyway
      const int nb = (g < a.dec.n_grp && s_nvalid[g] > 0) ? D.grp_nb[g] : 0;
      s_nb[g] = nb;
      if (nb > 0) steps = max(steps, a.dec.layer_len[g]);
      s_nb[8 + g] = (g < a.ext.n_grp) ? D.exit_nb[g] : 0;
    }
    s_steps = steps;
    s_seen = 0;
    s_edone[0] = s_edone[1] = s_edone[2] = s_edone[3] = 0;
    s_qhead = s_qtail = 0;
    s_cdone = 0;
    // Attention families that are live AT THE SAME TIME: here the stages' attention work is spread in time (a stage's
    // heads become ready as its QKV tiles are finalized, stage after stage), so the chunk ranges are sized as if ONE
    // stage were live - the last stage's tasks are what the O projection waits for, and they find the grid idle.
    int lm = 0;
    for (int m = 0; m < D.N; ++m) {
      int lm_m = 0;
      for (int s = 0; s < D.max_seqs; ++s) {
        const SeqState st = D.seqs[s];
        if (!r_seq_live(st) || st.q < m) continue;
        lm_m += PT ? (r_stage_count(st.q, m) * (D.nh / D.nkv) + 15) / 16 : 1;
      }
      lm = max(lm, lm_m);
    }
    s_live_ms = lm;
    s_cum[0] = 0;
    for (int m = 0; m < kMaxGrp; ++m)
      s_cum[m + 1] = s_cum[m] + ((PT && m < D.N) ? D.max_seqs * ((cap_of(D.N, m) * (D.nh / D.nkv) + 15) / 16) : 0);
    for (int i = 0; i < NS; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&tfull[i], 1);
      mbar_init(&tempty[i], 4);
    }
    fence_mbar_init();
    for (int i = 0; i < (D.ad_m > 0 ? 7 : 5); ++i) tma_prefetch_desc(&tm.w[i]);
    for (int i = 0; i < 4; ++i) tma_prefetch_desc(&tm.x[i]);
    tma_prefetch_desc(&tm.wgu2);
  }
  if (warp == kWarpM) {
    tmem_alloc(tmem_slot, 2 * a.acc_cols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t lo_off = (!a.stacked && D.planes == 2) ? (uint32_t)a.x_cap : 0u;   // lo-plane accumulator columns (gemm_dev.cuh)

  FSeq sq;
  sq.a = &a; sq.s_nb = s_nb; sq.s_perm = s_perm; sq.n_steps = s_steps; sq.n_ad_ops = (D.ad_m > 0 && D.N >= 2) ? 2 : 0;
  sq.G = gridDim.x; sq.cta = blockIdx.x; sq.gu_half = (D.ffn + 127) / 128;
  const unsigned G = gridDim.x;
  int* const ctr = D.flow_ctr;
  // ---- the layer micro-ops (one projection of one live stage at one layer-step) in SKEWED order: micro-op (j, kind k,
  // live-stage rank m) has key (4j + k) n + 2m (n = live stages), ties to the lower stage.  Every stage's own chain
  // QKV -> O -> gate/up -> down -> next QKV stays in order, and between two dependent micro-ops of a stage lie n - 1
  // micro-ops of the others: their streams cover its attention tasks and last-arriver finalizations (with the plain
  // stage-major order the O projection of the LAST stage followed its QKV projection by three short ops and waited tens
  // of microseconds for its attention).
  __shared__ int s_n_layer;
  int* const mops = reinterpret_cast<int*>(smem + a.attn_smem_off);    // prologue scratch: the attention buffers
  int* const opn = mops + kMaxOps;
  unsigned char* const opi0 = reinterpret_cast<unsigned char*>(opn + kMaxOps + 1);
  if (threadIdx.x == 0) {
    int live[kMaxGrp], n = 0, cnt = 0;
    for (int g = 0; g < a.dec.n_grp; ++g)
      if (s_nb[g] > 0) live[n++] = g;
    if (n > 0) {
      const int key_end = 4 * n * s_steps + 2 * n;
      for (int key = 0; key < key_end; ++key)
        for (int m = 0; m < n; ++m) {
          const int rem = key - 2 * m;
          if (rem < 0 || rem % n) continue;
          const int jk = rem / n, j = jk >> 2, k = jk & 3;
          if (j < a.dec.layer_len[live[m]] && cnt < kMaxOps - 3) mops[cnt++] = (j << 8) | (k << 4) | live[m];
        }
    }
    s_n_layer = cnt;
  }
  __syncthreads();
  sq.mops = mops; sq.n_layer = s_n_layer;
  sq.n_ops = sq.n_layer + sq.n_ad_ops + 1;
  const int n_layer_ops = sq.n_layer;

  // ---- decode this CTA's items once (items are dealt round-robin, continuing across ops)
  sq.recs = reinterpret_cast<const FRec*>(D.item_recs) + (size_t)blockIdx.x * D.item_cap;
  sq.n_my = 0;
  if (s_steps > 0) {
    FRec* my = reinterpret_cast<FRec*>(D.item_recs) + (size_t)blockIdx.x * D.item_cap;
    for (int t = threadIdx.x; t < sq.n_ops; t += blockDim.x) {
      FOp o;
      sq.op_info(t, o);
      opn[t] = o.n_items;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int rr = 0, start = 0;
      for (int t = 0; t < sq.n_ops; ++t) {
        const int n = opn[t], i0 = (sq.cta + sq.G - rr) % sq.G;
        opi0[t] = (unsigned char)i0;
        opn[t] = start;
        start += n > i0 ? (n - i0 + sq.G - 1) / sq.G : 0;
        rr = (rr + n) % sq.G;
      }
      opn[sq.n_ops] = start;
      if (start > D.item_cap || sq.n_ops > kMaxOps) __trap();
    }
    __syncthreads();
    sq.n_my = opn[sq.n_ops];
    for (int k = threadIdx.x; k < sq.n_my; k += blockDim.x) {
      int lo = 0, hi = sq.n_ops;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (opn[mid] <= k) lo = mid; else hi = mid;
      }
      FOp o;
      FItem it;
      sq.op_info(lo, o);
      sq.decode(o, (int)opi0[lo] + (k - opn[lo]) * sq.G, it);
      FRec r;
      r.c1 = it.c1; r.col0 = it.col0; r.c2 = (short)it.c2; r.t = (short)lo; r.kb0 = (short)it.kb0; r.kb1 = (short)it.kb1;
      r.nb = (short)it.nb; r.row0 = (short)it.row0; r.row_end = (short)it.row_end; r.cnt_idx = (short)it.cnt_idx;
      r.g = (unsigned char)it.g; r.split = (unsigned char)it.split; r.which = (unsigned char)o.which;
      r.cnt_target = (unsigned char)it.cnt_target; r.j = o.j;
      my[k] = r;
    }
    __syncthreads();
  }

  if (s_steps > 0) {
    if (warp == kWarpW) {
      // ===================== weight producer: always as far ahead as the ring allows =====================
      FRecWalker w;
      unsigned st = 0, ph = 0;
      bool wrapped = false;
      for (w.start(sq); w.valid; w.next(sq)) {
        const CUtensorMap* desc = (w.t < n_layer_ops && w.o.which == 2) ? &tm.wgu2 : &tm.w[w.o.which];
        const uint32_t tx = kABytes + D.planes * w.it.nb * 128;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          if (wrapped) mbar_wait(&empty[st], ph ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(&full[st], tx);
            tma_load_3d(smem + (size_t)st * stage_bytes, desc, &full[st], kb * kTileK, w.it.c1, w.it.c2, kEvictFirst);
          }
          __syncwarp();
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; wrapped = true; }
        }
      }
    } else if (warp == kWarpA) {
      // ===================== activation producer: waits for the K slice of its item =====================
      // The counter of item i + 1 is requested (relaxed load) before the boxes of item i are issued and consumed after
      // them, so its L2 round trip (microseconds under the weight stream) is off the critical path.  The load is
      // relaxed: what depends on it are async-proxy (TMA) reads issued after fence.proxy.async, of data the finalizer
      // released at gpu scope before it bumped the counter; a gpu-scope acquire fence here stalls on the SM's
      // in-flight TMA traffic (measured: every fence.acq_rel.gpu costs microseconds of stream).
      FRecWalker w, wn;
      unsigned st = 0, ph = 0;
      bool wrapped = false;
      unsigned seen = 0;
      const int sl_x = a.op[0].kbps * kTileK, sl_o = a.op[1].kbps * kTileK, sl_f = a.op[3].kbps * kTileK;
      auto dep_of = [&](const FRecWalker& x, const int*& flag, int& target) {
        flag = nullptr; target = 0;
        if (!x.valid || x.t >= n_layer_ops) return;
        const int which = x.o.which, m = x.it.g, s = x.it.split, j = x.o.j;
        if (which == 0) {
          flag = ctr + kFcXa + m * kFlowSlices + s;
          target = j * tiles_in_slice(D.d, sl_x, s);
        } else if (which == 1) {
          flag = ctr + kFcAo + m * kFlowSlices + s;
          const int hs = (min((s + 1) * sl_o, D.nh * D.hd) - s * sl_o) / D.hd;
          target = (j + 1) * s_nvalid[m] * hs;
        } else if (which == 2) {
          flag = ctr + kFcXf + m * kFlowSlices + s;
          target = (j + 1) * tiles_in_slice(D.d, sl_x, s);
        } else {
          flag = ctr + kFcF + m * kFlowSlices + s;
          target = (j + 1) * tiles_in_slice(D.ffn, sl_f, s);
        }
      };
      w.start(sq);
      const int* f_cur;
      int t_cur, v_cur = 0;
      dep_of(w, f_cur, t_cur);
      if (t_cur > 0) v_cur = ld_relaxed_s32(f_cur);
      while (w.valid) {
        const int which = w.o.which;
        if (w.t < n_layer_ops) {
          if (t_cur > 0) {
            unsigned spins = 0;
            while (v_cur < t_cur) {
              __nanosleep(20);
              v_cur = ld_relaxed_s32(f_cur);
              if (++spins > 20000000u) flow_die(D, 1, which, (w.it.g << 16) | w.it.split, w.o.j, t_cur);
            }
            fence_proxy_async();
          }
        } else {
          // tail ops (adapters, exit head): published by grid barriers, as in k_round
          const int k = w.t - n_layer_ops;
          const unsigned need = sq.n_ad_ops ? (k == 0 ? 1u : (k == 1 ? 3u : 5u)) : 1u;
          if (seen < need) {
            unsigned spins = 0;
            while ((seen = *reinterpret_cast<volatile unsigned*>(&s_seen)) < need) {
              __nanosleep(32);
              if (++spins > 100000000u) __trap();
            }
            __threadfence_block();
            fence_proxy_async();
          }
        }
        wn = w;
        wn.next(sq);
        const int* f_n;
        int t_n, v_n = 0;
        dep_of(wn, f_n, t_n);
        if (t_n > 0) v_n = ld_relaxed_s32(f_n);              // consumed after this item's boxes are issued
        const CUtensorMap* desc = &tm.x[(which == 0 || which == 2 || which == 5) ? 0 : (which == 1 ? 1 : (which == 4 ? 3 : 2))];
        const int row0 = w.it.row0, nb = w.it.nb;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          if (wrapped) mbar_wait(&empty[st], ph ^ 1u);
          if (elect_one()) {
            uint8_t* sB = smem + (size_t)st * stage_bytes + kABytes;
            if (a.stacked) {
              for (int r = 0; r < nb; r += kBoxRows)
                tma_load_3d(sB + r * 256, desc, &full[st], kb * kTileK, row0 + r, 0, kEvictLast);
            } else {
              for (int p = 0; p < D.planes; ++p)
                for (int r = 0; r < nb; r += kBoxRows)
                  tma_load_3d(sB + p * plane_bytes + r * 128, desc, &full[st], kb * kTileK, row0 + r, p, kEvictLast);
            }
          }
          __syncwarp();
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; wrapped = true; }
        }
        w = wn; f_cur = f_n; t_cur = t_n; v_cur = v_n;
      }
    } else if (warp == kWarpM) {
      // ===================== MMA issuer =====================
      FRecWalker w;
      unsigned st = 0, ph = 0;
      int n_it = 0;
      const bool stacked = a.stacked != 0;
      for (w.start(sq); w.valid; w.next(sq), ++n_it) {
        const int as = n_it & 1;
        mbar_wait(&tempty[as], ((n_it >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * a.acc_cols;
        const uint32_t idesc = make_idesc_bf16_m128(stacked ? 2 * w.it.nb : w.it.nb);
        uint32_t acc = 0;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          mbar_wait(&full[st], ph);
          tc_fence_after();
          if (elect_one()) {
            mma_stage(smem_u32(smem + (size_t)st * stage_bytes), plane_bytes, D.planes, stacked, d_tmem, lo_off, idesc, acc);
            umma_commit(&empty[st]);
          }
          __syncwarp();
          acc = 1;
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; }
        }
        if (elect_one()) umma_commit(&tfull[as]);
        __syncwarp();
      }
    } else if (warp >= kWarpE0 && warp < kWarpE0 + 4) {
      // ===================== epilogue: TMEM -> partials of the op's own region / exit arg-max =====================
      const int quarter = warp & 3;
      EpiCtx ec;
      ec.rows = D.rows; ec.s_valid = s_valid; ec.vocab = D.vocab; ec.best_key = D.best_key;
      ec.ref_tile = D.ref_tile; ec.ref_tiles = D.ref_tiles; ec.dev = &D; ec.exit_map = D.exit_map;
      FRecWalker w;
      int n_it = 0;
      for (w.start(sq); w.valid; w.next(sq), ++n_it) {
        const int which = w.o.which;
        const OpDesc& od = a.op[which];
        ec.mode = which == 4 ? 1 : 0;
        ec.part = D.part + (w.t < n_layer_ops ? a.part_off[which] : 0);
        ec.part_ld = od.part_ld; ec.split_stride = od.split_stride; ec.out_dim = w.it.col_end;
        const int as = n_it & 1;
        mbar_wait(&tfull[as], (n_it >> 1) & 1);
        tc_fence_after();
        const uint32_t t_addr = tmem_base + as * a.acc_cols + ((uint32_t)(quarter * 32) << 16);
        epilogue_item(ec, t_addr, a.stacked != 0, lo_off, w.it.nb, w.it.row0, w.it.row_end, w.it.tile, w.it.col0, w.it.split, quarter, lane);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(&tempty[as]);
          red_release_cta_shared_add(&s_edone[quarter], 1u); // this warp's partials of the item are written
        }
      }
    } else if (warp == kWarpC) {
      // ===================== counter warp =====================
      // Every finished item of this CTA (all four epilogue warps have written its partials) is counted into its out
      // tile's counter; the arrival that completes the tile queues it for the finalizer group.  Lane l of a batch
      // handles item n_counted + l: the atomics of a batch are in flight together.
      FRecWalker wf;
      wf.start(sq);
      unsigned n_counted = 0, head = 0;
      int n_stamp = 0;
      if (D.taps && blockIdx.x == 0 && lane == 0) D.tap_times[n_stamp] = (unsigned long long)clock64();
      ++n_stamp;
      unsigned idle = 0;
      while (wf.valid && wf.t < n_layer_ops) {
        unsigned done = ld_acquire_cta_shared(&s_edone[lane & 3]);
        done = min(done, __shfl_xor_sync(0xffffffffu, done, 1));
        done = min(done, __shfl_xor_sync(0xffffffffu, done, 2));
        if (done <= n_counted) {
          __nanosleep(200);
          if (++idle > 30000000u) flow_die(D, 2, (int)n_counted, (int)done, wf.t, wf.i);
          continue;
        }
        idle = 0;
        const int n = (int)min(done - n_counted, 32u);
        FJob mine;
        int* cnt = nullptr;
        int target = 0, taken = 0;
        for (int i = 0; i < n && wf.valid && wf.t < n_layer_ops; ++i) {
          if (i == lane) {
            mine.which = wf.o.which; mine.m = wf.it.g; mine.idx = wf.it.cnt_idx; mine.j = wf.o.j;
            mine.row0 = wf.it.row0; mine.row_hi = min(wf.it.row0 + wf.it.nb, wf.it.row_end);
            cnt = ctr + kFcTile + (mine.which * kMaxGrp + mine.m) * kFlowTiles + mine.idx;
            target = (mine.j + 1) * wf.it.cnt_target;
          }
          const int t_before = wf.t;
          wf.next(sq);
          ++taken;
          if (D.taps && blockIdx.x == 0 && (!wf.valid || wf.t != t_before)) {
            if (lane == 0 && n_stamp < 20 * D.max_len + 60) D.tap_times[n_stamp] = (unsigned long long)clock64();
            ++n_stamp;                                        // CTA 0 counted its last item of an op
          }
        }
        n_counted += taken;
        bool last = false;
        // release: publishes this CTA's partials of the item.  The acquire side (an L1 invalidation on this SM, which
        // also costs the TMA units their cached descriptors) is paid only by an arrival that completes a tile.
        if (lane < taken) last = atom_acq_rel_add_s32(cnt, 1) + 1 == target;
        const unsigned bal = __ballot_sync(0xffffffffu, last);
        const unsigned bal_all = bal;
        const unsigned bal_own = PT ? 0u : __ballot_sync(0xffffffffu, last && mine.row_hi - mine.row0 <= 16 && s_nvalid[mine.m] <= 1);
        const unsigned bal_q = bal_all & ~bal_own;
        if (bal_own) {
          // Narrow lattices (a stage has a few rows): this warp finalizes the tiles its arrivals completed right away -
          // the finalizer group may be inside an attention task for tens of microseconds, and every finalization sits on
          // the dependency chain of the next op.  Warp unit = (row, 128 columns), the bodies of round_dev.cuh.
          const int sl_x = a.op[0].kbps * kTileK, sl_f = a.op[3].kbps * kTileK;
          for (unsigned rest = bal_own; rest; rest &= rest - 1) {
            const int b = __ffs(rest) - 1;
            const int which = __shfl_sync(0xffffffffu, mine.which, b), m = __shfl_sync(0xffffffffu, mine.m, b);
            const int idx = __shfl_sync(0xffffffffu, mine.idx, b), j = __shfl_sync(0xffffffffu, mine.j, b);
            const int row0 = __shfl_sync(0xffffffffu, mine.row0, b), row_hi = __shfl_sync(0xffffffffu, mine.row_hi, b);
            const float* part = D.part + a.part_off[which];
            if (which == 0) {
              const int hpt = kTileM / D.hd, h0 = idx * hpt;
              for (int u = 0; u < (row_hi - row0) * hpt; ++u) {
                const int r = row0 + u / hpt, hh = h0 + u % hpt;
                if (!((s_valid[r >> 5] >> (r & 31)) & 1u)) continue;
                if (D.hd == 128) unit_qkv<128>(a, j, part, r, hh, lane); else unit_qkv<64>(a, j, part, r, hh, lane);
              }
            } else {
              for (int r = row0; r < row_hi; ++r) {
                if (!((s_valid[r >> 5] >> (r & 31)) & 1u)) continue;
                if (which == 2) unit_silu(a, j, a.op[2], part, r, idx, lane);
                else unit_add_norm(a, j, which == 1 ? 0 : 1, a.op[which], part, r, idx, lane);
              }
            }
            fence_proxy_async();                             // operand planes are read by TMA
            __syncwarp();
            if (lane == 0) {
              if (which == 0) {
                for (int g = s_glo[idx]; g <= s_ghi[idx]; ++g) red_release_add_s32(ctr + kFcQkv + m * kFlowSlices + g, 1);
              } else if (which == 1) {
                red_release_add_s32(ctr + kFcXf + m * kFlowSlices + (idx * kTileM) / sl_x, 1);
              } else if (which == 2) {
                red_release_add_s32(ctr + kFcF + m * kFlowSlices + (idx * kTileM) / sl_f, 1);
              } else {
                red_release_add_s32(ctr + kFcXa + m * kFlowSlices + (idx * kTileM) / sl_x, 1);
              }
            }
            __syncwarp();
          }
        }
        if (bal_q) {
          const unsigned bal = bal_q;
          const bool last = (bal >> lane) & 1u;
          const int n_new = __popc(bal);
          unsigned spins = 0;
          while (head + n_new - ld_acquire_cta_shared(&s_qtail) > (unsigned)kFlowQueue) {   // queue space
            __nanosleep(32);
            if (++spins > 100000000u) __trap();
          }
          if (last) s_queue[(head + __popc(bal & ((1u << lane) - 1u))) % kFlowQueue] = mine;
          __syncwarp();
          head += n_new;
          if (lane == 0) asm volatile("st.release.cta.shared.u32 [%0], %1;\n" ::"r"(smem_u32(&s_qhead)), "r"(head) : "memory");
        }
      }
      // this CTA's item counts through the adapter ops (the finalizer group waits for their partials in the tail)
      for (int k = 0; k < 2; ++k) {
        while (wf.valid && wf.t == n_layer_ops + k && sq.n_ad_ops) { wf.next(sq); ++n_counted; }
        if (lane == 0) s_tail_items[k] = n_counted;
      }
      __syncwarp();
      if (lane == 0) asm volatile("st.release.cta.shared.u32 [%0], %1;\n" ::"r"(smem_u32(&s_cdone)), "r"(1u) : "memory");
      if (D.taps && blockIdx.x == 0 && lane == 0 && n_stamp < 20 * D.max_len + 60) D.tap_times[n_stamp] = (unsigned long long)clock64();
    } else if (flow_fin_index(warp) >= 0) {
      // ===================== finalizer group (warps 7-10) =====================
      const int we = flow_fin_index(warp), tid_f = we * 32 + lane;
      constexpr int GT = kFT;
      AttnPlan pl;
      attn_plan<PT>(a, G, s_live_ms, s_cum, pl);
      // A CTA runs its attention tasks in order, each waiting for its head's QKV counter: the order must follow the op
      // order (stage-major within a layer-step).  k_round's heaviest-range-first deal puts tasks of LATER stages first,
      // and such a task blocks one that an earlier op is waiting for: deadlock on lattices with more tasks than CTAs.
      pl.lpt = 0;
      const int sl_x = a.op[0].kbps * kTileK, sl_f = a.op[3].kbps * kTileK, sl_o = a.op[1].kbps * kTileK;
      void* const asm_ = smem + a.attn_smem_off;
      // warp 0 of the group owns the cursors: queue tail, next attention task
      unsigned tail = 0;
      int att_j = 0, att_u = blockIdx.x;
      AttnTask tk;
      bool have = false;
      unsigned it_no = 0, idle = 0;
      for (;; ++it_no) {
        FDec* dec = &s_dec[it_no & 1];
        if (we == 0) {
          int kind = 0;
          const unsigned cdone = ld_acquire_cta_shared(&s_cdone);      // read BEFORE the head: done => head is final
          const unsigned head = ld_acquire_cta_shared(&s_qhead);
          if (tail < head) {
            kind = 1;
            if (lane == 0) {
              dec->job = s_queue[tail % kFlowQueue];
              asm volatile("st.release.cta.shared.u32 [%0], %1;\n" ::"r"(smem_u32(&s_qtail)), "r"(tail + 1) : "memory");
            }
            ++tail;
          } else {
            // next live attention task of this CTA (dead ones are skipped without waiting); decoded once, then only
            // its counter is polled
            while (!have && att_j < sq.n_steps) {
              if (att_u >= pl.n_tasks) { ++att_j; att_u = blockIdx.x; continue; }
              attn_task_of<PT>(a, pl, s_cum, G, att_u, tk);
              const SeqState sst = s_seq[tk.s];
              if (!r_seq_live(sst) || sst.q < tk.m || att_j >= a.dec.layer_len[tk.m] || s_nb[tk.m] == 0) { att_u += G; continue; }
              have = true;
            }
            if (have) {
              int v = 0;
              if (lane == 0) v = ld_relaxed_s32(ctr + kFcQkv + tk.m * kFlowSlices + tk.g);
              v = __shfl_sync(0xffffffffu, v, 0);
              if (v >= s_qtarget[tk.g] * (att_j + 1)) {
                // polled with relaxed loads (an acquire costs the SM an L1 invalidation every time); ONE acquire load of
                // the counter that has reached its target
                if (lane == 0) v = ld_acquire_s32(ctr + kFcQkv + tk.m * kFlowSlices + tk.g);
                kind = 2;
                if (lane == 0) { dec->tk = tk; dec->j = att_j; }
                att_u += G;
                have = false;
              }
            } else if (cdone) {
              kind = 3;
            }
          }
          if (lane == 0) dec->kind = kind;
        }
        bar_f<GT>();
        const int kind = dec->kind;
        if (kind == 3) break;
        if (kind == 1) {
          idle = 0;
          const int which = dec->job.which, m = dec->job.m, idx = dec->job.idx, j = dec->job.j;
          const int row0 = dec->job.row0, row_hi = dec->job.row_hi;
          const float* part = D.part + a.part_off[which];
          if (which == 0) {
            const int hpt = kTileM / D.hd, h0 = idx * hpt;    // heads of the fused QKV output in this tile
            for (int u = we; u < (row_hi - row0) * hpt; u += GT / 32) {
              const int r = row0 + u / hpt, hh = h0 + u % hpt;
              if (D.hd == 128) unit_qkv<128>(a, j, part, r, hh, lane); else unit_qkv<64>(a, j, part, r, hh, lane);
            }
          } else if (which == 2) {
            for (int r = row0 + we; r < row_hi; r += GT / 32) unit_silu(a, j, a.op[2], part, r, idx, lane);
          } else {
            for (int r = row0 + we; r < row_hi; r += GT / 32) unit_add_norm(a, j, which == 1 ? 0 : 1, a.op[which], part, r, idx, lane);
          }
          fence_proxy_async();                               // operand planes are read by TMA
          bar_f<GT>();
          if (tid_f == 0) {
            if (which == 0) {
              for (int g = s_glo[idx]; g <= s_ghi[idx]; ++g) red_release_add_s32(ctr + kFcQkv + m * kFlowSlices + g, 1);
            } else if (which == 1) {
              red_release_add_s32(ctr + kFcXf + m * kFlowSlices + (idx * kTileM) / sl_x, 1);
            } else if (which == 2) {
              red_release_add_s32(ctr + kFcF + m * kFlowSlices + (idx * kTileM) / sl_f, 1);
            } else {
              red_release_add_s32(ctr + kFcXa + m * kFlowSlices + (idx * kTileM) / sl_x, 1);
            }
          }
        } else if (kind == 2) {
          idle = 0;
          const AttnTask tk = dec->tk;
          const int j = dec->j;
          if (tid_f < kFlowSlices) s_ao_cnt[tid_f] = 0;
          bar_f<GT>();
          if (D.hd == 128) attn_run<128, GT, PT>(a, pl, tk, j, tid_f, lane, we, reinterpret_cast<AttnSmem<128>*>(asm_), s_ao_cnt, sl_o, s_seq);
          else attn_run<64, GT, PT>(a, pl, tk, j, tid_f, lane, we, reinterpret_cast<AttnSmem<64>*>(asm_), s_ao_cnt, sl_o, s_seq);
          fence_proxy_async();                               // act_o is read by TMA
          bar_f<GT>();
          if (tid_f < kFlowSlices) {
            const int c = s_ao_cnt[tid_f];
            if (c > 0) red_release_add_s32(ctr + kFcAo + tk.m * kFlowSlices + tid_f, c);
          }
        } else {
          __nanosleep(200);
          if (++idle > 30000000u) flow_die(D, 3, (int)tail, att_j, att_u, (int)ld_acquire_cta_shared(&s_cdone));   // protocol bug
        }
      }
      // ---- tail of the round: grid barriers publish the operands of the adapters / the exit head (as in k_round)
      unsigned gb = 0;
      ++gb; grid_bar<GT>(D.gbar, gb * G, tid_f, &s_seen, gb);        // every layer-step finalization is done
      if (sq.n_ad_ops) {
        const int gw = blockIdx.x * (GT / 32) + we, n_gw = gridDim.x * (GT / 32);
        for (int k = 0; k < 2; ++k) {
          // wait until this CTA's epilogue warps have written the partials of all of its items of adapter op k
          if (tid_f == 0) {
            const unsigned need = s_tail_items[k];
            unsigned spins = 0;
            while (min(min(ld_acquire_cta_shared(&s_edone[0]), ld_acquire_cta_shared(&s_edone[1])),
                       min(ld_acquire_cta_shared(&s_edone[2]), ld_acquire_cta_shared(&s_edone[3]))) < need) {
              __nanosleep(32);
              if (++spins > 100000000u) __trap();
            }
          }
          ++gb; grid_bar<GT>(D.gbar, gb * G, tid_f, &s_seen, gb);
          if (k == 0) glue_ad1(a, a.op[5], gw, n_gw, lane); else glue_ad2(a, a.op[6], gw, n_gw, lane);
          ++gb; grid_bar<GT>(D.gbar, gb * G, tid_f, &s_seen, gb);
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == kWarpM) tmem_dealloc(tmem_base, 2 * a.acc_cols);
}

cudaError_t flow_init() {
  cudaError_t e = cudaFuncSetAttribute(k_flow<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 223 * 1024);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_flow<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 223 * 1024);
}

// Cooperative launch: all CTAs must be co-resident (they wait on one another's counters).
cudaError_t launch_flow(const TmSet& tm, const RoundArgs& a, int grid, size_t smem_bytes, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kFlowThreads);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  if (cap_of(a.D.N, 0) * (a.D.nh / a.D.nkv) > kAttnPairs) return cudaLaunchKernelEx(&cfg, k_flow<true>, tm, a);
  return cudaLaunchKernelEx(&cfg, k_flow<false>, tm, a);
}

}  // namespace dexk
