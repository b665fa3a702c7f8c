// kernels.cu — everything of the DEX step that is not the weight-streaming GEMM:
// lattice bookkeeping (expand / insert / validate_and_commit / collapse / advance, PAPER.md:143-190,
// 196-208), RMSNorm / RoPE / SwiGLU glue, the lattice-masked paged decode attention
// (north_star (b)) and the commit-and-collapse kernels (north_star (d)).
#include "common.cuh"

namespace dexk {

// ------------------------------------------------------------------------------------------
// helpers
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// Block-wide sum with a fixed reduction tree (deterministic for a given blockDim).
__device__ __forceinline__ float block_sum(float v, float* red /*[33]*/) {
  v = warp_sum(v);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  if (w == 0) {
    float t = (l < nw) ? red[l] : 0.f;
    t = warp_sum(t);
    if (l == 0) red[32] = t;
  }
  __syncthreads();
  return red[32];
}
// Programmatic dependent launch: every kernel between the first segment GEMM and the exit GEMM
// is launched with programmatic stream serialization; it lets its dependents start early
// (pdl_trigger) and waits for its own predecessor before touching anything that predecessor
// wrote (pdl_wait).  Row tables / grp_nb are written before k_gather_norm, which is a normal
// launch, so they are complete for every later kernel of the round.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 add4(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
// sum of the split-K partials, added in split order (fixed order: H3)
__device__ __forceinline__ float4 sum_splits4(const float* p, int ksplit, size_t split_stride) {
  float4 acc = ld4(p);
#pragma unroll 4
  for (int s = 1; s < ksplit; ++s) acc = add4(acc, ld4(p + (size_t)s * split_stride));
  return acc;
}
__device__ __forceinline__ void split_store4(__nv_bfloat16* base, size_t plane_stride, size_t idx, float4 v, int planes) {
  __nv_bfloat162 h0 = __floats2bfloat162_rn(v.x, v.y), h1 = __floats2bfloat162_rn(v.z, v.w);
  uint2 pk;
  pk.x = *reinterpret_cast<uint32_t*>(&h0);
  pk.y = *reinterpret_cast<uint32_t*>(&h1);
  *reinterpret_cast<uint2*>(base + idx) = pk;
  if (planes > 1) {
    const float2 f0 = __bfloat1622float2(h0), f1 = __bfloat1622float2(h1);
    __nv_bfloat162 l0 = __floats2bfloat162_rn(v.x - f0.x, v.y - f0.y), l1 = __floats2bfloat162_rn(v.z - f1.x, v.w - f1.y);
    pk.x = *reinterpret_cast<uint32_t*>(&l0);
    pk.y = *reinterpret_cast<uint32_t*>(&l1);
    *reinterpret_cast<uint2*>(base + plane_stride + idx) = pk;
  }
}

__device__ __forceinline__ bool seq_live(const SeqState& s) { return s.active && !s.done && !s.pending; }
__device__ __forceinline__ int round16(int v) { return (v + 15) & ~15; }

// rows of stage m that are live for a sequence at FSM state q (2^{q-1-m}, stage q: 1)
__device__ __forceinline__ int stage_count(int q, int m) { return m > q ? 0 : (m == q ? 1 : (1 << (q - 1 - m))); }

// ------------------------------------------------------------------------------------------
// a0: expand bookkeeping.  ONE block, one thread per row slot of the decode plan (R_cap <= 1024): the valid rows are
// ranked with a block-wide scan, which gives every row its DENSE exit row (the exit head then streams the LM head once
// per exit_chunk valid rows instead of once per exit_chunk row slots: at N = 8 the slots of a low-q round span both
// chunks although a handful of rows are live).
__global__ void __launch_bounds__(1024) k_rows_decode(Dev D, Plan plan) {
  __shared__ int s_wcnt[32];
  const int r = threadIdx.x;
  for (int i = r; i < kFcTotal; i += blockDim.x) D.flow_ctr[i] = 0;   // k_flow: arrival counters / ready flags
  if (r == 0) {
    *D.gbar = 0u;                                     // grid-barrier counter of this round's k_round
    // live row extent of every stage group
    for (int m = 0; m < kMaxGrp; ++m) {
      int ext = 0;
      if (m < D.N) {
        const int cap = cap_of(D.N, m);
        for (int s = 0; s < D.max_seqs; ++s) {
          const SeqState st = D.seqs[s];
          if (seq_live(st) && st.q >= m) ext = max(ext, s * cap + stage_count(st.q, m));
        }
      }
      D.grp_nb[m] = round16(ext);
    }
  }
  const bool in_range = r < D.R_cap;
  if (in_range) D.best_key[r] = 0ull;
  RowInfo ri;
  ri.valid = 0;
  ri.seq = 0; ri.node = -1; ri.pos = -1; ri.grp = 0; ri.slot = 0; ri.n_paged = 0; ri.n_anc = 0;   // a clean dead row
  ri.parent_row = -1; ri.tok_in = 0; ri.is_ref = 0; ri.n_mask = 0;
  if (in_range && r < D.R_dec) {
    int m = 0;
    while (m + 1 < D.N && r >= plan.row_base[m + 1]) ++m;
    const int cap = cap_of(D.N, m);
    const int local = r - plan.row_base[m];
    const int s = local / cap, j = local % cap;
    if (s < D.max_seqs) {
      const SeqState st = D.seqs[s];
      const int q = st.q;
      const int o = (m == q) ? 0 : ((j << (m + 1)) | (1 << m));
      bool expand = seq_live(st) && j < stage_count(q, m);
      // sparse lattice (R26): within P positions of the commit position, under an expanded parent (B holds its token)
      if (expand && D.lookahead > 0 && q > 0)
        expand = __popc(o) <= D.lookahead && D.B[s * D.n_nodes + node_id(q - 1, o >> 1)] >= 0;
      if (expand) {
        ri.valid = 1;
        ri.seq = s;
        ri.node = node_id(q, o);
        ri.pos = st.ctx_len + __popc(o);
        ri.grp = m;
        ri.n_paged = st.ctx_len;
        // ancestor slots: the slot of the node at which each position move on the root path was taken
        int na = 0, lvl = 0, off = 0;
        for (int b = q - 1; b >= 0; --b) {
          const int mv = (o >> b) & 1;
          if (mv) {
            const int ms = stage_of(lvl, off);                     // strip trailing depth moves
            ri.anc[na++] = compact_slot(node_id(lvl - ms, off >> ms));
          }
          off = (off << 1) | mv;
          ++lvl;
        }
        ri.n_anc = na;
        for (int i = na; i < kMaxAnc; ++i) ri.anc[i] = 0;
        ri.slot = compact_slot(node_id(q - m, o >> m));
        // input: root <- last committed token; depth child <- parent's hidden; position child <- parent's candidate
        if (q == 0) {
          ri.parent_row = -1;
          ri.tok_in = st.last_tok;
        } else if ((o & 1) == 0) {
          const int op = o >> 1, mp = stage_of(q - 1, op);
          ri.parent_row = plan.row_base[mp] + s * cap_of(D.N, mp) + idx_in_stage(q - 1, op, mp);
          ri.tok_in = -1;
        } else {
          ri.parent_row = -1;
          ri.tok_in = D.B[s * D.n_nodes + node_id(q - 1, o >> 1)];
        }
        // DECS mask (Alg. 2 lines 1-7): tokens of shallower nodes of the same slot chain; the
        // final-depth reference node 2^{N-1}-1 is never masked.
        ri.is_ref = (q == D.N - 1 && o == 0) ? 1 : 0;
        int nm = 0;
        if (D.decs && !ri.is_ref) {
          for (int i = 0; i < m; ++i) ri.mask_tok[nm++] = D.B[s * D.n_nodes + node_id(q - m + i, (o >> m) << i)];
        }
        ri.n_mask = nm;
        for (int i = nm; i < kMaxAnc; ++i) ri.mask_tok[i] = -1;
      }
    }
  }
  // dense rank of the valid rows (ascending row index) = exit row
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  const unsigned bal = __ballot_sync(0xffffffffu, ri.valid != 0);
  if (lane == 0) s_wcnt[wp] = __popc(bal);
  __syncthreads();
  int base = 0, total = 0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
    base += w < wp ? s_wcnt[w] : 0;
    total += s_wcnt[w];
  }
  const int rank = base + __popc(bal & ((1u << lane) - 1u));
  ri.exit_row = ri.valid ? rank : 0;
  ri.pad[0] = ri.pad[1] = ri.pad[2] = 0;
  if (in_range) {
    D.rows[r] = ri;
    if (ri.valid) D.exit_map[rank] = r;
    if (r >= total) D.exit_map[r] = -1;
  }
  if (r < kMaxGrp) {                                  // live extent of every exit chunk of the dense rows
    const int e = min(D.exit_chunk, total - D.exit_chunk * r);
    D.exit_nb[r] = e > 0 ? round16(e) : 0;
  }
}

// Prefill rows: positions p0 .. p0+R-1 of the prompt as one causal chunk.
__global__ void k_rows_prefill(Dev D, int seq, int p0, int R) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) {
    for (int m = 0; m < kMaxGrp; ++m) {
      D.grp_nb[m] = (m == 0) ? round16(R) : 0;
      D.exit_nb[m] = 0;
    }
  }
  if (r >= D.R_cap) return;
  RowInfo ri;
  ri.valid = 0;
  if (r < R) {
    ri.valid = 1;
    ri.seq = seq;
    ri.node = -1;
    ri.pos = p0 + r;
    ri.grp = 0;
    ri.slot = -1;
    ri.n_paged = p0 + R;
    ri.n_anc = 0;
    for (int i = 0; i < kMaxAnc; ++i) ri.anc[i] = 0, ri.mask_tok[i] = -1;
    ri.parent_row = -1;
    ri.tok_in = D.tokens[seq * (D.max_ctx + 1) + p0 + r];
    ri.is_ref = 0;
    ri.n_mask = 0;
  }
  ri.exit_row = r;                                    // no exit op in prefill; keeps the last norm's (unused) operand row in range
  D.exit_map[r] = -1;
  D.rows[r] = ri;
}

__global__ void k_seq_init(Dev D, int seq, int n) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    SeqState st;
    st.active = 1;
    st.q = 0;
    st.ctx_len = n - 1;
    st.n_tok = n;
    st.last_tok = D.tokens[seq * (D.max_ctx + 1) + n - 1];
    st.pending = 0;
    st.done = (n >= D.max_ctx) ? 1 : 0;               // same rule as the host mirror (dex_prefill / dex_rewind)
    st.pad = 0;
    D.seqs[seq] = st;
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < D.n_nodes; i += gridDim.x * blockDim.x)
    D.B[seq * D.n_nodes + i] = -1;
}

__global__ void k_rope_table(Dev D, double theta, int n_pos) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int half = D.hd / 2;
  if (i >= n_pos * half) return;
  const int pos = i / half, f = i % half;
  const double ang = (double)pos * pow(theta, -2.0 * (double)f / (double)D.hd);
  D.rope[i] = make_float2((float)cos(ang), (float)sin(ang));
}

// ------------------------------------------------------------------------------------------
// a1 + first RMSNorm: h_in = parent's frontier hidden (depth expansion) or Embed[tok]
// (position expansion), then a = RMSNorm(h_in; w_attn[first layer of the stage]).
__global__ void __launch_bounds__(1024) k_gather_norm(Dev D, Plan plan) {
  const int r = blockIdx.x;
  const RowInfo ri = D.rows[r];
  if (!ri.valid) return;
  float* x = D.x_cur + (size_t)r * D.d;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  const int n_seg = (D.d + 127) / 128;
  const float* w = D.norm_attn + (size_t)plan.layer_lo[ri.grp] * D.d;
  const size_t ps = (size_t)D.R_cap * D.d;
  // Warp unit = 128-element segment, lane = 4 consecutive elements, sum of squares per segment: the SAME reduction as
  // the add+norm units of the round kernels and k_add_norm (deferred RMSNorm scale, H3: a row's norm must not depend
  // on which kernel produced it)
  for (int seg = warp; seg < kSsSeg; seg += n_warps) {
    float ss = 0.f;
    const int i = seg * 128 + lane * 4;
    if (seg < n_seg && i < D.d) {
      float4 v;
      if (ri.parent_row >= 0) {
        v = ld4(D.x_front + (size_t)ri.parent_row * D.d + i);
      } else {
        const uint2 pk = *reinterpret_cast<const uint2*>(D.embed + (size_t)ri.tok_in * D.d + i);
        const float2 a = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&pk.x));
        const float2 b = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&pk.y));
        v = make_float4(a.x, a.y, b.x, b.y);
      }
      *reinterpret_cast<float4*>(x + i) = v;
      ss = sumsq4(v);
      const float4 wv = ld4(w + i);
      split_store4(D.act_a, ps, (size_t)r * D.d + i, make_float4(v.x * wv.x, v.y * wv.y, v.z * wv.z, v.w * wv.w), D.planes);
    }
    ss = warp_sum(ss);
    if (lane == 0) D.ss_part[(size_t)r * kSsSeg + seg] = ss;                 // unused segments hold 0
  }
}

// x += sum_s part[s]; then RMSNorm into the next GEMM's operand planes.
//   mode 0 (after o_proj):    w = norm_ffn[l]                      -> act_a
//   mode 1 (after down_proj): w = norm_attn[l+1] if the stage continues -> act_a,
//                             else the shared final norm (exit) -> act_e
// One CTA per row; warp unit = 128-element segment (see k_gather_norm), all split loads of a unit in flight at once.
__global__ void __launch_bounds__(1024) k_add_norm(Dev D, Plan plan, int step, int mode, int ksplit, size_t split_stride, int ld) {
  pdl_trigger();
  const int r = blockIdx.x;
  const RowInfo ri = D.rows[r];
  if (!ri.valid || step >= plan.layer_len[ri.grp]) return;
  const int layer = plan.layer_lo[ri.grp] + step;
  float* x = D.x_cur + (size_t)r * D.d;
  const float* p = D.part + (size_t)r * ld;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  const int n_seg = (D.d + 127) / 128;
  const float* w;
  __nv_bfloat16* dst = D.act_a;
  if (mode == 0) {
    w = D.norm_ffn + (size_t)layer * D.d;
  } else if (step + 1 < plan.layer_len[ri.grp]) {
    w = D.norm_attn + (size_t)(layer + 1) * D.d;
  } else {
    w = D.norm_final;
    dst = D.act_e;
  }
  const size_t ps = (size_t)D.R_cap * D.d;
  pdl_wait();
  for (int seg = warp; seg < n_seg; seg += n_warps) {
    float ss = 0.f;
    const int i = seg * 128 + lane * 4;
    if (i < D.d) {
      const float4 a = sum_splits4(p + i, ksplit, split_stride);
      const float4 v = add4(ld4(x + i), a);
      *reinterpret_cast<float4*>(x + i) = v;
      ss = sumsq4(v);
      if (mode == 1 && D.taps) *reinterpret_cast<float4*>(D.tap_hidden + ((size_t)r * D.max_len + step) * D.d + i) = v;
      const float4 wv = ld4(w + i);
      split_store4(dst, ps, (size_t)(dst == D.act_e ? ri.exit_row : r) * D.d + i, make_float4(v.x * wv.x, v.y * wv.y, v.z * wv.z, v.w * wv.w), D.planes);
    }
    ss = warp_sum(ss);
    if (lane == 0) D.ss_part[(size_t)r * kSsSeg + seg] = ss;
  }
}

// q,k,v = sum of split-K partials; RoPE (rotate-half, R13) on q,k; q -> fp32 buffer; k,v -> bf16
// into the row's slot K/V (branch-private) or, for prefill rows, straight into committed pages.
// grid (rows, blocks): a thread owns 4 consecutive dims of one head (and their rotate-half partners).
__global__ void __launch_bounds__(256) k_rope_kv(Dev D, Plan plan, int step, int ksplit, size_t split_stride, int ld) {
  pdl_trigger();
  const int r = blockIdx.x;
  const RowInfo ri = D.rows[r];
  if (!ri.valid || step >= plan.layer_len[ri.grp]) return;
  const int layer = plan.layer_lo[ri.grp] + step;
  const int hd = D.hd, half = hd / 2, qd = half / 4;     // qd: float4 groups per half head
  const float* p = D.part + (size_t)r * ld;
  const float2* rt = D.rope + (size_t)ri.pos * half;
  const size_t kvo = (ri.slot >= 0) ? slot_off(D, ri.seq, ri.slot, layer) : page_off(D, ri.seq, layer, ri.pos);
  __nv_bfloat16* kd = ((ri.slot >= 0) ? D.kslot : D.kpool) + kvo;
  __nv_bfloat16* vd = ((ri.slot >= 0) ? D.vslot : D.vpool) + kvo;
  const int nq = D.nh * hd, nk = D.nkv * hd;
  const int n_rot = (D.nh + D.nkv) * qd;                 // rotated float4 pair groups
  const int n_v = nk / 4;
  pdl_wait();
  const float inv = inv_rms(D, r);                       // deferred RMSNorm scale of the QKV input
  for (int t = blockIdx.y * blockDim.x + threadIdx.x; t < n_rot + n_v; t += gridDim.y * blockDim.x) {
    if (t < n_rot) {
      const int h = t / qd, i = (t % qd) * 4;
      const int i1 = h * hd + i, i2 = i1 + half;
      float4 a = sum_splits4(p + i1, ksplit, split_stride);
      float4 b = sum_splits4(p + i2, ksplit, split_stride);
      a.x *= inv; a.y *= inv; a.z *= inv; a.w *= inv;
      b.x *= inv; b.y *= inv; b.z *= inv; b.w *= inv;
      const float2 c0 = rt[i], c1 = rt[i + 1], c2 = rt[i + 2], c3 = rt[i + 3];
      const float4 o1 = make_float4(a.x * c0.x - b.x * c0.y, a.y * c1.x - b.y * c1.y, a.z * c2.x - b.z * c2.y, a.w * c3.x - b.w * c3.y);
      const float4 o2 = make_float4(b.x * c0.x + a.x * c0.y, b.y * c1.x + a.y * c1.y, b.z * c2.x + a.z * c2.y, b.w * c3.x + a.w * c3.y);
      if (h < D.nh) {
        *reinterpret_cast<float4*>(D.qbuf + (size_t)r * nq + i1) = o1;
        *reinterpret_cast<float4*>(D.qbuf + (size_t)r * nq + i2) = o2;
      } else {
        __nv_bfloat162 x0 = __floats2bfloat162_rn(o1.x, o1.y), x1 = __floats2bfloat162_rn(o1.z, o1.w);
        __nv_bfloat162 y0 = __floats2bfloat162_rn(o2.x, o2.y), y1 = __floats2bfloat162_rn(o2.z, o2.w);
        *reinterpret_cast<__nv_bfloat162*>(kd + i1 - nq) = x0;
        *reinterpret_cast<__nv_bfloat162*>(kd + i1 - nq + 2) = x1;
        *reinterpret_cast<__nv_bfloat162*>(kd + i2 - nq) = y0;
        *reinterpret_cast<__nv_bfloat162*>(kd + i2 - nq + 2) = y1;
      }
    } else {
      const int i = (t - n_rot) * 4;
      const float4 a = sum_splits4(p + nq + nk + i, ksplit, split_stride);
      *reinterpret_cast<__nv_bfloat162*>(vd + i) = __floats2bfloat162_rn(a.x * inv, a.y * inv);
      *reinterpret_cast<__nv_bfloat162*>(vd + i + 2) = __floats2bfloat162_rn(a.z * inv, a.w * inv);
    }
  }
}

// act = SiLU(gate) * up  (SwiGLU), from the split-K partials of the fused gate/up projection.
__global__ void __launch_bounds__(256) k_silu_mul(Dev D, Plan plan, int step, int ksplit, size_t split_stride, int ld) {
  pdl_trigger();
  const int r = blockIdx.x;
  const RowInfo ri = D.rows[r];
  if (!ri.valid || step >= plan.layer_len[ri.grp]) return;
  const float* p = D.part + (size_t)r * ld;
  const size_t ps = (size_t)D.R_cap * D.ffn;
  pdl_wait();
  const float inv = inv_rms(D, r);                       // deferred RMSNorm scale of the gate/up input
  for (int i = (blockIdx.y * blockDim.x + threadIdx.x) * 4; i < D.ffn; i += gridDim.y * blockDim.x * 4) {
    float4 g = sum_splits4(p + i, ksplit, split_stride);
    float4 u = sum_splits4(p + D.ffn + i, ksplit, split_stride);
    g.x *= inv; g.y *= inv; g.z *= inv; g.w *= inv;
    u.x *= inv; u.y *= inv; u.z *= inv; u.w *= inv;
    float4 a;
    a.x = g.x / (1.0f + expf(-g.x)) * u.x;
    a.y = g.y / (1.0f + expf(-g.y)) * u.y;
    a.z = g.z / (1.0f + expf(-g.z)) * u.z;
    a.w = g.w / (1.0f + expf(-g.w)) * u.w;
    split_store4(D.act_f, ps, (size_t)r * D.ffn + i, a, D.planes);
  }
}

// ------------------------------------------------------------------------------------------
// a3: lattice-masked decode attention, split over fixed 64-position chunks of ABSOLUTE position.
// CTA = (chunk, kv head, (group, sequence)): the committed-prefix K/V of the chunk is staged in
// shared memory once (128-bit loads, XOR-swizzled rows) and applied to every branch row of that
// (stage, sequence) and every query head of the GQA group.  Positions >= n_paged are the row's
// branch-private suffix: K/V of its ancestor slots and its own slot, picked per row from the
// ancestry list (the "ancestry bitmask" of north_star (b), stored as a slot list).  A position's
// arithmetic is identical wherever its K/V lives, so a row gives the same bits before and after
// its ancestors are committed.  row_split > 1 (prefill: 128 causal rows per (chunk, head)) deals the rows of a
// (stage, sequence) to that many CTAs, each staging the chunk for itself: the per-row arithmetic is unchanged.
template <int HD>
__global__ void __launch_bounds__(128) k_attn(Dev D, Plan plan, int step, int kv_static, int row_split) {
  constexpr int CPR = HD / 8;                       // 16-byte chunks per K/V row
  __shared__ __align__(16) __nv_bfloat16 sK[kChunk * HD];
  __shared__ __align__(16) __nv_bfloat16 sV[kChunk * HD];
  __shared__ __align__(16) float sQ[4][HD];
  __shared__ float sP[4][kChunk];
  __shared__ int row_list[256];
  __shared__ int n_rows_s, max_pos_s, n_paged_s;

  pdl_trigger();
  const int c = blockIdx.x, g = blockIdx.y;
  const int sub = blockIdx.z % row_split, zz = blockIdx.z / row_split;
  const int m = zz / D.max_seqs, s = zz % D.max_seqs;
  if (m >= plan.n_grp || step >= plan.layer_len[m]) return;
  const int nb = D.grp_nb[m];
  if (nb == 0) return;
  const int per = (nb + row_split - 1) / row_split;
  const int r_lo = plan.row_base[m] + sub * per, r_hi = min(r_lo + per, plan.row_base[m] + nb);
  const int layer = plan.layer_lo[m] + step;
  const int c0 = c * kChunk;

  if (threadIdx.x == 0) {
    n_rows_s = 0;
    max_pos_s = -1;
    n_paged_s = 0;
  }
  __syncthreads();
  for (int r = r_lo + threadIdx.x; r < r_hi; r += blockDim.x) {
    const RowInfo* ri = &D.rows[r];
    if (ri->valid && ri->grp == m && ri->seq == s && ri->pos >= c0) {
      int k = atomicAdd(&n_rows_s, 1);
      row_list[k] = r;
      atomicMax(&max_pos_s, ri->pos);
      atomicMax(&n_paged_s, ri->n_paged);
    }
  }
  __syncthreads();
  const int n_rows = n_rows_s;
  if (n_rows == 0) return;
  const int n_paged = n_paged_s;
  const int n_shared = max(0, min(kChunk, min(n_paged, max_pos_s + 1) - c0));

  // stage the committed part of the chunk (one page: page_size % 64 == 0).  Decode: committed
  // pages do not change during the round, so they are fetched before the dependency wait.
  if (!kv_static) pdl_wait();
  if (n_shared > 0) {
    const size_t base = page_off(D, s, layer, c0) + (size_t)g * HD;
    const int stride = D.nkv * HD;
    for (int ci = threadIdx.x; ci < n_shared * CPR; ci += blockDim.x) {
      const int pl = ci / CPR, cj = ci % CPR;
      const uint4 kk = *reinterpret_cast<const uint4*>(D.kpool + base + (size_t)pl * stride + cj * 8);
      const uint4 vv = *reinterpret_cast<const uint4*>(D.vpool + base + (size_t)pl * stride + cj * 8);
      const int dj = (cj ^ (pl & 7)) * 8;
      *reinterpret_cast<uint4*>(&sK[pl * HD + dj]) = kk;
      *reinterpret_cast<uint4*>(&sV[pl * HD + dj]) = vv;
    }
  }
  if (kv_static) pdl_wait();   // q and the slot K/V rows come from the predecessor
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = D.nh / D.nkv;
  const float scale = 1.0f / sqrtf((float)HD);
  for (int pair = warp; pair < n_rows * G; pair += 4) {
    const int r = row_list[pair / G];
    const int h = g * G + pair % G;
    const RowInfo* ri = &D.rows[r];
    const int p_row = ri->pos, n_anc = ri->n_anc;
    __syncwarp();
    for (int i = lane; i < HD; i += 32) sQ[warp][i] = D.qbuf[(size_t)r * D.nh * HD + h * HD + i];
    __syncwarp();

    float sc[2];
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
      const int pl = pass * 32 + lane, pos = c0 + pl;
      float acc = -INFINITY;
      if (pos <= p_row) {
        const __nv_bfloat16* kp;
        int swz = 0;
        if (pos < n_paged) {
          kp = &sK[pl * HD];
          swz = pl & 7;
        } else {
          const int ai = pos - n_paged;
          const int slot = (ai < n_anc) ? ri->anc[ai] : ri->slot;
          kp = D.kslot + slot_off(D, s, slot, layer) + (size_t)g * HD;
        }
        float a = 0.f;
#pragma unroll
        for (int j = 0; j < CPR; ++j) {
          const uint4 kk = *reinterpret_cast<const uint4*>(kp + ((j ^ swz) * 8));
          const __nv_bfloat162* k2 = reinterpret_cast<const __nv_bfloat162*>(&kk);
          const float4 q0 = *reinterpret_cast<const float4*>(&sQ[warp][j * 8]);
          const float4 q1 = *reinterpret_cast<const float4*>(&sQ[warp][j * 8 + 4]);
          float2 f;
          f = __bfloat1622float2(k2[0]); a = fmaf(q0.x, f.x, a); a = fmaf(q0.y, f.y, a);
          f = __bfloat1622float2(k2[1]); a = fmaf(q0.z, f.x, a); a = fmaf(q0.w, f.y, a);
          f = __bfloat1622float2(k2[2]); a = fmaf(q1.x, f.x, a); a = fmaf(q1.y, f.y, a);
          f = __bfloat1622float2(k2[3]); a = fmaf(q1.z, f.x, a); a = fmaf(q1.w, f.y, a);
        }
        acc = a * scale;
      }
      sc[pass] = acc;
    }
    const float mx = warp_max(fmaxf(sc[0], sc[1]));          // finite: position c0 <= p_row is visible
    const float e0 = (sc[0] == -INFINITY) ? 0.f : expf(sc[0] - mx);
    const float e1 = (sc[1] == -INFINITY) ? 0.f : expf(sc[1] - mx);
    const float lsum = warp_sum(e0 + e1);
    sP[warp][lane] = e0;
    sP[warp][32 + lane] = e1;
    __syncwarp();

    constexpr int DPL = HD / 32;                      // dims per lane
    float o[DPL];
#pragma unroll
    for (int t = 0; t < DPL; ++t) o[t] = 0.f;
    const int d0 = lane * DPL;
    const int n_vis = min(kChunk, p_row - c0 + 1);
    for (int pl = 0; pl < n_vis; ++pl) {
      const int pos = c0 + pl;
      const float pp = sP[warp][pl];
      const __nv_bfloat16* vp;
      if (pos < n_paged) {
        vp = &sV[pl * HD + (((d0 >> 3) ^ (pl & 7)) << 3) + (d0 & 7)];
      } else {
        const int ai = pos - n_paged;
        const int slot = (ai < n_anc) ? ri->anc[ai] : ri->slot;
        vp = D.vslot + slot_off(D, s, slot, layer) + (size_t)g * HD + d0;
      }
#pragma unroll
      for (int t = 0; t < DPL; t += 2) {
        const float2 f = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(vp + t));
        o[t] = fmaf(pp, f.x, o[t]);
        o[t + 1] = fmaf(pp, f.y, o[t + 1]);
      }
    }
    float* dst = D.attn_part + (((size_t)r * D.nh + h) * D.max_chunks + c) * (HD + 2);
#pragma unroll
    for (int t = 0; t < DPL; ++t) dst[d0 + t] = o[t];
    if (lane == 0) {
      dst[HD] = mx;
      dst[HD + 1] = lsum;
    }
  }
}

// Merge the per-chunk partials in ascending chunk order (fixed order: H3) -> bf16 operand planes.
template <int HD>
__global__ void __launch_bounds__(HD) k_attn_combine(Dev D, Plan plan, int step) {
  pdl_trigger();
  const int r = blockIdx.x, h = blockIdx.y, dd = threadIdx.x;
  const RowInfo* ri = &D.rows[r];
  if (!ri->valid || step >= plan.layer_len[ri->grp]) return;
  const int nc = ri->pos / kChunk + 1;
  pdl_wait();
  const float* src = D.attn_part + ((size_t)r * D.nh + h) * D.max_chunks * (HD + 2);
  float M = -INFINITY;
  for (int c = 0; c < nc; ++c) M = fmaxf(M, src[(size_t)c * (HD + 2) + HD]);
  float num = 0.f, den = 0.f;
  for (int c = 0; c < nc; ++c) {
    const float w = expf(src[(size_t)c * (HD + 2) + HD] - M);
    num = fmaf(w, src[(size_t)c * (HD + 2) + dd], num);
    den = fmaf(w, src[(size_t)c * (HD + 2) + HD + 1], den);
  }
  const int K = D.nh * HD;
  split_store(D.act_o, (size_t)D.R_cap * K, (size_t)r * K + h * HD + dd, num / den, D.planes);
}

// ------------------------------------------------------------------------------------------
// a5 insert + a6 validate_and_commit.  One warp per sequence.
__global__ void k_decide(Dev D, Plan plan, int auto_collapse) {
  const int s = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (s >= D.max_seqs) return;
  SeqState st = D.seqs[s];
  dex_step_result* res = &D.result_dev[s];
  CollapseCmd cmd;
  cmd.op = 0; cmd.k_sel = -1; cmd.token = -1; cmd.q_old = st.q;
  if (!seq_live(st)) {
    if (lane == 0) {
      res->active = 0; res->committed = 0; res->token = -1; res->match_k = -1;
      res->q_before = st.q; res->q_after = st.q; res->exit_rows = 0; res->critical_layers = 0;
      res->layer_evals = 0; res->n_tokens = st.n_tok; res->done = st.done; res->branch_mask = 0; res->reserved = 0;
      for (int i = 0; i < DEX_MAX_DEPTHS; ++i) res->rows_per_stage[i] = 0, res->anchor_tokens[i] = -1;
      res->ref_top1 = 0.f; res->ref_top2 = 0.f;
      D.cmd[s] = cmd;
    }
    return;
  }
  const int q = st.q, N = D.N;
  // insert: B[node] = u for every new node of level q
  int cnt[DEX_MAX_DEPTHS];                            // expanded rows per stage (sparse lattice: counted, not 2^{q-1-m})
#pragma unroll
  for (int m = 0; m < DEX_MAX_DEPTHS; ++m) cnt[m] = 0;
  for (int o = lane; o < (1 << q); o += 32) {
    const int m = stage_of(q, o);
    const int r = plan.row_base[m] + s * cap_of(N, m) + idx_in_stage(q, o, m);
    const unsigned long long key = D.best_key[r];      // 0 for a row that was not expanded -> B = -1 (empty)
    D.B[s * D.n_nodes + node_id(q, o)] = (int)(0xFFFFFFFFu - (uint32_t)(key & 0xFFFFFFFFull));
    const int live = D.rows[r].valid;
#pragma unroll
    for (int mm = 0; mm < DEX_MAX_DEPTHS; ++mm) cnt[mm] += (mm == m) ? live : 0;
  }
#pragma unroll
  for (int m = 0; m < DEX_MAX_DEPTHS; ++m)
    for (int off = 16; off > 0; off >>= 1) cnt[m] += __shfl_xor_sync(0xffffffffu, cnt[m], off);
  __syncwarp();
  // top-2 of the reference node's logits (reported; the oracle's margin decides flagging, R17)
  float t1 = -INFINITY, t2 = -INFINITY;
  if (q == N - 1) {
    for (int i = lane; i < D.ref_tiles; i += 32) {
      const float2 v = D.ref_tile[(size_t)s * D.ref_tiles + i];
      if (v.x > t1) { t2 = fmaxf(t1, v.y); t1 = v.x; } else { t2 = fmaxf(t2, v.x); }
    }
    for (int off = 16; off > 0; off >>= 1) {
      const float a1 = __shfl_xor_sync(0xffffffffu, t1, off), a2 = __shfl_xor_sync(0xffffffffu, t2, off);
      const float hi = fmaxf(t1, a1), lo = fminf(t1, a1);
      t2 = fmaxf(lo, fmaxf(t2, a2));
      t1 = hi;
    }
    // the exit head saw x*w_final: apply the deferred RMSNorm scale of the anchor row
    if (!D.sample) {                                    // sampling mode reports the perturbed values (already scaled)
      const float inv = inv_rms(D, plan.row_base[N - 1] + s * cap_of(N, N - 1));
      t1 *= inv;
      t2 *= inv;
    }
  }
  if (lane != 0) return;
  res->active = 1;
  res->q_before = q;
  long long evals = 0;
  int crit = 0, n_exit = 0;
#pragma unroll
  for (int m = 0; m < DEX_MAX_DEPTHS; ++m) {
    const int n = (m < N) ? cnt[m] : 0;
    n_exit += n;
    res->rows_per_stage[m] = n;
    if (n > 0) {
      const int len = D.depths[m] - (m ? D.depths[m - 1] : 0);
      evals += (long long)n * len;
      crit = max(crit, len);
    }
    res->anchor_tokens[m] = -1;
  }
  res->exit_rows = n_exit;
  res->layer_evals = evals;
  res->critical_layers = crit;
  res->branch_mask = 0; res->reserved = 0;
  res->committed = 0; res->token = -1; res->match_k = -1;
  res->ref_top1 = 0.f; res->ref_top2 = 0.f;
  res->n_tokens = st.n_tok; res->done = 0;
  if (q == N - 1) {                                   // ReachFinalDepth(q)
    int ref = D.B[s * D.n_nodes + node_id(N - 1, 0)];
    int k_sel = N - 1;                                // fallback b_{N-1}
    int explored = 0;                                 // branches whose continuation (position child of anchor k) exists
    for (int k = 0; k < N - 1; ++k)
      if (D.B[s * D.n_nodes + node_id(k + 1, 1)] >= 0) explored |= 1 << k;
    res->branch_mask = explored;
    for (int k = N - 2; k >= 0; --k)
      if (D.B[s * D.n_nodes + node_id(k, 0)] == ref && ((explored >> k) & 1)) k_sel = k;   // shallowest explored match (R6, R26)
    for (int k = 0; k < N; ++k) res->anchor_tokens[k] = D.B[s * D.n_nodes + node_id(k, 0)];
    res->token = ref; res->match_k = k_sel;
    res->ref_top1 = t1; res->ref_top2 = t2;
    cmd.k_sel = k_sel; cmd.token = ref;
    if (auto_collapse) {
      cmd.op = 2;
      res->committed = 1;
    } else {
      cmd.op = 3;
      D.seqs[s].pending = 1;
      res->q_after = q;
    }
  } else {
    cmd.op = 1;
  }
  D.cmd[s] = cmd;
}

__global__ void k_set_cmd(Dev D, int seq, int k_sel, int token) {
  CollapseCmd cmd;
  cmd.op = 2; cmd.k_sel = k_sel; cmd.token = token; cmd.q_old = D.seqs[seq].q;
  for (int s = 0; s < D.max_seqs; ++s) {
    if (s == seq) D.cmd[s] = cmd;
    else D.cmd[s].op = 0;
  }
}

// a7 (K/V part): append the root slot's K/V of every layer to the committed pages at position
// ctx_len, then compact the surviving slots in place.  grid (L, max_seqs), each thread owns the
// same 16-byte pieces of every slot, walks the new slots in ascending order (source index >
// destination index always, PAPER.md:206-208 sub-tree re-rooting) -> no cross-thread hazard.
__global__ void __launch_bounds__(256) k_collapse_kv(Dev D) {
  const int l = blockIdx.x, s = blockIdx.y;
  const CollapseCmd cmd = D.cmd[s];
  if (cmd.op != 2) return;
  const SeqState st = D.seqs[s];
  const int N = D.N;
  const int pieces = D.nkv * D.hd / 8;                // uint4 pieces per K (or V) row
  const size_t dst_off = page_off(D, s, l, st.ctx_len);
  const int q_new = (cmd.k_sel < N - 1) ? (N - 1 - cmd.k_sel) : 0;
  const int r_old = 2 << cmd.k_sel;                   // old root of the surviving sub-tree, 2^{k+1}
  const int n_new = (1 << q_new) - 1;                 // surviving nodes

  for (int pc = threadIdx.x; pc < pieces; pc += blockDim.x) {
    const size_t e = (size_t)pc * 8;
    // root slot (compact id 0) joins the committed context C
    *reinterpret_cast<uint4*>(D.kpool + dst_off + e) = *reinterpret_cast<const uint4*>(D.kslot + slot_off(D, s, 0, l) + e);
    *reinterpret_cast<uint4*>(D.vpool + dst_off + e) = *reinterpret_cast<const uint4*>(D.vslot + slot_off(D, s, 0, l) + e);
    // surviving slot roots: new node j (0 or even), ascending
    int j = 0;
    while (j < n_new) {
      uint4 kb[8], vb[8];
      int jd[8];
      int nbat = 0;
      while (j < n_new && nbat < 8) {
        const int lam = node_level(j);
        // the slot rooted at level lam has run stages 0 .. q_new-1-lam -> layers < depths[q_new-1-lam]
        if (l < D.depths[q_new - 1 - lam]) {
          const int o = j + 1 - (1 << lam);
          const int old = ((r_old + 1) << lam) + o - 1;
          kb[nbat] = *reinterpret_cast<const uint4*>(D.kslot + slot_off(D, s, compact_slot(old), l) + e);
          vb[nbat] = *reinterpret_cast<const uint4*>(D.vslot + slot_off(D, s, compact_slot(old), l) + e);
          jd[nbat] = compact_slot(j);
          ++nbat;
        }
        j = (j == 0) ? 2 : j + 2;
      }
      for (int b = 0; b < nbat; ++b) {
        *reinterpret_cast<uint4*>(D.kslot + slot_off(D, s, jd[b], l) + e) = kb[b];
        *reinterpret_cast<uint4*>(D.vslot + slot_off(D, s, jd[b], l) + e) = vb[b];
      }
    }
  }
}

// a7 (hidden part) / a8: frontier hidden rows for the next round.  advance: identity copy of this
// round's rows; collapse: gather the surviving frontier (old level N-1, path prefix D^k P).
__global__ void __launch_bounds__(256) k_collapse_hidden(Dev D, Plan plan) {
  const int r = blockIdx.x;
  if (r >= D.R_dec) return;
  int m = 0;
  while (m + 1 < D.N && r >= plan.row_base[m + 1]) ++m;
  const int cap = cap_of(D.N, m);
  const int local = r - plan.row_base[m];
  const int s = local / cap, j = local % cap;
  if (s >= D.max_seqs) return;
  const CollapseCmd cmd = D.cmd[s];
  int src = -1;
  if (cmd.op == 1) {
    if (D.rows[r].valid) src = r;
  } else if (cmd.op == 2 && cmd.k_sel < D.N - 1) {
    const int lam = D.N - 2 - cmd.k_sel;              // new frontier level q'-1
    if (m <= lam) {
      const int o = (m == lam) ? 0 : ((j << (m + 1)) | (1 << m));
      if ((m == lam && j == 0) || (m < lam && o < (1 << lam))) {
        const int o_old = (1 << lam) | o;
        src = plan.row_base[m] + s * cap + idx_in_stage(D.N - 1, o_old, m);
      }
    }
  }
  if (src < 0) return;
  const float4* a = reinterpret_cast<const float4*>(D.x_cur + (size_t)src * D.d);
  float4* b = reinterpret_cast<float4*>(D.x_front + (size_t)r * D.d);
  for (int i = threadIdx.x; i < D.d / 4; i += blockDim.x) b[i] = a[i];
}

// a7 (integer part) + a8 advance: FSM update, token append, B compaction.  One warp per sequence.
__global__ void k_apply(Dev D, int eos_id) {
  __shared__ int tmp[8][256];
  const int s = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (s >= D.max_seqs) return;
  const CollapseCmd cmd = D.cmd[s];
  if (cmd.op == 0 || cmd.op == 3) return;
  SeqState st = D.seqs[s];
  dex_step_result* res = &D.result_dev[s];
  int* B = D.B + s * D.n_nodes;
  if (cmd.op == 1) {
    if (lane == 0) {
      st.q += 1;                                      // advance (Alg. 1 line 15)
      D.seqs[s] = st;
      res->q_after = st.q;
    }
    return;
  }
  const int N = D.N;
  const int q_new = (cmd.k_sel < N - 1) ? (N - 1 - cmd.k_sel) : 0;
  const int n_new = (1 << q_new) - 1;
  const int r_old = 2 << cmd.k_sel;
  for (int j = lane; j < n_new; j += 32) {
    const int lam = node_level(j);
    tmp[s & 7][j] = B[((r_old + 1) << lam) + (j + 1 - (1 << lam)) - 1];
  }
  __syncwarp();
  for (int j = lane; j < D.n_nodes; j += 32) B[j] = (j < n_new) ? tmp[s & 7][j] : -1;
  if (lane == 0) {
    D.tokens[s * (D.max_ctx + 1) + st.n_tok] = cmd.token;       // Y <- Y || y
    st.n_tok += 1;
    st.ctx_len += 1;
    st.last_tok = cmd.token;
    st.q = q_new;
    st.pending = 0;
    if (st.n_tok >= D.max_ctx || cmd.token == eos_id) st.done = 1;
    D.seqs[s] = st;
    res->q_after = q_new;
    res->n_tokens = st.n_tok;
    res->done = st.done;
    res->committed = 1;
    res->token = cmd.token;
    res->match_k = cmd.k_sel;
  }
}

// ------------------------------------------------------------------------------------------
// debug taps (test-only paths; plain CUDA-core code)
__global__ void k_tap_logits(Dev D, int row, float* out) {
  const int v = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (v >= D.vocab) return;
  const __nv_bfloat16* w = D.lm_head + (size_t)v * D.d;
  const __nv_bfloat16* e = D.act_e + (size_t)D.rows[row].exit_row * D.d;
  const size_t ps = (size_t)D.R_cap * D.d;
  float acc = 0.f;
  for (int i = lane; i < D.d; i += 32) {
    float x = __bfloat162float(e[i]);
    if (D.planes > 1) x += __bfloat162float(e[ps + i]);
    acc = fmaf(x, __bfloat162float(w[i]), acc);
  }
  acc = warp_sum(acc);
  if (lane == 0) out[v] = acc * inv_rms(D, row);
}

// The fused exit's own per-block maxima of the final-depth anchor row (what the tcgen05 epilogue reduced: top-1 / top-2
// of every 32 consecutive vocabulary ids), with the deferred RMSNorm scale of the row applied.
__global__ void k_tap_ref_tiles(Dev D, int row, int seq, float2* out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= D.ref_tiles) return;
  const float inv = D.sample ? 1.f : inv_rms(D, row);
  const float2 v = D.ref_tile[(size_t)seq * D.ref_tiles + i];
  out[i] = make_float2(v.x * inv, v.y * inv);
}

__global__ void k_debug_rows(Dev D, int R) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0)
    for (int m = 0; m < kMaxGrp; ++m) D.grp_nb[m] = (m == 0) ? round16(R) : 0, D.exit_nb[m] = 0;
  if (r >= D.R_cap) return;
  RowInfo ri;
  ri.valid = r < R;
  ri.seq = 0; ri.node = -1; ri.pos = 0; ri.grp = 0; ri.slot = -1; ri.n_paged = 0; ri.n_anc = 0;
  ri.parent_row = -1; ri.tok_in = 0; ri.is_ref = 0; ri.n_mask = 0;
  for (int i = 0; i < kMaxAnc; ++i) ri.anc[i] = 0, ri.mask_tok[i] = -1;
  ri.exit_row = r;
  D.exit_map[r] = -1;
  D.rows[r] = ri;
}
__global__ void k_debug_split(const float* x, __nv_bfloat16* dst, int rows, int k, size_t plane_stride, int planes) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)rows * k) return;
  split_store(dst, plane_stride, i, x[i], planes);
}
__global__ void k_debug_sum(const float* part, float* y, int rows, int out, int part_ld, int ksplit, size_t split_stride) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)rows * out) return;
  const int r = (int)(i / out), c = (int)(i % out);
  float acc = 0.f;
  for (int s = 0; s < ksplit; ++s) acc += part[(size_t)s * split_stride + (size_t)r * part_ld + c];
  y[i] = acc;
}

// ------------------------------------------------------------------------------------------
// launch wrappers (called from api.cu)
#define DEX_LAUNCH_CHECK() return cudaGetLastError()

template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = 0;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

cudaError_t launch_rows_decode(const Dev& D, const Plan& p, cudaStream_t st) {
  if (D.R_cap > 1024) return cudaErrorInvalidValue;
  k_rows_decode<<<1, 1024, 0, st>>>(D, p);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_rows_prefill(const Dev& D, int seq, int p0, int R, cudaStream_t st) {
  k_rows_prefill<<<(D.R_cap + 127) / 128, 128, 0, st>>>(D, seq, p0, R);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_seq_init(const Dev& D, int seq, int n, cudaStream_t st) {
  k_seq_init<<<1, 256, 0, st>>>(D, seq, n);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_rope_table(const Dev& D, double theta, int n_pos, cudaStream_t st) {
  const int n = n_pos * (D.hd / 2);
  k_rope_table<<<(n + 255) / 256, 256, 0, st>>>(D, theta, n_pos);
  DEX_LAUNCH_CHECK();
}
static int norm_threads(int d) {
  int threads = ((d / 4 + 1) / 2 + 31) / 32 * 32;      // two float4 per thread cover d
  return threads < 64 ? 64 : (threads > 1024 ? 1024 : threads);
}
cudaError_t launch_gather_norm(const Dev& D, const Plan& p, int rows, cudaStream_t st) {
  k_gather_norm<<<rows, norm_threads(D.d), 0, st>>>(D, p);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_add_norm(const Dev& D, const Plan& p, int rows, int step, int mode, const OpDesc& o, cudaStream_t st) {
  return launch_pdl(k_add_norm, dim3(rows), dim3(norm_threads(D.d)), st, D, p, step, mode, o.ksplit, o.split_stride, o.part_ld);
}
cudaError_t launch_rope_kv(const Dev& D, const Plan& p, int rows, int step, const OpDesc& o, cudaStream_t st) {
  const int items = (D.nh + D.nkv) * (D.hd / 8) + D.nkv * D.hd / 4;
  return launch_pdl(k_rope_kv, dim3(rows, (items + 255) / 256), dim3(256), st, D, p, step, o.ksplit, o.split_stride, o.part_ld);
}
cudaError_t launch_silu_mul(const Dev& D, const Plan& p, int rows, int step, const OpDesc& o, cudaStream_t st) {
  return launch_pdl(k_silu_mul, dim3(rows, (D.ffn / 4 + 255) / 256), dim3(256), st, D, p, step, o.ksplit, o.split_stride, o.part_ld);
}
cudaError_t launch_attn(const Dev& D, const Plan& p, int rows, int step, int n_chunks, int kv_static, cudaStream_t st) {
  const int row_split = kv_static ? 1 : 8;      // prefill: up to 128 rows per (chunk, head) -> 16 per CTA
  dim3 g(n_chunks, D.nkv, p.n_grp * D.max_seqs * row_split);
  dim3 gc(rows, D.nh);
  cudaError_t e;
  if (D.hd == 128) {
    e = launch_pdl(k_attn<128>, g, dim3(128), st, D, p, step, kv_static, row_split);
    if (e != cudaSuccess) return e;
    return launch_pdl(k_attn_combine<128>, gc, dim3(128), st, D, p, step);
  }
  e = launch_pdl(k_attn<64>, g, dim3(128), st, D, p, step, kv_static, row_split);
  if (e != cudaSuccess) return e;
  return launch_pdl(k_attn_combine<64>, gc, dim3(64), st, D, p, step);
}
cudaError_t launch_decide(const Dev& D, const Plan& p, int auto_collapse, cudaStream_t st) {
  k_decide<<<1, 32 * D.max_seqs, 0, st>>>(D, p, auto_collapse);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_set_cmd(const Dev& D, int seq, int k, int tok, cudaStream_t st) {
  k_set_cmd<<<1, 1, 0, st>>>(D, seq, k, tok);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_collapse(const Dev& D, const Plan& p, int eos_id, cudaStream_t st) {
  dim3 g(D.L, D.max_seqs);
  k_collapse_kv<<<g, 256, 0, st>>>(D);
  k_collapse_hidden<<<D.R_dec, 256, 0, st>>>(D, p);
  k_apply<<<1, 32 * D.max_seqs, 0, st>>>(D, eos_id);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_tap_logits(const Dev& D, int row, float* out, cudaStream_t st) {
  k_tap_logits<<<(D.vocab + 7) / 8, 256, 0, st>>>(D, row, out);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_tap_ref_tiles(const Dev& D, int row, int seq, float2* out, cudaStream_t st) {
  k_tap_ref_tiles<<<(D.ref_tiles + 255) / 256, 256, 0, st>>>(D, row, seq, out);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_debug_rows(const Dev& D, int R, cudaStream_t st) {
  k_debug_rows<<<(D.R_cap + 127) / 128, 128, 0, st>>>(D, R);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_debug_split(const float* x, __nv_bfloat16* dst, int rows, int k, size_t ps, int planes, cudaStream_t st) {
  const size_t n = (size_t)rows * k;
  k_debug_split<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, dst, rows, k, ps, planes);
  DEX_LAUNCH_CHECK();
}
cudaError_t launch_debug_sum(const float* part, float* y, int rows, int out, int part_ld, int ksplit, size_t ss, cudaStream_t st) {
  const size_t n = (size_t)rows * out;
  k_debug_sum<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(part, y, rows, out, part_ld, ksplit, ss);
  DEX_LAUNCH_CHECK();
}

}  // namespace dexk
