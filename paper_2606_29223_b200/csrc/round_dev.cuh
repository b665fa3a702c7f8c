// round_dev.cuh — device pieces shared by the two persistent round kernels (k_round in round.cu: phases separated
// by grid barriers; k_flow in flow.cu: dataflow, flags instead of barriers): small helpers, the item walker of
// k_round, the glue units (split-K sum + RMSNorm operand / RoPE + slot K/V / SwiGLU / inducing adapters) and the
// lattice-masked decode attention (a3).
#pragma once
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_dev.cuh"

namespace dexk {

// warps: 0 weight TMA, 1 MMA, 2-5 GEMM epilogue + glue, 6 activation TMA, 7-10 glue only.  A lone warp per
// scheduler runs the glue phases latency-bound; two per scheduler measured best (12 glue warps push the kernel
// under 128 registers and spill).
constexpr int kRoundThreads = 352;

// ---------------------------------------------------------------- small device helpers
template <int GT>
__device__ __forceinline__ void bar_epi() { asm volatile("bar.sync 1, %0;\n" ::"n"(GT) : "memory"); }
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add(unsigned* p, unsigned v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}
// generic-proxy global writes <-> async-proxy (TMA) global reads; the .global form does not wait on the
// CTA's in-flight TMA traffic into shared memory
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.global;\n" ::: "memory"); }

__device__ __forceinline__ float4 r_ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 r_add4(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ float4 r_sum4(const float* p, int S, size_t stride) {
  float4 acc = r_ld4(p);
#pragma unroll 8
  for (int s = 1; s < S; ++s) acc = r_add4(acc, r_ld4(p + (size_t)s * stride));
  return acc;
}
// NV float4 split-K sums at once: the loads of up to 8 splits of all NV values are issued together (one
// round trip), then added in split order (H3).
template <int NV, int NB = 8>
__device__ __forceinline__ void r_sum4_batch(const float* const (&p)[NV], int S, size_t stride, float4 (&out)[NV]) {
#pragma unroll
  for (int v = 0; v < NV; ++v) out[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s0 = 0; s0 < S; s0 += NB) {
    float4 t[NB][NV];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int v = 0; v < NV; ++v)
        t[i][v] = (s0 + i < S) ? r_ld4(p[v] + (size_t)(s0 + i) * stride) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < NB; ++i)
      if (s0 + i < S) {
#pragma unroll
        for (int v = 0; v < NV; ++v) out[v] = r_add4(out[v], t[i][v]);
      }
  }
}
__device__ __forceinline__ float r_sum1(const float* p, int S, size_t stride) {
  float acc = p[0];
#pragma unroll 8
  for (int s = 1; s < S; ++s) acc += p[(size_t)s * stride];
  return acc;
}
__device__ __forceinline__ void r_split_store4(__nv_bfloat16* base, size_t plane_stride, size_t idx, float4 v, int planes) {
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
__device__ __forceinline__ bool r_seq_live(const SeqState& s) { return s.active && !s.done && !s.pending; }
__device__ __forceinline__ int r_stage_count(int q, int m) { return m > q ? 0 : (m == q ? 1 : (1 << (q - 1 - m))); }

// ---------------------------------------------------------------- the round's op / item sequence
// op t < 4*n_steps: step j = t/4, kind t%4 (qkv, o, gate/up, down); then, with inducing adapters,
// the two adapter projections W1 (kind 5) and W2 (kind 6) of every live non-final stage; last op: the exit head (kind 4).
struct OpI {
  int which, j, ext;
  unsigned mask;           // live groups of the op's plan
  int n_tiles, ksplit, kbps, kb_total, per_grp, n_items;
};
struct ItemI {
  int g, nb, tile, split, layer, kb0, kb1, row0, row_end;
};

struct Seq {               // shared by all roles: same deterministic walk
  const RoundArgs* a;
  const int* s_nb;         // [16] shared: decode group extents 0..7, exit chunk extents 8..15
  int n_steps, n_ops, n_ad_ops, G, cta;

  __device__ __forceinline__ int which_of(int t) const {
    return t < 4 * n_steps ? (t & 3) : (t < 4 * n_steps + n_ad_ops ? 5 + t - 4 * n_steps : 4);
  }
  __device__ __forceinline__ void op_info(int t, OpI& o) const {
    unsigned mask = 0;
    if (t < 4 * n_steps) {
      o.j = t >> 2; o.which = t & 3; o.ext = 0;
      for (int g = 0; g < a->dec.n_grp; ++g)
        if (s_nb[g] > 0 && o.j < a->dec.layer_len[g]) mask |= 1u << g;
    } else if (t < 4 * n_steps + n_ad_ops) {
      o.j = 0; o.which = 5 + t - 4 * n_steps; o.ext = 0;
      for (int g = 0; g + 1 < a->dec.n_grp; ++g)             // adapter g serves the rows leaving depth d_g, g < N-1
        if (s_nb[g] > 0) mask |= 1u << g;
    } else {
      o.j = 0; o.which = 4; o.ext = 1;
      for (int g = 0; g < a->ext.n_grp; ++g)
        if (s_nb[8 + g] > 0) mask |= 1u << g;
    }
    o.mask = mask;
    const OpDesc& d = a->op[o.which];
    o.n_tiles = d.n_tiles; o.ksplit = d.ksplit; o.kbps = d.kbps; o.kb_total = d.kb_total;
    o.per_grp = d.n_tiles * d.ksplit;
    o.n_items = __popc(mask) * o.per_grp;
  }
  __device__ __forceinline__ void decode(const OpI& o, int i, ItemI& it) const {
    const int gi = i / o.per_grp, rem = i - gi * o.per_grp;
    it.g = __fns(o.mask, 0, gi + 1);
    const Plan& p = o.ext ? a->ext : a->dec;
    it.nb = s_nb[(o.ext ? 8 : 0) + it.g];
    it.tile = rem / o.ksplit;
    it.split = rem - it.tile * o.ksplit;
    it.layer = o.ext ? 0 : (o.which >= 5 ? it.g : p.layer_lo[it.g] + o.j);
    it.kb0 = it.split * o.kbps;
    it.kb1 = min(it.kb0 + o.kbps, o.kb_total);
    it.row0 = p.row_base[it.g];
    it.row_end = it.row0 + p.rows_cap[it.g];
  }
  // grid barriers that must have completed before op t's operand may be read (9 per step: one after
  // every GEMM's epilogue, one after every glue phase; the QKV output takes two glue phases; an adapter op two)
  __device__ __forceinline__ unsigned dep(int t) const {
    if (t >= 4 * n_steps) return 9u * n_steps + 2u * min(t - 4 * n_steps, n_ad_ops);
    const int k = t & 3;
    return 9u * (t >> 2) + (k == 0 ? 0u : 2u * k + 1u);
  }
};

struct Walker {            // this CTA's items, in order
  int t, i, rr;
  bool valid;
  OpI o;
  ItemI it;
  __device__ __forceinline__ void start(const Seq& q) {
    t = 0; rr = 0;
    q.op_info(0, o);
    i = q.cta;
    settle(q);
  }
  __device__ __forceinline__ void settle(const Seq& q) {
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
  __device__ __forceinline__ void next(const Seq& q) {
    i += q.G;
    settle(q);
  }
};

// ---------------------------------------------------------------- grid barrier (epilogue groups)
// Every glue thread orders its generic-proxy global writes against later async-proxy (TMA) reads; the CTA barrier
// orders them before ONE thread's gpu-scope release (red.release: cumulative over what the barrier made visible to
// it), which arrives on the counter; the same thread spins with gpu-scope acquire loads and the second CTA barrier
// hands the acquired view to the group.  No separate fences: release / acquire + bar.sync compose in the PTX model.
template <int GT>
__device__ __forceinline__ void grid_bar(unsigned* gbar, unsigned target, int tid_e, volatile unsigned* s_seen, unsigned gb) {
  fence_proxy_async();
  bar_epi<GT>();
  if (tid_e == 0) {
    red_release_add(gbar, 1u);
    unsigned spins = 0;
    while (ld_acquire_u32(gbar) < target) {
      if (++spins > 400000000u) __trap();   // protocol bug: trap instead of hanging the box
    }
    __threadfence_block();
    *s_seen = gb;                // the activation producer of this CTA learns of the barrier without polling L2
  }
  bar_epi<GT>();
}

// ---------------------------------------------------------------- per-row record cached in shared memory
// The glue units need a row's (valid, stage, sequence, slot, position, exit row) before they can address anything that
// depends on the layer or the position (norm weights, RoPE table, slot K/V): read from the row table in global memory
// that is one more dependent L2 round trip per phase under the weight stream.  k_round copies the fields into shared
// memory once per round (8 bytes per row); callers without the cache (k_flow) pass nullptr.
struct RowLite {
  int pos;
  unsigned bits;           // valid | grp << 1 | seq << 4 | slot << 8 | exit_row << 16
};
constexpr int kRowCache = 544;   // rows cached (R_cap of every supported lattice: 4 x 128 + 16 slack + 16)
struct RowView {
  int valid, grp, seq, slot, pos, exit_row;
};
__device__ __forceinline__ RowLite row_lite_of(const RowInfo& ri) {
  RowLite l;
  l.pos = ri.pos;
  l.bits = (ri.valid ? 1u : 0u) | ((unsigned)ri.grp & 7u) << 1 | ((unsigned)ri.seq & 15u) << 4 | ((unsigned)ri.slot & 255u) << 8 |
           ((unsigned)ri.exit_row & 65535u) << 16;
  return l;
}
__device__ __forceinline__ RowView row_view(const Dev& D, const RowLite* cache, int r) {
  RowView v;
  if (cache != nullptr) {
    const RowLite l = cache[r];
    v.valid = l.bits & 1u; v.grp = (l.bits >> 1) & 7u; v.seq = (l.bits >> 4) & 15u; v.slot = (l.bits >> 8) & 255u;
    v.exit_row = l.bits >> 16; v.pos = l.pos;
  } else {
    const RowInfo* ri = &D.rows[r];
    v.valid = ri->valid; v.grp = ri->grp; v.seq = ri->seq; v.slot = ri->slot; v.pos = ri->pos; v.exit_row = ri->exit_row;
  }
  return v;
}

// ---------------------------------------------------------------- glue phases (epilogue group)
__device__ __forceinline__ float r_warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// Every glue phase is laid out for memory-level parallelism: a thread issues all of its loads in one or two
// batches (a dependent load under the weight stream costs microseconds), and the work is spread over all CTAs.

// x += sum_s part[s]; operand planes <- x * w (RMSNorm scale deferred: Dev::ss_part).  Warp unit = (row,
// 128-element segment).  mode 0: after o_proj (w = norm_ffn[l] -> act_a); mode 1: after down_proj (next layer's
// attention norm -> act_a, or the shared final norm -> act_e).
__device__ __forceinline__ void unit_add_norm(const RoundArgs& a, int j, int mode, const OpDesc& op, const float* part, int r, int seg,
                                              int lane, const RowLite* rc = nullptr) {
  const Dev& D = a.D;
  // the row table, x and the partials are loaded together (addresses depend on r only); w needs the layer (with the
  // shared-memory row cache it is known at once and w joins the same batch of loads)
  const RowView rv = row_view(D, rc, r);
  const int valid = rv.valid, grp = rv.grp, exit_row = rv.exit_row;
  const int i = seg * 128 + lane * 4;
  const bool in = i < D.d;
  float* x = D.x_cur + (size_t)r * D.d + (in ? i : 0);
  const float4 xv = r_ld4(x);
  const float* const pp[1] = {part + (size_t)r * op.part_ld + (in ? i : 0)};
  float4 sv[1];
  r_sum4_batch<1, 12>(pp, op.ksplit, op.split_stride, sv);
  if (!valid) return;
  if (j >= a.dec.layer_len[grp]) return;
  const int layer = a.dec.layer_lo[grp] + j;
  float ss = 0.f;
  if (in) {
    const float* w;
    __nv_bfloat16* dst = D.act_a;
    if (mode == 0) {
      w = D.norm_ffn + (size_t)layer * D.d;
    } else if (j + 1 < a.dec.layer_len[grp]) {
      w = D.norm_attn + (size_t)(layer + 1) * D.d;
    } else if (D.ad_m > 0 && grp + 1 < D.N) {
      w = D.ad_norm + (size_t)grp * D.d;       // adapter input RMSNorm(h; norm_k): same row, same deferred scale
    } else {
      w = D.norm_final;
      dst = D.act_e;
    }
    const float4 wv = r_ld4(w + i);
    const float4 s4 = sv[0];
    const float4 v = r_add4(xv, s4);
    *reinterpret_cast<float4*>(x) = v;
    ss = sumsq4(v);
    if (mode == 1 && D.taps) *reinterpret_cast<float4*>(D.tap_hidden + ((size_t)r * D.max_len + j) * D.d + i) = v;
    // the exit operand is indexed by the row's DENSE exit row (Dev::exit_map)
    r_split_store4(dst, (size_t)D.R_cap * D.d, (size_t)(dst == D.act_e ? exit_row : r) * D.d + i, make_float4(v.x * wv.x, v.y * wv.y, v.z * wv.z, v.w * wv.w),
                   D.planes);
  }
  ss = r_warp_sum(ss);
  if (lane == 0) D.ss_part[(size_t)r * kSsSeg + seg] = ss;
}
static __device__ void glue_add_norm(const RoundArgs& a, int j, int mode, const OpDesc& op, int gw, int n_gw, int lane, const RowLite* rc) {
  const Dev& D = a.D;
  const int n_seg = (D.d + 127) / 128;
  for (int u = gw; u < D.R_dec * n_seg; u += n_gw) {
    const int r = u / n_seg, seg = u - r * n_seg;
    unit_add_norm(a, j, mode, op, D.part, r, seg, lane, rc);
  }
}

// act_f = SiLU(gate) * up from the split-K partials of the fused gate/up projection (scaled by the deferred
// RMSNorm factor of the row).  Warp unit = (row, 128 elements).
__device__ __forceinline__ void unit_silu(const RoundArgs& a, int j, const OpDesc& op, const float* part, int r, int b, int lane) {
  const Dev& D = a.D;
  const size_t ps = (size_t)D.R_cap * D.ffn;
  const int i = b * 128 + lane * 4;
  if (i >= D.ffn) return;
  // the row table, the deferred norm scale and the partials are loaded together (addresses depend on r only)
  const RowInfo* ri = &D.rows[r];
  const int valid = ri->valid, grp = ri->grp;
  const float* p = part + (size_t)r * op.part_ld;
  const float* const pp[2] = {p + i, p + D.ffn + i};
  float4 gu[2];
  r_sum4_batch<2>(pp, op.ksplit, op.split_stride, gu);
  const float inv = inv_rms(D, r);
  if (!valid || j >= a.dec.layer_len[grp]) return;
  float4 g = gu[0], up = gu[1];
  g.x *= inv; g.y *= inv; g.z *= inv; g.w *= inv;
  up.x *= inv; up.y *= inv; up.z *= inv; up.w *= inv;
  float4 o;
  o.x = g.x / (1.0f + expf(-g.x)) * up.x;
  o.y = g.y / (1.0f + expf(-g.y)) * up.y;
  o.z = g.z / (1.0f + expf(-g.z)) * up.z;
  o.w = g.w / (1.0f + expf(-g.w)) * up.w;
  r_split_store4(D.act_f, ps, (size_t)r * D.ffn + i, o, D.planes);
}
static __device__ void glue_silu(const RoundArgs& a, int j, const OpDesc& op, int gw, int n_gw, int lane) {
  const Dev& D = a.D;
  const int nblk = (D.ffn + 127) / 128;
  for (int u = gw; u < D.R_dec * nblk; u += n_gw) {
    const int r = u / nblk, b = u - r * nblk;
    unit_silu(a, j, op, D.part, r, b, lane);
  }
}

// Inducing adapter of the non-final exits (reading R25), first half:
// act_f[:, 0..m) <- SiLU(inv_rms * (W1_k . (h * norm_k)) + b1_k).  Warp unit = (row, 128 elements of m).
static __device__ void glue_ad1(const RoundArgs& a, const OpDesc& op, int gw, int n_gw, int lane) {
  const Dev& D = a.D;
  const int m = D.ad_m, nblk = (m + 127) / 128;
  const size_t ps = (size_t)D.R_cap * D.ffn;
  for (int u = gw; u < D.R_dec * nblk; u += n_gw) {
    const int r = u / nblk, b = u - r * nblk;
    const int i = b * 128 + lane * 4;
    if (i >= m) continue;
    const RowInfo* ri = &D.rows[r];
    const int valid = ri->valid, grp = ri->grp;
    const float* const pp[1] = {D.part + (size_t)r * op.part_ld + i};
    float4 sv[1];
    r_sum4_batch<1, 8>(pp, op.ksplit, op.split_stride, sv);
    const float inv = inv_rms(D, r);
    if (!valid || grp + 1 >= D.N) continue;
    const float4 bv = r_ld4(D.ad_b1 + (size_t)grp * m + i);
    float4 t = make_float4(sv[0].x * inv + bv.x, sv[0].y * inv + bv.y, sv[0].z * inv + bv.z, sv[0].w * inv + bv.w);
    float4 o;
    o.x = t.x / (1.0f + expf(-t.x));
    o.y = t.y / (1.0f + expf(-t.y));
    o.z = t.z / (1.0f + expf(-t.z));
    o.w = t.w / (1.0f + expf(-t.w));
    r_split_store4(D.act_f, ps, (size_t)r * D.ffn + i, o, D.planes);
  }
}

// Second half: h~ = h + alpha_k (W2_k . act + b2_k); exit operand act_e <- h~ * norm_final with the deferred scale of
// h~ (ss_part rewritten).  x_cur keeps h: deeper stages continue from the un-induced hidden.
static __device__ void glue_ad2(const RoundArgs& a, const OpDesc& op, int gw, int n_gw, int lane) {
  const Dev& D = a.D;
  const int n_seg = (D.d + 127) / 128;
  for (int u = gw; u < D.R_dec * n_seg; u += n_gw) {
    const int r = u / n_seg, seg = u - r * n_seg;
    const RowInfo* ri = &D.rows[r];
    const int valid = ri->valid, grp = ri->grp;
    const int i = seg * 128 + lane * 4;
    const bool in = i < D.d;
    const float4 xv = r_ld4(D.x_cur + (size_t)r * D.d + (in ? i : 0));
    const float* const pp[1] = {D.part + (size_t)r * op.part_ld + (in ? i : 0)};
    float4 sv[1];
    r_sum4_batch<1, 16>(pp, op.ksplit, op.split_stride, sv);
    if (!valid || grp + 1 >= D.N) continue;
    float ss = 0.f;
    if (in) {
      const float al = D.ad_alpha[grp];
      const float4 bv = r_ld4(D.ad_b2 + (size_t)grp * D.d + i);
      const float4 wv = r_ld4(D.norm_final + i);
      const float4 v = make_float4(xv.x + al * (sv[0].x + bv.x), xv.y + al * (sv[0].y + bv.y), xv.z + al * (sv[0].z + bv.z),
                                   xv.w + al * (sv[0].w + bv.w));
      ss = sumsq4(v);
      r_split_store4(D.act_e, (size_t)D.R_cap * D.d, (size_t)ri->exit_row * D.d + i, make_float4(v.x * wv.x, v.y * wv.y, v.z * wv.z, v.w * wv.w),
                     D.planes);
    }
    ss = r_warp_sum(ss);
    if (lane == 0) D.ss_part[(size_t)r * kSsSeg + seg] = ss;
  }
}

__device__ __forceinline__ void cvt_bf16x16(const uint4& u0, const uint4& u1, float (&f)[16]) {
  const __nv_bfloat162* a = reinterpret_cast<const __nv_bfloat162*>(&u0);
  const __nv_bfloat162* b = reinterpret_cast<const __nv_bfloat162*>(&u1);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 x = __bfloat1622float2(a[i]), y = __bfloat1622float2(b[i]);
    f[2 * i] = x.x; f[2 * i + 1] = x.y;
    f[8 + 2 * i] = y.x; f[8 + 2 * i + 1] = y.y;
  }
}
__device__ __forceinline__ float bf16_rt(float v) { return __bfloat162float(__float2bfloat16_rn(v)); }

// Merge the sub-partials of (row, head) - one per 16 positions - in ascending position order (fixed order: H3)
// -> act_o planes.  The definition is the one-pass merge with a running maximum M:
//     for i ascending, sub-partial (o_i, m_i, l_i) present:  if m_i > M { s = exp(M - m_i); den *= s; num *= s; M = m_i }
//                                                            w = exp(m_i - M); num = fma(w, o_i, num); den = fma(w, l_i, den)
// computed here without its dependent chain of exponentials: the scalars (s_i, w_i) depend on the m_i alone, so the
// lanes of the warp take one sub-partial each, find the running maximum BEFORE theirs with an exclusive prefix max
// (exact in any order) and evaluate the same two expf on the same arguments; the data loop that follows is then
// multiplies and fmas only (s_i = 1 where the definition skips the rescale: x * 1 is exact).  Groups of 24
// sub-partials: their (m, l) and their o (two 8-byte loads per lane, coalesced: lane owns dims 2*lane, 2*lane + 1
// of every 64) are all issued in ONE batch, so a group costs one L2 round trip under the weight stream.  Measured on
// c2 (timing-only builds): the previous form - 16 per batch, four scalar loads per lane, exponentials in the loop -
// cost 7 us of a 28 us attention phase.
template <int HD>
__device__ __forceinline__ void attn_merge(const Dev& D, int r, int h, int n_sub, int lane) {
  constexpr int DPL = HD / 32, NV = DPL / 2, GB = 24;
  const float* src = D.attn_part + ((size_t)r * D.nh + h) * (size_t)(D.max_chunks * 4) * (HD + 2);
  float Mc = -INFINITY, den = 0.f, num[DPL];
#pragma unroll
  for (int t = 0; t < DPL; ++t) num[t] = 0.f;
  for (int g0 = 0; g0 < n_sub; g0 += GB) {
    const int n_g = min(GB, n_sub - g0);
    float mv = -INFINITY, lv = 0.f;
    if (lane < n_g) {
      const float2 ml = __ldcg(reinterpret_cast<const float2*>(src + (size_t)(g0 + lane) * (HD + 2) + HD));
      mv = ml.x; lv = ml.y;
    }
    float2 ov[GB][NV];
#pragma unroll
    for (int i = 0; i < GB; ++i) {
      const float* sc = src + (size_t)(g0 + i) * (HD + 2);
#pragma unroll
      for (int v = 0; v < NV; ++v)
        ov[i][v] = i < n_g ? __ldcg(reinterpret_cast<const float2*>(sc + v * 64 + 2 * lane)) : make_float2(0.f, 0.f);
    }
    // running maximum before this lane's sub-partial, within the group and from the groups before
    float incl = mv;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl = fmaxf(incl, t);
    }
    float excl = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) excl = -INFINITY;
    const float Mprev = fmaxf(Mc, excl);
    const float s_l = (mv > Mprev) ? expf(Mprev - mv) : 1.0f;    // exp(-inf) = 0 on the first one
    const float w_l = (mv == -INFINITY) ? 0.f : expf(mv - fmaxf(Mprev, mv));
    Mc = fmaxf(Mc, __shfl_sync(0xffffffffu, incl, 31));
#pragma unroll
    for (int i = 0; i < GB; ++i) {
      const float mi = __shfl_sync(0xffffffffu, mv, i);
      const float si = __shfl_sync(0xffffffffu, s_l, i), wi = __shfl_sync(0xffffffffu, w_l, i);
      const float li = __shfl_sync(0xffffffffu, lv, i);
      if (mi == -INFINITY) continue;                         // absent, or a tile without visible positions (warp-uniform)
      den *= si;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        num[2 * v] *= si;
        num[2 * v + 1] *= si;
        num[2 * v] = fmaf(wi, ov[i][v].x, num[2 * v]);
        num[2 * v + 1] = fmaf(wi, ov[i][v].y, num[2 * v + 1]);
      }
      den = fmaf(wi, li, den);
    }
  }
  const int K = D.nh * HD;
  const size_t ps = (size_t)D.R_cap * K;
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const size_t idx = (size_t)r * K + h * HD + v * 64 + 2 * lane;
    const float v0 = num[2 * v] / den, v1 = num[2 * v + 1] / den;
    const __nv_bfloat16 h0 = __float2bfloat16_rn(v0), h1 = __float2bfloat16_rn(v1);
    *reinterpret_cast<__nv_bfloat162*>(&D.act_o[idx]) = __halves2bfloat162(h0, h1);
    if (D.planes > 1)
      *reinterpret_cast<__nv_bfloat162*>(&D.act_o[ps + idx]) =
          __halves2bfloat162(__float2bfloat16_rn(v0 - __bfloat162float(h0)), __float2bfloat16_rn(v1 - __bfloat162float(h1)));
  }
}

// ---------------------------------------------------------------- QKV finalize + a3: lattice-masked decode attention
// Phase Q (warp = (row, head of the fused QKV output)): split-K sum, deferred RMSNorm scale, RoPE (rotate-half,
// R13); query heads -> fp32 qbuf, key / value heads -> bf16 into the row's branch-private slot.
template <int HD>
__device__ __forceinline__ void unit_qkv(const RoundArgs& a, int j, const float* part, int r, int hh, int lane,
                                         const RowLite* rc = nullptr) {
  constexpr int DPL = HD / 32, HH = HD / 2;
  const Dev& D = a.D;
  const OpDesc& op = a.op[0];
  const RowView rv = row_view(D, rc, r);
  if (!rv.valid) return;
  const int m = rv.grp;
  if (j >= a.dec.layer_len[m]) return;
  const int layer = a.dec.layer_lo[m] + j, pos = rv.pos;
  const float inv = inv_rms(D, r);
  const int d0 = lane * DPL;
  const float* p = part + (size_t)r * op.part_ld + (size_t)hh * HD + d0;
  float x[DPL];
#pragma unroll
  for (int t = 0; t < DPL; ++t) x[t] = 0.f;
  for (int s0 = 0; s0 < op.ksplit; s0 += 8) {              // all split-K partial loads of a pass in one batch
    float tv[8][DPL];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool on = s0 + i < op.ksplit;
      const size_t so = (size_t)(s0 + i) * op.split_stride;
#pragma unroll
      for (int t = 0; t < DPL; ++t) tv[i][t] = on ? p[so + t] : 0.f;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int t = 0; t < DPL; ++t)
        if (s0 + i < op.ksplit) x[t] += tv[i][t];          // split order (H3)
  }
  const bool is_v = hh >= D.nh + D.nkv;
  const bool lo = lane < 16;
  const float2* rt = D.rope + (size_t)pos * HH + (lo ? d0 : d0 - HH);
  float o[DPL];
#pragma unroll
  for (int t = 0; t < DPL; ++t) {
    const float xa = x[t] * inv;
    const float xb = __shfl_xor_sync(0xffffffffu, xa, 16); // rotate-half partner dim lives in lane ^ 16
    const float2 cs = is_v ? make_float2(1.f, 0.f) : rt[t];
    o[t] = is_v ? xa : (lo ? (xa * cs.x - xb * cs.y) : (xa * cs.x + xb * cs.y));
  }
  if (hh < D.nh) {
    float* q = D.qbuf + ((size_t)r * D.nh + hh) * HD + d0;
#pragma unroll
    for (int t = 0; t < DPL; ++t) q[t] = o[t];
  } else {
    const int g = is_v ? hh - D.nh - D.nkv : hh - D.nh;
    __nv_bfloat16* dst = (is_v ? D.vslot : D.kslot) + slot_off(D, rv.seq, rv.slot, layer) + (size_t)g * HD + d0;
#pragma unroll
    for (int t = 0; t < DPL; ++t) dst[t] = __float2bfloat16_rn(o[t]);
  }
}
template <int HD>
__device__ void glue_qkv_finalize(const RoundArgs& a, int j, int gw, int n_gw, int lane, const RowLite* rc) {
  const Dev& D = a.D;
  const int heads = D.nh + 2 * D.nkv;
  for (int u = gw; u < D.R_dec * heads; u += n_gw) {
    const int r = u / heads, hh = u - r * heads;
    unit_qkv<HD>(a, j, D.part, r, hh, lane, rc);
  }
}

// Phase A.  Task (one CTA's glue group) = (stage m, sequence s, KV head g, range of 64-position chunks of
// ABSOLUTE position).  The committed K/V of each chunk is staged in shared memory with cp.async (128-bit,
// double buffered, 16-byte pieces XOR-swizzled by row) and applied to up to 16 (row, query head) pairs of
// (m, s, g) at once on the tensor cores (mma.sync m16n8k16, bf16 x bf16 -> fp32):
//   S^T[pair][pos] = Q[pair][:] . K[pos][:]   A = q as bf16 hi + lo (two MMAs: fp32-grade products, R23),
//                                             B = K rows straight from the staged tile (ldmatrix)
//   softmax over the warp's 16 positions      fp32, in the accumulator fragment (quad shuffles)
//   O[pair][dim]  = P[pair][pos] . V[pos][:]  A = P as bf16 hi + lo (the score fragment IS the A fragment),
//                                             B = V rows (ldmatrix.trans)
// Warp w of the first four handles positions [16w, 16w+16) of the chunk and writes one (o, max, sum)
// sub-partial per pair.  Positions >= n_paged are a row's private suffix - its ancestor slots and its own
// slot, the "ancestry mask" of north_star (b): for the chunk(s) that hold them the rows are processed one
// lattice row at a time, after that row's private K/V rows are patched into the staged tile at their
// positions.  Every position therefore goes through the same instructions wherever its K/V lives (slot before
// commit, page after) and whatever else shares the MMA: DEX stream == AR stream (H3).  When all chunks of
// (row, head) are written, the last writer merges the sub-partials in ascending position order.
constexpr int kAttnPairs = 16;       // pairs per pass of a task (the M of the MMAs)
constexpr int kPageCache = 96;       // chunks of a range whose page index is cached in shared memory (longer ranges: table lookups)

template <int HD>
struct AttnSmem {
  __nv_bfloat16 kv[2][2][kChunk * HD];          // eight tile buffers of [K / V][16 positions][dim] (attn_run: NB per warp),
                                                // 16-byte pieces swizzled: j ^ (row & 7)
  __nv_bfloat16 qh[kAttnPairs][HD + 8];         // q hi / lo planes (row stride padded: conflict-free fragment loads)
  __nv_bfloat16 ql[kAttnPairs][HD + 8];
  int ppos[kAttnPairs];                         // position of the pair's row; -1: not in this pass
  int prow[kAttnPairs], phead[kAttnPairs];
  int rpos[kAttnPairs];                         // per LATTICE ROW of the pass (row rl = pair / Gq): its position and the slot
  int rslot[kAttnPairs][kMaxAnc + 1];           // that holds private position n_paged + i (ancestor slots, then its own): read
                                                // once per task, so the private-tile loop has ONE dependent load per row
  int n_vrow;                                   // sparse lattice (R26): the expanded rows of the task's (stage, sequence)
  short vrow[128];
  int unit_ctr;                                 // next work unit of the pass (claimed per warp)
  int cpage[kPageCache];                        // page of every 64-position chunk of the task's range
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};\n"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&v);
}

// Positions [c0 + 16*t, +16) of the staged chunk against the pass's pairs [p_lo, p_hi): one sub-partial per pair.
// kbase / vbase: shared-memory tiles whose row `row0 + i` holds position c*64 + 16*t + i.
template <int HD>
__device__ __forceinline__ void attn_tile(const Dev& D, AttnSmem<HD>* sm, uint32_t kbase, uint32_t vbase, int row0, int c, int t,
                                          int p_lo, int p_hi, int lane) {
  constexpr int KT = HD / 16, NT = HD / 8;
  const int c0 = c * kChunk;
  const int rq = lane >> 2, cq = (lane & 3) * 2;            // fragment row (pair) / column offset of this lane
  // ---- S^T = Q . K^T over the head dim
  // four independent accumulator chains per position half (q hi / lo planes x even / odd k-tiles), added in a
  // fixed order afterwards: a dependent mma.sync costs ~35 cycles
  float S[2][4], Sx[2][3][4];
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      S[j][e] = 0.f;
      Sx[j][0][e] = Sx[j][1][e] = Sx[j][2][e] = 0.f;
    }
  const int krow = row0 + (lane & 7) + ((lane >> 4) << 3);   // ldmatrix row of this lane: matrices 0,1 -> rows 0-7, 2,3 -> 8-15
  const int khalf = (lane >> 3) & 1;                           // matrices 1,3: second 16-byte piece of the k-tile
#pragma unroll
  for (int kt = 0; kt < KT; ++kt) {
    uint32_t ah[4], al[4], b[4];
    ah[0] = *reinterpret_cast<const uint32_t*>(&sm->qh[rq][kt * 16 + cq]);
    ah[1] = *reinterpret_cast<const uint32_t*>(&sm->qh[rq + 8][kt * 16 + cq]);
    ah[2] = *reinterpret_cast<const uint32_t*>(&sm->qh[rq][kt * 16 + 8 + cq]);
    ah[3] = *reinterpret_cast<const uint32_t*>(&sm->qh[rq + 8][kt * 16 + 8 + cq]);
    al[0] = *reinterpret_cast<const uint32_t*>(&sm->ql[rq][kt * 16 + cq]);
    al[1] = *reinterpret_cast<const uint32_t*>(&sm->ql[rq + 8][kt * 16 + cq]);
    al[2] = *reinterpret_cast<const uint32_t*>(&sm->ql[rq][kt * 16 + 8 + cq]);
    al[3] = *reinterpret_cast<const uint32_t*>(&sm->ql[rq + 8][kt * 16 + 8 + cq]);
    const int piece = (kt * 2 + khalf) ^ (krow & 7);
    ldsm_x4(kbase + (krow * HD + piece * 8) * 2, b);           // b[0],b[1]: positions 0-7 of the tile; b[2],b[3]: 8-15
    if (kt & 1) {
      mma_bf16(Sx[0][1], ah, b[0], b[1]);
      mma_bf16(Sx[0][2], al, b[0], b[1]);
      mma_bf16(Sx[1][1], ah, b[2], b[3]);
      mma_bf16(Sx[1][2], al, b[2], b[3]);
    } else {
      mma_bf16(S[0], ah, b[0], b[1]);
      mma_bf16(Sx[0][0], al, b[0], b[1]);
      mma_bf16(S[1], ah, b[2], b[3]);
      mma_bf16(Sx[1][0], al, b[2], b[3]);
    }
  }
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int e = 0; e < 4; ++e) S[j][e] = (S[j][e] + Sx[j][1][e]) + (Sx[j][0][e] + Sx[j][2][e]);
  // ---- mask, scale, softmax over the tile's 16 positions (fragment rows rq and rq + 8)
  const float scale = 1.0f / sqrtf((float)HD);
  const int pos_a = (rq >= p_lo && rq < p_hi) ? sm->ppos[rq] : -1;
  const int pos_b = (rq + 8 >= p_lo && rq + 8 < p_hi) ? sm->ppos[rq + 8] : -1;
  float mx_a = -INFINITY, mx_b = -INFINITY;
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int pp = c0 + t * 16 + j * 8 + cq + (e & 1);
      const int lim = (e < 2) ? pos_a : pos_b;
      const float v = (pp <= lim) ? S[j][e] * scale : -INFINITY;
      S[j][e] = v;
      if (e < 2) mx_a = fmaxf(mx_a, v); else mx_b = fmaxf(mx_b, v);
    }
#pragma unroll
  for (int o = 1; o < 4; o <<= 1) {
    mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, o));
    mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, o));
  }
  float l_a = 0.f, l_b = 0.f;
  uint32_t ph[4], pl[4];                                      // P as A fragments (hi / lo planes)
  {
    float p[2][4];
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float m = (e < 2) ? mx_a : mx_b;
        const float v = (S[j][e] == -INFINITY) ? 0.f : expf(S[j][e] - m);
        p[j][e] = v;
        if (e < 2) l_a += v; else l_b += v;
      }
#pragma unroll
    for (int j = 0; j < 2; ++j) {                             // a0a1 | a2a3 = positions 0-7 (rows rq | rq+8), a4a5 | a6a7 = 8-15
      const float h0 = bf16_rt(p[j][0]), h1 = bf16_rt(p[j][1]), h2 = bf16_rt(p[j][2]), h3 = bf16_rt(p[j][3]);
      ph[2 * j] = pack_bf16(h0, h1);
      ph[2 * j + 1] = pack_bf16(h2, h3);
      pl[2 * j] = pack_bf16(p[j][0] - h0, p[j][1] - h1);
      pl[2 * j + 1] = pack_bf16(p[j][2] - h2, p[j][3] - h3);
    }
  }
#pragma unroll
  for (int o = 1; o < 4; o <<= 1) {
    l_a += __shfl_xor_sync(0xffffffffu, l_a, o);
    l_b += __shfl_xor_sync(0xffffffffu, l_b, o);
  }
  // ---- O = P . V
  float O[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt)
#pragma unroll
    for (int e = 0; e < 4; ++e) O[nt][e] = 0.f;
  const int vrow = row0 + (lane & 7) + (((lane >> 3) & 1) << 3);   // matrices 0,2: positions 0-7; 1,3: 8-15
  const int vsel = lane >> 4;                                        // matrices 2,3: the next 8-dim piece
#pragma unroll
  for (int nt = 0; nt < NT; nt += 2) {
    uint32_t b[4];
    const int piece = (nt + vsel) ^ (vrow & 7);
    ldsm_x4_t(vbase + (vrow * HD + piece * 8) * 2, b);         // b[0],b[1]: dims nt*8..+8; b[2],b[3]: the next 8
    mma_bf16(O[nt], ph, b[0], b[1]);
    mma_bf16(O[nt], pl, b[0], b[1]);
    mma_bf16(O[nt + 1], ph, b[2], b[3]);
    mma_bf16(O[nt + 1], pl, b[2], b[3]);
  }
  // ---- one (o, max, sum) sub-partial per pair: sub index = 4*c + t
  const size_t sub = (size_t)(c * 4 + t) * (HD + 2);
  if (pos_a >= c0 + t * 16) {                                 // the row sees this tile
    float* dst = D.attn_part + ((size_t)sm->prow[rq] * D.nh + sm->phead[rq]) * (size_t)(D.max_chunks * 4) * (HD + 2) + sub;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) *reinterpret_cast<float2*>(dst + nt * 8 + cq) = make_float2(O[nt][0], O[nt][1]);
    if ((lane & 3) == 0) { dst[HD] = mx_a; dst[HD + 1] = l_a; }
  }
  if (pos_b >= c0 + t * 16) {
    float* dst = D.attn_part + ((size_t)sm->prow[rq + 8] * D.nh + sm->phead[rq + 8]) * (size_t)(D.max_chunks * 4) * (HD + 2) + sub;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) *reinterpret_cast<float2*>(dst + nt * 8 + cq) = make_float2(O[nt][2], O[nt][3]);
    if ((lane & 3) == 0) { dst[HD] = mx_b; dst[HD + 1] = l_b; }
  }
}

// PT (pass tasks): a task also fixes ONE pass of <= 16 (row, head) pairs of its (stage, sequence).  Passes re-stage
// the chunks anyway, and as tasks of their own a wide stage (64 rows at N = 8, 16 passes with GQA) spreads over
// the grid instead of running its passes back to back on one CTA; with more tasks than CTAs the ranges are dealt
// from the LAST one (private positions, merges: the heaviest tasks first).  A separate instantiation because
// lattices whose stages all fit one pass (N <= 5 at MHA) keep the simpler loop and its register allocation.
// How the attention work of one layer-step is cut into tasks (shared by every CTA: same deterministic split).
struct AttnPlan {
  int tail_own, n_body, CR, n_ranges, Gq, per_ms, fam, n_tasks;
  int lpt;                 // pass tasks dealt heaviest range first (k_round); k_flow needs stage-major task order
};
struct AttnTask {
  int m, s, g, rg, pb_task;
};
template <bool PT>
__device__ __forceinline__ void attn_plan(const RoundArgs& a, int G, int n_live_ms, const int* cum, AttnPlan& p) {
  const Dev& D = a.D;
  const int n_msg = max(1, n_live_ms) * D.nkv;
  // ranges of chunks per (stage, sequence, KV head): as many as fill the grid once.  With >= 2 ranges the LAST
  // chunk (the one with the private positions, the per-row passes and usually the final merge) is a range of
  // its own and the others share the rest; more families than CTAs: 3-chunk ranges dealt round-robin.
  const int nr_fit = G / n_msg;
  const bool tail_own = nr_fit >= 2 && a.n_chunks >= 2;
  const int n_body = tail_own ? a.n_chunks - 1 : a.n_chunks;
  const int nr_body = tail_own ? nr_fit - 1 : max(nr_fit, 1);
  // more families than CTAs: ranges sized for about four tasks per CTA (a task's fixed cost - q staging, first
  // stage, counters, merges - is several chunks' worth), at least 3 chunks
  const int nr_many = max(1, (4 * G) / n_msg);
  const int CR = nr_fit >= 1 ? max(1, (n_body + nr_body - 1) / nr_body) : max(3, (n_body + nr_many - 1) / nr_many);
  p.tail_own = tail_own; p.n_body = n_body; p.CR = CR;
  p.n_ranges = (n_body + CR - 1) / CR + (tail_own ? 1 : 0);
  p.Gq = D.nh / D.nkv;
  p.per_ms = D.nkv * p.n_ranges;
  p.fam = PT ? cum[D.N] * D.nkv : 0;                         // cum[m]: (sequence, pass) slots of the stages before m (shared memory)
  p.n_tasks = PT ? p.fam * p.n_ranges : D.N * D.max_seqs * p.per_ms;
  p.lpt = PT && p.n_tasks > G;                             // one wave: range fastest, as without pass tasks
}
template <bool PT>
__device__ __forceinline__ void attn_task_of(const RoundArgs& a, const AttnPlan& p, const int* cum, int G, int u, AttnTask& t) {
  const Dev& D = a.D;
  t.pb_task = 0;
  if constexpr (PT) {
    const bool lpt = p.lpt != 0;
    t.rg = lpt ? p.n_ranges - 1 - u / p.fam : u % p.n_ranges;
    const int rem = lpt ? u % p.fam : u / p.n_ranges;
    const int psi = rem / D.nkv;
    t.g = rem - psi * D.nkv;
    int m = 0;
    while (psi >= cum[m + 1]) ++m;
    const int pp_m = (cum[m + 1] - cum[m]) / D.max_seqs;
    t.m = m;
    t.s = (psi - cum[m]) / pp_m;
    t.pb_task = ((psi - cum[m]) % pp_m) * kAttnPairs;
  } else {
    const int ms = u / p.per_ms, rem = u - ms * p.per_ms;
    t.m = ms / D.max_seqs; t.s = ms - t.m * D.max_seqs;
    t.g = rem / p.n_ranges; t.rg = rem - t.g * p.n_ranges;
  }
}

// One task by one glue group of GT threads (we = warp of the group, tid_e = thread of the group).  s_ao_cnt (k_flow
// only, else nullptr): shared counters of the (row, head) pairs this task merged, per ao_slice_cols columns of act_o.
template <int HD, int GT, bool PT>
__device__ void attn_run(const RoundArgs& a, const AttnPlan& pl, const AttnTask& tk, int j, int tid_e, int lane, int we,
                         AttnSmem<HD>* sm, int* s_ao_cnt, int ao_slice_cols, const SeqState* seq_sm) {
  constexpr int CPR = HD / 8;                                // 16-byte pieces per K/V row
  constexpr int kEpiThreads = GT;
  constexpr int NW = GT / 32, NB = NW >= 8 ? 1 : 2;          // warps of the group; 16-position tile buffers per warp
  static_assert(NW * NB <= 8, "the K/V staging area holds eight 16-position tile pairs");
  const Dev& D = a.D;
  const int m = tk.m, s = tk.s, g = tk.g, rg = tk.rg, pb_task = tk.pb_task;
  const bool tail_own = pl.tail_own != 0;
  const int n_body = pl.n_body, CR = pl.CR, n_ranges = pl.n_ranges, Gq = pl.Gq;
  const size_t kv_stride = (size_t)D.nkv * HD;
  const SeqState st = seq_sm[s];                            // the round's FSM snapshot in shared memory (constant for the round)
  if (!r_seq_live(st) || st.q < m || j >= a.dec.layer_len[m]) return;
  const bool is_tail = tail_own && rg == n_ranges - 1;
  const int ca = is_tail ? n_body : rg * CR;
  const int cb = min(is_tail ? a.n_chunks : min(ca + CR, n_body), (st.ctx_len + st.q) / kChunk + 1);   // no row lies beyond ctx_len + q
  if (ca >= cb) return;
  int cnt = r_stage_count(st.q, m);
  const int layer = a.dec.layer_lo[m] + j;
  const int r0 = a.dec.row_base[m] + s * cap_of(D.N, m);
  const int n_paged = st.ctx_len;
  const bool sparse = D.lookahead > 0;
  if (sparse) {                                            // compact list of the rows that were expanded (ascending)
    if (we == 0) {
      int base = 0;
      for (int i0 = 0; i0 < cnt; i0 += 32) {
        const int i = i0 + lane;
        const bool v = i < cnt && D.rows[r0 + i].valid;
        const unsigned bal = __ballot_sync(0xffffffffu, v);
        if (v) sm->vrow[base + __popc(bal & ((1u << lane) - 1u))] = (short)i;
        base += __popc(bal);
      }
      if (lane == 0) sm->n_vrow = base;
    }
    bar_epi<GT>();
    cnt = sm->n_vrow;
    bar_epi<GT>();                                           // every warp has read n_vrow before warp 0 may rewrite it (next task)
  }
  auto row_of = [&](int i) { return r0 + (sparse ? (int)sm->vrow[i] : i); };
  const int n_pairs = cnt * Gq;
  if (PT && pb_task >= n_pairs) return;                  // this pass has no pairs at the sequence's FSM state

  for (int pb = pb_task; pb < (PT ? min(n_pairs, pb_task + kAttnPairs) : n_pairs); pb += kAttnPairs) {
    const int np = min(kAttnPairs, n_pairs - pb);
    // ---- work units of the pass.  The range's 16-position tiles [4 ca, 4 cb) are independent of one another: every
    // (tile, pair) writes a sub-partial of its own and the merge below adds them in position order, so which warp runs
    // a tile, and when, cannot change a bit (H3).  Each warp owns NB tile buffers (K and V of 16 positions, 64 KB for
    // the group), claims units from a shared counter, loads the tile with cp.async and computes it on its own: no
    // CTA-wide barrier inside the loop, and the 8 warps' loads are in flight under one another's MMAs (the chunk-wide
    // double buffer had ONE 32 KB stage in flight per CTA and was bound by its latency).
    //   shared tile  (all 16 positions committed): one attn_tile over every pair of the pass
    //   private unit (tile, rank of nk): the tile holds private positions; the unit takes lattice rows rank, rank + nk, ...
    //     one at a time, patching the row's ancestor / own K/V rows (from their slots) into its copy of the tile IN PLACE.
    //     Rows above the row's own position keep finite data (zeros or an earlier row's patch): they are masked and
    //     enter the P.V MMA with weight 0.  Private units come first in the claim order (they are the long ones).
    const int T0 = ca * 4;
    const int T_end = min(cb * 4, (st.ctx_len + st.q) / 16 + 1);          // no row sees a tile beyond ctx_len + q
    const int T_sh = min(T_end, max(T0, n_paged / 16));                    // tiles [T0, T_sh) are fully committed
    const int n_priv = T_end - T_sh;
    const int n_rl = (np + Gq - 1) / Gq;
    const int nk = n_priv > 0 ? max(1, min(n_rl, NW / n_priv)) : 1;
    const int n_pu = n_priv * nk;
    const int n_units = n_pu + (T_sh - T0);
    if (tid_e == 0) sm->unit_ctr = 0;
    for (int i = tid_e; i < min(cb - ca, kPageCache); i += kEpiThreads)     // page of every chunk of the range (one per chunk:
      sm->cpage[i] = D.page_table[s * D.pages_per_seq + ((ca + i) * kChunk) / D.page_size];   // page_size % 64 == 0)
    bar_epi<GT>();
    auto claim = [&]() {
      int u = 0;
      if (lane == 0) u = atomicAdd(&sm->unit_ctr, 1);
      return __shfl_sync(0xffffffffu, u, 0);
    };
    auto tile_of = [&](int u) { return u < n_pu ? T_sh + u / nk : T0 + (u - n_pu); };
    auto kbuf = [&](int b) { return &sm->kv[0][0][0] + (size_t)((we * NB + b) * 2) * (16 * HD); };
    auto load_unit = [&](int u, int b) {                  // committed rows of the unit's tile -> the warp's buffer b, zeros above
      if (u < n_units) {
        const int T = tile_of(u), p0 = T * 16, ci = T / 4 - ca;
        const int n_rows = max(0, min(16, n_paged - p0));
        __nv_bfloat16* kd = kbuf(b);
        __nv_bfloat16* vd = kd + 16 * HD;
        if (n_rows > 0) {
          const int pg = ci < kPageCache ? sm->cpage[ci] : D.page_table[s * D.pages_per_seq + p0 / D.page_size];
          const size_t base = (size_t)layer * kv_layer_elems(D) + (size_t)pg * kv_page_elems(D) + (size_t)(p0 % D.page_size) * kv_stride + (size_t)g * HD;
          for (int id = lane; id < n_rows * CPR; id += 32) {
            const int pl = id / CPR, cj = id - pl * CPR;
            const int dj = (cj ^ (pl & 7)) * 8;
            cp_async16(kd + pl * HD + dj, D.kpool + base + (size_t)pl * kv_stride + cj * 8);
            cp_async16(vd + pl * HD + dj, D.vpool + base + (size_t)pl * kv_stride + cj * 8);
          }
        }
        for (int id = lane; id < (16 - n_rows) * CPR; id += 32) {
          const int pl = n_rows + id / CPR, cj = id % CPR;
          *reinterpret_cast<uint4*>(kd + pl * HD + cj * 8) = make_uint4(0u, 0u, 0u, 0u);
          *reinterpret_cast<uint4*>(vd + pl * HD + cj * 8) = make_uint4(0u, 0u, 0u, 0u);
        }
      }
      cp_async_commit();
    };
    int u0 = claim(), u1 = n_units;
    load_unit(u0, 0);
    if (NB == 2) { u1 = claim(); load_unit(u1, 1); }
    // ---- q of the pass's pairs (phase Q wrote it) -> bf16 hi / lo planes, in flight together with the first tiles
    for (int id = tid_e; id < kAttnPairs * HD; id += kEpiThreads) {
      const int pi = id / HD, t = id - pi * HD;
      float v = 0.f;
      if (pi < np) {
        const int r = row_of((pb + pi) / Gq), h = g * Gq + (pb + pi) % Gq;
        v = D.qbuf[((size_t)r * D.nh + h) * HD + t];
      }
      const __nv_bfloat16 hi = __float2bfloat16_rn(v);
      sm->qh[pi][t] = hi;
      sm->ql[pi][t] = __float2bfloat16_rn(v - __bfloat162float(hi));
    }
    if (tid_e < kAttnPairs) {
      const int pi = tid_e;
      int pos = -1, r = 0, h = 0;
      if (pi < np) {
        r = row_of((pb + pi) / Gq);
        h = g * Gq + (pb + pi) % Gq;
        pos = D.rows[r].pos;
        if (pos < ca * kChunk) pos = -1;                   // the row ends before this range
      }
      sm->ppos[pi] = pos;
      sm->prow[pi] = r;
      sm->phead[pi] = h;
      if (pi < np && (pb + pi) % Gq == 0) {                  // first pair of a lattice row: the row's private-suffix table
        const int rl = pi / Gq;
        const RowInfo* ri = &D.rows[r];
        const int n_anc = ri->n_anc, own = ri->slot;
        sm->rpos[rl] = ri->pos;
#pragma unroll
        for (int i = 0; i <= kMaxAnc; ++i) sm->rslot[rl][i] = (i < n_anc && i < kMaxAnc) ? ri->anc[i] : own;
      }
    }
    bar_epi<GT>();                                           // q planes and the row tables are written
    for (int k = 0;; ++k) {
      const int b = NB == 2 ? (k & 1) : 0;
      const int u = b ? u1 : u0;
      if (u >= n_units) break;                               // claims only grow: nothing later is valid either
      cp_async_wait<NB - 1>();
      __syncwarp();
      {
        const int T = tile_of(u), c = T >> 2, t = T & 3, p0 = T * 16;
        __nv_bfloat16* kd = kbuf(b);
        const uint32_t kbt = smem_u32(kd), vbt = smem_u32(kd + 16 * HD);
        if (u >= n_pu) {
          attn_tile<HD>(D, sm, kbt, vbt, 0, c, t, 0, np, lane);   // every pair shares a committed tile
        } else {
          const int i_lo = max(n_paged - p0, 0);
          for (int rl = u % nk; rl < n_rl; rl += nk) {
            const int pos = sm->rpos[rl];
            if (pos < p0) continue;                        // the row does not see this tile (warp-uniform)
            const int i_hi = min(pos - p0, 15);
            for (int id = lane; id < (i_hi - i_lo + 1) * CPR; id += 32) {
              const int i = i_lo + id / CPR, cj = id % CPR;
              const int ai = p0 + i - n_paged;
              const int slot = sm->rslot[rl][min(ai, kMaxAnc)];
              const size_t so = slot_off(D, s, slot, layer) + (size_t)g * HD + cj * 8;
              const int dj = (cj ^ (i & 7)) * 8;
              *reinterpret_cast<uint4*>(kd + i * HD + dj) = *reinterpret_cast<const uint4*>(D.kslot + so);
              *reinterpret_cast<uint4*>(kd + 16 * HD + i * HD + dj) = *reinterpret_cast<const uint4*>(D.vslot + so);
            }
            __syncwarp();
            attn_tile<HD>(D, sm, kbt, vbt, 0, c, t, rl * Gq, min(np, (rl + 1) * Gq), lane);
            __syncwarp();
          }
        }
      }
      __syncwarp();                                          // every lane is done with buffer b before it is refilled
      const int un = claim();
      load_unit(un, b);
      if (b) u1 = un; else u0 = un;
    }
    cp_async_wait<0>();
    // ---- all sub-partials of this pass are written: count the chunks in; the last writer of (row, head) merges
    bar_epi<GT>();                                           // orders every warp's sub-partial stores before the counter's release
    for (int pi = we; pi < np; pi += GT / 32) {
      const int pos = sm->ppos[pi];
      if (pos < 0) continue;
      const int r = sm->prow[pi], h = sm->phead[pi];
      const int mine = min(cb, pos / kChunk + 1) - ca;     // chunks of this range visible to the row
      if (mine <= 0) continue;
      const int nc = pos / kChunk + 1;
      // this range holds EVERY chunk the row sees: sole writer, no counter (the CTA barrier above already orders this
      // CTA's sub-partial stores before the merge's loads) - saves the atomic's round trip on the lattice rounds, whose
      // (stage, head) families fill the grid with one range each
      const bool sole = mine == nc;
      int old = 0;
      if (!sole && lane == 0)                                // release our sub-partials, acquire the other ranges'
        asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], %2;\n" : "=r"(old) : "l"(&D.attn_cnt[r * D.nh + h]), "r"(mine) : "memory");
      old = __shfl_sync(0xffffffffu, old, 0);
      if (sole || old + mine == nc) {
        attn_merge<HD>(D, r, h, pos / 16 + 1, lane);           // reads with ld.global.cg (L2)
        if (lane == 0) {
          if (!sole) D.attn_cnt[r * D.nh + h] = 0;
          if (s_ao_cnt) atomicAdd(&s_ao_cnt[(h * HD) / ao_slice_cols], 1);   // k_flow: merged (row, head) pairs per O-operand slice
        }
      }
    }
    bar_epi<GT>();
  }
}

template <int HD, int GT, bool PT>
__device__ void glue_attention(const RoundArgs& a, int j, int tid_e, int lane, int we, int cta, int G,
                               AttnSmem<HD>* sm, int n_live_ms, const int* cum, const SeqState* seq_sm) {
  AttnPlan pl;
  attn_plan<PT>(a, G, n_live_ms, cum, pl);
  for (int u = cta; u < pl.n_tasks; u += G) {
    AttnTask tk;
    attn_task_of<PT>(a, pl, cum, G, u, tk);
    attn_run<HD, GT, PT>(a, pl, tk, j, tid_e, lane, we, sm, nullptr, 1, seq_sm);
  }
}

}  // namespace dexk
