// round.cu — k_round: ONE persistent kernel for the whole expand + exit part of a DEX round
// (Alg. 1 lines 5-6): for every layer-step j all live stages run
//   QKV GEMM -> RoPE + slot-KV write + lattice attention -> O GEMM + residual + RMSNorm ->
//   gate/up GEMM -> SwiGLU -> down GEMM + residual + RMSNorm,
// then the fused exit (final RMSNorm done by the last step, LM-head GEMM, DECS arg-max).
//
// Why one kernel: at <= 16 stacked rows every op is a pure HBM stream of its weights (5-30 us at
// 7B), so launch boundaries and dependency bubbles, not bytes, set the speed.  Here one CTA per SM
// stays resident; its TMA producer walks the round's whole (op, tile, K-split) item list and keeps
// requesting weight tiles as far ahead as the shared-memory ring allows - weights do not depend on
// activations - while the dependent part (activation boxes, MMAs, epilogue, glue) trails behind
// grid-wide barriers.  The HBM stream therefore continues across op boundaries, glue phases and
// the barrier latency itself.
//
//   warp 0      producer: weight tiles (always ahead) + activation boxes (after the op's inputs
//               are published by a grid barrier)
//   warp 1      tcgen05.mma issuer (one lane), owns TMEM (two accumulator stages)
//   warps 2..5  epilogue group: TMEM -> split-K partials / exit arg-max, then the glue phase of
//               the step (attention, combine, add+norm, SwiGLU) spread over all CTAs, then the
//               grid barrier that publishes the next op's operand
//
// Items are dealt round-robin to CTAs continuing across ops, so the per-op remainder rotates and
// every CTA streams the same bytes per round to within one item.  The K split is fixed per
// operator shape and partials are added in split order: a row's bits do not depend on which rows
// or stages share the round (H3).
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_dev.cuh"

namespace dexk {

constexpr int kRoundThreads = 224;      // warps: 0 weight TMA, 1 MMA, 2-5 epilogue/glue, 6 activation TMA
constexpr int kEpiThreads = 128;

// ---------------------------------------------------------------- small device helpers
__device__ __forceinline__ void bar_epi() { asm volatile("bar.sync 1, 128;\n" ::: "memory"); }
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
#pragma unroll 4
  for (int s = 1; s < S; ++s) acc = r_add4(acc, r_ld4(p + (size_t)s * stride));
  return acc;
}
__device__ __forceinline__ float r_sum1(const float* p, int S, size_t stride) {
  float acc = p[0];
#pragma unroll 4
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
// op t < 4*n_steps: step j = t/4, kind t%4 (qkv, o, gate/up, down); op 4*n_steps: the exit head.
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
  int n_steps, n_ops, G, cta;

  __device__ __forceinline__ void op_info(int t, OpI& o) const {
    unsigned mask = 0;
    if (t < 4 * n_steps) {
      o.j = t >> 2; o.which = t & 3; o.ext = 0;
      for (int g = 0; g < a->dec.n_grp; ++g)
        if (s_nb[g] > 0 && o.j < a->dec.layer_len[g]) mask |= 1u << g;
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
    it.layer = o.ext ? 0 : p.layer_lo[it.g] + o.j;
    it.kb0 = it.split * o.kbps;
    it.kb1 = min(it.kb0 + o.kbps, o.kb_total);
    it.row0 = p.row_base[it.g];
    it.row_end = it.row0 + p.rows_cap[it.g];
  }
  // grid barriers that must have completed before op t's operand may be read (9 per step)
  __device__ __forceinline__ unsigned dep(int t) const {
    if (t >= 4 * n_steps) return 9u * n_steps;
    const int k = t & 3;
    return 9u * (t >> 2) + (k == 0 ? 0u : (k == 1 ? 3u : (k == 2 ? 5u : 7u)));
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
__device__ __forceinline__ void grid_bar(unsigned* gbar, unsigned target, int tid_e, volatile unsigned* s_seen, unsigned gb, int dbg = 0) {
  if (dbg & 2) return;
  __threadfence();
  fence_proxy_async();           // generic-proxy writes (operand planes) -> later TMA reads
  bar_epi();
  if (tid_e == 0) {
    red_release_add(gbar, 1u);
    unsigned spins = 0;
    while (ld_acquire_u32(gbar) < target) {
      __nanosleep(32);
      if (++spins > 100000000u) __trap();   // protocol bug: trap instead of hanging the box
    }
    __threadfence();
    *s_seen = gb;                // the producer of this CTA learns of the barrier without polling HBM/L2
  }
  bar_epi();
}

// ---------------------------------------------------------------- glue phases (epilogue group)
__device__ __forceinline__ float r_warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float group_sum(float v, float* red /*[4]*/, int tid_e) {
  v = r_warp_sum(v);
  bar_epi();
  if ((tid_e & 31) == 0) red[tid_e >> 5] = v;
  bar_epi();
  return (red[0] + red[1]) + (red[2] + red[3]);
}

// x += sum_s part[s]; RMSNorm -> operand planes.  mode 0: after o_proj (w = norm_ffn[l] -> act_a);
// mode 1: after down_proj (next layer's attention norm -> act_a, or the shared final norm -> act_e).
__device__ void glue_add_norm(const RoundArgs& a, int j, int mode, const OpDesc& op, float* red, int tid_e, int cta, int G) {
  const Dev& D = a.D;
  const int nv = D.d >> 2;
  for (int r = cta; r < D.R_dec; r += G) {
    const RowInfo* ri = &D.rows[r];
    if (!ri->valid) continue;
    const int grp = ri->grp;
    if (j >= a.dec.layer_len[grp]) continue;
    const int layer = a.dec.layer_lo[grp] + j;
    float* x = D.x_cur + (size_t)r * D.d;
    const float* p = D.part + (size_t)r * op.part_ld;
    float ss = 0.f;
    for (int i = tid_e; i < nv; i += kEpiThreads) {
      const float4 s4 = r_sum4(p + 4 * i, op.ksplit, op.split_stride);
      const float4 v = r_add4(r_ld4(x + 4 * i), s4);
      *reinterpret_cast<float4*>(x + 4 * i) = v;
      ss += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
      if (mode == 1 && D.taps) *reinterpret_cast<float4*>(D.tap_hidden + ((size_t)r * D.max_len + j) * D.d + 4 * i) = v;
    }
    ss = group_sum(ss, red, tid_e);
    const float inv = 1.0f / sqrtf(ss / (float)D.d + D.eps);
    const float* w;
    __nv_bfloat16* dst = D.act_a;
    if (mode == 0) {
      w = D.norm_ffn + (size_t)layer * D.d;
    } else if (j + 1 < a.dec.layer_len[grp]) {
      w = D.norm_attn + (size_t)(layer + 1) * D.d;
    } else {
      w = D.norm_final;
      dst = D.act_e;
    }
    const size_t ps = (size_t)D.R_cap * D.d;
    for (int i = tid_e; i < nv; i += kEpiThreads) {
      const float4 v = r_ld4(x + 4 * i), wv = r_ld4(w + 4 * i);   // own writes of the loop above
      r_split_store4(dst, ps, (size_t)r * D.d + 4 * i,
                     make_float4(v.x * inv * wv.x, v.y * inv * wv.y, v.z * inv * wv.z, v.w * inv * wv.w), D.planes);
    }
  }
}

// act_f = SiLU(gate) * up from the split-K partials of the fused gate/up projection.
__device__ void glue_silu(const RoundArgs& a, int j, const OpDesc& op, int tid_e, int cta, int G) {
  const Dev& D = a.D;
  const int blk = kEpiThreads * 4;
  const int nblk = (D.ffn + blk - 1) / blk;
  const size_t ps = (size_t)D.R_cap * D.ffn;
  for (int u = cta; u < D.R_dec * nblk; u += G) {
    const int r = u / nblk, b = u - r * nblk;
    const RowInfo* ri = &D.rows[r];
    if (!ri->valid || j >= a.dec.layer_len[ri->grp]) continue;
    const int i = b * blk + tid_e * 4;
    if (i >= D.ffn) continue;
    const float* p = D.part + (size_t)r * op.part_ld;
    const float4 g = r_sum4(p + i, op.ksplit, op.split_stride);
    const float4 up = r_sum4(p + D.ffn + i, op.ksplit, op.split_stride);
    float4 o;
    o.x = g.x / (1.0f + expf(-g.x)) * up.x;
    o.y = g.y / (1.0f + expf(-g.y)) * up.y;
    o.z = g.z / (1.0f + expf(-g.z)) * up.z;
    o.w = g.w / (1.0f + expf(-g.w)) * up.w;
    r_split_store4(D.act_f, ps, (size_t)r * D.ffn + i, o, D.planes);
  }
}

// Merge the per-chunk attention partials in ascending chunk order -> act_o planes.  Warp per (row, head).
template <int HD>
__device__ void glue_combine(const RoundArgs& a, int j, int gw, int n_gw, int lane) {
  const Dev& D = a.D;
  constexpr int DPL = HD / 32;
  const int K = D.nh * HD;
  for (int u = gw; u < D.R_dec * D.nh; u += n_gw) {
    const int r = u / D.nh, h = u - r * D.nh;
    const RowInfo* ri = &D.rows[r];
    if (!ri->valid || j >= a.dec.layer_len[ri->grp]) continue;
    const int nc = ri->pos / kChunk + 1;
    const float* src = D.attn_part + ((size_t)r * D.nh + h) * D.max_chunks * (HD + 2);
    float M = -INFINITY;
    for (int c = 0; c < nc; ++c) M = fmaxf(M, src[(size_t)c * (HD + 2) + HD]);
    float num[DPL], den = 0.f;
#pragma unroll
    for (int t = 0; t < DPL; ++t) num[t] = 0.f;
    for (int c = 0; c < nc; ++c) {
      const float* sc = src + (size_t)c * (HD + 2);
      const float w = expf(sc[HD] - M);
#pragma unroll
      for (int t = 0; t < DPL; ++t) num[t] = fmaf(w, sc[lane * DPL + t], num[t]);
      den = fmaf(w, sc[HD + 1], den);
    }
    const size_t ps = (size_t)D.R_cap * K;
    const size_t idx = (size_t)r * K + h * HD + lane * DPL;
#pragma unroll
    for (int t = 0; t < DPL; ++t) {
      const float v = num[t] / den;
      const __nv_bfloat16 hi = __float2bfloat16_rn(v);
      D.act_o[idx + t] = hi;
      if (D.planes > 1) D.act_o[ps + idx + t] = __float2bfloat16_rn(v - __bfloat162float(hi));
    }
  }
}

// 16 consecutive bf16 (two 16-byte loads) -> fp32
__device__ __forceinline__ void ld_bf16x16(const __nv_bfloat16* p, float (&f)[16]) {
  const uint4 u0 = *reinterpret_cast<const uint4*>(p), u1 = *reinterpret_cast<const uint4*>(p + 8);
  const __nv_bfloat162* a = reinterpret_cast<const __nv_bfloat162*>(&u0);
  const __nv_bfloat162* b = reinterpret_cast<const __nv_bfloat162*>(&u1);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 x = __bfloat1622float2(a[i]), y = __bfloat1622float2(b[i]);
    f[2 * i] = x.x; f[2 * i + 1] = x.y;
    f[8 + 2 * i] = y.x; f[8 + 2 * i + 1] = y.y;
  }
}

// a3: one warp = one unit (stage m, sequence s, KV head g, 64-position chunk c of ABSOLUTE position).
// The warp first finishes K/V of the rows whose own position lies in the chunk (split-K sum, RoPE,
// bf16 store into the row's slot), then attends up to 4 (row, query head) pairs at a time: LP lanes
// share a position (16 dims each), 32/LP positions per pass, so the committed K/V of the chunk is
// loaded once for the 4 pairs.  Positions >= n_paged are the row's private suffix (ancestor slots,
// own slot) and are fetched per pair.  fp32 scores, warp-shuffle softmax, per-chunk (o, max, sum).
template <int HD>
__device__ void attn_unit(const RoundArgs& a, int j, int m, int s, int g, int c, int lane, const OpDesc& op) {
  constexpr int LP = HD / 16, PI = 32 / LP, NIT = kChunk / PI, HALF = HD / 2;
  constexpr int PB = (HD == 128) ? 2 : 4;                   // (row, head) pairs per pass (register budget)
  const Dev& D = a.D;
  const SeqState st = D.seqs[s];
  if (!r_seq_live(st) || st.q < m || j >= a.dec.layer_len[m]) return;
  const int c0 = c * kChunk;
  if (c0 > st.ctx_len + st.q) return;                       // beyond every row's position
  const int cnt = r_stage_count(st.q, m);
  const int layer = a.dec.layer_lo[m] + j;
  const int r0 = a.dec.row_base[m] + s * cap_of(D.N, m);
  const int n_paged = st.ctx_len;
  const int G = D.nh / D.nkv;
  const int nq = D.nh * HD, nk = D.nkv * HD;
  const int sub = lane % LP, pg = lane / LP;
  const int S = op.ksplit;
  const size_t sst = op.split_stride;

  // (1) own K/V of rows positioned in this chunk
  for (int jr = 0; jr < cnt; ++jr) {
    const RowInfo* ri = &D.rows[r0 + jr];
    const int pos = ri->pos;
    if (pos < c0 || pos >= c0 + kChunk) continue;
    const float* p = D.part + (size_t)(r0 + jr) * op.part_ld;
    const float2* rt = D.rope + (size_t)pos * HALF;
    const size_t kvo = slot_off(D, s, ri->slot, layer) + (size_t)g * HD;
    __nv_bfloat16* kd = D.kslot + kvo;
    __nv_bfloat16* vd = D.vslot + kvo;
    for (int e = lane; e < HALF; e += 32) {
      const float x1 = r_sum1(p + nq + g * HD + e, S, sst), x2 = r_sum1(p + nq + g * HD + e + HALF, S, sst);
      const float2 cs = rt[e];
      kd[e] = __float2bfloat16_rn(x1 * cs.x - x2 * cs.y);
      kd[e + HALF] = __float2bfloat16_rn(x2 * cs.x + x1 * cs.y);
    }
    for (int e = lane; e < HD; e += 32) vd[e] = __float2bfloat16_rn(r_sum1(p + nq + nk + g * HD + e, S, sst));
  }
  __syncwarp();

  const float scale = 1.0f / sqrtf((float)HD);
  const int n_pairs = cnt * G;
  const size_t kv_stride = (size_t)D.nkv * HD;
  const size_t page_base = (c0 < n_paged) ? page_off(D, s, layer, c0) + (size_t)g * HD + sub * 16 : 0;

  for (int pb = 0; pb < n_pairs; pb += PB) {
    int prow[PB], phead[PB], ppos[PB];
    float q[PB][16];
#pragma unroll
    for (int p = 0; p < PB; ++p) {
      prow[p] = -1; phead[p] = 0; ppos[p] = -1;
      if (pb + p < n_pairs) {
        const int row = r0 + (pb + p) / G;
        const int pos = D.rows[row].pos;
        if (pos >= c0) {
          prow[p] = row; phead[p] = g * G + (pb + p) % G; ppos[p] = pos;
          // q = RoPE(sum of split-K partials), this lane's 16 dims
          const float* pr = D.part + (size_t)row * op.part_ld + phead[p] * HD;
          const float2* rt = D.rope + (size_t)pos * HALF;
          const int i0 = sub * 16;
          const bool lo = i0 < HALF;
          const int ia = lo ? i0 : i0 - HALF;              // index in the first half
#pragma unroll
          for (int e = 0; e < 16; e += 4) {
            const float4 x1 = r_sum4(pr + ia + e, S, sst), x2 = r_sum4(pr + ia + e + HALF, S, sst);
            const float2 c0_ = rt[ia + e], c1_ = rt[ia + e + 1], c2_ = rt[ia + e + 2], c3_ = rt[ia + e + 3];
            if (lo) {
              q[p][e] = x1.x * c0_.x - x2.x * c0_.y; q[p][e + 1] = x1.y * c1_.x - x2.y * c1_.y;
              q[p][e + 2] = x1.z * c2_.x - x2.z * c2_.y; q[p][e + 3] = x1.w * c3_.x - x2.w * c3_.y;
            } else {
              q[p][e] = x2.x * c0_.x + x1.x * c0_.y; q[p][e + 1] = x2.y * c1_.x + x1.y * c1_.y;
              q[p][e + 2] = x2.z * c2_.x + x1.z * c2_.y; q[p][e + 3] = x2.w * c3_.x + x1.w * c3_.y;
            }
          }
        }
      }
    }
    bool any = false;
#pragma unroll
    for (int p = 0; p < PB; ++p) any |= prow[p] >= 0;
    if (!any) continue;

    // scores
    float sc[PB][NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const int pl = it * PI + pg, pos = c0 + pl;
      const bool shared_it = (c0 + it * PI + PI - 1) < n_paged;     // warp-uniform
      float kf[16];
      if (shared_it) ld_bf16x16(D.kpool + page_base + (size_t)pl * kv_stride, kf);
#pragma unroll
      for (int p = 0; p < PB; ++p) {
        float dot = -INFINITY;
        if (prow[p] >= 0) {                                            // warp-uniform
          bool vis = true;
          if (!shared_it) {
            vis = pos <= ppos[p];
            if (vis) {
              const __nv_bfloat16* kp;
              if (pos < n_paged) {
                kp = D.kpool + page_base + (size_t)pl * kv_stride;
              } else {
                const RowInfo* ri = &D.rows[prow[p]];
                const int ai = pos - n_paged;
                const int slot = (ai < ri->n_anc) ? ri->anc[ai] : ri->slot;
                kp = D.kslot + slot_off(D, s, slot, layer) + (size_t)g * HD + sub * 16;
              }
              ld_bf16x16(kp, kf);
            }
          }
          float acc = 0.f;
          if (vis) {
#pragma unroll
            for (int e = 0; e < 16; ++e) acc = fmaf(q[p][e], kf[e], acc);
          }
#pragma unroll
          for (int o = 1; o < LP; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
          dot = vis ? acc * scale : -INFINITY;
        }
        sc[p][it] = dot;
      }
    }
    // softmax statistics of the chunk
    float mx[PB], lsum[PB];
#pragma unroll
    for (int p = 0; p < PB; ++p) {
      float v = -INFINITY;
#pragma unroll
      for (int it = 0; it < NIT; ++it) v = fmaxf(v, sc[p][it]);
#pragma unroll
      for (int o = LP; o < 32; o <<= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
      mx[p] = v;                                   // finite for an active pair: position c0 <= ppos is visible
      float t = 0.f;
#pragma unroll
      for (int it = 0; it < NIT; ++it) {
        const float e = (sc[p][it] == -INFINITY) ? 0.f : expf(sc[p][it] - v);
        sc[p][it] = e;
        t += e;
      }
#pragma unroll
      for (int o = LP; o < 32; o <<= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      lsum[p] = t;
    }
    // P.V (q[][] is dead: reuse as the output accumulator)
#pragma unroll
    for (int p = 0; p < PB; ++p)
#pragma unroll
      for (int e = 0; e < 16; ++e) q[p][e] = 0.f;
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const int pl = it * PI + pg, pos = c0 + pl;
      const bool shared_it = (c0 + it * PI + PI - 1) < n_paged;
      float vf[16];
      if (shared_it) ld_bf16x16(D.vpool + page_base + (size_t)pl * kv_stride, vf);
#pragma unroll
      for (int p = 0; p < PB; ++p) {
        if (prow[p] < 0) continue;
        const float pr = sc[p][it];
        if (!shared_it) {
          if (pos > ppos[p]) continue;
          const __nv_bfloat16* vp;
          if (pos < n_paged) {
            vp = D.vpool + page_base + (size_t)pl * kv_stride;
          } else {
            const RowInfo* ri = &D.rows[prow[p]];
            const int ai = pos - n_paged;
            const int slot = (ai < ri->n_anc) ? ri->anc[ai] : ri->slot;
            vp = D.vslot + slot_off(D, s, slot, layer) + (size_t)g * HD + sub * 16;
          }
          ld_bf16x16(vp, vf);
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) q[p][e] = fmaf(pr, vf[e], q[p][e]);
      }
    }
#pragma unroll
    for (int p = 0; p < PB; ++p) {
      if (prow[p] < 0) continue;
#pragma unroll
      for (int e = 0; e < 16; ++e) {
        float v = q[p][e];
#pragma unroll
        for (int o = LP; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        q[p][e] = v;
      }
      float* dst = D.attn_part + (((size_t)prow[p] * D.nh + phead[p]) * D.max_chunks + c) * (HD + 2);
      if (pg == 0) {
#pragma unroll
        for (int e = 0; e < 16; e += 4)
          *reinterpret_cast<float2*>(dst + sub * 16 + e) = make_float2(q[p][e], q[p][e + 1]),
          *reinterpret_cast<float2*>(dst + sub * 16 + e + 2) = make_float2(q[p][e + 2], q[p][e + 3]);
      }
      if (lane == 0) {
        dst[HD] = mx[p];
        dst[HD + 1] = lsum[p];
      }
    }
  }
}

template <int HD>
__device__ void glue_attention(const RoundArgs& a, int j, int gw, int n_gw, int lane) {
  const Dev& D = a.D;
  const OpDesc& op = a.op[0];
  const int per_ms = D.nkv * a.n_chunks;
  const int n_units = D.N * D.max_seqs * per_ms;
  for (int u = gw; u < n_units; u += n_gw) {
    const int ms = u / per_ms, rem = u - ms * per_ms;
    const int m = ms / D.max_seqs, s = ms - m * D.max_seqs;
    const int g = rem / a.n_chunks, c = rem - g * a.n_chunks;
    attn_unit<HD>(a, j, m, s, g, c, lane, op);
  }
}

// ---------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(kRoundThreads, 1) k_round(const __grid_constant__ TmSet tm, const __grid_constant__ RoundArgs a) {
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
  __shared__ float s_red[4];
  __shared__ int s_steps;
  __shared__ unsigned s_seen;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x < 32) s_valid[threadIdx.x] = 0;
  __syncthreads();
  for (int r = threadIdx.x; r < D.R_cap; r += kRoundThreads)
    if (D.rows[r].valid) atomicOr(&s_valid[r >> 5], 1u << (r & 31));
  if (threadIdx.x == 0) {
    int steps = 0;
    for (int g = 0; g < 8; ++g) {
      const int nb = (g < a.dec.n_grp) ? D.grp_nb[g] : 0;
      s_nb[g] = nb;
      if (nb > 0) steps = max(steps, a.dec.layer_len[g]);
      s_nb[8 + g] = (g < a.ext.n_grp) ? D.exit_nb[g] : 0;
    }
    s_steps = steps;
    s_seen = 0;
    for (int i = 0; i < NS; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&tfull[i], 1);
      mbar_init(&tempty[i], 4);
    }
    fence_mbar_init();
    for (int i = 0; i < 5; ++i) tma_prefetch_desc(&tm.w[i]);
    for (int i = 0; i < 4; ++i) tma_prefetch_desc(&tm.x[i]);
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, 2 * a.acc_cols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  Seq sq;
  sq.a = &a; sq.s_nb = s_nb; sq.n_steps = s_steps; sq.n_ops = 4 * s_steps + 1; sq.G = gridDim.x; sq.cta = blockIdx.x;
  const unsigned G = gridDim.x;

  if (s_steps > 0) {
    // The three single-issuer roles run warp-uniformly (all lanes walk the item list) and elect one lane
    // only around the TMA / MMA instructions, so those are issued from converged code.
    if (warp == 0) {
      // ===================== weight producer: always as far ahead as the ring allows =====================
      Walker w;
      unsigned st = 0, ph = 0;
      bool wrapped = false;
      const bool tiled = (a.dbg & 4) != 0;
      for (w.start(sq); w.valid; w.next(sq)) {
        const CUtensorMap* desc = tiled ? &tm.wt[w.o.which] : &tm.w[w.o.which];
        const uint32_t tx = kABytes + ((a.dbg & 8) ? 0 : D.planes * w.it.nb * 128);
        const int c1 = w.it.tile * kTileM, c2 = w.it.layer;
        const int tbase = (w.it.layer * (w.o.n_tiles - (a.op[w.o.which].out_dim % kTileM ? 1 : 0)) + min(w.it.tile, w.o.n_tiles - 2)) * (a.op[w.o.which].k_dim / kTileK);
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          if (wrapped) mbar_wait(&empty[st], ph ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(&full[st], tx);
            if (tiled) tma_load_3d(smem + (size_t)st * stage_bytes, desc, &full[st], 0, 0, tbase + min(kb, a.op[w.o.which].k_dim / kTileK - 1), kEvictFirst);
            else tma_load_3d(smem + (size_t)st * stage_bytes, desc, &full[st], kb * kTileK, c1, c2, kEvictFirst);
          }
          __syncwarp();
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; wrapped = true; }
        }
      }
    } else if (warp == 6) {
      // ===================== activation producer: trails behind the grid barriers =====================
      Walker w;
      unsigned st = 0, ph = 0;
      bool wrapped = false;
      unsigned seen = 0;
      for (w.start(sq); w.valid; w.next(sq)) {
        const unsigned need = (a.dbg & 2) ? 0u : sq.dep(w.t);
        if (seen < need) {
          unsigned spins = 0;
          while ((seen = *reinterpret_cast<volatile unsigned*>(&s_seen)) < need) {
            __nanosleep(32);
            if (++spins > 100000000u) __trap();
          }
          __threadfence();
          fence_proxy_async();
        }
        const int which = w.o.which;
        const CUtensorMap* desc = &tm.x[which == 0 ? 0 : (which == 1 ? 1 : (which == 2 ? 0 : (which == 3 ? 2 : 3)))];
        const int row0 = w.it.row0, nb = w.it.nb;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          // slot free (its previous tile consumed) => full[st] is in this tile's phase; the bytes may
          // land before the weight producer arms the phase (tx-count goes negative, arrival still pending)
          if (wrapped) mbar_wait(&empty[st], ph ^ 1u);
          if (!(a.dbg & 8) && elect_one()) {
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
      }
    } else if (warp == 1) {
      // ===================== MMA issuer =====================
      Walker w;
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
            mma_stage(smem_u32(smem + (size_t)st * stage_bytes), plane_bytes, D.planes, stacked, d_tmem, idesc, acc);
            umma_commit(&empty[st]);     // frees the ring slot when these MMAs have read it
          }
          __syncwarp();
          acc = 1;
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; }
        }
        if (elect_one()) umma_commit(&tfull[as]);   // accumulator complete -> epilogue
        __syncwarp();
      }
    } else if (warp < 6) {
      // ===================== epilogue group: GEMM epilogues + glue + grid barriers =====================
      const int tid_e = threadIdx.x - 64, we = warp - 2;
      const int quarter = warp & 3;
      const int gw = blockIdx.x * 4 + we, n_gw = gridDim.x * 4;
      EpiCtx ec;
      ec.rows = D.rows; ec.s_valid = s_valid; ec.part = D.part; ec.vocab = D.vocab; ec.best_key = D.best_key;
      ec.ref_tile = D.ref_tile; ec.ref_tiles = D.ref_tiles;
      Walker w;
      w.start(sq);
      int n_it = 0;
      unsigned gb = 0;
      int n_stamp = 0;
      auto stamp = [&]() {
        if (D.taps && blockIdx.x == 0 && tid_e == 0) {
          D.tap_times[n_stamp] = (unsigned long long)clock64();   // SM cycles of CTA 0's SM
        }
        ++n_stamp;
      };
      stamp();
      auto run_items = [&](int t) {
        const OpDesc& od = a.op[t < 4 * sq.n_steps ? (t & 3) : 4];
        ec.mode = (t < 4 * sq.n_steps) ? 0 : 1;
        ec.part_ld = od.part_ld; ec.split_stride = od.split_stride; ec.out_dim = od.out_dim;
        for (; w.valid && w.t == t; w.next(sq), ++n_it) {
          const int as = n_it & 1;
          mbar_wait(&tfull[as], (n_it >> 1) & 1);
          tc_fence_after();
          const uint32_t t_addr = tmem_base + as * a.acc_cols + ((uint32_t)(quarter * 32) << 16);
          epilogue_item(ec, t_addr, a.stacked != 0, w.it.nb, w.it.row0, w.it.row_end, w.it.tile, w.it.split, quarter, lane);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty[as]);
        }
      };
      for (int j = 0; j < sq.n_steps; ++j) {
        run_items(4 * j); stamp();
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        if (!(a.dbg & 1)) { if (D.hd == 128) glue_attention<128>(a, j, gw, n_gw, lane); else glue_attention<64>(a, j, gw, n_gw, lane); }
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        if (!(a.dbg & 1)) { if (D.hd == 128) glue_combine<128>(a, j, gw, n_gw, lane); else glue_combine<64>(a, j, gw, n_gw, lane); }
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        run_items(4 * j + 1); stamp();
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        if (!(a.dbg & 1)) glue_add_norm(a, j, 0, a.op[1], s_red, tid_e, blockIdx.x, G);
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        run_items(4 * j + 2); stamp();
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        if (!(a.dbg & 1)) glue_silu(a, j, a.op[2], tid_e, blockIdx.x, G);
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        run_items(4 * j + 3); stamp();
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
        if (!(a.dbg & 1)) glue_add_norm(a, j, 1, a.op[3], s_red, tid_e, blockIdx.x, G);
        ++gb; grid_bar(D.gbar, gb * G, tid_e, &s_seen, gb, a.dbg); stamp();
      }
      run_items(4 * sq.n_steps); stamp();
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 2 * a.acc_cols);
}

cudaError_t round_init() {
  return cudaFuncSetAttribute(k_round, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
}

// Cooperative launch: all CTAs must be co-resident (they meet at grid barriers).
cudaError_t launch_round(const TmSet& tm, const RoundArgs& a, int grid, size_t smem_bytes, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kRoundThreads);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_round, tm, a);
}

}  // namespace dexk
