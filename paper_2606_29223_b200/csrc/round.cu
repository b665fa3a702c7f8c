// round.cu — k_round: ONE persistent kernel for the whole expand + exit part of a DEX round
// (Alg. 1 lines 5-6): for every layer-step j all live stages run
//   QKV GEMM -> QKV finalize (scale, RoPE, slot-KV write) -> lattice attention -> O GEMM -> residual + norm operand ->
//   gate/up GEMM -> SwiGLU -> down GEMM -> residual + norm operand,
// then the fused exit (LM-head GEMM + DECS arg-max on the final-norm operand of every new row).
//
// Why one kernel: at <= 16 stacked rows every op is a pure HBM stream of its weights (5-30 us at
// 7B), so launch boundaries and dependency bubbles, not bytes, set the speed.  Here one CTA per SM
// stays resident; its weight producer walks the round's whole (op, tile, K-split) item list and keeps
// requesting weight tiles as far ahead as the shared-memory ring allows - weights do not depend on
// activations - while the dependent part (activation boxes, MMAs, epilogue, glue) trails behind
// grid-wide barriers.  The HBM stream therefore continues across op boundaries, glue phases and
// the barrier latency itself.
//
//   warp 0      weight producer (TMA, always ahead)
//   warp 6      activation producer (TMA, after the grid barrier that publishes the op's operand)
//   warp 1      tcgen05.mma issuer (one elected lane), owns TMEM (two accumulator stages)
//   warps 2..5  GEMM epilogue: TMEM -> split-K partials / exit arg-max; then part of the glue group
//   warps 2..5, 7..10  glue group: the step's glue phases (QKV finalize, attention, add+norm, SwiGLU) spread
//               over all CTAs, each followed by the grid barrier that publishes the next op's operand
//
// Items are dealt round-robin to CTAs continuing across ops, so the per-op remainder rotates and
// every CTA streams the same bytes per round to within one item.  The K split is fixed per
// operator shape and partials are added in split order: a row's bits do not depend on which rows
// or stages share the round (H3).
#include "round_dev.cuh"

namespace dexk {

// ---------------------------------------------------------------- the kernel
template <int kMaxThreads, bool PT>
__global__ void __launch_bounds__(kMaxThreads, 1) k_round(const __grid_constant__ TmSet tm, const __grid_constant__ RoundArgs a) {
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
  __shared__ int s_live_ms;
  __shared__ int s_cum[kMaxGrp + 1];
  __shared__ int s_steps;
  __shared__ unsigned s_seen;
  __shared__ RowLite s_row[kRowCache];   // per-row record of the glue units (round_dev.cuh)
  __shared__ SeqState s_seq[8];          // the round's FSM snapshot (attention tasks read it instead of global memory)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x < 32) s_valid[threadIdx.x] = 0;
  if (threadIdx.x >= 32 && threadIdx.x < 40) {
    const int s_ = threadIdx.x - 32;
    SeqState z;
    z.active = 0; z.q = 0; z.ctx_len = 0; z.n_tok = 0; z.last_tok = 0; z.pending = 0; z.done = 1; z.pad = 0;
    s_seq[s_] = s_ < D.max_seqs ? D.seqs[s_] : z;
  }
  __syncthreads();
  for (int r = threadIdx.x; r < D.R_cap; r += blockDim.x) {
    const RowInfo ri = D.rows[r];
    if (ri.valid) atomicOr(&s_valid[r >> 5], 1u << (r & 31));
    if (r < kRowCache) s_row[r] = row_lite_of(ri);
  }
  const RowLite* const rc = D.R_cap <= kRowCache ? s_row : nullptr;
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
    int lm = 0;
    for (int s = 0; s < D.max_seqs; ++s) {                   // live (stage, sequence[, 16-pair pass]) attention families
      const SeqState st = D.seqs[s];
      if (!r_seq_live(st)) continue;
      if constexpr (PT) {
        for (int m = 0; m <= min(st.q, D.N - 1); ++m) lm += (r_stage_count(st.q, m) * (D.nh / D.nkv) + 15) / 16;
      } else {
        lm += min(st.q, D.N - 1) + 1;
      }
    }
    s_live_ms = lm;
    if constexpr (PT) {
      s_cum[0] = 0;
      for (int m = 0; m < kMaxGrp; ++m)
        s_cum[m + 1] = s_cum[m] + (m < D.N ? D.max_seqs * ((cap_of(D.N, m) * (D.nh / D.nkv) + 15) / 16) : 0);
    }
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
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, 2 * a.acc_cols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t lo_off = (!a.stacked && D.planes == 2) ? (uint32_t)a.x_cap : 0u;   // lo-plane accumulator columns (gemm_dev.cuh)

  Seq sq;
  sq.a = &a; sq.s_nb = s_nb; sq.n_steps = s_steps; sq.n_ad_ops = (D.ad_m > 0 && D.N >= 2) ? 2 : 0;
  sq.n_ops = 4 * s_steps + sq.n_ad_ops + 1; sq.G = gridDim.x; sq.cta = blockIdx.x;
  const unsigned G = gridDim.x;

  if (s_steps > 0) {
    // The three single-issuer roles run warp-uniformly (all lanes walk the item list) and elect one lane
    // only around the TMA / MMA instructions, so those are issued from converged code.
    if (warp == 0) {
      // ===================== weight producer: always as far ahead as the ring allows =====================
      Walker w;
      unsigned st = 0, ph = 0;
      bool wrapped = false;
      for (w.start(sq); w.valid; w.next(sq)) {
        const CUtensorMap* desc = &tm.w[w.o.which];
        const uint32_t tx = kABytes + D.planes * w.it.nb * 128;
        const int c1 = w.it.tile * kTileM, c2 = w.it.layer;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          if (wrapped) mbar_wait(&empty[st], ph ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(&full[st], tx);
            tma_load_3d(smem + (size_t)st * stage_bytes, desc, &full[st], kb * kTileK, c1, c2, kEvictFirst);
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
        const unsigned need = sq.dep(w.t);
        if (seen < need) {
          unsigned spins = 0;
          while ((seen = *reinterpret_cast<volatile unsigned*>(&s_seen)) < need) {
            __nanosleep(32);
            if (++spins > 100000000u) __trap();
          }
          __threadfence_block();           // pairs with the cta-scope release before the flag store in grid_bar
          fence_proxy_async();
        }
        const int which = w.o.which;
        // operand of the op: act_a (qkv, gate/up, adapter W1), act_o (o), act_f (down, adapter W2), act_e (exit)
        const CUtensorMap* desc = &tm.x[(which == 0 || which == 2 || which == 5) ? 0 : (which == 1 ? 1 : (which == 4 ? 3 : 2))];
        const int row0 = w.it.row0, nb = w.it.nb;
        for (int kb = w.it.kb0; kb < w.it.kb1; ++kb) {
          // slot free (its previous tile consumed) => full[st] is in this tile's phase; the bytes may
          // land before the weight producer arms the phase (tx-count goes negative, arrival still pending)
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
            mma_stage(smem_u32(smem + (size_t)st * stage_bytes), plane_bytes, D.planes, stacked, d_tmem, lo_off, idesc, acc);
            umma_commit(&empty[st]);     // frees the ring slot when these MMAs have read it
          }
          __syncwarp();
          acc = 1;
          if (++st == (unsigned)NS) { st = 0; ph ^= 1u; }
        }
        if (elect_one()) umma_commit(&tfull[as]);   // accumulator complete -> epilogue
        __syncwarp();
      }
    } else {
      // ===================== glue group (12 warps): GEMM epilogues (warps 2-5) + glue + grid barriers =====================
      const int we = warp < 6 ? warp - 2 : warp - 3;        // 0 .. glue warps - 1
      const int tid_e = we * 32 + lane;
      constexpr int GT = kMaxThreads - 96, kGlueWarps = GT / 32;   // glue threads / warps
      const int quarter = warp & 3;
      const int gw = blockIdx.x * kGlueWarps + we, n_gw = gridDim.x * kGlueWarps;
      EpiCtx ec;
      ec.rows = D.rows; ec.s_valid = s_valid; ec.part = D.part; ec.vocab = D.vocab; ec.best_key = D.best_key;
      ec.ref_tile = D.ref_tile; ec.ref_tiles = D.ref_tiles; ec.dev = &D; ec.exit_map = D.exit_map;
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
        const int which = sq.which_of(t);
        const OpDesc& od = a.op[which];
        ec.mode = which == 4 ? 1 : 0;
        ec.part_ld = od.part_ld; ec.split_stride = od.split_stride; ec.out_dim = od.out_dim;
        if (we >= 4) return;                                 // TMEM lane quarters belong to warps 2-5
        for (; w.valid && w.t == t; w.next(sq), ++n_it) {
          const int as = n_it & 1;
          mbar_wait(&tfull[as], (n_it >> 1) & 1);
          tc_fence_after();
          const uint32_t t_addr = tmem_base + as * a.acc_cols + ((uint32_t)(quarter * 32) << 16);
          epilogue_item(ec, t_addr, a.stacked != 0, lo_off, w.it.nb, w.it.row0, w.it.row_end, w.it.tile, w.it.tile * kTileM, w.it.split, quarter, lane);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty[as]);
        }
      };
      for (int j = 0; j < sq.n_steps; ++j) {
        run_items(4 * j); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        if (D.hd == 128) glue_qkv_finalize<128>(a, j, gw, n_gw, lane, rc); else glue_qkv_finalize<64>(a, j, gw, n_gw, lane, rc);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        {
          void* asm_ = smem + a.attn_smem_off;
          if (D.hd == 128) glue_attention<128, GT, PT>(a, j, tid_e, lane, we, blockIdx.x, G, reinterpret_cast<AttnSmem<128>*>(asm_), s_live_ms, s_cum, s_seq);
          else glue_attention<64, GT, PT>(a, j, tid_e, lane, we, blockIdx.x, G, reinterpret_cast<AttnSmem<64>*>(asm_), s_live_ms, s_cum, s_seq);
        }
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        run_items(4 * j + 1); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        glue_add_norm(a, j, 0, a.op[1], gw, n_gw, lane, rc);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        run_items(4 * j + 2); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        glue_silu(a, j, a.op[2], gw, n_gw, lane);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        run_items(4 * j + 3); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        glue_add_norm(a, j, 1, a.op[3], gw, n_gw, lane, rc);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
      }
      int t_exit = 4 * sq.n_steps;
      if (sq.n_ad_ops) {                                     // inducing adapters of the non-final exits
        run_items(t_exit); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        glue_ad1(a, a.op[5], gw, n_gw, lane);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        run_items(t_exit + 1); stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        glue_ad2(a, a.op[6], gw, n_gw, lane);
        stamp();
        ++gb; grid_bar<GT>(D.gbar, gb * G, tid_e, &s_seen, gb); stamp();
        t_exit += 2;
      }
      run_items(t_exit); stamp();
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 2 * a.acc_cols);
}

size_t round_attn_smem(int hd) { return hd == 128 ? sizeof(AttnSmem<128>) : sizeof(AttnSmem<64>); }

cudaError_t round_init() {
  cudaError_t e = cudaFuncSetAttribute(k_round<kRoundThreads, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 222 * 1024);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_round<kRoundThreads, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 222 * 1024);
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
  // pass tasks only where a (stage, sequence) can hold more than one 16-pair pass
  if (cap_of(a.D.N, 0) * (a.D.nh / a.D.nkv) > kAttnPairs) return cudaLaunchKernelEx(&cfg, k_round<kRoundThreads, true>, tm, a);
  return cudaLaunchKernelEx(&cfg, k_round<kRoundThreads, false>, tm, a);
}

}  // namespace dexk
