// gemm_dev.cuh — device pieces of the weight-streaming GEMM shared by the per-op kernel (k_gemm,
// gemm.cu) and the persistent round kernel (k_round, round.cu): the MMA issue of one pipeline
// stage and the epilogue of one work item (TMEM -> split-K partials, or the fused exit arg-max).
#pragma once
#include "common.cuh"
#include "ptx.cuh"

namespace dexk {

constexpr uint32_t kABytes = kTileM * kTileK * 2;  // 16 KiB weight tile per ring stage

struct EpiCtx {
  int mode;                // 0: split-K partials, 1: DECS-masked arg-max (Alg. 2 lines 1-9)
  const RowInfo* rows;
  const uint32_t* s_valid; // live-row bitmap in shared memory
  float* part;
  int part_ld;
  size_t split_stride;
  int out_dim, vocab;
  unsigned long long* best_key;
  float2* ref_tile;
  int ref_tiles;
  const Dev* dev;          // sampling mode only (k_round): deferred norm scale, temperature, seed
  const int* exit_map;     // mode 1: the operand rows are DENSE exit rows; exit_map[row] = lattice row (-1: none)
};

// One ring stage: (kTileK/16) MMAs of M=128, K=16 into d_tmem.  Activation planes (bf16 hi / lo, R23):
//   stacked   one TMA box {64 K, 16 rows, 2 planes} per 16 rows, so the stage's B tile is
//             [rows 0-15 hi | rows 0-15 lo | rows 16-31 hi | ...]: ONE B operand of N = 2*nb.  hi products of
//             row r accumulate in TMEM column 32*(r/16) + r%16, lo products 16 columns further, the epilogue
//             adds the two.  Half the MMA and TMA instructions of the plane-by-plane form.
//   otherwise (2*nb > 256, or one plane): plane p at byte offset p*plane_bytes, N = nb; the lo plane accumulates in
//             columns of its own, lo_off columns after the hi plane's, and the epilogue adds the two - the SAME
//             arithmetic as the stacked form (sum of hi products + sum of lo products), so a row's bits do not depend
//             on which layout the context's row capacity selects (H3: a 256-row DEX context and its AR baseline).
__device__ __forceinline__ void mma_stage(uint32_t sA, uint32_t plane_bytes, int planes, bool stacked, uint32_t d_tmem,
                                          uint32_t lo_off, uint32_t idesc, uint32_t acc) {
  const uint32_t sB = sA + kABytes;
  const uint64_t da = make_sw128_kmajor_desc(sA);
  const int np = stacked ? 1 : planes;
  for (int p = 0; p < np; ++p) {
    const uint64_t db = make_sw128_kmajor_desc(sB + p * plane_bytes);
    uint32_t ac = acc;
#pragma unroll
    for (int k = 0; k < kTileK / 16; ++k) {
      umma_bf16(d_tmem + p * lo_off, da + (k * 32 >> 4), db + (k * 32 >> 4), idesc, ac);
      ac = 1;
    }
  }
}

// Epilogue of one item by one warp: TMEM lanes 32*quarter..+31 = out features tile*128 + 32*quarter + lane,
// TMEM columns 0..nb-1 = rows row0..row0+nb-1 (rows >= row_end belong to other groups: skipped).
// stacked: see mma_stage (hi at column 2*c0 + i, lo 16 columns further; added here).
// col0: out feature (partial column / vocabulary id) of TMEM lane 0; columns >= e.out_dim are not stored.
// lo_off > 0 (two planes, not stacked): the lo plane's sums sit lo_off columns after the hi plane's.
__device__ __forceinline__ void epilogue_item(const EpiCtx& e, uint32_t t_addr, bool stacked, uint32_t lo_off, int nb, int row0,
                                              int row_end, int tile, int col0, int split, int quarter, int lane) {
  const int col = col0 + quarter * 32 + lane;            // out feature / vocabulary id
  for (int c0 = 0; c0 < nb; c0 += 16) {
    if (row0 + c0 >= row_end) break;
    uint32_t v[16];
    tmem_ld16(t_addr + (stacked ? 2 * c0 : c0), v);
    if (stacked || lo_off) {
      uint32_t v2[16];
      tmem_ld16(stacked ? t_addr + 2 * c0 + 16 : t_addr + lo_off + c0, v2);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) + __uint_as_float(v2[i]));
    } else {
      tmem_ld_wait();
    }
    if (e.mode == 0) {
      float* dst = e.part + (size_t)split * e.split_stride + (size_t)(row0 + c0) * e.part_ld + col;
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const int rr = row0 + c0 + i;
        if (rr < row_end && ((e.s_valid[rr >> 5] >> (rr & 31)) & 1u) && col < e.out_dim)
          dst[(size_t)i * e.part_ld] = __uint_as_float(v[i]);
      }
    } else {
      // sampling mode (Alg. 2 line 13): the logit needs its deferred RMSNorm scale before the noise is added;
      // lane i computes the scale of row c0 + i once per block of 16 rows
      // the operand rows of the exit head are dense exit rows: lane i looks up the lattice row of row c0 + i
      int lr_lane = -1;
      if (lane < 16 && row0 + c0 + lane < row_end) lr_lane = e.exit_map[row0 + c0 + lane];
      float inv_lane = 1.f;
      const bool sampling = e.dev != nullptr && e.dev->sample;
      if (sampling && lr_lane >= 0) inv_lane = inv_rms(*e.dev, lr_lane) * e.dev->inv_tau;
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const int rr = __shfl_sync(0xffffffffu, lr_lane, i);
        const float inv_i = __shfl_sync(0xffffffffu, inv_lane, i);
        if (rr < 0) continue;                                                        // warp-uniform
        const RowInfo* ri = &e.rows[rr];
        float val = __uint_as_float(v[i]);
        if (sampling) val = val * inv_i + gumbel_noise(e.dev->sample_seed, ri->seq, ri->pos + 1, col);
        bool dead = col >= e.vocab;
        const int nm = ri->n_mask;                      // Alg. 2 lines 5-7: mask prior proposals
        for (int t = 0; t < nm; ++t) dead |= (ri->mask_tok[t] == col);
        uint32_t key = dead ? 0u : f2key(val);
        uint32_t best = __reduce_max_sync(0xffffffffu, key);
        uint32_t who = __ballot_sync(0xffffffffu, key == best);
        int wl = __ffs(who) - 1;                        // lowest lane = lowest token id (R11)
        if (best != 0u && lane == wl) {
          unsigned long long k64 = ((unsigned long long)best << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)col);
          atomicMax(&e.best_key[rr], k64);
        }
        if (ri->is_ref) {                               // top-2 of the reference node, for margin reporting
          uint32_t key2 = (lane == wl) ? 0u : key;
          uint32_t second = __reduce_max_sync(0xffffffffu, key2);
          if (lane == 0)
            e.ref_tile[(size_t)ri->seq * e.ref_tiles + tile * 4 + quarter] =
                make_float2(best ? key2f(best) : -INFINITY, second ? key2f(second) : -INFINITY);
        }
      }
    }
  }
}

}  // namespace dexk
