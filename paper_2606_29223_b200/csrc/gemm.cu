// gemm.cu — the weight-streaming grouped GEMM of the DEX layer segment (north_star (a), (c)).
//
//   Y_g[rows_g, out] = X_g[rows_g, K] . W[layer_g][out, K]^T      for every live group g
//
// One persistent launch covers all live stages Pi_m of the round (every
// frontier node through its next stage) so each stage's weights leave HBM once for all of
// its stacked branch rows.  "Swap-AB": the weight tile is the MMA M operand (128 out rows),
// the <=256 stacked branch rows are the MMA N operand, accumulators live in TMEM.
//
//   warp 0      TMA producer: weight tile [128 x 64] + activation boxes [16 x 64] per plane
//   warp 1      tcgen05.mma issuer (one lane), owns the TMEM allocation
//   warps 2..5  epilogue: tcgen05.ld -> (mode 0) fp32 split-K partials to HBM/L2
//                                        (mode 1) masked arg-max over the vocabulary tile, packed
//                                                 (value, ~index) atomicMax - no logits to HBM
//
// Work item = (group, 128-row out tile, K split); item i of CTA b is b + i * gridDim.x.  The
// K split depends on the operator shape only, so a row's arithmetic never depends on how many
// rows or stages share the launch (H3: DEX stream == AR stream).
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_dev.cuh"

namespace dexk {

constexpr int kGemmThreads = 192;

struct Item {
  int g, tile, split, nb, layer, kb0, kb1;
};

__device__ __forceinline__ int build_live(const GemmArgs& a, int* live_g, int* live_nb) {
  int n = 0;
  for (int g = 0; g < a.plan.n_grp; ++g) {
    int nb = a.grp_nb[g];
    if (nb > 0 && a.step < a.plan.layer_len[g]) {
      live_g[n] = g;
      live_nb[n] = nb;
      ++n;
    }
  }
  return n;
}

__device__ __forceinline__ Item decode_item(const GemmArgs& a, int item, const int* live_g, const int* live_nb) {
  Item it;
  int per_grp = a.n_tiles * a.ksplit;
  int gi = item / per_grp;
  int rem = item - gi * per_grp;
  it.g = live_g[gi];
  it.nb = live_nb[gi];
  it.tile = rem / a.ksplit;
  it.split = rem - it.tile * a.ksplit;
  it.layer = a.plan.layer_lo[it.g] + a.step;
  it.kb0 = it.split * a.kb_per_split;
  it.kb1 = min(it.kb0 + a.kb_per_split, a.kb_total);
  return it;
}

__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmX, const GemmArgs a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t plane_bytes = a.x_cap * 128;
  const uint32_t stage_bytes = kABytes + a.planes * plane_bytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)a.n_stages * stage_bytes);
  uint64_t* full = bars;
  uint64_t* empty = bars + a.n_stages;
  uint64_t* tfull = bars + 2 * a.n_stages;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");

  __shared__ int live_g[kMaxGrp], live_nb[kMaxGrp];
  __shared__ int n_live_s;
  __shared__ uint32_t s_valid[32];                 // live-row bitmap (R_cap <= 1024)
  if (threadIdx.x < 32) s_valid[threadIdx.x] = 0;
  __syncthreads();
  for (int r = threadIdx.x; r < a.n_rows; r += kGemmThreads)
    if (a.rows[r].valid) atomicOr(&s_valid[r >> 5], 1u << (r & 31));
  if (threadIdx.x == 0) {
    n_live_s = build_live(a, live_g, live_nb);
    for (int i = 0; i < a.n_stages; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&tfull[i], 1);
      mbar_init(&tempty[i], 4);
    }
    fence_mbar_init();
    tma_prefetch_desc(&tmW);
    tma_prefetch_desc(&tmX);
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, a.n_acc * a.acc_cols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int n_items = n_live_s * a.n_tiles * a.ksplit;
  const uint32_t lo_off = (!a.stacked && a.planes == 2) ? (uint32_t)a.x_cap : 0u;   // lo-plane accumulator columns (gemm_dev.cuh)

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      // Weights do not depend on the preceding kernel: the first ring-full of weight tiles is
      // requested BEFORE waiting on the programmatic dependency, the activation boxes after it.
      int pre = 0;
      for (int item = blockIdx.x; item < n_items && pre < a.n_stages; item += gridDim.x) {
        Item it = decode_item(a, item, live_g, live_nb);
        const uint32_t tx = kABytes + a.planes * it.nb * 128;
        for (int kb = it.kb0; kb < it.kb1 && pre < a.n_stages; ++kb, ++pre) {
          mbar_expect_tx(&full[pre], tx);
          tma_load_3d(smem + (size_t)pre * stage_bytes, &tmW, &full[pre], kb * kTileK, it.tile * kTileM, it.layer, kEvictFirst);
        }
      }
      asm volatile("griddepcontrol.wait;\n" ::: "memory");
      int stage = 0, issued = 0;
      uint32_t phase = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        Item it = decode_item(a, item, live_g, live_nb);
        const int row0 = a.plan.row_base[it.g];
        const uint32_t tx = kABytes + a.planes * it.nb * 128;
        for (int kb = it.kb0; kb < it.kb1; ++kb, ++issued) {
          uint8_t* sA = smem + (size_t)stage * stage_bytes;
          uint8_t* sB = sA + kABytes;
          if (issued >= pre) {
            mbar_wait(&empty[stage], phase ^ 1);
            mbar_expect_tx(&full[stage], tx);
            tma_load_3d(sA, &tmW, &full[stage], kb * kTileK, it.tile * kTileM, it.layer, kEvictFirst);
          }
          if (a.stacked) {
            for (int r = 0; r < it.nb; r += kBoxRows)
              tma_load_3d(sB + r * 256, &tmX, &full[stage], kb * kTileK, row0 + r, 0, kEvictLast);
          } else {
            for (int p = 0; p < a.planes; ++p)
              for (int r = 0; r < it.nb; r += kBoxRows)
                tma_load_3d(sB + p * plane_bytes + r * 128, &tmX, &full[stage], kb * kTileK, row0 + r, p, kEvictLast);
          }
          if (++stage == a.n_stages) {
            stage = 0;
            phase ^= 1;
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int n_it = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++n_it) {
        Item it = decode_item(a, item, live_g, live_nb);
        const int as = n_it % a.n_acc;
        const uint32_t aphase = (n_it / a.n_acc) & 1;
        mbar_wait(&tempty[as], aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * a.acc_cols;
        const uint32_t idesc = make_idesc_bf16_m128(a.stacked ? 2 * it.nb : it.nb);
        uint32_t acc = 0;
        for (int kb = it.kb0; kb < it.kb1; ++kb) {
          mbar_wait(&full[stage], phase);
          tc_fence_after();
          mma_stage(smem_u32(smem + (size_t)stage * stage_bytes), plane_bytes, a.planes, a.stacked != 0, d_tmem, lo_off, idesc, acc);
          acc = 1;
          umma_commit(&empty[stage]);   // frees the ring slot when these MMAs have read it
          if (++stage == a.n_stages) {
            stage = 0;
            phase ^= 1;
          }
        }
        umma_commit(&tfull[as]);        // accumulator complete -> epilogue
      }
    }
    __syncwarp();
  } else {
    // ===================== epilogue (warps 2..5) =====================
    const int quarter = warp & 3;       // TMEM lanes 32*quarter .. +31 are this warp's
    EpiCtx ec;
    ec.mode = a.mode; ec.rows = a.rows; ec.s_valid = s_valid; ec.part = a.part; ec.part_ld = a.part_ld;
    ec.split_stride = a.part_split_stride; ec.out_dim = a.out_dim; ec.vocab = a.vocab; ec.best_key = a.best_key;
    ec.ref_tile = a.ref_tile; ec.ref_tiles = a.ref_tiles; ec.dev = nullptr; ec.exit_map = a.exit_map;
    int n_it = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++n_it) {
      Item it = decode_item(a, item, live_g, live_nb);
      const int as = n_it % a.n_acc;
      const uint32_t aphase = (n_it / a.n_acc) & 1;
      mbar_wait(&tfull[as], aphase);
      tc_fence_after();
      const uint32_t t_addr = tmem_base + as * a.acc_cols + ((uint32_t)(quarter * 32) << 16);
      const int row0 = a.plan.row_base[it.g];
      epilogue_item(ec, t_addr, a.stacked != 0, lo_off, it.nb, row0, row0 + a.plan.rows_cap[it.g], it.tile, it.tile * kTileM, it.split, quarter, lane);
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty[as]);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, a.n_acc * a.acc_cols);
}

cudaError_t gemm_init() {
  return cudaFuncSetAttribute(k_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, 216 * 1024);
}

// Host-side launcher (called from api.cu).
cudaError_t launch_gemm(const CUtensorMap& tmW, const CUtensorMap& tmX, const GemmArgs& a, int grid, size_t smem_bytes,
                        cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kGemmThreads);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_gemm, tmW, tmX, a);
}

}  // namespace dexk
