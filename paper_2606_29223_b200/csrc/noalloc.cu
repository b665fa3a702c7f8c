// noalloc.cu — dex_gemm_noalloc: the weight-streaming GEMM (k_gemm, gemm.cu) through an entry point that allocates
// NOTHING.  For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it) and have no dex context with its caller-allocated workspace at hand.
//
//   y[rows, out] (f32) = x[rows, k] (f32) . W[out, k]^T (bf16)
//
// k_gemm needs scratch: the bf16 hi / lo operand planes of x, the row table and group extent it reads, and the fp32
// split-K partials it writes.  Here all of that lives in ONE file-scope `static __device__` array of a fixed, stated
// size (kNaScratchBytes = 10 MiB + 8 KiB), which every GPU that loads the library holds until the process exits.  The
// kernel itself is the unchanged k_gemm (same tiles, same fixed K split, so the same bits as the context path); the
// variant is where its scratch comes from.
//
// Rules of the shared array
//   * In HOST code the array's name is a host-side stand-in, not a device address.  The address is taken once per
//     device, with that device current, by cudaGetSymbolAddress (na_device_state) and passed to the kernels / the
//     tensor map; device code in this file names the array directly.
//   * Every call shares the array and it keeps the last call's contents: the set-up kernel rewrites the whole row
//     table and ZEROES the operand rows between `rows` and the 16-row box boundary (they enter the MMA); partials are
//     only read where this call's epilogue wrote them.
//   * Calls that overlap on the GPU (two streams, two threads) RACE on the array.  Calls on one stream are ordered.
//   * Limits (DEX_ECAPACITY beyond them): rows <= 32, k <= 16384, out <= 262144,
//     ceil(k / 512) * round16(rows) * round4(out) <= 2 Mi partial floats.
#include <cstdio>
#include <cstring>
#include <mutex>

#include "common.cuh"

namespace dexk {
cudaError_t gemm_init();
cudaError_t launch_gemm(const CUtensorMap&, const CUtensorMap&, const GemmArgs&, int, size_t, cudaStream_t);
void set_global_error(const char* msg);          // api.cu: the string dex_last_error(NULL) returns
}  // namespace dexk

using namespace dexk;

namespace {

constexpr int kNaMaxRows = 32;                    // stacked rows per call
constexpr int kNaMaxK = 16384;                    // reduction dimension
constexpr int kNaMaxOut = 262144;
constexpr size_t kNaMaxPartFloats = (size_t)2 << 20;            // 8 MiB of split-K partials
constexpr int kNaKbPerSplit = 8;                  // the decode split of api.cu (split_fine): items of <= 8 K-blocks
// layout of the array (byte offsets)
constexpr size_t kNaOffRows = 0;                                 // RowInfo[32]
constexpr size_t kNaOffNb = kNaOffRows + sizeof(RowInfo) * kNaMaxRows;   // int[kMaxGrp] (+ pad to 8 KiB)
constexpr size_t kNaOffPlanes = 8192;                            // bf16 [2][round16(rows)][k]
constexpr size_t kNaPlaneBytes = (size_t)2 * kNaMaxRows * kNaMaxK * 2;   // 2 MiB
constexpr size_t kNaOffPart = kNaOffPlanes + kNaPlaneBytes;      // f32 [ksplit][round16(rows)][round4(out)]
constexpr size_t kNaScratchBytes = kNaOffPart + kNaMaxPartFloats * sizeof(float);   // 10 MiB + 8 KiB
static_assert(kNaOffNb + sizeof(int) * kMaxGrp <= kNaOffPlanes, "row table and extents fit the first 8 KiB");

static __device__ __align__(256) unsigned char g_na_scratch[kNaScratchBytes];

// Row table, group extent and operand planes of this call.  Device code: names the array directly.
__global__ void k_na_setup(const float* __restrict__ x, int rows, int x_cap, int k_dim, int planes) {
  RowInfo* rt = reinterpret_cast<RowInfo*>(g_na_scratch + kNaOffRows);
  int* nb = reinterpret_cast<int*>(g_na_scratch + kNaOffNb);
  __nv_bfloat16* pl = reinterpret_cast<__nv_bfloat16*>(g_na_scratch + kNaOffPlanes);
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (size_t)gridDim.x * blockDim.x;
  if (tid < (size_t)kNaMaxRows) {
    RowInfo ri;
    ri.valid = (int)tid < rows;
    ri.seq = 0; ri.node = -1; ri.pos = 0; ri.grp = 0; ri.slot = -1; ri.n_paged = 0; ri.n_anc = 0;
    ri.parent_row = -1; ri.tok_in = 0; ri.is_ref = 0; ri.n_mask = 0;
    for (int i = 0; i < kMaxAnc; ++i) ri.anc[i] = 0, ri.mask_tok[i] = -1;
    for (int i = 0; i < 4; ++i) ri.pad[i] = 0;
    rt[tid] = ri;
  }
  if (tid < (size_t)kMaxGrp) nb[tid] = tid == 0 ? x_cap : 0;
  const size_t n = (size_t)x_cap * k_dim, ps = n;             // plane stride in elements
  for (size_t i = tid; i < n; i += nthr) {
    const int r = (int)(i / k_dim);
    const float v = r < rows ? x[i] : 0.f;                   // rows up to the box boundary are cleared every call
    split_store(pl, ps, i, v, planes);
  }
}

// y = sum over the K splits, in split order (the fixed order of every consumer of split-K partials in this library).
__global__ void k_na_reduce(float* __restrict__ y, int rows, int out_dim, int part_ld, int ksplit, size_t split_stride) {
  const float* part = reinterpret_cast<const float*>(g_na_scratch + kNaOffPart);
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)rows * out_dim) return;
  const int r = (int)(i / out_dim), c = (int)(i % out_dim);
  float acc = 0.f;
  for (int s = 0; s < ksplit; ++s) acc += part[(size_t)s * split_stride + (size_t)r * part_ld + c];
  y[i] = acc;
}

}  // namespace

namespace {

typedef CUresult (*NaEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct NaDevice {            // per-device set-up, done once with that device current
  bool ready = false;
  unsigned char* scratch = nullptr;      // DEVICE address of g_na_scratch on this device
  int n_sms = 0;
  NaEncodeFn encode = nullptr;
};
constexpr int kNaMaxDevices = 64;
NaDevice g_na_dev[kNaMaxDevices];
std::mutex g_na_mutex;

int na_fail(int code, const char* fmt, long long a = 0, long long b = 0, long long c = 0) {
  char buf[320];
  snprintf(buf, sizeof buf, fmt, a, b, c);
  set_global_error(buf);
  return code;
}

// The array's device address on the CURRENT device.  No allocation: the array is part of the loaded module.
int na_device_state(NaDevice** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0) return na_fail(DEX_ECUDA, "dex_gemm_noalloc: no CUDA device (there is no CPU fallback)");
  if (dev >= kNaMaxDevices) return na_fail(DEX_ECAPACITY, "dex_gemm_noalloc: device index %lld beyond %lld", dev, kNaMaxDevices);
  std::lock_guard<std::mutex> lock(g_na_mutex);
  NaDevice& d = g_na_dev[dev];
  if (!d.ready) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_na_scratch);            // host code must NOT pass g_na_scratch itself to a kernel
    if (e != cudaSuccess || !ptr) {
      char buf[256];
      snprintf(buf, sizeof buf, "dex_gemm_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
      set_global_error(buf);
      return DEX_ECUDA;
    }
    if (cudaDeviceGetAttribute(&d.n_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || d.n_sms < 1)
      return na_fail(DEX_ECUDA, "dex_gemm_noalloc: cannot read the SM count");
    void* fnp = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fnp, cudaEnableDefault, &qres) != cudaSuccess || !fnp)
      return na_fail(DEX_ECUDA, "dex_gemm_noalloc: cuTensorMapEncodeTiled entry point not found");
    if (gemm_init() != cudaSuccess)
      return na_fail(DEX_ECUDA, "dex_gemm_noalloc: cannot raise the GEMM kernel's dynamic shared memory limit");
    d.scratch = static_cast<unsigned char*>(ptr);
    d.encode = reinterpret_cast<NaEncodeFn>(fnp);
    d.ready = true;
  }
  *out = &d;
  return DEX_OK;
}

bool na_encode(NaEncodeFn fn, CUtensorMap* tm, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint32_t box1, uint32_t box2) {
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
  cuuint32_t box[3] = {(cuuint32_t)kTileK, box1, box2};
  cuuint32_t es[3] = {1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

extern "C" int32_t dex_gemm_noalloc(const void* w_dev, const float* x_dev, int32_t rows, int32_t out_dim, int32_t k_dim,
                                    int32_t act_planes, float* y_dev, void* cuda_stream) {
  if (!w_dev || !x_dev || !y_dev) return na_fail(DEX_EINVAL, "dex_gemm_noalloc: null pointer");
  if ((reinterpret_cast<uintptr_t>(w_dev) & 15) || (reinterpret_cast<uintptr_t>(x_dev) & 3) || (reinterpret_cast<uintptr_t>(y_dev) & 3))
    return na_fail(DEX_EINVAL, "dex_gemm_noalloc: w must be 16-byte aligned, x and y 4-byte aligned");
  if (rows < 1 || out_dim < 1 || k_dim < 8 || k_dim % 8)
    return na_fail(DEX_EINVAL, "dex_gemm_noalloc: need rows >= 1, out >= 1, k a positive multiple of 8 (got %lld, %lld, %lld)", rows, out_dim, k_dim);
  if (act_planes != 1 && act_planes != 2) return na_fail(DEX_EINVAL, "dex_gemm_noalloc: act_planes must be 1 or 2");
  if (rows > kNaMaxRows || k_dim > kNaMaxK || out_dim > kNaMaxOut)
    return na_fail(DEX_ECAPACITY, "dex_gemm_noalloc: rows %lld / k %lld / out %lld exceed the static scratch's maximum (32 rows, k 16384, out 262144)",
                   rows, k_dim, out_dim);
  const int x_cap = (rows + 15) & ~15;
  const int kb_total = (k_dim + kTileK - 1) / kTileK;
  const int kbps = kb_total < kNaKbPerSplit ? kb_total : kNaKbPerSplit;
  const int ksplit = (kb_total + kbps - 1) / kbps;
  const int part_ld = (out_dim + 3) & ~3;
  const size_t split_stride = (size_t)x_cap * part_ld;
  if ((size_t)ksplit * split_stride > kNaMaxPartFloats)
    return na_fail(DEX_ECAPACITY, "dex_gemm_noalloc: %lld split-K partial floats exceed the static scratch's %lld (ceil(k/512) * round16(rows) * round4(out))",
                   (long long)((size_t)ksplit * split_stride), (long long)kNaMaxPartFloats);
  NaDevice* d = nullptr;
  int rc = na_device_state(&d);
  if (rc) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

  // ring / TMEM geometry of one group of x_cap rows: the rules of api.cu's make_ring
  const size_t stage = 16384 + (size_t)act_planes * x_cap * 128;
  size_t n_stages = (200 * 1024) / stage;
  n_stages = n_stages < 2 ? 2 : (n_stages > 12 ? 12 : n_stages);
  const int stacked = (act_planes == 2 && 2 * x_cap <= 256) ? 1 : 0;
  int acc_cols = 32;
  while (acc_cols < act_planes * x_cap) acc_cols *= 2;

  CUtensorMap tmW, tmX;
  if (!na_encode(d->encode, &tmW, w_dev, (uint64_t)k_dim, (uint64_t)out_dim, 1, kTileM, 1) ||
      !na_encode(d->encode, &tmX, d->scratch + kNaOffPlanes, (uint64_t)k_dim, (uint64_t)x_cap, (uint64_t)act_planes, kBoxRows, stacked ? 2 : 1))
    return na_fail(DEX_ECUDA, "dex_gemm_noalloc: cuTensorMapEncodeTiled failed");

  GemmArgs a;
  memset(&a, 0, sizeof a);
  a.plan.n_grp = 1;
  a.plan.row_base[0] = 0; a.plan.rows_cap[0] = x_cap; a.plan.layer_lo[0] = 0; a.plan.layer_len[0] = 1;
  a.step = 0;
  a.out_dim = out_dim; a.k_dim = k_dim;
  a.n_tiles = (out_dim + kTileM - 1) / kTileM;
  a.ksplit = ksplit; a.kb_per_split = kbps; a.kb_total = kb_total;
  a.planes = act_planes; a.mode = 0;
  a.x_cap = x_cap; a.n_stages = (int)n_stages; a.acc_cols = acc_cols; a.n_acc = 2 * acc_cols <= 512 ? 2 : 1; a.stacked = stacked;
  a.grp_nb = reinterpret_cast<const int*>(d->scratch + kNaOffNb);
  a.rows = reinterpret_cast<const RowInfo*>(d->scratch + kNaOffRows);
  a.n_rows = x_cap;
  a.part = reinterpret_cast<float*>(d->scratch + kNaOffPart);
  a.part_ld = part_ld; a.part_split_stride = split_stride;
  a.best_key = nullptr; a.ref_tile = nullptr; a.ref_tiles = 0; a.vocab = out_dim;

  const size_t n_el = (size_t)x_cap * k_dim;
  const int setup_blocks = (int)((n_el + 255) / 256 < 1184 ? (n_el + 255) / 256 : 1184);
  k_na_setup<<<setup_blocks, 256, 0, stream>>>(x_dev, rows, x_cap, k_dim, act_planes);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = launch_gemm(tmW, tmX, a, d->n_sms, n_stages * stage + 1024 + 512, stream);
  if (e == cudaSuccess) {
    const size_t n_out = (size_t)rows * out_dim;
    k_na_reduce<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(y_dev, rows, out_dim, part_ld, ksplit, split_stride);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    char buf[256];
    snprintf(buf, sizeof buf, "dex_gemm_noalloc: launch failed: %s", cudaGetErrorString(e));
    set_global_error(buf);
    return DEX_ECUDA;
  }
  return DEX_OK;                                             // enqueued on the caller's stream, not synchronised
}
