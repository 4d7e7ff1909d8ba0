// uts_sort.cu — F3: stable LSD radix sort of ((tile, rho), i) pairs (Alg.1 l.15 PAPER.md:560; radial-depth ordering
// PAPER.md:112; reading A9/A10) and F4: per-tile ranges (Alg.1 l.16 PAPER.md:561).
//
// Key = (view*N_tile + tile) << 32 | float_bits(rho); rho > 0 so the IEEE-754 pattern orders as an unsigned integer.
// 8-bit digits, least significant first; only the bytes that can differ are sorted: 4 depth bytes plus
// ceil(log2(V*N_tile)/8) tile bytes.  Each pass is reduce-then-scan (no inter-block spinning):
//   upsweep   : per-block digit histogram                              reads  8 B/pair
//   scan      : exclusive scan over [digit][block]                     ~1 KB per block
//   downsweep : stable in-block ranking (warp match), reorder in shared memory, scatter in digit runs
//                                                                      reads 12 B/pair, writes 12 B/pair
// Stability: inside a block keys are ranked in (warp, item, lane) order, which is their memory order; blocks are
// ordered by the scan.  So equal keys keep their emission order = ascending Gaussian id.
#include "uts_internal.cuh"
#include "uts_scan.cuh"

namespace uts {

constexpr int kSortThreads = 256;
#ifndef UTS_SORT_ITEMS
#define UTS_SORT_ITEMS 12
#endif
#ifndef UTS_SORT_MINB
#define UTS_SORT_MINB 4
#endif
constexpr int kSortItems = UTS_SORT_ITEMS;
constexpr int kSortTile = kSortThreads * kSortItems;     // 3072 pairs per block (47 KB of static shared memory)
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kRadix = 256;

__device__ __forceinline__ uint32_t digit_of(uint64_t key, int shift) { return (uint32_t)(key >> shift) & (kRadix - 1); }

// counts[digit * nb + block]
__global__ void __launch_bounds__(kSortThreads)
sort_upsweep(const uint64_t* __restrict__ keys, uint64_t n, int shift, uint32_t nb, uint32_t* __restrict__ counts) {
  __shared__ uint32_t hist[kSortWarps][kRadix];
  const int wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < kSortWarps * kRadix; i += kSortThreads) (&hist[0][0])[i] = 0;
  __syncthreads();
  const uint64_t base = (uint64_t)blockIdx.x * kSortTile;
#pragma unroll 4
  for (int j = 0; j < kSortItems; ++j) {
    const uint64_t idx = base + (uint64_t)j * kSortThreads + threadIdx.x;
    if (idx < n) atomicAdd(&hist[wid][digit_of(__ldg(keys + idx), shift)], 1u);
  }
  __syncthreads();
  for (int d = threadIdx.x; d < kRadix; d += kSortThreads) {
    uint32_t s = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) s += hist[w][d];
    counts[(uint64_t)d * nb + blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(kSortThreads, UTS_SORT_MINB)
sort_downsweep(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in, uint64_t* __restrict__ keys_out,
               uint32_t* __restrict__ vals_out, uint64_t n, int shift, uint32_t nb, const uint64_t* __restrict__ offsets) {
  __shared__ uint32_t whist[kSortWarps][kRadix];      // per-warp digit counts, then per-warp exclusive bases
  __shared__ uint32_t dstart[kRadix];                 // start of each digit's run inside the block
  __shared__ uint64_t gbase[kRadix];                  // global start of this block's run of each digit
  extern __shared__ uint64_t sort_dyn[];
  uint64_t* skeys = sort_dyn;                                            // [kSortTile]
  uint32_t* svals = reinterpret_cast<uint32_t*>(sort_dyn + kSortTile);   // [kSortTile]
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  for (int i = threadIdx.x; i < kSortWarps * kRadix; i += kSortThreads) (&whist[0][0])[i] = 0;
  for (int d = threadIdx.x; d < kRadix; d += kSortThreads) gbase[d] = offsets[(uint64_t)d * nb + blockIdx.x];
  __syncthreads();

  // Memory order inside the block: warp-major, then item, then lane (each warp owns a contiguous 512-pair segment).
  const uint64_t wbase = (uint64_t)blockIdx.x * kSortTile + (uint64_t)wid * (32 * kSortItems);
  uint64_t key[kSortItems];
  uint16_t rank[kSortItems];
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const uint64_t idx = wbase + (uint64_t)j * 32 + lane;
    const bool ok = idx < n;
    key[j] = ok ? __ldg(keys_in + idx) : ~0ull;
  }
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const uint64_t idx = wbase + (uint64_t)j * 32 + lane;
    const bool ok = idx < n;
    const uint32_t d = digit_of(key[j], shift);
    const uint32_t peers = __match_any_sync(0xffffffffu, ok ? d : 0xffffffffu);
    const uint32_t before = whist[wid][d & (kRadix - 1)];
    rank[j] = (uint16_t)(before + __popc(peers & lt_mask));
    __syncwarp();
    if (ok && (peers & lt_mask) == 0) whist[wid][d] = before + __popc(peers);   // leader of each digit group
    __syncwarp();
  }
  __syncthreads();
  // per digit: exclusive scan over warps; block totals -> dstart
  uint32_t my_total = 0;
  if (threadIdx.x < kRadix) {
    const int d = threadIdx.x;
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) { const uint32_t c = whist[w][d]; whist[w][d] = run; run += c; }
    my_total = run;
  }
  {  // exclusive scan of the 256 digit totals (kSortThreads == kRadix)
    __shared__ uint32_t wsum[kSortWarps];
    uint32_t incl = my_total;
#pragma unroll
    for (int dlt = 1; dlt < 32; dlt <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, dlt); if (lane >= dlt) incl += y; }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    uint32_t before = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) if (w < wid) before += wsum[w];
    dstart[threadIdx.x] = before + incl - my_total;
  }
  __syncthreads();
  // reorder in shared memory so that each digit's keys are contiguous and in stable order
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const uint64_t idx = wbase + (uint64_t)j * 32 + lane;
    if (idx < n) {
      const uint32_t d = digit_of(key[j], shift);
      const uint32_t pos = dstart[d] + whist[wid][d] + rank[j];
      skeys[pos] = key[j]; svals[pos] = __ldg(vals_in + idx);      // values are fetched only now: 12 fewer live registers
    }
  }
  __syncthreads();
  const uint64_t tile_base = (uint64_t)blockIdx.x * kSortTile;
  const uint32_t cnt = (uint32_t)((n - tile_base) < (uint64_t)kSortTile ? (n - tile_base) : (uint64_t)kSortTile);
#pragma unroll 4
  for (int j = 0; j < kSortItems; ++j) {
    const uint32_t pos = j * kSortThreads + threadIdx.x;
    if (pos < cnt) {
      const uint64_t kk = skeys[pos];
      const uint32_t d = digit_of(kk, shift);
      const uint64_t dst = gbase[d] + (pos - dstart[d]);
      keys_out[dst] = kk; vals_out[dst] = svals[pos];
    }
  }
}

__global__ void copy_pairs(const uint64_t* __restrict__ ki, const uint32_t* __restrict__ vi, uint64_t* __restrict__ ko,
                           uint32_t* __restrict__ vo, uint64_t n) {
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    ko[i] = ki[i]; vo[i] = vi[i];
  }
}

// F4.  One thread per pair: a pair that differs from its predecessor in the (view,tile) field opens a range, one that
// differs from its successor closes it.  `ranges` is zeroed first so that empty tiles read (0,0).
__global__ void __launch_bounds__(256)
tile_ranges_kernel(const uint64_t* __restrict__ keys, uint64_t n, uint64_t* __restrict__ ranges) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const uint32_t id = (uint32_t)(__ldg(keys + j) >> 32);
  const uint32_t prev = j > 0 ? (uint32_t)(__ldg(keys + j - 1) >> 32) : ~id;
  const uint32_t next = j + 1 < n ? (uint32_t)(__ldg(keys + j + 1) >> 32) : ~id;
  if (prev != id) ranges[2 * (uint64_t)id] = j;
  if (next != id) ranges[2 * (uint64_t)id + 1] = j + 1;
}

// F4 for long lists: one thread per (view, tile) finds its range by two binary searches on the sorted keys' high words — 2 log2(n)
// reads per tile instead of one read per pair (config 4's 41 M small pairs over 49 152 tiles: 0.11 -> 0.02 ms).  Same output.
__global__ void __launch_bounds__(256)
tile_ranges_search_kernel(const uint64_t* __restrict__ keys, uint64_t n, uint64_t ids, uint64_t* __restrict__ ranges) {
  const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ids) return;
  auto lower = [&](uint64_t id) {                      // first j with high word >= id
    uint64_t lo = 0, hi = n;
    while (lo < hi) { const uint64_t mid = (lo + hi) >> 1; if ((__ldg(keys + mid) >> 32) < id) lo = mid + 1; else hi = mid; }
    return lo;
  };
  const uint64_t a = lower(t), b = lower(t + 1);
  if (b > a) { ranges[2 * t] = a; ranges[2 * t + 1] = b; }
}

static int tile_bits_of(const uts_config* cfg) {
  const uint64_t ids = ((uint64_t)12 << (2 * (cfg->order - cfg->tile_log2))) * (uint64_t)cfg->n_views;
  int b = 0;
  while (((uint64_t)1 << b) < ids) ++b;
  return b;
}

}  // namespace uts

using namespace uts;

extern "C" {

size_t uts_sort_scratch_bytes(uint64_t n_pairs) {
  const uint64_t nb = (n_pairs + kSortTile - 1) / kSortTile;
  const uint64_t m = nb * kRadix;                     // histogram entries
  return (size_t)(((m * 4 + 255) / 256) * 256 + ((m + 1) * 8 + 255) / 256 * 256) + scan_scratch_bytes((int64_t)m);
}

}  // extern "C"

namespace uts {
// LSD passes over key bytes [first_byte, first_byte + n_bytes); result left in keys/vals.
static int radix_sort_bytes(uint64_t n_pairs, uint64_t* keys, uint32_t* vals, uint64_t* keys_tmp, uint32_t* vals_tmp, void* scratch,
                            int first_byte, int n_bytes, cudaStream_t s) {
  const uint32_t nb = (uint32_t)((n_pairs + kSortTile - 1) / kSortTile);
  const uint64_t m = (uint64_t)nb * kRadix;
  char* sp = reinterpret_cast<char*>(scratch);
  uint32_t* counts = reinterpret_cast<uint32_t*>(sp);            sp += ((m * 4 + 255) / 256) * 256;
  uint64_t* offs = reinterpret_cast<uint64_t*>(sp);              sp += (((m + 1) * 8 + 255) / 256) * 256;
  uint64_t* block_sums = reinterpret_cast<uint64_t*>(sp);
  uint64_t* kin = keys; uint32_t* vin = vals; uint64_t* kout = keys_tmp; uint32_t* vout = vals_tmp;
  DeviceCtx* ctx = device_ctx();
  if (!ctx) return UTS_ERR_CUDA;
  {
    std::lock_guard<std::recursive_mutex> lock(ctx->mu);
    if (!ctx->attrs_set[1]) {                                    // once per device
      UTS_CUDA(cudaFuncSetAttribute(sort_downsweep, cudaFuncAttributeMaxDynamicSharedMemorySize, kSortTile * 12));
      ctx->attrs_set[1] = true;
    }
  }
  for (int pass = 0; pass < n_bytes; ++pass) {
    const int shift = 8 * (first_byte + pass);
    sort_upsweep<<<nb, kSortThreads, 0, s>>>(kin, n_pairs, shift, nb, counts);
    UTS_LAUNCH_CHECK();
    int st = exclusive_scan_u32(counts, (int64_t)m, offs, block_sums, s);
    if (st) return st;
    sort_downsweep<<<nb, kSortThreads, kSortTile * 12, s>>>(kin, vin, kout, vout, n_pairs, shift, nb, offs);
    UTS_LAUNCH_CHECK();
    uint64_t* tk = kin; kin = kout; kout = tk;
    uint32_t* tv = vin; vin = vout; vout = tv;
  }
  if (kin != keys) {
    copy_pairs<<<ctx->sms * 8, 256, 0, s>>>(kin, vin, keys, vals, n_pairs);
    UTS_LAUNCH_CHECK();
  }
  return UTS_OK;
}

// keys[k] = (view << 32) | float_bits(rho[k]),  vals[k] = k
__global__ void depth_keys_kernel(const float* __restrict__ rho, int64_t n, int P, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  keys[k] = ((uint64_t)(k / P) << 32) | (uint64_t)__float_as_uint(__ldg(rho + k));
  vals[k] = (uint32_t)k;
}
__global__ void invert_kernel(const uint32_t* __restrict__ order, int64_t n, uint32_t* __restrict__ rank) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) rank[order[j]] = (uint32_t)j;
}
}  // namespace uts

extern "C" {

int uts_sort(const uts_config* cfg, uint64_t n_pairs, uint64_t* keys, uint32_t* vals, uint64_t* keys_tmp, uint32_t* vals_tmp,
             int depth_presorted, void* scratch, size_t scratch_bytes, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (n_pairs == 0) return UTS_OK;
  if (!keys || !vals || !keys_tmp || !vals_tmp || !scratch) return UTS_ERR_INVALID_ARG;
  if (scratch_bytes < uts_sort_scratch_bytes(n_pairs) || ((uintptr_t)scratch & 255)) return UTS_ERR_INVALID_ARG;
  if (n_pairs > ((uint64_t)1 << 40)) return UTS_ERR_UNSUPPORTED;
  const int tile_bytes = (tile_bits_of(cfg) + 7) / 8;
  // stable LSD: when the pairs already arrive in (view, depth, id) order only the (view, tile) bytes need sorting
  return depth_presorted ? radix_sort_bytes(n_pairs, keys, vals, keys_tmp, vals_tmp, scratch, 4, tile_bytes, (cudaStream_t)stream)
                         : radix_sort_bytes(n_pairs, keys, vals, keys_tmp, vals_tmp, scratch, 0, 4 + tile_bytes, (cudaStream_t)stream);
}

size_t uts_depth_order_scratch_bytes(const uts_config* cfg) {
  if (check_config(cfg) != UTS_OK) return 0;
  const uint64_t n = (uint64_t)cfg->n_gauss * cfg->n_views;
  return (size_t)(2 * ((n * 8 + 255) / 256 * 256) + 2 * ((n * 4 + 255) / 256 * 256)) + uts_sort_scratch_bytes(n) + 256;
}

int uts_depth_order(const uts_config* cfg, const float* rho, uint32_t* emit_rank, void* scratch, size_t scratch_bytes, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  const int64_t n = (int64_t)cfg->n_gauss * cfg->n_views;
  if (n == 0) return UTS_OK;
  if (!rho || !emit_rank || !scratch) return UTS_ERR_INVALID_ARG;
  if (scratch_bytes < uts_depth_order_scratch_bytes(cfg) || ((uintptr_t)scratch & 255)) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  char* sp = reinterpret_cast<char*>(scratch);
  const size_t kb = ((size_t)n * 8 + 255) / 256 * 256, vb = ((size_t)n * 4 + 255) / 256 * 256;
  uint64_t* keys = reinterpret_cast<uint64_t*>(sp); sp += kb;
  uint64_t* keys_tmp = reinterpret_cast<uint64_t*>(sp); sp += kb;
  uint32_t* vals = reinterpret_cast<uint32_t*>(sp); sp += vb;
  uint32_t* vals_tmp = reinterpret_cast<uint32_t*>(sp); sp += vb;
  depth_keys_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(rho, n, cfg->n_gauss, keys, vals);
  UTS_LAUNCH_CHECK();
  int view_bits = 0;
  while ((1 << view_bits) < cfg->n_views) ++view_bits;
  if ((st = radix_sort_bytes((uint64_t)n, keys, vals, keys_tmp, vals_tmp, sp, 0, 4 + (view_bits + 7) / 8, s))) return st;
  invert_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(vals, n, emit_rank);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_tile_ranges(const uts_config* cfg, uint64_t n_pairs, const uint64_t* keys, uint64_t* ranges, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (!ranges || (n_pairs && !keys)) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const uint64_t ids = ((uint64_t)12 << (2 * (cfg->order - cfg->tile_log2))) * (uint64_t)cfg->n_views;
  UTS_CUDA(cudaMemsetAsync(ranges, 0, ids * 2 * sizeof(uint64_t), s));
  if (n_pairs == 0) return UTS_OK;
  if (n_pairs >= 64 * ids) tile_ranges_search_kernel<<<(unsigned)((ids + 255) / 256), 256, 0, s>>>(keys, n_pairs, ids, ranges);
  else tile_ranges_kernel<<<(unsigned)((n_pairs + 255) / 256), 256, 0, s>>>(keys, n_pairs, ranges);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

// ------------------------------------------------------------------------------------- uts_depth_order without caller scratch
// For callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the scratch of
// uts_depth_order lives in a file-scope device array of the library, 7 MiB, enough for UTS_DEPTH_ORDER_STATIC_MAX (view, Gaussian)
// records; every GPU that loads the library holds it until the process exits.  In host code `g_depth_order_scratch` is only a
// stand-in for the symbol, NOT a device address: its device address is looked up once per device, with that device current, by
// cudaGetSymbolAddress (checked), and that pointer is what the kernels get.
}  // extern "C"

namespace uts {
constexpr size_t kDepthOrderStaticBytes = (size_t)7 << 20;
static __device__ __align__(256) unsigned char g_depth_order_scratch[kDepthOrderStaticBytes];

// device address of g_depth_order_scratch on the current device (looked up once per device), or nullptr (last CUDA error set)
static void* depth_order_static_scratch() {
  constexpr int kMaxDevices = 64;
  static void* table[kMaxDevices] = {};
  static std::mutex mu;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) { set_last_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidDevice); return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!table[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_depth_order_scratch);
    if (e != cudaSuccess || !ptr) { set_last_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidSymbol); return nullptr; }
    table[dev] = ptr;
  }
  return table[dev];
}
}  // namespace uts

extern "C" {

uint64_t uts_depth_order_static_max(void) { return (uint64_t)UTS_DEPTH_ORDER_STATIC_MAX; }

int uts_depth_order_static(const uts_config* cfg, const float* rho, uint32_t* emit_rank, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  const uint64_t n = (uint64_t)cfg->n_gauss * (uint64_t)cfg->n_views;
  // beyond the array: refused before anything is enqueued (UTS_ERR_CAPACITY; uts_depth_order_static_max() is the limit)
  if (n > (uint64_t)UTS_DEPTH_ORDER_STATIC_MAX || uts_depth_order_scratch_bytes(cfg) > kDepthOrderStaticBytes) return UTS_ERR_CAPACITY;
  if (n == 0) return UTS_OK;
  if (!rho || !emit_rank) return UTS_ERR_INVALID_ARG;
  void* scratch = depth_order_static_scratch();
  if (!scratch) return UTS_ERR_CUDA;
  // Nothing in the scratch has to start at zero: every region (keys, values, digit counts, scan sums) is written by a kernel of this
  // call before a later kernel of this call reads it, so the previous call's contents are never seen.
  return uts_depth_order(cfg, rho, emit_rank, scratch, kDepthOrderStaticBytes, stream);
}

}  // extern "C"
