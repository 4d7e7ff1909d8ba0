// uts_common.cu — status handling, config validation, rho_max table, pixel-centre export and the FoV-mask builder.
#include "uts_internal.cuh"
#include <atomic>
#include <mutex>

namespace uts {

static std::atomic<int> g_last_cuda_error{0};
void set_last_cuda_error(cudaError_t e) { g_last_cuda_error.store((int)e); }
static std::atomic<unsigned long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

// One context per device, created under a table lock on first use and never destroyed (the streams and events live as long as
// the process; include/uts.h "Library state").
DeviceCtx* device_ctx() {
  constexpr int kMaxDevices = 64;
  static DeviceCtx* table[kMaxDevices] = {};
  static std::mutex table_mu;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) { set_last_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidDevice); return nullptr; }
  std::lock_guard<std::mutex> lock(table_mu);
  if (table[dev]) return table[dev];
  DeviceCtx* c = new DeviceCtx();
  c->device = dev;
  if (cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || c->sms <= 0) c->sms = 148;
  bool ok = true;
  for (int i = 0; i < 2 && ok; ++i)
    ok = cudaStreamCreateWithFlags(&c->aux[i], cudaStreamNonBlocking) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->join[i], cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&c->copy, cudaStreamNonBlocking) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->side_fork, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->side_join, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->side_mid, cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; i < 4 && ok; ++i) ok = cudaEventCreateWithFlags(&c->ev[i], cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaHostAlloc(reinterpret_cast<void**>(&c->pin), 64, cudaHostAllocDefault) == cudaSuccess;
  if (!ok) { set_last_cuda_error(cudaGetLastError()); delete c; return nullptr; }
  table[dev] = c;
  return c;
}

int sm_count() {
  DeviceCtx* c = device_ctx();
  return c ? c->sms : 148;
}

int check_config(const uts_config* c) {
  if (!c) return UTS_ERR_INVALID_ARG;
  if (c->tile_log2 != kTileLog2) return UTS_ERR_UNSUPPORTED;
  if (c->order < c->tile_log2 || c->order > kMaxOrder) return UTS_ERR_INVALID_ARG;
  if (c->query_refine_log2 < 0 || c->query_refine_log2 > c->tile_log2) return UTS_ERR_INVALID_ARG;
  if (c->sh_degree < 0 || c->sh_degree > 3) return UTS_ERR_INVALID_ARG;
  if (c->query_mode != UTS_QUERY_NESTED && c->query_mode != UTS_QUERY_RING) return UTS_ERR_INVALID_ARG;
  if (c->n_gauss < 0 || c->n_views < 1) return UTS_ERR_INVALID_ARG;
  if ((int64_t)c->n_gauss * c->n_views > (int64_t)0x7fffffff) return UTS_ERR_UNSUPPORTED;
  if ((((int64_t)12 << (2 * (c->order - c->tile_log2))) * c->n_views) > (int64_t)0xffffffffll) return UTS_ERR_UNSUPPORTED;
  if (!(c->alpha_min >= 0.f) || !(c->alpha_max <= 1.f) || !(c->t_eps >= 0.f) || !(c->cov_dilation_px2 >= 0.f))
    return UTS_ERR_INVALID_ARG;
  if (!(c->alpha_min <= c->alpha_max) || !isfinite(c->r_near)) return UTS_ERR_INVALID_ARG;
  for (int i = 0; i < 3; ++i) if (!isfinite(c->bg[i])) return UTS_ERR_INVALID_ARG;
  return UTS_OK;
}

int check_mask(const uts_config* c, const uts_mask& m) {
  const bool none = !m.active_tiles && !m.slot_of_tile && !m.pixel_mask_bits;
  if (none) return (m.n_active == -1 || m.n_active == 0) ? UTS_OK : UTS_ERR_INVALID_ARG;
  if (!m.active_tiles || !m.slot_of_tile || !m.pixel_mask_bits) return UTS_ERR_INVALID_ARG;
  const int64_t nt = (int64_t)12 << (2 * (c->order - c->tile_log2));
  if (m.n_active < 0 || m.n_active > nt) return UTS_ERR_INVALID_ARG;
  return UTS_OK;
}

// rho_max(o): the largest angle between an order-o pixel centre and one of its own corners (Alg.2's PixRad, reading A6).
// It is attained by the pixel of the first equatorial ring next to a face's northern corner: centre (z = 2/3,
// lambda = pi/(4N)), corner on the face boundary meridian lambda = 0 at 1 - z = (1 - 1/N)^2 / 3.  Angle from the chord.
static void fill_rho_max(double* t) {
  for (int o = 0; o <= kMaxOrder; ++o) {
    const double N = (double)((int64_t)1 << o);
    const double zc = 2.0 / 3.0, sc = sqrt(1.0 - zc * zc), lc = kPi / (4.0 * N);
    const double w = (1.0 - 1.0 / N) * (1.0 - 1.0 / N) / 3.0;
    const double zk = 1.0 - w, sk = sqrt(w * (2.0 - w));
    const double dx = sc * cos(lc) - sk, dy = sc * sin(lc), dz = zc - zk;
    t[o] = 2.0 * asin(0.5 * sqrt(dx * dx + dy * dy + dz * dz));
  }
}
const double* rho_max_table_host() {
  static double table[kMaxOrder + 1];
  static std::once_flag once;
  std::call_once(once, [] { fill_rho_max(table); });
  return table;
}

// ------------------------------------------------------------------------------------------- kernels
__global__ void pixel_centers_kernel(int order, uint64_t first, uint64_t n, double* __restrict__ out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double x, y, z;
  pix_center_cam(order, first + i, x, y, z);
  out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}

struct MaskParams { int kind; double p[11]; double cos_half; };

// One thread per 32-pixel word of the bitmap; one block of 256 threads covers 8192 pixels = 32 tiles.
__global__ void mask_bits_kernel(int order, MaskParams mp, uint32_t* __restrict__ bits, uint64_t n_words) {
  uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_words) return;
  uint32_t word = 0;
  for (int b = 0; b < 32; ++b) {
    double vx, vy, vz;
    pix_center_cam(order, w * 32 + b, vx, vy, vz);
    bool on;
    if (mp.kind == 0) {
      on = (vx * mp.p[0] + vy * mp.p[1] + vz * mp.p[2]) >= mp.cos_half;
    } else {
      const double x = vx * mp.p[0] + vy * mp.p[1] + vz * mp.p[2];
      const double y = vx * mp.p[3] + vy * mp.p[4] + vz * mp.p[5];
      const double z = vx * mp.p[6] + vy * mp.p[7] + vz * mp.p[8];
      on = z > 0 && fabs(x) <= mp.p[9] * z && fabs(y) <= mp.p[10] * z;
    }
    if (on) word |= 1u << b;
  }
  bits[w] = word;
}

// Tile active <=> any of its 256 pixels visible (reading A19).  Ascending compaction with a single block so that the
// slot order is the tile order; N_tile <= 805 306 368 / 256, this is not on the per-frame path.
__global__ void mask_tiles_kernel(const uint32_t* __restrict__ bits, int64_t n_tile, int32_t* __restrict__ slot_of_tile,
                                  uint32_t* __restrict__ active_tiles, int* __restrict__ n_active_out) {
  __shared__ int warp_sums[32];
  __shared__ int base;
  if (threadIdx.x == 0) base = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int64_t t0 = 0; t0 < n_tile; t0 += blockDim.x) {
    const int64_t t = t0 + threadIdx.x;
    int on = 0;
    if (t < n_tile) {
      uint32_t acc = 0;
      const uint4* w = reinterpret_cast<const uint4*>(bits + t * 8);
      uint4 a = w[0], b = w[1];
      acc = a.x | a.y | a.z | a.w | b.x | b.y | b.z | b.w;
      on = acc != 0;
    }
    const unsigned ball = __ballot_sync(0xffffffffu, on);
    if (lane == 0) warp_sums[wid] = __popc(ball);
    __syncthreads();
    int before = base;
    for (int w2 = 0; w2 < wid; ++w2) before += warp_sums[w2];
    const int my = before + __popc(ball & ((1u << lane) - 1));
    if (t < n_tile) {
      slot_of_tile[t] = on ? my : -1;
      if (on) active_tiles[my] = (uint32_t)t;
    }
    __syncthreads();
    if (threadIdx.x == 0) { int s = 0; for (int w2 = 0; w2 < nw; ++w2) s += warp_sums[w2]; base += s; }
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_active_out = base;
}

// active-tile list and slot table of a pixel bitmap (shared by uts_build_mask and uts_build_camera_mask); synchronises s
int build_mask_tiles(const Dims& d, uint32_t* pixel_mask_bits, int32_t* slot_of_tile, uint32_t* active_tiles, int* h_n_active, cudaStream_t s) {
  int* d_count = reinterpret_cast<int*>(active_tiles + d.n_tile);     // entry N_tile of the caller's buffer receives n_active
  mask_tiles_kernel<<<1, 1024, 0, s>>>(pixel_mask_bits, d.n_tile, slot_of_tile, active_tiles, d_count);
  UTS_LAUNCH_CHECK();
  UTS_CUDA(cudaMemcpyAsync(h_n_active, d_count, sizeof(int), cudaMemcpyDeviceToHost, s));
  UTS_CUDA(cudaStreamSynchronize(s));
  return UTS_OK;
}

}  // namespace uts

using namespace uts;

extern "C" {

int uts_last_cuda_error(void) { return g_last_cuda_error.load(); }
uint64_t uts_launch_count(void) { return (uint64_t)g_launches.load(); }

const char* uts_strerror(int s) {
  switch (s) {
    case UTS_OK: return "ok";
    case UTS_ERR_INVALID_ARG: return "invalid argument";
    case UTS_ERR_CAPACITY: return "caller buffer too small";
    case UTS_ERR_CUDA: return "CUDA runtime error (see uts_last_cuda_error)";
    case UTS_ERR_UNSUPPORTED: return "unsupported device or configuration";
    default: return "unknown status";
  }
}

const char* uts_version(void) { return "uts 0.1 (sm_100a)"; }

int uts_rho_max_table(double* h_out14) {
  if (!h_out14) return UTS_ERR_INVALID_ARG;
  const double* t = rho_max_table_host();
  for (int o = 0; o <= kMaxOrder; ++o) h_out14[o] = t[o];
  return UTS_OK;
}

int uts_pixel_centers(int order, uint64_t first, uint64_t n, double* out_xyz, void* stream) {
  if (order < 0 || order > kMaxOrder || !out_xyz) return UTS_ERR_INVALID_ARG;
  if (first + n > ((uint64_t)12 << (2 * order))) return UTS_ERR_INVALID_ARG;
  if (n == 0) return UTS_OK;
  pixel_centers_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(order, first, n, out_xyz);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_build_mask(const uts_config* cfg, int kind, const double* h_params, uint32_t* pixel_mask_bits,
                   int32_t* slot_of_tile, uint32_t* active_tiles, int* h_n_active, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((kind != 0 && kind != 1) || !h_params || !pixel_mask_bits || !slot_of_tile || !active_tiles || !h_n_active)
    return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, nullptr);
  MaskParams mp; mp.kind = kind;
  const int np = kind == 0 ? 4 : 11;
  for (int i = 0; i < 11; ++i) mp.p[i] = i < np ? h_params[i] : 0.0;
  mp.cos_half = kind == 0 ? cos(h_params[3]) : 0.0;
  cudaStream_t s = (cudaStream_t)stream;
  const uint64_t n_words = (uint64_t)d.n_pix / 32;
  mask_bits_kernel<<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(d.k, mp, pixel_mask_bits, n_words);
  UTS_LAUNCH_CHECK();
  return build_mask_tiles(d, pixel_mask_bits, slot_of_tile, active_tiles, h_n_active, s);
}

}  // extern "C"
