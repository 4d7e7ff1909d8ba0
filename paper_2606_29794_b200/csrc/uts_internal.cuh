// uts_internal.cuh — shared by the CUDA translation units of libuts.so (not part of the ABI).
// Holds: status / launch helpers, derived sizes of a uts_config, and the library's own HEALPix NESTED indexing
// (§3.1; Gorski et al. as cited at PAPER.md:23).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>
#include <mutex>
#include "uts.h"

namespace uts {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr int kMaxOrder = 13;
constexpr int kTileLog2 = 4;          // B = 16 (Table 6): the only tile size implemented
constexpr int kTilePix = 256;         // B*B pixels per tile == threads per blend block

// ------------------------------------------------------------------------------------------------ status
void set_last_cuda_error(cudaError_t e);
#define UTS_CUDA(call)                                                      \
  do {                                                                      \
    cudaError_t e__ = (call);                                               \
    if (e__ != cudaSuccess) { ::uts::set_last_cuda_error(e__); return UTS_ERR_CUDA; } \
  } while (0)
void count_launch();                     // uts_launch_count(): one tick per kernel launch of this library
#define UTS_LAUNCH_CHECK() do { ::uts::count_launch(); UTS_CUDA(cudaGetLastError()); } while (0)

int check_config(const uts_config* c);   // UTS_OK / UTS_ERR_INVALID_ARG / UTS_ERR_UNSUPPORTED
int check_mask(const uts_config* c, const uts_mask& m);
int sm_count();                          // of the current device (from its context)

// The library's per-device state (include/uts.h "Library state"): created on the first call made with the device current, kept
// until the process ends.  `mu` is held by a call while it enqueues on the streams below (fork ... join), so concurrent callers
// never interleave their event records; the streams themselves only order work.
struct DeviceCtx {
  std::recursive_mutex mu;            // recursive: uts_host_forward_backward holds it around the stage calls
  int device = -1, sms = 148;
  cudaStream_t aux[2] = {nullptr, nullptr};         // tile query: the three work shapes run side by side
  cudaEvent_t fork = nullptr, join[2] = {nullptr, nullptr};
  cudaStream_t side = nullptr;                      // uts_tile_lists: matrix transpose + popcount beside the small pairs' emit + sort
  cudaEvent_t side_fork = nullptr, side_join = nullptr, side_mid = nullptr;
  cudaStream_t copy = nullptr;                      // uts_host_forward_backward: copies off the critical path
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  unsigned long long* pin = nullptr;                // 8 pinned host words: small device -> host reads in one copy (under mu)
  bool attrs_set[4] = {false, false, false, false}; // cudaFuncSetAttribute done, per translation unit (under mu)
  static constexpr int kOccSlots = 32;              // cached cudaOccupancyMaxActiveBlocksPerMultiprocessor results (under mu)
  uint64_t occ_key[kOccSlots] = {}; int occ_val[kOccSlots] = {}; int occ_n = 0;
};
DeviceCtx* device_ctx();                 // nullptr when the CUDA runtime fails (last error set)
// blocks per SM of `kernel` at (threads, dynamic smem), looked up in / added to ctx's cache; the caller holds ctx->mu
template <class K>
inline int cached_occupancy(DeviceCtx* ctx, int kernel_id, K kernel, int threads, size_t smem) {
  const uint64_t key = ((uint64_t)kernel_id << 48) | ((uint64_t)threads << 36) | (uint64_t)smem;
  for (int i = 0; i < ctx->occ_n; ++i) if (ctx->occ_key[i] == key) return ctx->occ_val[i];
  int occ = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess || occ < 1) occ = 1;
  if (ctx->occ_n < DeviceCtx::kOccSlots) { ctx->occ_key[ctx->occ_n] = key; ctx->occ_val[ctx->occ_n] = occ; ++ctx->occ_n; }
  return occ;
}

// --------------------------------------------------------------------------------------------- derived
struct Dims {
  int k, kt, kq, P, V, M;
  int64_t n_pix, n_tile;
  int64_t n_slot;       // tiles that get a thread block: n_active or n_tile
};
inline Dims dims_of(const uts_config* c, const uts_mask* m) {
  Dims d;
  d.k = c->order; d.kt = c->order - c->tile_log2; d.kq = d.kt + c->query_refine_log2;
  d.P = c->n_gauss; d.V = c->n_views; d.M = (c->sh_degree + 1) * (c->sh_degree + 1);
  d.n_pix = (int64_t)12 << (2 * d.k);
  d.n_tile = (int64_t)12 << (2 * d.kt);
  d.n_slot = (m && m->active_tiles) ? m->n_active : d.n_tile;
  return d;
}

// rho_max(o) table (host, computed once): uts_common.cu, fill_rho_max()
const double* rho_max_table_host();

// ------------------------------------------------------------------------------------- HEALPix (device)
// NESTED index p at order o  ->  face f and in-face integer coordinates (x,y): x in the even bits, y in the odd
// bits of p mod 4^o.
__host__ __device__ __forceinline__ uint32_t squeeze_even_bits(uint64_t v) {
  v &= 0x5555555555555555ull;
  v = (v | (v >> 1)) & 0x3333333333333333ull;
  v = (v | (v >> 2)) & 0x0f0f0f0f0f0f0f0full;
  v = (v | (v >> 4)) & 0x00ff00ff00ff00ffull;
  v = (v | (v >> 8)) & 0x0000ffff0000ffffull;
  v = (v | (v >> 16)) & 0x00000000ffffffffull;
  return (uint32_t)v;
}

struct PixGeom {        // what fixes a pixel centre: z (or 1-|z| in the caps) and longitude in quarter-turn units
  double z;             // sin(latitude) = HEALPix polar coordinate
  double sth;           // cos(latitude)
  double lam;           // longitude (radians), not wrapped
};

// Centre of NESTED pixel p at order o.
// Derivation used here: inside face f = 4*r + c the centre sits at v = x + y - (N-1) half-rings above the face's
// middle ring and h = x - y half-steps east of the face's central meridian.  Ring number from the north pole is
// i = (r+1) N - v.  A ring holds 4*n pixels with n = min(i, N, 4N - i); the z of a ring is 1 - i^2/(3N^2) in the north
// cap (i < N), 2(2N - i)/(3N) in the equatorial belt, and mirrored in the south cap.  The face's central meridian is
// at (2c + 1 - (r & 1)) quarter-turns/2, and one half-step in a ring of 4n pixels is pi/(4n), so
//      lambda = (pi/4) * ((2c + 1 - (r&1)) + h / n).
__host__ __device__ __forceinline__ PixGeom pix_geom(int o, uint64_t p) {
  const int64_t N = (int64_t)1 << o;
  const int f = (int)(p >> (2 * o));
  const uint64_t m = p & (((uint64_t)1 << (2 * o)) - 1);
  const int64_t x = squeeze_even_bits(m), y = squeeze_even_bits(m >> 1);
  const int r = f >> 2, c = f & 3;
  const int64_t i = (int64_t)(r + 1) * N - (x + y - (N - 1));
  const int64_t h = x - y;
  PixGeom g;
  int64_t n;
  const double inv3N2 = 1.0 / (3.0 * (double)N * (double)N);
  if (i < N) {                       // north polar cap
    n = i;
    const double w = (double)(n * n) * inv3N2;        // 1 - z
    g.z = 1.0 - w; g.sth = sqrt(w * (2.0 - w));
  } else if (i > 3 * N) {            // south polar cap
    n = 4 * N - i;
    const double w = (double)(n * n) * inv3N2;        // 1 + z
    g.z = w - 1.0; g.sth = sqrt(w * (2.0 - w));
  } else {                           // equatorial belt
    n = N;
    g.z = (double)(2 * (2 * N - i)) / (double)(3 * N);
    g.sth = sqrt((1.0 - g.z) * (1.0 + g.z));
  }
  g.lam = (kPi / 4) * ((double)(2 * c + 1 - (r & 1)) + (double)h / (double)n);
  return g;
}

// Camera-frame unit vector of a pixel centre.  Frame (reading A1): polar axis = camera +y, longitude 0 at camera +z,
// longitude = omega = atan2(t_x, t_z)  =>  (x,y,z)_cam = (cos(lat) sin(lam), sin(lat), cos(lat) cos(lam)).
__device__ __forceinline__ void pix_center_cam(int o, uint64_t p, double& vx, double& vy, double& vz) {
  PixGeom g = pix_geom(o, p);
  double s, c;
  sincos(g.lam, &s, &c);
  vx = g.sth * s; vy = g.z; vz = g.sth * c;
}

// Single-precision pixel centre (absolute error about 1e-6 per component): used only to pre-classify quadtree nodes with a
// safety margin; every decision that defines an output is re-taken in double when it falls inside the margin.
// A NESTED index at order <= 13 fits 32 bits (12 * 4^13 < 2^32).
__host__ __device__ __forceinline__ uint32_t squeeze_even_bits32(uint32_t v) {
  v &= 0x55555555u;
  v = (v | (v >> 1)) & 0x33333333u;
  v = (v | (v >> 2)) & 0x0f0f0f0fu;
  v = (v | (v >> 4)) & 0x00ff00ffu;
  v = (v | (v >> 8)) & 0x0000ffffu;
  return v;
}

__device__ __forceinline__ void pix_center_cam_f32(int o, uint32_t p, float& vx, float& vy, float& vz) {
  const int N = 1 << o;
  const int f = (int)(p >> (2 * o));
  const uint32_t m = p & ((1u << (2 * o)) - 1u);
  const int x = (int)squeeze_even_bits32(m), y = (int)squeeze_even_bits32(m >> 1);
  const int r = f >> 2, c = f & 3;
  const int i = (r + 1) * N - (x + y - (N - 1));
  const int h = x - y;
  const float invN = __int_as_float((127 - o) << 23);          // 2^-o, exact
  const float inv3N2 = 0.333333343f * invN * invN;
  float z, sth, q;
  if (i < N) { const float fn = (float)i; const float w = fn * fn * inv3N2; z = 1.0f - w; sth = sqrtf(w * (2.0f - w)); q = __fdividef((float)h, fn); }
  else if (i > 3 * N) { const float fn = (float)(4 * N - i); const float w = fn * fn * inv3N2; z = w - 1.0f; sth = sqrtf(w * (2.0f - w)); q = __fdividef((float)h, fn); }
  else { z = (float)(2 * (2 * N - i)) * (0.333333343f * invN); sth = sqrtf((1.0f - z) * (1.0f + z)); q = (float)h * invN; }
  // longitude in quarter turns, reduced to (-4, 4] so that the fast sincos sees |lam| <= pi (absolute error < 5e-7 there)
  q += (float)(2 * c + 1 - (r & 1));
  if (q > 4.0f) q -= 8.0f;
  float s, cs;
  __sincosf(q * 0.78539816339744831f, &s, &cs);
  vx = sth * s; vy = z; vz = sth * cs;
}

// Packed fp32 pairs (sm_100: fma / mul / add .f32x2 — one instruction, two IEEE roundings, the same results as the scalar forms).
// A pair is a 64-bit register; f2_bc(s) = (s, s) costs nothing (ptxas folds it into a scalar operand of FFMA2 / FMUL2 / FADD2).
typedef unsigned long long f2_t;
__device__ __forceinline__ f2_t f2_pack(float lo, float hi) { f2_t d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d; }
__device__ __forceinline__ f2_t f2_bc(float s) { return f2_pack(s, s); }
__device__ __forceinline__ void f2_unpack(f2_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f2_t f2_fma(f2_t a, f2_t b, f2_t c) { f2_t d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f2_t f2_mul(f2_t a, f2_t b) { f2_t d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2_t f2_add(f2_t a, f2_t b) { f2_t d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

}  // namespace uts
