// uts_render.cu — F5/F6: front-to-back alpha blending at every HEALPix pixel centre with the FoV mask
// (Alg.1 l.17-30 PAPER.md:563-587; Eq.6; SphericalOffset PAPER.md:112; mask PAPER.md:62, 129), and
// B1: its backward.
//
// One thread block of 256 / PX threads per active tile; every thread owns PX pixels (p & 255 = 32 (PX warp + j) + lane, j < PX: a
// warp owns PX consecutive 8x4 "patches" of 32 pixels in NESTED order), so that one staged list entry read from shared memory
// serves PX pixel evaluations — two at a time in packed fp32 pairs (FFMA2 / FMUL2 / FADD2, sm_100) — and, in the backward, one warp
// reduction + one set of atomics serves up to 32 PX pixels.  Patches are what the early exit, the patch cull, the marks and the
// backward's visit list are kept for.  The tile's sorted list is staged through shared memory in batches of 256 entries.
//
// SphericalOffset without inverse trigonometry and without fp32 cancellation:  with Gaussian direction u
// and its east/north unit vectors e, n, and pixel direction w,
//     a = e.w, b = n.w, c = u.w,  sin(d_gc) = sqrt(a^2+b^2),  (d_x,d_y) = (d_gc / sin d_gc) (a,b)
// is the haversine distance + bearing decomposition of PAPER.md:112 in vector form.  Because e.u = n.u = 0,
// a = e.(w-u) and b = n.(w-u): the difference w-u = (c_tile - u) + (w - c_tile) is formed in double precision once per
// (tile, Gaussian) and once per pixel, then everything per (pixel, Gaussian) is fp32 FMAs on small, exactly known
// differences.  k = d_gc/sin d_gc = P(c) rsqrt(1+c) with a degree-7 polynomial P for c = cos d_gc >= 0 (out of line beyond 90
// degrees, still without atan).  (A polynomial in t = sin^2 d_gc alone, which needs no c on the near side, was measured and
// dropped: on the paper's kind of scene the entries a pixel consumes before it saturates are the nearest, largest Gaussians, and
// 64 % of the evaluated pairs of config 4 lie beyond 30 degrees of the Gaussian's centre, 22 % beyond 60.)
// power*log2(e) = k^2 (qa a^2 + qb a b + qc b^2) with the conic pre-scaled at staging; alpha uses ex2, and an entry whose power is
// below log2(alpha_min / o) (minus a margin far above the ex2 error) is skipped before the ex2: the same decision as
// alpha < alpha_min, taken identically by forward and backward.
#include "uts_internal.cuh"

namespace uts {

struct RenderParams {
  int k, P;
  int64_t n_tile, n_slot;
  float amin, amax, teps, bg[3];
};

constexpr float kLog2e = 1.4426950408889634f;
// Pixels per thread (PX) of the two kernels: a block has 256 / PX threads and a warp owns PX consecutive patches of 32 pixels.
// Measured on config 4 (B200): with scalar arithmetic the forward is bound by the per-evaluation instructions, not by the
// shared-memory reads or the loop (the same 2.9e9 warp instructions at PX = 1 and 4), and more pixels per thread only cost
// occupancy; with PX = 2 the two pixels' evaluations go through packed fp32 pairs (FFMA2 / FMUL2, eval_entry2): half the
// arithmetic instructions per pixel, 2.53 -> 2.10 ms.  The backward gains from PX = 4 because one warp reduction + one set of
// atomics then serves the four patches of a warp.
#ifndef UTS_FWD_PX
#define UTS_FWD_PX 2
#endif
#ifndef UTS_BWD_PX
#define UTS_BWD_PX 4
#endif
constexpr int kFwdPx = UTS_FWD_PX, kBwdPx = UTS_BWD_PX;
constexpr int kBatch = 256;                          // list entries staged per batch

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Bare MUFU forms (no denormal / range fix-up code around them: the arguments here are never denormal or huge).
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// Broadcast reads of the staged entries with the shared-window address kept in a register by the caller.
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void red_add_global(float* p, float v) {       // p is a global address (cudaMalloc'ed gradient buffer)
  asm volatile("red.global.add.f32 [%0], %1;" :: "l"(p), "f"(v) : "memory");
}

// k = d_gc / sin(d_gc).  For cos(d_gc) = c >= 0:  acos(c) = sqrt(1-c) P(c) with P analytic on [0,1], so
// k = acos(c) / sqrt((1-c)(1+c)) = P(c) rsqrt(1+c): no cancellation (1-c never formed), one MUFU.
// P is a degree-7 Chebyshev fit of acos(c)/sqrt(1-c) on [0,1] (own fit; max relative error of k in fp32: 1.7e-7).
// Beyond 90 degrees (c < 0; only the far tail of very large Gaussians): acos(c) = pi - acos(|c|) and
// sqrt(1-|c|) = sin / sqrt(1+|c|), so k = (pi - sin P(|c|) rsqrt(1+|c|)) / sin with sin = sqrt(t): still no cancellation.
// That branch is out of line so that the common path stays straight.
__device__ __forceinline__ float acos_poly(float c) {
  float p = -0.00115729403f;
  p = fmaf(p, c, 0.00628544204f);
  p = fmaf(p, c, -0.016528869f);
  p = fmaf(p, c, 0.0304812621f);
  p = fmaf(p, c, -0.0500148833f);
  p = fmaf(p, c, 0.0889478773f);
  p = fmaf(p, c, -0.214596227f);
  return fmaf(p, c, 1.57079625f);
}
__device__ __noinline__ float arc_over_sin_far(float t, float c) {
  if (!(t > 0.f)) return 1.0f;                      // antipode: never reached by a finite conic (alpha underflows first)
  const float is = rsqrt_approx(t), s = t * is, ac = -c;
  return (3.14159274f - s * acos_poly(ac) * rsqrt_approx(1.0f + ac)) * is;
}
__device__ __forceinline__ float arc_over_sin(float t, float c) {
  if (c >= 0.f) return acos_poly(c) * rsqrt_approx(1.0f + c);
  return arc_over_sin_far(t, c);
}

// What one (tile, Gaussian) list entry contributes to every pixel of the tile, staged once per entry as float4 rows:
//   g0 = (a0, b0, c0, th)     a0 = e.(c_tile-u), b0 = n.(c_tile-u), c0 = uhat.c_tile; th = log2(alpha_min / o) - margin
//   g1 = (ex, ez, nx, ny)     e = (ex, 0, ez)
//   g2 = (nz, ux, uy, uz)     uhat
//   g3 = (qa, qb, qc, o)      -0.5 A log2e, -B log2e, -0.5 C log2e; opacity
//   g4 = (r, g, b, id | 1/rho)  colour; backward: Gaussian index as raw bits; forward with the depth channel: 1 / rho
//   g5 = (sin phi, cos phi, 1/rho)   backward;  (L, -, -, -) forward: L = sqrt(lambda_max) of the scaled conic, for the patch cull
constexpr uint32_t kRow = kBatch * 16u;               // bytes between rows
struct TileFrame { double cx, cy, cz; };              // tile centre direction (order k_t pixel centre)

template <bool BWD>
struct __align__(16) SEntries { float4 g[6][kBatch]; };

template <bool BWD>
__device__ __forceinline__ void stage_entry(SEntries<BWD>& S, int i, const TileFrame& tf, float amin, uint32_t id, float ux, float uy,
                                            float uz, float4 co, float r, float g, float b, float inv_r) {
  const float dxf = (float)(tf.cx - (double)ux), dyf = (float)(tf.cy - (double)uy), dzf = (float)(tf.cz - (double)uz);
  const float rxz2 = ux * ux + uz * uz;
  float ex = 1.f, ez = 0.f;
  if (rxz2 > 0.f) { const float inv = rsqrtf(rxz2); ex = uz * inv; ez = -ux * inv; }    // pole guard: reading A22
  const float invn = rsqrtf(rxz2 + uy * uy);
  const float hx = ux * invn, hy = uy * invn, hz = uz * invn;
  const float nx = hy * ez, ny = hz * ex - hx * ez, nz = -hy * ex;                       // n = uhat x e
  // alpha = o 2^p2 < alpha_min  <=>  p2 < log2(alpha_min / o); the 1e-3 margin (0.07 % in alpha) is far above the error of
  // lg2.approx / ex2.approx, so p2 < th implies alpha < alpha_min and the exact test settles everything else
  float th = -3.0e38f;
  if (amin > 0.f) th = co.w > 0.f ? __log2f(amin / co.w) - 1e-3f : 3.0e38f;
  S.g[0][i] = make_float4(ex * dxf + ez * dzf, nx * dxf + ny * dyf + nz * dzf, hx * (float)tf.cx + hy * (float)tf.cy + hz * (float)tf.cz, th);
  S.g[1][i] = make_float4(ex, ez, nx, ny);
  S.g[2][i] = make_float4(nz, hx, hy, hz);
  S.g[3][i] = make_float4(-0.5f * kLog2e * co.x, -kLog2e * co.y, -0.5f * kLog2e * co.z, co.w);
  S.g[4][i] = make_float4(r, g, b, BWD ? __uint_as_float(id) : inv_r);
  if (BWD) S.g[5][i] = make_float4(hy, sqrtf(hx * hx + hz * hz), inv_r, 0.f);
  else {
    // -q(d) = d^T K d with K = [[-qa, -qb/2], [-qb/2, -qc]] positive definite: sqrt(-q) is a norm, bounded by L |d|
    const float A = 0.5f * kLog2e * co.x, B = 0.5f * kLog2e * co.y, C = 0.5f * kLog2e * co.z;
    const float hd = 0.5f * (A - C);
    S.g[5][i] = make_float4(sqrtf(0.5f * (A + C) + sqrtf(fmaf(hd, hd, B * B))) * 1.00001f, 0.f, 0.f, 0.f);
  }
}

struct Eval { float a, b, c, t, k, p2; };

// Shared by forward and backward so that both take the same skip / clamp decisions.
__device__ __forceinline__ void eval_entry(const float4 g0, const float4 g1, const float4 g2, const float4 g3, float px, float py, float pz,
                                           Eval& ev) {
  ev.a = fmaf(g1.x, px, fmaf(g1.y, pz, g0.x));
  ev.b = fmaf(g1.z, px, fmaf(g1.w, py, fmaf(g2.x, pz, g0.y)));
  ev.c = fmaf(g2.y, px, fmaf(g2.z, py, fmaf(g2.w, pz, g0.z)));
  ev.t = fmaf(ev.a, ev.a, ev.b * ev.b);
  ev.k = arc_over_sin(ev.t, ev.c);
  const float q = fmaf(ev.a, fmaf(g3.x, ev.a, g3.y * ev.b), g3.z * ev.b * ev.b);     // qa a^2 + qb a b + qc b^2
  ev.p2 = q * ev.k * ev.k;
}
// Alg.1 l.23 (reading A7): power > 0 skipped; power below the alpha_min cut skipped (see stage_entry)
__device__ __forceinline__ bool may_contribute(const Eval& ev, float th) { return !(ev.p2 > 0.f) && ev.p2 >= th; }

// eval_entry for two pixels at once: the same operations in the same order on packed pairs, so a, b, c, k and p2 are bit-identical to
// two scalar calls (the backward and the counted forward keep the scalar form and rely on that; a test compares the images bit by bit).
struct Eval2 { f2_t a, b, c, k, p2; };
__device__ __forceinline__ void eval_entry2(const float4 g0, const float4 g1, const float4 g2, const float4 g3, f2_t px, f2_t py, f2_t pz,
                                            Eval2& ev) {
  const f2_t a = f2_fma(f2_bc(g1.x), px, f2_fma(f2_bc(g1.y), pz, f2_bc(g0.x)));
  const f2_t b = f2_fma(f2_bc(g1.z), px, f2_fma(f2_bc(g1.w), py, f2_fma(f2_bc(g2.x), pz, f2_bc(g0.y))));
  const f2_t c = f2_fma(f2_bc(g2.y), px, f2_fma(f2_bc(g2.z), py, f2_fma(f2_bc(g2.w), pz, f2_bc(g0.z))));
  float c0, c1;
  f2_unpack(c, c0, c1);
  f2_t k;
  if (c0 >= 0.f && c1 >= 0.f) {                        // acos_poly(c) * rsqrt(1 + c), both pixels
    f2_t p = f2_fma(f2_bc(-0.00115729403f), c, f2_bc(0.00628544204f));
    p = f2_fma(p, c, f2_bc(-0.016528869f));
    p = f2_fma(p, c, f2_bc(0.0304812621f));
    p = f2_fma(p, c, f2_bc(-0.0500148833f));
    p = f2_fma(p, c, f2_bc(0.0889478773f));
    p = f2_fma(p, c, f2_bc(-0.214596227f));
    p = f2_fma(p, c, f2_bc(1.57079625f));
    float s0, s1;
    f2_unpack(f2_add(f2_bc(1.0f), c), s0, s1);
    k = f2_mul(p, f2_pack(rsqrt_approx(s0), rsqrt_approx(s1)));
  } else {                                             // a pixel beyond 90 degrees: the scalar form
    float a0, a1, b0, b1;
    f2_unpack(a, a0, a1); f2_unpack(b, b0, b1);
    k = f2_pack(arc_over_sin(fmaf(a0, a0, b0 * b0), c0), arc_over_sin(fmaf(a1, a1, b1 * b1), c1));
  }
  const f2_t q = f2_fma(a, f2_fma(f2_bc(g3.x), a, f2_mul(f2_bc(g3.y), b)), f2_mul(f2_mul(f2_bc(g3.z), b), b));
  ev.a = a; ev.b = b; ev.c = c; ev.k = k;
  ev.p2 = f2_mul(f2_mul(q, k), k);
}
__device__ __forceinline__ bool may_contribute(float p2, float th) { return !(p2 > 0.f) && p2 >= th; }

// Pixel and tile set-up common to both kernels.
template <int PX>
struct TileSetup { bool on[PX]; float px[PX], py[PX], pz[PX]; size_t out0; uint64_t start, end; int v; int64_t tile; };

template <int PX>
__device__ __forceinline__ void setup_tile(const RenderParams& rp, const uint32_t* __restrict__ active_tiles,
                                           const uint32_t* __restrict__ mask_bits, const uint64_t* __restrict__ ranges,
                                           TileFrame* s_tf, TileSetup<PX>& ts) {
  constexpr int kThreads = kTilePix / PX;
  const int64_t slot = blockIdx.x % rp.n_slot;
  ts.v = (int)(blockIdx.x / rp.n_slot);
  const int64_t tile = active_tiles ? (int64_t)__ldg(active_tiles + slot) : slot;
  ts.tile = tile;
  const uint32_t pix0 = (threadIdx.x >> 5) * (32u * PX) + (threadIdx.x & 31u);  // a warp owns PX consecutive patches of 32 pixels
  ts.out0 = ((size_t)ts.v * rp.n_slot + slot) * kTilePix + pix0;                 // pixel j of this thread: out0 + 32 j
  const uint64_t rix = 2 * ((uint64_t)ts.v * rp.n_tile + tile);
  ts.start = __ldg(ranges + rix); ts.end = __ldg(ranges + rix + 1);
  if (threadIdx.x == 0) pix_center_cam(rp.k - kTileLog2, (uint64_t)tile, s_tf->cx, s_tf->cy, s_tf->cz);
  double wx[PX], wy[PX], wz[PX];
#pragma unroll
  for (int j = 0; j < PX; ++j) {
    const uint64_t p = (uint64_t)tile * kTilePix + pix0 + 32u * j;
    ts.on[j] = mask_bits ? ((__ldg(mask_bits + (p >> 5)) >> (p & 31)) & 1u) != 0 : true;
    pix_center_cam(rp.k, p, wx[j], wy[j], wz[j]);
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < PX; ++j) {
    ts.px[j] = (float)(wx[j] - s_tf->cx); ts.py[j] = (float)(wy[j] - s_tf->cy); ts.pz[j] = (float)(wz[j] - s_tf->cz);
  }
}

// Marks (uts_render_fwd_marked / uts_render_bwd_marked): one bit per (patch, list entry), set by the forward when at least one
// of the patch's 32 pixels blended the entry.  Patch (warp, j) — pixels 32 (PX warp + j) + lane, a warp owns PX consecutive patches —
// is plane PX warp + j of 8, whatever PX the forward and the backward were built with; the bits
// of (view, tile) vt start at word (start_vt >> 5) + vt of the plane, entry i of the list at bit i of that run — runs of
// different tiles never share a word.  The backward visits an entry only for the patches whose bit is set: on the paper's kind of
// scene half of the (patch, entry) visits would re-evaluate alpha just to find that no pixel of the patch took the entry.
template <int PX>
__device__ __forceinline__ uint64_t mark_base(const RenderParams& rp, const TileSetup<PX>& ts) {
  return (ts.start >> 5) + (uint64_t)ts.v * (uint64_t)rp.n_tile + (uint64_t)ts.tile;
}

// Every thread stages PX entries of the batch, one after the other (issuing the gathers of several entries together was measured:
// the extra registers cost more occupancy than the overlapped latency gives back).  Up to three null entries follow the last real
// one, so that the walk can take entries four at a time: a = 1, qa = 1 give power > 0, which Alg.1 l.23 skips whatever the thresholds.
template <int PX, bool BWD, bool DEPTH>
__device__ __forceinline__ void stage_batch(SEntries<BWD>& S, const TileFrame& tf, const RenderParams& rp, const float* __restrict__ dir,
                                            const float* __restrict__ conic_opac, const float* __restrict__ rgb, const float* __restrict__ rho,
                                            const uint32_t* __restrict__ vals, uint64_t first, uint64_t n, size_t gbase) {
  constexpr int kThreads = kTilePix / PX;
#pragma unroll 1
  for (uint32_t e = threadIdx.x; e < (uint32_t)kBatch; e += kThreads) {
    if ((uint64_t)e < n) {
      const uint32_t id = __ldg(vals + first + e);
      const size_t gi = gbase + id;
      stage_entry<BWD>(S, (int)e, tf, rp.amin, id, __ldg(dir + 3 * gi), __ldg(dir + 3 * gi + 1), __ldg(dir + 3 * gi + 2),
                       __ldg(reinterpret_cast<const float4*>(conic_opac) + gi), __ldg(rgb + 3 * gi), __ldg(rgb + 3 * gi + 1),
                       __ldg(rgb + 3 * gi + 2), DEPTH ? __fdiv_rn(1.0f, __ldg(rho + gi)) : 0.f);
    } else {
      if ((uint64_t)e < n + 3) {
        S.g[0][e] = make_float4(1.f, 0.f, 1.f, -3.0e38f); S.g[1][e] = make_float4(0.f, 0.f, 0.f, 0.f);
        S.g[2][e] = make_float4(0.f, 0.f, 0.f, 0.f); S.g[3][e] = make_float4(1.f, 0.f, 0.f, 0.f);
      }
      break;
    }
  }
}

// COUNT (uts_render_fwd_counted, measurement only): the walk WITHOUT the patch cull (every entry is evaluated: the reference for its
// bit-identity), adding to work[0..3] the (pixel, entry) pairs of Alg.1's loop, those that contribute, those the production kernel
// evaluates (they pass the patch cull) and those a patch-level early out on q alone would still leave (not taken: see below).
// DEPTH (uts_render_fwd_depth): a fourth blended channel, the inverse radial depth 1 / rho_i (reading A29).
template <int PX, bool MARK, bool COUNT = false, bool DEPTH = false>
__global__ void __launch_bounds__(kTilePix / PX)
render_fwd_kernel(RenderParams rp, const float* __restrict__ dir, const float* __restrict__ conic_opac, const float* __restrict__ rgb,
                  const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ mask_bits,
                  const uint64_t* __restrict__ ranges, const uint32_t* __restrict__ vals, float* __restrict__ color,
                  float* __restrict__ alpha_out, float* __restrict__ trans_out, uint32_t* __restrict__ n_last_out,
                  uint32_t* __restrict__ marks, uint64_t plane_words, unsigned long long* __restrict__ work = nullptr,
                  const float* __restrict__ rho = nullptr, float* __restrict__ depth_out = nullptr) {
  constexpr int kThreads = kTilePix / PX, kWarps = kThreads / 32;
  __shared__ SEntries<false> S;
  uint32_t n_eval = 0, n_contrib = 0, n_cull = 0, n_full = 0;      // COUNT only
  __shared__ TileFrame s_tf;
  TileSetup<PX> ts;
  setup_tile<PX>(rp, active_tiles, mask_bits, ranges, &s_tf, ts);
  const TileFrame tf = s_tf;
  const size_t gbase = (size_t)ts.v * rp.P;
  const int wid = threadIdx.x >> 5;

  float T[PX], Cr[PX], Cg[PX], Cb[PX], Cd[PX];
  uint32_t n_last[PX];
  uint32_t open = 0;                                  // bit j: pixel j still takes entries
#pragma unroll
  for (int j = 0; j < PX; ++j) { T[j] = 1.f; Cr[j] = Cg[j] = Cb[j] = Cd[j] = 0.f; n_last[j] = 0; if (ts.on[j]) open |= 1u << j; }
  const uint64_t len = ts.end - ts.start;
  uint32_t sS = (uint32_t)__cvta_generic_to_shared(&S);
  asm volatile("" : "+r"(sS));                       // keep the window address in a register (otherwise it is rebuilt from CgaCtaId at every entry)
  uint32_t* mark_w = nullptr;                         // plane PX wid of this tile's run; patch j is j planes further
  if (MARK) mark_w = marks + (uint64_t)(PX * wid) * plane_words + mark_base<PX>(rp, ts);
  // Patch cull (PX = 1: a warp is one 8x4 patch).  At the start of a group of 32 entries lane l asks whether entry l can reach the
  // patch at all: with the patch's centre pc and radius r (in the tile frame; the map to the Gaussian's (a, b) plane is an
  // isometry of the chord), sqrt(-q) >= N(pc) - r L everywhere on the patch, so N(pc) - r L > sqrt(-th) means every pixel's power
  // is below the alpha_min cut.  The warp walks the ballot's survivors only.  No per-pixel
  // decision changes (such an entry fails may_contribute() at every pixel); the margin 1.0001 covers the fp32 rounding of the
  // bound.  A warp whose last tested group kept >= 30 of 32 entries skips the test for 3 groups (a test costs about
  // as much as half a visit, so it pays as soon as one entry in 32 is culled: threshold 24 -> 30, config 4 2.00 -> 1.92 ms).
  constexpr bool kCull = PX <= 2;                     // per patch j of the warp (PX = 2: an entry is walked when it reaches either)
  float pcx[PX], pcy[PX], pcz[PX], prad[PX];
  int skip_tests = 0;
#pragma unroll
  for (int j = 0; j < PX; ++j) {
    pcx[j] = pcy[j] = pcz[j] = prad[j] = 0.f;
    if (kCull) {
      float sx = ts.px[j], sy = ts.py[j], sz = ts.pz[j];
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, d); sy += __shfl_xor_sync(0xffffffffu, sy, d); sz += __shfl_xor_sync(0xffffffffu, sz, d);
      }
      pcx[j] = sx * (1.f / 32.f); pcy[j] = sy * (1.f / 32.f); pcz[j] = sz * (1.f / 32.f);
      const float ex = ts.px[j] - pcx[j], ey = ts.py[j] - pcy[j], ez = ts.pz[j] - pcz[j];
      float r = sqrtf(ex * ex + ey * ey + ez * ez);
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, d));
      prad[j] = r * 1.00001f;
    }
  }
  f2_t px2 = 0, py2 = 0, pz2 = 0;                     // PX = 2: the two pixels' coordinates, T and colour sums as packed pairs
  f2_t T2 = f2_bc(1.f), Cr2 = 0, Cg2 = 0, Cb2 = 0, Cd2 = 0;
  if (PX == 2) { px2 = f2_pack(ts.px[0], ts.px[PX - 1]); py2 = f2_pack(ts.py[0], ts.py[PX - 1]); pz2 = f2_pack(ts.pz[0], ts.pz[PX - 1]); }
  for (uint64_t b0 = 0; b0 < len; b0 += kBatch) {
    if (__syncthreads_and(open == 0)) break;          // every pixel of the tile saturated (or masked)
    const uint64_t left_n = len - b0;
    stage_batch<PX, false, DEPTH>(S, tf, rp, dir, conic_opac, rgb, rho, vals, ts.start + b0, left_n, gbase);
    __syncthreads();
    const int nb = (int)(left_n < (uint64_t)kBatch ? left_n : (uint64_t)kBatch);
    // The batch is walked in groups of 32 entries, one mark word per patch each.  Every four entries the warp finds out which
    // of its patches still have an open pixel (one redux); the vote only ends a patch's walk early, every skip / clamp decision
    // is per pixel.  The list is padded with null entries to a multiple of four.
    bool left = false;
    for (int g0 = 0; g0 < nb && !left; g0 += 32) {
      uint32_t mw[PX];                                // this lane's marks of the group, per patch
#pragma unroll
      for (int j = 0; j < PX; ++j) mw[j] = 0u;
      const int ge = min(nb, g0 + 32);
      uint32_t live = 0xffffffffu;                    // bit e: entry g0 + e may reach a patch of this warp
      if (kCull) {
        if (skip_tests > 0) --skip_tests;
        else {
          const int e = g0 + (int)(threadIdx.x & 31);
          bool reach = false;
          if (e < nb) {
            const uint32_t se = sS + (uint32_t)e * 16u;
            const float4 h0 = lds128(se), h1 = lds128(se + kRow), h2 = lds128(se + 2u * kRow), h3 = lds128(se + 3u * kRow), h5 = lds128(se + 5u * kRow);
#pragma unroll
            for (int j = 0; j < PX; ++j) {
              const float ac = fmaf(h1.x, pcx[j], fmaf(h1.y, pcz[j], h0.x));
              const float bc = fmaf(h1.z, pcx[j], fmaf(h1.w, pcy[j], fmaf(h2.x, pcz[j], h0.y)));
              const float nq = -fmaf(ac, fmaf(h3.x, ac, h3.y * bc), h3.z * bc * bc);   // -q at the patch centre
              const float slack = sqrtf(fmaxf(nq, 0.f)) - prad[j] * h5.x;
              reach = reach || !(slack > 0.f && slack * slack > -h0.w * 1.0002f);
            }
          }
          live = __ballot_sync(0xffffffffu, reach);
          if (__popc(live) >= 30) skip_tests = 3;
        }
      }
      // The entries of the group this warp visits (the cull's survivors), front to back; culled entries cost nothing.  Measured
      // against testing the bit of every entry inside a walk unrolled by four with immediate addresses: config 4 (32 % culled)
      // 1.98 -> 2.03 ms, config 5 (70 % culled) 2.61 -> 2.48 ms, config 3 0.50 -> 0.48 ms.
      uint32_t walk = COUNT ? 0xffffffffu : live;
      if (ge - g0 < 32) walk &= (1u << (ge - g0)) - 1u;
      while (walk) {
        const uint32_t alive = __reduce_or_sync(0xffffffffu, open);
        if (alive == 0) { left = true; break; }       // every pixel of the warp is saturated
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (!walk) break;
          const int jj = g0 + __ffs((int)walk) - 1;
          walk &= walk - 1u;
          const uint32_t sa = sS + (uint32_t)jj * 16u;
          const float4 g0v = lds128(sa), g1 = lds128(sa + kRow), g2 = lds128(sa + 2u * kRow), g3 = lds128(sa + 3u * kRow);
          float p2[PX];
          uint32_t cand = 0;                          // bit j: pixel j may blend this entry
          if (PX == 2 && !COUNT) {                    // both pixels in packed arithmetic
            Eval2 ev2;
            eval_entry2(g0v, g1, g2, g3, px2, py2, pz2, ev2);
            f2_unpack(ev2.p2, p2[0], p2[PX - 1]);
            bool c0 = (open & 1u) && may_contribute(p2[0], g0v.w), c1 = (open & 2u) && may_contribute(p2[PX - 1], g0v.w);
            if (!(c0 || c1)) continue;
            // The blend of both pixels, packed and branch-free: a pixel that does not take the entry gets alpha = 0, which leaves its
            // T and colour sums exactly as they were (w = T 0 = 0, C + 0 c = C, T (1 - 0) = T).
            const float4 g4 = lds128(sa + 4u * kRow);
            float a0 = fminf(rp.amax, g3.w * ex2_approx(p2[0])), a1 = fminf(rp.amax, g3.w * ex2_approx(p2[PX - 1]));
            c0 = c0 && !(a0 < rp.amin); c1 = c1 && !(a1 < rp.amin);
            a0 = c0 ? a0 : 0.f; a1 = c1 ? a1 : 0.f;
            const f2_t al = f2_pack(a0, a1);
            const f2_t w = f2_mul(T2, al);              // Eq.6: c_i alpha_i prod_{j<i} (1 - alpha_j)
            Cr2 = f2_fma(w, f2_bc(g4.x), Cr2); Cg2 = f2_fma(w, f2_bc(g4.y), Cg2); Cb2 = f2_fma(w, f2_bc(g4.z), Cb2);
            if (DEPTH) Cd2 = f2_fma(w, f2_bc(g4.w), Cd2);
            T2 = f2_mul(T2, f2_fma(al, f2_bc(-1.f), f2_bc(1.f)));
            float t0, t1;
            f2_unpack(T2, t0, t1);
            const uint32_t bit = 1u << (jj - g0), nl = (uint32_t)(b0 + jj) + 1u;
            if (c0) { if (MARK) mw[0] |= bit; n_last[0] = nl; if (t0 < rp.teps) open &= ~1u; }      // Alg.1 l.27: test after the update
            if (c1) { if (MARK) mw[PX - 1] |= bit; n_last[PX - 1] = nl; if (t1 < rp.teps) open &= ~2u; }
            continue;
          } else
#pragma unroll
          for (int j = 0; j < PX; ++j) {
            p2[j] = 1.f;
            if (PX == 1 || (alive & (1u << j))) {     // warp-uniform
              Eval ev;
              if (PX == 1 && COUNT) {
                // Informational: k >= 1, so power = q k^2 <= q for q <= 0; where q is below the alpha_min cut for every open
                // pixel of the patch, c and k would not be needed.  The production kernel does NOT take this early out: after the
                // patch cull it removes 7 % (config 4) to 30 % (config 5) of the visits and the vote costs every visit 8
                // instructions: 2.73 -> 2.53 ms and 3.29 -> 3.21 ms without it.  work[3] says what it would save.
                ev.a = fmaf(g1.x, ts.px[j], fmaf(g1.y, ts.pz[j], g0v.x));
                ev.b = fmaf(g1.z, ts.px[j], fmaf(g1.w, ts.py[j], fmaf(g2.x, ts.pz[j], g0v.y)));
                const float q = fmaf(ev.a, fmaf(g3.x, ev.a, g3.y * ev.b), g3.z * ev.b * ev.b);
                const bool maybe = open && !(q > 0.f) && q * 0.999999f >= g0v.w;
                const bool pass = __any_sync(0xffffffffu, maybe);
                if (open && (uint64_t)jj < left_n && ((live >> (jj - g0)) & 1u)) { ++n_cull; if (pass) ++n_full; }
              }
              eval_entry(g0v, g1, g2, g3, ts.px[j], ts.py[j], ts.pz[j], ev);
              p2[j] = ev.p2;
              if (COUNT && ((open >> j) & 1u) && (uint64_t)jj < left_n) ++n_eval;       // null padding entries are not Alg.1's
              if (((open >> j) & 1u) && may_contribute(ev, g0v.w)) cand |= 1u << j;
            }
          }
          if (PX > 2 && !__any_sync(0xffffffffu, cand != 0)) continue;
          if (PX <= 2 && cand == 0) continue;
          const float4 g4 = lds128(sa + 4u * kRow);
          const uint32_t bit = 1u << (jj - g0);
#pragma unroll
          for (int j = 0; j < PX; ++j) {
            if (!((cand >> j) & 1u)) continue;
            const float a = fminf(rp.amax, g3.w * ex2_approx(p2[j]));
            if (a < rp.amin) continue;
            if (MARK) mw[j] |= bit;                   // this pixel blended the entry
            if (COUNT) ++n_contrib;
            const float w = T[j] * a;                 // Eq.6: c_i alpha_i prod_{j<i} (1 - alpha_j)
            Cr[j] = fmaf(w, g4.x, Cr[j]); Cg[j] = fmaf(w, g4.y, Cg[j]); Cb[j] = fmaf(w, g4.z, Cb[j]);
            if (DEPTH) Cd[j] = fmaf(w, g4.w, Cd[j]);  // D = sum_i T_i alpha_i / rho_i, no background term
            T[j] = T[j] * (1.f - a);
            n_last[j] = (uint32_t)(b0 + jj) + 1u;
            if (T[j] < rp.teps) open &= ~(1u << j);   // Alg.1 l.27: test after the update
          }
        }
      }
      if (MARK) {                                     // the patches' words of the group (written even when 0: the buffer is not cleared)
#pragma unroll
        for (int j = 0; j < PX; ++j) {
          const uint32_t gw = __reduce_or_sync(0xffffffffu, mw[j]);
          if ((threadIdx.x & 31) == 0) mark_w[(uint64_t)j * plane_words + ((b0 + (uint64_t)g0) >> 5)] = gw;
        }
      }
    }
  }
  if (PX == 2 && !COUNT) {
    f2_unpack(T2, T[0], T[PX - 1]); f2_unpack(Cr2, Cr[0], Cr[PX - 1]); f2_unpack(Cg2, Cg[0], Cg[PX - 1]); f2_unpack(Cb2, Cb[0], Cb[PX - 1]);
    if (DEPTH) f2_unpack(Cd2, Cd[0], Cd[PX - 1]);
  }
  if (COUNT) {
    const uint32_t e = __reduce_add_sync(0xffffffffu, n_eval), c = __reduce_add_sync(0xffffffffu, n_contrib);
    const uint32_t u = __reduce_add_sync(0xffffffffu, n_cull), f = __reduce_add_sync(0xffffffffu, n_full);
    if ((threadIdx.x & 31) == 0) {
      atomicAdd(work, (unsigned long long)e); atomicAdd(work + 1, (unsigned long long)c);
      atomicAdd(work + 2, (unsigned long long)u); atomicAdd(work + 3, (unsigned long long)f);
    }
  }
#pragma unroll
  for (int j = 0; j < PX; ++j) {
    const size_t o = ts.out0 + (size_t)32 * j;
    if (ts.on[j]) {
      color[3 * o] = fmaf(T[j], rp.bg[0], Cr[j]); color[3 * o + 1] = fmaf(T[j], rp.bg[1], Cg[j]); color[3 * o + 2] = fmaf(T[j], rp.bg[2], Cb[j]);
      alpha_out[o] = 1.f - T[j]; trans_out[o] = T[j]; n_last_out[o] = n_last[j];
      if (DEPTH) depth_out[o] = Cd[j];
    } else {
      color[3 * o] = 0.f; color[3 * o + 1] = 0.f; color[3 * o + 2] = 0.f;
      alpha_out[o] = 0.f; trans_out[o] = 1.f; n_last_out[o] = 0u;
      if (DEPTH) depth_out[o] = 0.f;
    }
  }
}

// ------------------------------------------------------------------------------------------------ backward
__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
  return x;
}

#ifndef UTS_BWD_MINB
#define UTS_BWD_MINB 8   // 8 blocks of 64 threads per SM: 128 registers; at 138 registers (7 blocks) the kernel takes 5.0 instead of 4.4 ms
#endif
template <int PX, bool MARK, bool DEPTH = false>
__global__ void __launch_bounds__(kTilePix / PX, UTS_BWD_MINB)
render_bwd_kernel(RenderParams rp, const float* __restrict__ dir, const float* __restrict__ conic_opac, const float* __restrict__ rgb,
                  const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ mask_bits,
                  const uint64_t* __restrict__ ranges, const uint32_t* __restrict__ vals, const float* __restrict__ trans,
                  const uint32_t* __restrict__ n_last_in, const float* __restrict__ dL_dcolor, const float* __restrict__ dL_dalpha,
                  float* __restrict__ dL_drgb, float* __restrict__ dL_dconic, float* __restrict__ dL_dmu2, float* __restrict__ dL_dopac,
                  const uint32_t* __restrict__ marks, uint64_t plane_words, const float* __restrict__ rho = nullptr,
                  const float* __restrict__ dL_ddepth = nullptr, float* __restrict__ dL_dinvr = nullptr) {
  constexpr int kThreads = kTilePix / PX, kWarps = kThreads / 32;
  __shared__ SEntries<true> S;
  __shared__ TileFrame s_tf;
  __shared__ uint32_t s_max[kWarps];
  TileSetup<PX> ts;
  setup_tile<PX>(rp, active_tiles, mask_bits, ranges, &s_tf, ts);
  const TileFrame tf = s_tf;
  const size_t gbase = (size_t)ts.v * rp.P;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;

  uint32_t nl[PX];
  float T[PX], Sr[PX], Sg[PX], Sb[PX], gr[PX], gg[PX], gb[PX], ga_T[PX];
  float Sd[PX], gd[PX];                                 // DEPTH: depth accumulated behind the entry; upstream dL/dD
  uint32_t m = 0;
#pragma unroll
  for (int j = 0; j < PX; ++j) {
    const size_t o = ts.out0 + (size_t)32 * j;
    const bool on = ts.on[j];
    nl[j] = on ? __ldg(n_last_in + o) : 0u;
    const float Tfin = on ? __ldg(trans + o) : 1.f;
    gr[j] = on ? __ldg(dL_dcolor + 3 * o) : 0.f; gg[j] = on ? __ldg(dL_dcolor + 3 * o + 1) : 0.f; gb[j] = on ? __ldg(dL_dcolor + 3 * o + 2) : 0.f;
    ga_T[j] = (dL_dalpha && on) ? __ldg(dL_dalpha + o) * Tfin : 0.f;          // dL/dalpha_out * T_final
    T[j] = Tfin;                                        // transmittance after the entry being visited
    Sr[j] = Tfin * rp.bg[0]; Sg[j] = Tfin * rp.bg[1]; Sb[j] = Tfin * rp.bg[2];  // colour accumulated behind it
    Sd[j] = 0.f; gd[j] = (DEPTH && on) ? __ldg(dL_ddepth + o) : 0.f;
    m = max(m, nl[j]);
  }
  // PX even: the per-pixel state as packed pairs (pixels 2p, 2p + 1), walked with packed arithmetic (visit below)
  constexpr bool kPack = (PX % 2) == 0;
  constexpr int NP = kPack ? PX / 2 : 1;
  f2_t px2[NP], py2[NP], pz2[NP], T2[NP], Sr2[NP], Sg2[NP], Sb2[NP], Sd2[NP], gr2[NP], gg2[NP], gb2[NP], gaT2[NP], gd2[NP];
#pragma unroll
  for (int q = 0; q < NP; ++q) {
    const int j0 = kPack ? 2 * q : 0, j1 = kPack ? 2 * q + 1 : 0;
    px2[q] = f2_pack(ts.px[j0], ts.px[j1]); py2[q] = f2_pack(ts.py[j0], ts.py[j1]); pz2[q] = f2_pack(ts.pz[j0], ts.pz[j1]);
    T2[q] = f2_pack(T[j0], T[j1]); Sr2[q] = f2_pack(Sr[j0], Sr[j1]); Sg2[q] = f2_pack(Sg[j0], Sg[j1]); Sb2[q] = f2_pack(Sb[j0], Sb[j1]);
    Sd2[q] = 0; gr2[q] = f2_pack(gr[j0], gr[j1]); gg2[q] = f2_pack(gg[j0], gg[j1]); gb2[q] = f2_pack(gb[j0], gb[j1]);
    gaT2[q] = f2_pack(ga_T[j0], ga_T[j1]); gd2[q] = f2_pack(gd[j0], gd[j1]);
  }
  // block maximum of n_last: entries beyond it were reached by no pixel
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
  if (lane == 0) s_max[wid] = m;
  __syncthreads();
  uint32_t max_nl = 0;
#pragma unroll
  for (int w = 0; w < kWarps; ++w) max_nl = max(max_nl, s_max[w]);
  if (max_nl == 0) return;

  // the gradient word this lane owns after the butterfly below (lanes 4j: value j), as base pointer + stride per Gaussian:
  // bit4 -> +4, bit3 -> +2, bit2 -> +1  (0 r, 1 g, 2 b, 3 A, 4 B, 5 C, 6 omega, 7 phi)
  const int vi = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
  float* lane_dst = (vi < 3 ? dL_drgb + vi : vi < 6 ? dL_dconic + (vi - 3) : dL_dmu2 + (vi - 6)) + (size_t)(vi < 6 ? 3 : 2) * gbase;
  uint32_t lane_stride = vi < 6 ? 3u : 2u;
  if (lane == 1) { lane_dst = dL_dopac; lane_stride = 1u; }                    // lane 1 owns the opacity sum (summed over views)
  if (DEPTH && lane == 2) { lane_dst = dL_dinvr + gbase; lane_stride = 1u; }   // lane 2 the 1/rho sum
  const bool lane_owns = (lane & 3) == 0 || lane == 1 || (DEPTH && lane == 2);
  asm volatile("" : "+l"(lane_dst));                   // keep the per-view base folded into the pointer (one IMAD.WIDE per atomic)
  const uint32_t sS = (uint32_t)__cvta_generic_to_shared(&S);   // (pinning it in a register as in the forward costs two registers: 3.54 -> 3.58 ms)

  const int n_batch = (int)((max_nl + kBatch - 1) / kBatch);
  // lane 8 j + g (j < PX) reads word g of patch j's plane, kWarps j + wid
  const uint32_t* mark_w = nullptr;
  if (MARK && lane < 8 * PX) mark_w = marks + (uint64_t)(PX * wid + (lane >> 3)) * plane_words + mark_base<PX>(rp, ts);
  for (int bi = n_batch - 1; bi >= 0; --bi) {
    const uint32_t b0 = (uint32_t)bi * kBatch;
    // The forward wrote a patch's words up to the last entry any of its pixels blended; words beyond that hold whatever the
    // buffer held (it is never cleared) — a set bit there only costs the evaluation, because no pixel of the patch reaches
    // such an entry (jl < nl below).
    uint32_t myw = 0u;
    if (MARK && lane < 8 * PX) myw = __ldg(mark_w + (size_t)bi * 8 + (lane & 7));
    __syncthreads();
    stage_batch<PX, true, DEPTH>(S, tf, rp, dir, conic_opac, rgb, rho, vals, ts.start + b0, (uint64_t)(max_nl - b0), gbase);
    __syncthreads();
    const int nb = (int)min((uint32_t)kBatch, max_nl - b0);
    // one list entry for the patches in pm (bit j: patch j of this warp)
    auto visit = [&](const int jj, const uint32_t pm) {
      const uint32_t jl = b0 + (uint32_t)jj;
      const uint32_t sa = sS + (uint32_t)jj * 16u;
      const float4 g0v = lds128(sa), g1 = lds128(sa + kRow), g2 = lds128(sa + 2u * kRow), g3 = lds128(sa + 3u * kRow), g4 = lds128(sa + 4u * kRow);
      float d_r = 0.f, d_g = 0.f, d_b = 0.f, d_A = 0.f, d_B = 0.f, d_C = 0.f, d_o = 0.f, d_om = 0.f, d_ph = 0.f, d_i = 0.f;
      const float2 g5 = *reinterpret_cast<const float2*>(&S.g[5][jj]);
      const float inv_r = DEPTH ? S.g[5][jj].z : 0.f;
      bool any_used = false;
      if constexpr (kPack) {
        // Two pixels (patches 2q, 2q + 1 of the warp) per step in packed fp32 pairs, branch-free: a pixel that did not take the
        // entry gets alpha = 0 and zero gradient weights, which leave its state and every sum exactly as they were.
        f2_t s_r = 0, s_g = 0, s_b = 0, s_A = 0, s_B = 0, s_C = 0, s_o = 0, s_om = 0, s_ph = 0, s_i = 0;
        const float cA = -2.f / kLog2e * g3.x, cB = -1.f / kLog2e * g3.y, cC = -2.f / kLog2e * g3.z;   // conic (A,B,C)
        const float sp = g5.x, cp = g5.y;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          if (!((pm >> (2 * q)) & 3u)) continue;       // warp-uniform: neither patch has the entry marked
          Eval2 ev;
          eval_entry2(g0v, g1, g2, g3, px2[q], py2[q], pz2[q], ev);
          float p20, p21;
          f2_unpack(ev.p2, p20, p21);
          bool u0 = ((pm >> (2 * q)) & 1u) && jl < nl[2 * q] && may_contribute(p20, g0v.w);
          bool u1 = ((pm >> (2 * q + 1)) & 1u) && jl < nl[2 * q + 1] && may_contribute(p21, g0v.w);
          const float e20 = ex2_approx(p20), e21 = ex2_approx(p21);
          const float raw0 = g3.w * e20, raw1 = g3.w * e21;
          float a0 = fminf(rp.amax, raw0), a1 = fminf(rp.amax, raw1);
          u0 = u0 && !(a0 < rp.amin); u1 = u1 && !(a1 < rp.amin);
          if (!(u0 || u1)) continue;
          any_used = true;
          a0 = u0 ? a0 : 0.f; a1 = u1 ? a1 : 0.f;
          const f2_t al = f2_pack(a0, a1);
          float m0, m1;
          f2_unpack(f2_fma(al, f2_bc(-1.f), f2_bc(1.f)), m0, m1);                        // 1 - alpha
          const float i0 = u0 ? rcp_approx(fmaxf(m0, 1e-7f)) : 1.f, i1 = u1 ? rcp_approx(fmaxf(m1, 1e-7f)) : 1.f;
          const f2_t inv = f2_pack(i0, i1), ninv = f2_pack(-i0, -i1);
          const f2_t Tb = f2_mul(T2[q], inv);            // transmittance before this entry
          const f2_t w = f2_mul(Tb, al);
          s_r = f2_fma(w, gr2[q], s_r); s_g = f2_fma(w, gg2[q], s_g); s_b = f2_fma(w, gb2[q], s_b);
          f2_t dLa = f2_mul(gr2[q], f2_fma(Tb, f2_bc(g4.x), f2_mul(Sr2[q], ninv)));
          dLa = f2_fma(gg2[q], f2_fma(Tb, f2_bc(g4.y), f2_mul(Sg2[q], ninv)), dLa);
          dLa = f2_fma(gb2[q], f2_fma(Tb, f2_bc(g4.z), f2_mul(Sb2[q], ninv)), dLa);
          dLa = f2_fma(gaT2[q], inv, dLa);
          Sr2[q] = f2_fma(w, f2_bc(g4.x), Sr2[q]); Sg2[q] = f2_fma(w, f2_bc(g4.y), Sg2[q]); Sb2[q] = f2_fma(w, f2_bc(g4.z), Sb2[q]);
          if (DEPTH) {
            s_i = f2_fma(w, gd2[q], s_i);
            dLa = f2_fma(gd2[q], f2_fma(Tb, f2_bc(inv_r), f2_mul(Sd2[q], ninv)), dLa);
            Sd2[q] = f2_fma(w, f2_bc(inv_r), Sd2[q]);
          }
          T2[q] = Tb;
          // reading A7: no gradient through a clamped alpha
          const bool h0 = u0 && !(raw0 > rp.amax), h1 = u1 && !(raw1 > rp.amax);
          s_o = f2_fma(f2_pack(h0 ? e20 : 0.f, h1 ? e21 : 0.f), dLa, s_o);               // exp(power) dL/dalpha
          const f2_t ngp = f2_mul(f2_pack(h0 ? -a0 : 0.f, h1 ? -a1 : 0.f), dLa);         // - dL/dpower
          const f2_t dx = f2_mul(ev.k, ev.a), dy = f2_mul(ev.k, ev.b);
          s_A = f2_fma(f2_mul(f2_mul(f2_bc(0.5f), dx), dx), ngp, s_A);
          s_B = f2_fma(f2_mul(dx, dy), ngp, s_B);
          s_C = f2_fma(f2_mul(f2_mul(f2_bc(0.5f), dy), dy), ngp, s_C);
          const f2_t gdx = f2_mul(f2_fma(f2_bc(cA), dx, f2_mul(f2_bc(cB), dy)), ngp);
          const f2_t gdy = f2_mul(f2_fma(f2_bc(cB), dx, f2_mul(f2_bc(cC), dy)), ngp);
          // (dx,dy) = k(s,c) (a,b):  dk/ds / s = (c/den - k)/t,  dk/dc = -1/den,  den = s^2 + c^2;  t = 0: g_a = k gdx = gdx, g_c = 0
          const f2_t t = f2_fma(ev.a, ev.a, f2_mul(ev.b, ev.b));
          float t0, t1, den0, den1;
          f2_unpack(t, t0, t1);
          f2_unpack(f2_fma(ev.c, ev.c, t), den0, den1);
          const f2_t iden = f2_pack(rcp_approx(den0), rcp_approx(den1));
          const f2_t rt = f2_pack(t0 > 0.f ? rcp_approx(t0) : 0.f, t1 > 0.f ? rcp_approx(t1) : 0.f);
          const f2_t gk = f2_fma(gdx, ev.a, f2_mul(gdy, ev.b));
          const f2_t gkkp = f2_mul(gk, f2_mul(f2_fma(ev.c, iden, f2_mul(ev.k, f2_bc(-1.f))), rt));
          const f2_t g_a = f2_fma(gkkp, ev.a, f2_mul(ev.k, gdx));
          const f2_t g_b = f2_fma(gkkp, ev.b, f2_mul(ev.k, gdy));
          const f2_t g_c = f2_mul(f2_mul(gk, f2_bc(-1.f)), iden);
          // a = e.w, b = n.w, c = u.w with de/dom = -hh, dn/dom = -sin(phi) e, du/dom = cos(phi) e, dn/dphi = -u, du/dphi = n,
          // and hh.w = cos(phi) c - sin(phi) b
          s_om = f2_fma(g_a, f2_fma(f2_bc(-cp), ev.c, f2_mul(f2_bc(sp), ev.b)), s_om);
          s_om = f2_fma(f2_mul(g_b, f2_bc(-sp)), ev.a, s_om);
          s_om = f2_fma(f2_mul(g_c, f2_bc(cp)), ev.a, s_om);
          s_ph = f2_fma(g_c, ev.b, s_ph);
          s_ph = f2_fma(f2_mul(g_b, f2_bc(-1.f)), ev.c, s_ph);
        }
        float lo, hi;
        f2_unpack(s_r, lo, hi); d_r = lo + hi; f2_unpack(s_g, lo, hi); d_g = lo + hi; f2_unpack(s_b, lo, hi); d_b = lo + hi;
        f2_unpack(s_A, lo, hi); d_A = lo + hi; f2_unpack(s_B, lo, hi); d_B = lo + hi; f2_unpack(s_C, lo, hi); d_C = lo + hi;
        f2_unpack(s_o, lo, hi); d_o = lo + hi; f2_unpack(s_om, lo, hi); d_om = lo + hi; f2_unpack(s_ph, lo, hi); d_ph = lo + hi;
        if (DEPTH) { f2_unpack(s_i, lo, hi); d_i = lo + hi; }
      } else
#pragma unroll
      for (int j = 0; j < PX; ++j) {
        if (PX > 1 && !((pm >> j) & 1u)) continue;     // warp-uniform
        Eval ev;
        eval_entry(g0v, g1, g2, g3, ts.px[j], ts.py[j], ts.pz[j], ev);
        bool used = jl < nl[j] && may_contribute(ev, g0v.w);       // jl < nl: this pixel's forward pass got this far
        float e2 = 0.f, raw = 0.f, a = 0.f;
        if (used) { e2 = ex2_approx(ev.p2); raw = g3.w * e2; a = fminf(rp.amax, raw); used = !(a < rp.amin); }
        if (!used) continue;
        any_used = true;
        const float inv1a = rcp_approx(fmaxf(1.f - a, 1e-7f));      // alpha = 1 (alpha_max = 1, opacity 1 at the centre): finite
        const float Tb = T[j] * inv1a;                 // transmittance before this entry
        const float w = Tb * a;
        d_r = fmaf(w, gr[j], d_r); d_g = fmaf(w, gg[j], d_g); d_b = fmaf(w, gb[j], d_b);
        float dLa = gr[j] * (Tb * g4.x - Sr[j] * inv1a) + gg[j] * (Tb * g4.y - Sg[j] * inv1a) + gb[j] * (Tb * g4.z - Sb[j] * inv1a) +
                    ga_T[j] * inv1a;
        Sr[j] = fmaf(w, g4.x, Sr[j]); Sg[j] = fmaf(w, g4.y, Sg[j]); Sb[j] = fmaf(w, g4.z, Sb[j]);
        if (DEPTH) {                                   // the fourth channel, same algebra as a colour channel with c_i = 1 / rho_i
          d_i = fmaf(w, gd[j], d_i);
          dLa = fmaf(gd[j], Tb * inv_r - Sd[j] * inv1a, dLa);
          Sd[j] = fmaf(w, inv_r, Sd[j]);
        }
        T[j] = Tb;
        if (raw > rp.amax) continue;                   // reading A7: no gradient through a clamped alpha
        d_o = fmaf(e2, dLa, d_o);                      // exp(power) dL/dalpha
        const float gp = a * dLa;                      // dL/dpower
        const float dx = ev.k * ev.a, dy = ev.k * ev.b;
        const float cA = -2.f / kLog2e * g3.x, cB = -1.f / kLog2e * g3.y, cC = -2.f / kLog2e * g3.z;   // conic (A,B,C)
        d_A = fmaf(-0.5f * dx * dx, gp, d_A); d_B = fmaf(-dx * dy, gp, d_B); d_C = fmaf(-0.5f * dy * dy, gp, d_C);
        const float gdx = -(cA * dx + cB * dy) * gp, gdy = -(cB * dx + cC * dy) * gp;
        // (dx,dy) = k(s,c) (a,b):  dk/ds / s = (c/den - k)/t,  dk/dc = -1/den,  den = s^2 + c^2
        float g_a = gdx, g_b = gdy, g_c = 0.f;
        if (ev.t > 0.f) {
          const float den = ev.t + ev.c * ev.c;
          const float gk = gdx * ev.a + gdy * ev.b;
          const float iden = rcp_approx(den);
          const float kp = (ev.c * iden - ev.k) * rcp_approx(ev.t);
          g_a = fmaf(gk * kp, ev.a, ev.k * gdx);
          g_b = fmaf(gk * kp, ev.b, ev.k * gdy);
          g_c = -gk * iden;
        }
        // a = e.w, b = n.w, c = u.w with de/dom = -hh, dn/dom = -sin(phi) e, du/dom = cos(phi) e, dn/dphi = -u, du/dphi = n,
        // and hh.w = cos(phi) c - sin(phi) b
        const float sp = g5.x, cp = g5.y;
        d_om += -g_a * (cp * ev.c - sp * ev.b) - g_b * sp * ev.a + g_c * cp * ev.a;
        d_ph += g_c * ev.b - g_b * ev.c;
      }
      if (!__any_sync(0xffffffffu, any_used)) return;
      // 9 sums over the warp (each lane already holds the sum over its PX pixels).  Eight of them go through a transposing
      // butterfly: at each of the first three steps a lane keeps half of its values and hands the other half to its partner, so
      // 4+2+1 shuffles leave every lane with ONE value summed over 8 lanes, and two more steps finish it: 9 shuffles instead of
      // 40.  Lane 4*j ends up owning value j.
      float v0 = d_r, v1 = d_g, v2 = d_b, v3 = d_A, v4 = d_B, v5 = d_C, v6 = d_om, v7 = d_ph;
      {
        const bool hi = lane & 16;
        const float s0 = hi ? v0 : v4, s1 = hi ? v1 : v5, s2 = hi ? v2 : v6, s3 = hi ? v3 : v7;
        const float k0 = hi ? v4 : v0, k1 = hi ? v5 : v1, k2 = hi ? v6 : v2, k3 = hi ? v7 : v3;
        v0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 16); v1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 16);
        v2 = k2 + __shfl_xor_sync(0xffffffffu, s2, 16); v3 = k3 + __shfl_xor_sync(0xffffffffu, s3, 16);
      }
      {
        const bool hi = lane & 8;
        const float s0 = hi ? v0 : v2, s1 = hi ? v1 : v3;
        const float k0 = hi ? v2 : v0, k1 = hi ? v3 : v1;
        v0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 8); v1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 8);
      }
      {
        const bool hi = lane & 4;
        const float s0 = hi ? v0 : v1, k0 = hi ? v1 : v0;
        v0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 4);
      }
      v0 += __shfl_xor_sync(0xffffffffu, v0, 2);
      v0 += __shfl_xor_sync(0xffffffffu, v0, 1);
      d_o = warp_sum(d_o);
      if (DEPTH) d_i = warp_sum(d_i);
      if (lane_owns) red_add_global(lane_dst + (size_t)__float_as_uint(g4.w) * lane_stride, lane == 1 ? d_o : ((DEPTH && lane == 2) ? d_i : v0));
    };
    if (MARK) {
      for (int grp = (nb - 1) >> 5; grp >= 0; --grp) {
        uint32_t w[PX], wb = 0;
#pragma unroll
        for (int j = 0; j < PX; ++j) { w[j] = __shfl_sync(0xffffffffu, myw, 8 * j + grp); wb |= w[j]; }
        if (nb - 32 * grp < 32) wb &= (1u << (nb - 32 * grp)) - 1u;   // entries >= nb: beyond the tile's largest n_last
        while (wb) {                                                  // back to front over the marked entries
          const int bit = 31 - __clz((int)wb);
          wb &= ~(1u << bit);
          uint32_t pm = 0;
#pragma unroll
          for (int j = 0; j < PX; ++j) pm |= ((w[j] >> bit) & 1u) << j;
          visit(32 * grp + bit, pm);
        }
      }
    } else {
      for (int jj = nb - 1; jj >= 0; --jj) {
        const uint32_t jl = b0 + (uint32_t)jj;
        uint32_t reach = 0;
#pragma unroll
        for (int j = 0; j < PX; ++j) reach |= (jl < nl[j] ? 1u : 0u) << j;
        const uint32_t pm = __reduce_or_sync(0xffffffffu, reach);     // patches with a pixel that got this far
        if (pm) visit(jj, pm);
      }
    }
  }
}

static RenderParams make_params(const uts_config* cfg, const Dims& d) {
  RenderParams rp;
  rp.k = d.k; rp.P = d.P; rp.n_tile = d.n_tile; rp.n_slot = d.n_slot;
  rp.amin = cfg->alpha_min; rp.amax = cfg->alpha_max; rp.teps = cfg->t_eps;
  rp.bg[0] = cfg->bg[0]; rp.bg[1] = cfg->bg[1]; rp.bg[2] = cfg->bg[2];
  return rp;
}

}  // namespace uts

using namespace uts;

extern "C" {

static uint64_t mark_plane_words(const uts_config* cfg, uint64_t pair_capacity) {
  const uint64_t n_vt = (uint64_t)cfg->n_views * ((uint64_t)12 << (2 * (cfg->order - cfg->tile_log2)));
  return (pair_capacity >> 5) + n_vt + 16;            // runs start at (start >> 5) + vt; a batch read takes 8 words
}

size_t uts_render_marks_bytes(const uts_config* cfg, uint64_t pair_capacity) {
  if (check_config(cfg) != UTS_OK) return 0;
  return (size_t)mark_plane_words(cfg, pair_capacity) * 8 * sizeof(uint32_t);
}

static int render_fwd_impl(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                           float* color, float* alpha, float* trans, uint32_t* n_last, uint32_t* marks, uint64_t plane_words, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!in.dir || !in.conic_opac || !in.rgb || !ranges || !color || !alpha || !trans || !n_last) return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, &mask);
  if (d.n_slot == 0) return UTS_OK;
  if (d.n_slot * d.V > 0x7fffffffll) return UTS_ERR_UNSUPPORTED;
  RenderParams rp = make_params(cfg, d);
  if (marks)
    render_fwd_kernel<kFwdPx, true><<<(unsigned)(d.n_slot * d.V), kTilePix / kFwdPx, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, color, alpha, trans, n_last, marks, plane_words);
  else
    render_fwd_kernel<kFwdPx, false><<<(unsigned)(d.n_slot * d.V), kTilePix / kFwdPx, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, color, alpha, trans, n_last, nullptr, 0);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_render_fwd(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                   float* color, float* alpha, float* trans, uint32_t* n_last, void* stream) {
  return render_fwd_impl(cfg, in, mask, ranges, vals, color, alpha, trans, n_last, nullptr, 0, stream);
}

int uts_render_fwd_counted(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                           float* color, float* alpha, float* trans, uint32_t* n_last, uint64_t* work, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!in.dir || !in.conic_opac || !in.rgb || !ranges || !color || !alpha || !trans || !n_last || !work) return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, &mask);
  if (d.n_slot == 0) return UTS_OK;
  if (d.n_slot * d.V > 0x7fffffffll) return UTS_ERR_UNSUPPORTED;
  RenderParams rp = make_params(cfg, d);
  render_fwd_kernel<1, false, true><<<(unsigned)(d.n_slot * d.V), kTilePix, 0, (cudaStream_t)stream>>>(
      rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, color, alpha, trans, n_last, nullptr, 0,
      reinterpret_cast<unsigned long long*>(work));
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_render_fwd_marked(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                          uint64_t pair_capacity, float* color, float* alpha, float* trans, uint32_t* n_last, uint32_t* marks,
                          size_t marks_bytes, void* stream) {
  if (!marks || check_config(cfg) != UTS_OK) return UTS_ERR_INVALID_ARG;
  const uint64_t pw = mark_plane_words(cfg, pair_capacity);
  if (marks_bytes < (size_t)pw * 8 * sizeof(uint32_t)) return UTS_ERR_CAPACITY;
  return render_fwd_impl(cfg, in, mask, ranges, vals, color, alpha, trans, n_last, marks, pw, stream);
}

static int render_bwd_impl(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                           const float* trans, const uint32_t* n_last, const float* dL_dcolor, const float* dL_dalpha,
                           float* dL_drgb, float* dL_dconic, float* dL_dmu2, float* dL_dopac, const uint32_t* marks, uint64_t plane_words,
                           void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!in.dir || !in.conic_opac || !in.rgb || !ranges || !trans || !n_last || !dL_dcolor) return UTS_ERR_INVALID_ARG;
  if (!dL_drgb || !dL_dconic || !dL_dmu2 || !dL_dopac) return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, &mask);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t vp = (size_t)d.V * d.P;
  UTS_CUDA(cudaMemsetAsync(dL_drgb, 0, vp * 3 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dconic, 0, vp * 3 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dmu2, 0, vp * 2 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dopac, 0, (size_t)d.P * sizeof(float), s));
  if (d.n_slot == 0 || d.P == 0) return UTS_OK;
  if (d.n_slot * d.V > 0x7fffffffll) return UTS_ERR_UNSUPPORTED;
  RenderParams rp = make_params(cfg, d);
  if (marks)
    render_bwd_kernel<kBwdPx, true><<<(unsigned)(d.n_slot * d.V), kTilePix / kBwdPx, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, trans, n_last, dL_dcolor,
        dL_dalpha, dL_drgb, dL_dconic, dL_dmu2, dL_dopac, marks, plane_words);
  else
    render_bwd_kernel<kBwdPx, false><<<(unsigned)(d.n_slot * d.V), kTilePix / kBwdPx, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, trans, n_last, dL_dcolor,
        dL_dalpha, dL_drgb, dL_dconic, dL_dmu2, dL_dopac, nullptr, 0);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_render_bwd(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                   const float* trans, const uint32_t* n_last, const float* dL_dcolor, const float* dL_dalpha,
                   float* dL_drgb, float* dL_dconic, float* dL_dmu2, float* dL_dopac, void* stream) {
  return render_bwd_impl(cfg, in, mask, ranges, vals, trans, n_last, dL_dcolor, dL_dalpha, dL_drgb, dL_dconic, dL_dmu2, dL_dopac, nullptr, 0,
                         stream);
}

int uts_render_bwd_marked(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                          uint64_t pair_capacity, const float* trans, const uint32_t* n_last, const uint32_t* marks,
                          const float* dL_dcolor, const float* dL_dalpha, float* dL_drgb, float* dL_dconic, float* dL_dmu2,
                          float* dL_dopac, void* stream) {
  if (!marks || check_config(cfg) != UTS_OK) return UTS_ERR_INVALID_ARG;
  return render_bwd_impl(cfg, in, mask, ranges, vals, trans, n_last, dL_dcolor, dL_dalpha, dL_drgb, dL_dconic, dL_dmu2, dL_dopac, marks,
                         mark_plane_words(cfg, pair_capacity), stream);
}

// ---- colour + inverse radial depth in one blend pass
int uts_render_fwd_depth(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                         uint64_t pair_capacity, float* color, float* alpha, float* trans, uint32_t* n_last, float* depth,
                         uint32_t* marks, size_t marks_bytes, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!in.dir || !in.conic_opac || !in.rgb || !in.rho || !ranges || !color || !alpha || !trans || !n_last || !depth) return UTS_ERR_INVALID_ARG;
  uint64_t pw = 0;
  if (marks) {
    pw = mark_plane_words(cfg, pair_capacity);
    if (marks_bytes < (size_t)pw * 8 * sizeof(uint32_t)) return UTS_ERR_CAPACITY;
  }
  Dims d = dims_of(cfg, &mask);
  if (d.n_slot == 0) return UTS_OK;
  if (d.n_slot * d.V > 0x7fffffffll) return UTS_ERR_UNSUPPORTED;
  RenderParams rp = make_params(cfg, d);
  const unsigned grid = (unsigned)(d.n_slot * d.V);
  cudaStream_t s = (cudaStream_t)stream;
  if (marks)
    render_fwd_kernel<kFwdPx, true, false, true><<<grid, kTilePix / kFwdPx, 0, s>>>(rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits,
                                                                                   ranges, vals, color, alpha, trans, n_last, marks, pw, nullptr, in.rho, depth);
  else
    render_fwd_kernel<kFwdPx, false, false, true><<<grid, kTilePix / kFwdPx, 0, s>>>(rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits,
                                                                                    ranges, vals, color, alpha, trans, n_last, nullptr, 0, nullptr, in.rho, depth);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_render_bwd_depth(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                         uint64_t pair_capacity, const float* trans, const uint32_t* n_last, const uint32_t* marks,
                         const float* dL_dcolor, const float* dL_dalpha, const float* dL_ddepth, float* dL_drgb, float* dL_dconic,
                         float* dL_dmu2, float* dL_dopac, float* dL_dinvr, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!in.dir || !in.conic_opac || !in.rgb || !in.rho || !ranges || !trans || !n_last || !dL_dcolor || !dL_ddepth) return UTS_ERR_INVALID_ARG;
  if (!dL_drgb || !dL_dconic || !dL_dmu2 || !dL_dopac || !dL_dinvr) return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, &mask);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t vp = (size_t)d.V * d.P;
  UTS_CUDA(cudaMemsetAsync(dL_drgb, 0, vp * 3 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dconic, 0, vp * 3 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dmu2, 0, vp * 2 * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dopac, 0, (size_t)d.P * sizeof(float), s));
  UTS_CUDA(cudaMemsetAsync(dL_dinvr, 0, vp * sizeof(float), s));
  if (d.n_slot == 0 || d.P == 0) return UTS_OK;
  if (d.n_slot * d.V > 0x7fffffffll) return UTS_ERR_UNSUPPORTED;
  RenderParams rp = make_params(cfg, d);
  const unsigned grid = (unsigned)(d.n_slot * d.V);
  if (marks)
    render_bwd_kernel<kBwdPx, true, true><<<grid, kTilePix / kBwdPx, 0, s>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, trans, n_last, dL_dcolor, dL_dalpha, dL_drgb,
        dL_dconic, dL_dmu2, dL_dopac, marks, mark_plane_words(cfg, pair_capacity), in.rho, dL_ddepth, dL_dinvr);
  else
    render_bwd_kernel<kBwdPx, false, true><<<grid, kTilePix / kBwdPx, 0, s>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, trans, n_last, dL_dcolor, dL_dalpha, dL_drgb,
        dL_dconic, dL_dmu2, dL_dopac, nullptr, 0, in.rho, dL_ddepth, dL_dinvr);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // extern "C"
