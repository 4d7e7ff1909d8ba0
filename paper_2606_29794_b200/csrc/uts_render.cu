// uts_render.cu — F5/F6: front-to-back alpha blending at every HEALPix pixel centre with the FoV mask
// (Alg.1 l.17-30 PAPER.md:563-587; Eq.6; SphericalOffset PAPER.md:112; mask PAPER.md:62, 129), and
// B1: its backward.
//
// One thread block per active tile, one thread per pixel (thread id = p & 255, the NESTED low bits, so a warp is a
// compact 8x4 pixel patch).  The tile's sorted list is staged through shared memory in batches of 256 entries.
//
// SphericalOffset without inverse trigonometry in the common case, and without fp32 cancellation (DESIGN.md
// "Kernels/F5"):  with Gaussian direction u and its east/north unit vectors e, n, and pixel direction w,
//     a = e.w, b = n.w, c = u.w,  sin(d_gc) = sqrt(a^2+b^2),  (d_x,d_y) = (d_gc / sin d_gc) (a,b)
// is the haversine distance + bearing decomposition of PAPER.md:112 in vector form.  Because e.u = n.u = 0,
// a = e.(w-u) and b = n.(w-u): the difference w-u = (c_tile - u) + (w - c_tile) is formed in double precision once per
// (tile, Gaussian) and once per pixel, then everything per (pixel, Gaussian) is fp32 FMAs on small, exactly known
// differences.  k = d_gc/sin d_gc = P(c) rsqrt(1+c) with a degree-7 polynomial P for c = cos d_gc >= 0 (atan2f beyond
// 90 degrees).  power*log2(e) = k^2 (qa a^2 + qb a b + qc b^2) with the conic pre-scaled at staging; alpha uses ex2.
#include "uts_internal.cuh"

namespace uts {

struct RenderParams {
  int k, P;
  int64_t n_tile, n_slot;
  float amin, amax, teps, bg[3];
};

constexpr float kLog2e = 1.4426950408889634f;

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
__device__ __forceinline__ float2 lds64(uint32_t addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
  return v;
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

// What one (tile, Gaussian) list entry contributes to every pixel of the tile, staged once per entry.
struct Entry {
  float a0, b0, c0, o;          // e.(c_tile-u), n.(c_tile-u), uhat.c_tile, opacity
  float ex, ez, nx, ny;         // e = (ex, 0, ez)
  float nz, ux, uy, uz;         // uhat
  float qa, qb, qc, r;          // -0.5 A log2e, -B log2e, -0.5 C log2e, red
  float g, bl;                  // green, blue
};

struct TileFrame { double cx, cy, cz; };              // tile centre direction (order k_t pixel centre)

__device__ __forceinline__ void stage_entry(const TileFrame& tf, float ux, float uy, float uz, float4 co, float r, float g,
                                            float b, Entry& E) {
  const float dxf = (float)(tf.cx - (double)ux), dyf = (float)(tf.cy - (double)uy), dzf = (float)(tf.cz - (double)uz);
  const float rxz2 = ux * ux + uz * uz;
  float ex = 1.f, ez = 0.f;
  if (rxz2 > 0.f) { const float inv = rsqrtf(rxz2); ex = uz * inv; ez = -ux * inv; }    // pole guard: reading A22
  const float invn = rsqrtf(rxz2 + uy * uy);
  const float hx = ux * invn, hy = uy * invn, hz = uz * invn;
  const float nx = hy * ez, ny = hz * ex - hx * ez, nz = -hy * ex;                       // n = uhat x e
  E.a0 = ex * dxf + ez * dzf;
  E.b0 = nx * dxf + ny * dyf + nz * dzf;
  E.c0 = hx * (float)tf.cx + hy * (float)tf.cy + hz * (float)tf.cz;
  E.o = co.w;
  E.ex = ex; E.ez = ez; E.nx = nx; E.ny = ny; E.nz = nz; E.ux = hx; E.uy = hy; E.uz = hz;
  E.qa = -0.5f * kLog2e * co.x; E.qb = -kLog2e * co.y; E.qc = -0.5f * kLog2e * co.z;
  E.r = r; E.g = g; E.bl = b;
}

struct SEntry {                                       // shared-memory layout: broadcast reads of float4
  float4 f0[kTilePix], f1[kTilePix], f2[kTilePix], f3[kTilePix];
  float2 f4[kTilePix];
};

__device__ __forceinline__ void put_entry(SEntry& S, int i, const Entry& E) {
  S.f0[i] = make_float4(E.a0, E.b0, E.c0, E.o);
  S.f1[i] = make_float4(E.ex, E.ez, E.nx, E.ny);
  S.f2[i] = make_float4(E.nz, E.ux, E.uy, E.uz);
  S.f3[i] = make_float4(E.qa, E.qb, E.qc, E.r);
  S.f4[i] = make_float2(E.g, E.bl);
}

struct Eval { float a, b, c, t, k, p2; };

// Shared by forward and backward so that both take the same skip / clamp decisions.
__device__ __forceinline__ void eval_entry(const float4 f0, const float4 f1, const float4 f2, const float4 f3, float px,
                                           float py, float pz, Eval& ev) {
  ev.a = fmaf(f1.x, px, fmaf(f1.y, pz, f0.x));
  ev.b = fmaf(f1.z, px, fmaf(f1.w, py, fmaf(f2.x, pz, f0.y)));
  ev.c = fmaf(f2.y, px, fmaf(f2.z, py, fmaf(f2.w, pz, f0.z)));
  ev.t = fmaf(ev.a, ev.a, ev.b * ev.b);
  ev.k = arc_over_sin(ev.t, ev.c);
  const float q = fmaf(ev.a, fmaf(f3.x, ev.a, f3.y * ev.b), f3.z * ev.b * ev.b);     // qa a^2 + qb a b + qc b^2
  ev.p2 = q * ev.k * ev.k;
}

// Pixel and tile set-up common to both kernels.
struct PixelSetup { float px, py, pz; bool on; size_t out; uint64_t start, end; int v; int64_t tile; };

__device__ __forceinline__ void setup_pixel(const RenderParams& rp, const uint32_t* __restrict__ active_tiles,
                                            const uint32_t* __restrict__ mask_bits, const uint64_t* __restrict__ ranges,
                                            TileFrame* s_tf, PixelSetup& ps) {
  const int64_t slot = blockIdx.x % rp.n_slot;
  ps.v = (int)(blockIdx.x / rp.n_slot);
  const int64_t tile = active_tiles ? (int64_t)__ldg(active_tiles + slot) : slot;
  const uint64_t p = (uint64_t)tile * kTilePix + threadIdx.x;
  ps.tile = tile;
  ps.on = mask_bits ? ((__ldg(mask_bits + (p >> 5)) >> (p & 31)) & 1u) != 0 : true;
  ps.out = ((size_t)ps.v * rp.n_slot + slot) * kTilePix + threadIdx.x;
  const uint64_t rix = 2 * ((uint64_t)ps.v * rp.n_tile + tile);
  ps.start = __ldg(ranges + rix); ps.end = __ldg(ranges + rix + 1);
  if (threadIdx.x == 0) pix_center_cam(rp.k - kTileLog2, (uint64_t)tile, s_tf->cx, s_tf->cy, s_tf->cz);
  double wx, wy, wz;
  pix_center_cam(rp.k, p, wx, wy, wz);
  __syncthreads();
  ps.px = (float)(wx - s_tf->cx); ps.py = (float)(wy - s_tf->cy); ps.pz = (float)(wz - s_tf->cz);
}

// Marks (uts_render_fwd_marked / uts_render_bwd_marked): one bit per (warp of the tile's block, list entry), set by the forward
// when at least one of the warp's 32 pixels blended the entry.  Plane w (of 8) holds warp w's bits; the bits of (view, tile) vt
// start at word (start_vt >> 5) + vt of the plane, entry j of the list at bit j of that run — runs of different tiles never share a
// word.  The backward walks only the set bits: on the paper's kind of scene half of the (warp, entry) visits re-evaluate alpha just
// to find that no pixel of the warp took the entry.
__device__ __forceinline__ uint64_t mark_base(const RenderParams& rp, const PixelSetup& ps, int64_t tile) {
  return (ps.start >> 5) + (uint64_t)ps.v * (uint64_t)rp.n_tile + (uint64_t)tile;
}

template <bool MARK>
__global__ void __launch_bounds__(kTilePix)
render_fwd_kernel(RenderParams rp, const float* __restrict__ dir, const float* __restrict__ conic_opac, const float* __restrict__ rgb,
                  const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ mask_bits,
                  const uint64_t* __restrict__ ranges, const uint32_t* __restrict__ vals, float* __restrict__ color,
                  float* __restrict__ alpha_out, float* __restrict__ trans_out, uint32_t* __restrict__ n_last_out,
                  uint32_t* __restrict__ marks, uint64_t plane_words) {
  __shared__ SEntry S;
  __shared__ TileFrame s_tf;
  PixelSetup ps;
  setup_pixel(rp, active_tiles, mask_bits, ranges, &s_tf, ps);
  const TileFrame tf = s_tf;
  const size_t gbase = (size_t)ps.v * rp.P;

  float T = 1.f, Cr = 0.f, Cg = 0.f, Cb = 0.f;
  uint32_t n_last = 0;
  bool done = !ps.on;
  const uint64_t len = ps.end - ps.start;
  const uint32_t sS = (uint32_t)__cvta_generic_to_shared(&S);
  uint32_t* mark_w = nullptr;                         // this warp's run of mark words for the tile
  if (MARK) mark_w = marks + (uint64_t)(threadIdx.x >> 5) * plane_words + mark_base(rp, ps, ps.tile);
  for (uint64_t b0 = 0; b0 < len; b0 += kTilePix) {
    if (__syncthreads_and(done)) break;               // every pixel of the tile saturated (or masked)
    const uint64_t j = b0 + threadIdx.x;
    if (j < len) {
      const size_t gi = gbase + __ldg(vals + ps.start + j);
      Entry E;
      stage_entry(tf, __ldg(dir + 3 * gi), __ldg(dir + 3 * gi + 1), __ldg(dir + 3 * gi + 2),
                  __ldg(reinterpret_cast<const float4*>(conic_opac) + gi), __ldg(rgb + 3 * gi), __ldg(rgb + 3 * gi + 1),
                  __ldg(rgb + 3 * gi + 2), E);
      put_entry(S, threadIdx.x, E);
    } else if (j < len + 3) {
      // null entries pad the list to a multiple of 4: a = 1, qa = 1 give power > 0, which Alg.1 l.23 skips whatever the thresholds
      S.f0[threadIdx.x] = make_float4(1.f, 0.f, 0.f, 0.f); S.f1[threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
      S.f2[threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f); S.f3[threadIdx.x] = make_float4(1.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
    const int nb = (int)((len - b0) < (uint64_t)kTilePix ? (len - b0) : (uint64_t)kTilePix);
    // four entries per warp vote: the vote only ends the walk early, every skip / clamp decision is per lane.  The batch is walked
    // in groups of 32 entries, one mark word each.
    bool left = false;
    for (int g0 = 0; g0 < nb && !left; g0 += 32) {
      uint32_t mw = 0;                                // this lane's marks of the group
      const int ge = min(nb, g0 + 32);
      for (int j4 = g0; j4 < ge; j4 += 4) {
        if (__all_sync(0xffffffffu, done)) { left = true; break; }     // warp vote: the whole 8x4 patch is saturated
        const uint32_t bit4 = 1u << (j4 - g0);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int jj = j4 + u;
          const uint32_t sa = sS + (uint32_t)jj * 16u;
          const float4 f0 = lds128(sa), f1 = lds128(sa + 0x1000u), f2 = lds128(sa + 0x2000u), f3 = lds128(sa + 0x3000u);
          Eval ev;
          eval_entry(f0, f1, f2, f3, ps.px, ps.py, ps.pz, ev);
          if (done || ev.p2 > 0.f) continue;          // Alg.1 l.23: power > 0 skipped (reading A7)
          const float a = fminf(rp.amax, f0.w * ex2_approx(ev.p2));
          if (a < rp.amin) continue;
          if (MARK) mw |= bit4 << u;                  // this lane blended the entry
          const float2 f4 = lds64(sS + 0x4000u + (uint32_t)jj * 8u);
          const float w = T * a;                      // Eq.6: c_i alpha_i prod_{j<i} (1 - alpha_j)
          Cr = fmaf(w, f3.w, Cr); Cg = fmaf(w, f4.x, Cg); Cb = fmaf(w, f4.y, Cb);
          T = T * (1.f - a);
          n_last = (uint32_t)(b0 + jj) + 1u;
          if (T < rp.teps) done = true;               // Alg.1 l.27: test after the update
        }
      }
      if (MARK) {                                     // the warp's word of the group (written even when 0: the buffer is not cleared)
        const uint32_t gw = __reduce_or_sync(0xffffffffu, mw);
        if ((threadIdx.x & 31) == 0) mark_w[(b0 + (uint64_t)g0) >> 5] = gw;
      }
    }
  }
  if (ps.on) {
    color[3 * ps.out] = fmaf(T, rp.bg[0], Cr); color[3 * ps.out + 1] = fmaf(T, rp.bg[1], Cg); color[3 * ps.out + 2] = fmaf(T, rp.bg[2], Cb);
    alpha_out[ps.out] = 1.f - T; trans_out[ps.out] = T; n_last_out[ps.out] = n_last;
  } else {
    color[3 * ps.out] = 0.f; color[3 * ps.out + 1] = 0.f; color[3 * ps.out + 2] = 0.f;
    alpha_out[ps.out] = 0.f; trans_out[ps.out] = 1.f; n_last_out[ps.out] = 0u;
  }
}

// ------------------------------------------------------------------------------------------------ backward
__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
  return x;
}

struct SEntryBwd {
  float4 f0[kTilePix], f1[kTilePix], f2[kTilePix], f3[kTilePix];
  float4 f5[kTilePix];                                 // green, blue, sin(phi), cos(phi)
  uint32_t id[kTilePix];
};

template <bool MARK>
__global__ void __launch_bounds__(kTilePix)
render_bwd_kernel(RenderParams rp, const float* __restrict__ dir, const float* __restrict__ conic_opac, const float* __restrict__ rgb,
                  const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ mask_bits,
                  const uint64_t* __restrict__ ranges, const uint32_t* __restrict__ vals, const float* __restrict__ trans,
                  const uint32_t* __restrict__ n_last_in, const float* __restrict__ dL_dcolor, const float* __restrict__ dL_dalpha,
                  float* __restrict__ dL_drgb, float* __restrict__ dL_dconic, float* __restrict__ dL_dmu2, float* __restrict__ dL_dopac,
                  const uint32_t* __restrict__ marks, uint64_t plane_words) {
  __shared__ SEntryBwd S;
  __shared__ TileFrame s_tf;
  __shared__ uint32_t s_max[kTilePix / 32];
  PixelSetup ps;
  setup_pixel(rp, active_tiles, mask_bits, ranges, &s_tf, ps);
  const TileFrame tf = s_tf;
  const size_t gbase = (size_t)ps.v * rp.P;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;

  const uint32_t nl = ps.on ? __ldg(n_last_in + ps.out) : 0u;
  const float Tfin = ps.on ? __ldg(trans + ps.out) : 1.f;
  const float gr = ps.on ? __ldg(dL_dcolor + 3 * ps.out) : 0.f, gg = ps.on ? __ldg(dL_dcolor + 3 * ps.out + 1) : 0.f,
              gb = ps.on ? __ldg(dL_dcolor + 3 * ps.out + 2) : 0.f;
  const float ga_T = (dL_dalpha && ps.on) ? __ldg(dL_dalpha + ps.out) * Tfin : 0.f;      // dL/dalpha_out * T_final
  // block maximum of n_last: entries beyond it were reached by no pixel
  uint32_t m = nl;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
  if (lane == 0) s_max[wid] = m;
  __syncthreads();
  uint32_t max_nl = 0;
#pragma unroll
  for (int w = 0; w < kTilePix / 32; ++w) max_nl = max(max_nl, s_max[w]);
  if (max_nl == 0) return;

  // the gradient word this lane owns after the butterfly below (lanes 4j: value j), as base pointer + stride per Gaussian:
  // bit4 -> +4, bit3 -> +2, bit2 -> +1  (0 r, 1 g, 2 b, 3 A, 4 B, 5 C, 6 omega, 7 phi)
  const int vi = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
  float* lane_dst = (vi < 3 ? dL_drgb + vi : vi < 6 ? dL_dconic + (vi - 3) : dL_dmu2 + (vi - 6)) + (size_t)(vi < 6 ? 3 : 2) * gbase;
  uint32_t lane_stride = vi < 6 ? 3u : 2u;
  if (lane == 1) { lane_dst = dL_dopac; lane_stride = 1u; }                    // lane 1 owns the opacity sum (summed over views)
  const bool lane_owns = (lane & 3) == 0 || lane == 1;
  asm volatile("" : "+l"(lane_dst));                   // keep the per-view base folded into the pointer (one IMAD.WIDE per atomic)
  const uint32_t sS = (uint32_t)__cvta_generic_to_shared(&S);

  float T = Tfin;                                      // transmittance after the entry being visited
  float Sr = Tfin * rp.bg[0], Sg = Tfin * rp.bg[1], Sb = Tfin * rp.bg[2];                // colour accumulated behind it
  const int n_batch = (int)((max_nl + kTilePix - 1) / kTilePix);
  const uint32_t* mark_w = nullptr;                    // this warp's run of mark words for the tile (see render_fwd_kernel)
  if (MARK) mark_w = marks + (uint64_t)wid * plane_words + mark_base(rp, ps, ps.tile);
  for (int bi = n_batch - 1; bi >= 0; --bi) {
    const uint32_t b0 = (uint32_t)bi * kTilePix;
    // lane g < 8: the marks of entries b0 + 32 g .. + 31.  The forward wrote this warp's words up to the last entry any of its
    // pixels blended; words beyond that hold whatever the buffer held (it is never cleared) — a set bit there only costs the
    // visit's first vote, because no pixel of the warp reaches such an entry.
    uint32_t myw = 0u;
    if (MARK && lane < 8) myw = __ldg(mark_w + (size_t)bi * 8 + lane);
    __syncthreads();
    const uint32_t j = b0 + threadIdx.x;
    if (j < max_nl) {
      const uint32_t id = __ldg(vals + ps.start + j);
      const size_t gi = gbase + id;
      const float ux = __ldg(dir + 3 * gi), uy = __ldg(dir + 3 * gi + 1), uz = __ldg(dir + 3 * gi + 2);
      Entry E;
      stage_entry(tf, ux, uy, uz, __ldg(reinterpret_cast<const float4*>(conic_opac) + gi), __ldg(rgb + 3 * gi),
                  __ldg(rgb + 3 * gi + 1), __ldg(rgb + 3 * gi + 2), E);
      S.f0[threadIdx.x] = make_float4(E.a0, E.b0, E.c0, E.o);
      S.f1[threadIdx.x] = make_float4(E.ex, E.ez, E.nx, E.ny);
      S.f2[threadIdx.x] = make_float4(E.nz, E.ux, E.uy, E.uz);
      S.f3[threadIdx.x] = make_float4(E.qa, E.qb, E.qc, E.r);
      S.f5[threadIdx.x] = make_float4(E.g, E.bl, E.uy, sqrtf(E.ux * E.ux + E.uz * E.uz));
      S.id[threadIdx.x] = id;
    }
    __syncthreads();
    const int nb = (int)min((uint32_t)kTilePix, max_nl - b0);
    auto visit = [&](const int jj) {
      const uint32_t jl = b0 + (uint32_t)jj;
      const bool reach = jl < nl;                      // this pixel's forward pass got this far
      if (!__any_sync(0xffffffffu, reach)) return;
      const uint32_t sa = sS + (uint32_t)jj * 16u;
      const float4 f0 = lds128(sa), f1 = lds128(sa + 0x1000u), f2 = lds128(sa + 0x2000u), f3 = lds128(sa + 0x3000u), f5 = lds128(sa + 0x4000u);
      Eval ev;
      eval_entry(f0, f1, f2, f3, ps.px, ps.py, ps.pz, ev);
      float e2 = 0.f, raw = 0.f, a = 0.f;
      bool used = reach && !(ev.p2 > 0.f);
      if (used) { e2 = ex2_approx(ev.p2); raw = f0.w * e2; a = fminf(rp.amax, raw); used = !(a < rp.amin); }
      if (!__any_sync(0xffffffffu, used)) return;
      float d_r = 0.f, d_g = 0.f, d_b = 0.f, d_A = 0.f, d_B = 0.f, d_C = 0.f, d_o = 0.f, d_om = 0.f, d_ph = 0.f;
      if (used) {
        const float inv1a = rcp_approx(1.f - a);
        const float Tb = T * inv1a;                    // transmittance before this entry
        const float w = Tb * a;
        d_r = w * gr; d_g = w * gg; d_b = w * gb;
        float dLa = gr * (Tb * f3.w - Sr * inv1a) + gg * (Tb * f5.x - Sg * inv1a) + gb * (Tb * f5.y - Sb * inv1a) + ga_T * inv1a;
        Sr = fmaf(w, f3.w, Sr); Sg = fmaf(w, f5.x, Sg); Sb = fmaf(w, f5.y, Sb);
        T = Tb;
        if (!(raw > rp.amax)) {                        // reading A7: no gradient through a clamped alpha
          d_o = e2 * dLa;                              // exp(power) dL/dalpha
          const float gp = a * dLa;                    // dL/dpower
          const float dx = ev.k * ev.a, dy = ev.k * ev.b;
          const float cA = -2.f / kLog2e * f3.x, cB = -1.f / kLog2e * f3.y, cC = -2.f / kLog2e * f3.z;   // conic (A,B,C)
          d_A = -0.5f * dx * dx * gp; d_B = -dx * dy * gp; d_C = -0.5f * dy * dy * gp;
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
          const float sp = f5.z, cp = f5.w;
          d_om = -g_a * (cp * ev.c - sp * ev.b) - g_b * sp * ev.a + g_c * cp * ev.a;
          d_ph = g_c * ev.b - g_b * ev.c;
        }
      }
      // 9 sums over the warp.  Eight of them go through a transposing butterfly: at each of the first three steps a lane
      // keeps half of its values and hands the other half to its partner, so 4+2+1 shuffles leave every lane with ONE value
      // summed over 8 lanes, and two more steps finish it: 9 shuffles instead of 40.  Lane 4*j ends up owning value j.
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
      {
        const uint32_t id = S.id[jj];
        if (lane_owns) red_add_global(lane_dst + (size_t)id * lane_stride, lane == 1 ? d_o : v0);
      }
    };
    if (MARK) {
      for (int grp = (nb - 1) >> 5; grp >= 0; --grp) {
        uint32_t wb = __shfl_sync(0xffffffffu, myw, grp);
        if (nb - 32 * grp < 32) wb &= (1u << (nb - 32 * grp)) - 1u;   // entries >= nb: beyond the tile's largest n_last
        while (wb) {                                                  // back to front over the marked entries
          const int bit = 31 - __clz((int)wb);
          wb &= ~(1u << bit);
          visit(32 * grp + bit);
        }
      }
    } else {
      for (int jj = nb - 1; jj >= 0; --jj) visit(jj);
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
    render_fwd_kernel<true><<<(unsigned)(d.n_slot * d.V), kTilePix, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, color, alpha, trans, n_last, marks, plane_words);
  else
    render_fwd_kernel<false><<<(unsigned)(d.n_slot * d.V), kTilePix, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, color, alpha, trans, n_last, nullptr, 0);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_render_fwd(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                   float* color, float* alpha, float* trans, uint32_t* n_last, void* stream) {
  return render_fwd_impl(cfg, in, mask, ranges, vals, color, alpha, trans, n_last, nullptr, 0, stream);
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
    render_bwd_kernel<true><<<(unsigned)(d.n_slot * d.V), kTilePix, 0, (cudaStream_t)stream>>>(
        rp, in.dir, in.conic_opac, in.rgb, mask.active_tiles, mask.pixel_mask_bits, ranges, vals, trans, n_last, dL_dcolor,
        dL_dalpha, dL_drgb, dL_dconic, dL_dmu2, dL_dopac, marks, plane_words);
  else
    render_bwd_kernel<false><<<(unsigned)(d.n_slot * d.V), kTilePix, 0, (cudaStream_t)stream>>>(
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

}  // extern "C"
