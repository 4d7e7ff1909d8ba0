// uts_ring_query.cuh — ring-interval evaluation of the tile set (F2; Alg.1 l.9-14 PAPER.md:548-559).
//
// The set to compute (reading A6 for Alg.2, Alg.3 for the RING mode) is
//     T = { q >> 2(k_q - k_t) : q an order-k_q pixel, u . centre(q) >= cos R }.
// Alg.2 reaches it by a quadtree descent, one node test per step; the paper's Alg.3 (Eq.5) notes that on an
// iso-latitude ring the in-disc centres form ONE longitude interval.  This file uses that structure for both modes:
//   phase 1  per ring i of order k_q that the disc can reach: the exact interval [first, last] of in-disc pixel positions
//            (an fp32 estimate from Eq.5 in chord form, then the ends are settled by testing pixels — fp32 chord with a margin,
//            the defining double-precision predicate inside the margin), so all floating point work is O(rings), not O(tiles);
//   phase 2  per (face, tile diagonal S = X+Y) "tile row": a tile (X,Y) owns, on each of the 2m-1 rings it spans
//            (m = 2^(k_q-k_t)), a run of pixel positions; it belongs to T iff one of those runs meets that ring's interval.
//            This is integer interval arithmetic and yields a bit mask of the row's tiles — no per-tile geometry at all.
// Coordinates: a pixel of ring i sits at the integer position g = F2*n_r + (x - y) (mod 8 n_r), longitude (pi/4) g / n_r, with
// n_r = min(i, N, 4N - i), F2 = 2c + 1 - (r & 1) for face f = 4r + c, and ring i = (r + 2) N - 1 - (x + y)  (HEALPix ring form,
// Gorski et al. as cited at PAPER.md:23).  All pixels of a ring share the parity of g.
// Everything here is __host__ __device__ so that the same code is checked on the CPU against the oracle's sets
// (tests/test_ring_query_host.py) before it runs in a kernel.
#pragma once
#include "uts_internal.cuh"

namespace uts {

constexpr float kRingDelta = 4e-6f;       // fp32 chord margin, as in the descent's zone tests
constexpr int kRingFull = 1 << 28;        // |first|, |last| of a ring that lies entirely inside the disc

struct RingDisc {
  float dir[3];                           // the record's direction as stored (fp32)
  double un[3];                           // the same, normalised in double: what the defining predicate uses
  double R, cosR;                         // min(pi, r_s + rho_q) and its cosine
  float lq;                               // longitude in eighth-ring units: g_c = lq * n_r, lq in [0,8)
  float dq;                               // the disc's longitude half-extent in the same units (4 = everywhere)
  float zc, sc, T2, T2lo, T2hi;           // z and sin(colatitude) of u; chord thresholds T^2, (T -+ delta)^2, T = 2 sin(R/2)
  int i_lo, i_hi;                         // rings that can hold an in-disc centre (superset)
  bool all;                               // R >= pi: every tile (reading A24)
};

__host__ __device__ __forceinline__ int ring_n(int N, int i) { return min(i, min(N, 4 * N - i)); }
__host__ __device__ __forceinline__ int ring_parity(int N, int i) { return (i < N || i > 3 * N) ? 1 : ((N + 1 + i) & 1); }

// sin(t) for |t| <= pi/2 + 0.05 with relative error 1e-7 (own fit of sin(t)/t in t^2); independent of --use_fast_math
__host__ __device__ __forceinline__ float sin_poly(float t) {
  const float x = t * t;
  return t * (0.99999999416f + x * (-0.16666655522f + x * (0.00833299300f + x * (-0.000198048254f + x * 2.5956970e-06f))));
}

// real-valued ring coordinate of colatitude theta (ring i sits at coordinate i); fp32, good to a small fraction of a ring
__host__ __device__ __forceinline__ float ring_coord(int N, float theta) {
  const float z = cosf(theta);
  if (z >= 0.6666667f) return (float)N * 2.4494897f * sinf(0.5f * theta);
  if (z <= -0.6666667f) return 4.0f * (float)N - (float)N * 2.4494897f * cosf(0.5f * theta);
  return (float)N * (2.0f - 1.5f * z);
}

// dir: the projected record's unit direction (fp32); lon, lat: its (omega, phi) of Eq.1 (fp32, from the same record).
// The fp32 quantities only steer estimates and margin-guarded tests; the defining predicate uses dir and R in double.
__host__ __device__ __forceinline__ void make_ring_disc(int kq, const float dir[3], float lon, float lat, double R, RingDisc& D) {
  const int N = 1 << kq;
  D.dir[0] = dir[0]; D.dir[1] = dir[1]; D.dir[2] = dir[2];
  {
    const double ux = (double)dir[0], uy = (double)dir[1], uz = (double)dir[2];
    const double nrm = sqrt(ux * ux + uy * uy + uz * uz);
    D.un[0] = ux / nrm; D.un[1] = uy / nrm; D.un[2] = uz / nrm;
  }
  D.R = R;
  D.cosR = cos(R);
  D.all = R >= kPi;
  const float Rf = (float)R;
  const float T = 2.0f * sin_poly(0.5f * Rf);
  D.T2 = T * T;
  D.T2lo = T > kRingDelta ? (T - kRingDelta) * (T - kRingDelta) : -1.0f;
  D.T2hi = (T + kRingDelta) * (T + kRingDelta);
  D.zc = dir[1]; D.sc = sqrtf(dir[0] * dir[0] + dir[2] * dir[2]);
  float lq = lon * 1.2732395447351628f;
  if (lq < 0.0f) lq += 8.0f;
  if (!(lq < 8.0f)) lq = 0.0f;
  D.lq = lq;
  const float th = 1.5707963267948966f - lat;
  const float t0 = th - Rf - 4e-6f, t1 = th + Rf + 4e-6f;
  D.i_lo = max(1, (int)ceilf(ring_coord(N, fmaxf(0.0f, t0))) - 1);
  D.i_hi = min(4 * N - 1, (int)floorf(ring_coord(N, fminf(3.14159265f, t1))) + 1);
  // longitude extent: a disc that holds no pole stays within asin(sin R / sin theta_c) of its centre's meridian
  if (t0 <= 1e-5f || t1 >= 3.14158f || !(D.sc > 0.0f)) D.dq = 4.0f;
  else D.dq = asinf(fminf(1.0f, sinf(Rf) / D.sc)) * 1.2732395447351628f + 1e-3f;
}

// can face f hold a tile of the disc?  (its pixels lie within one eighth-ring unit of F2 on every ring)
__host__ __device__ __forceinline__ bool face_in_extent(const RingDisc& D, int f) {
  const int F2 = 2 * (f & 3) + 1 - ((f >> 2) & 1);
  float d = fabsf(D.lq - (float)F2);
  if (d > 4.0f) d = 8.0f - d;
  return d <= 1.0f + D.dq;
}

// the defining predicate  u . centre >= cos R  for the pixel at position g of ring i, in double.  With the centre
// (sth sin(lam), z, sth cos(lam)), sth = sqrt(s2) >= 0:  sth A >= B  with  A = u_x sin(lam) + u_z cos(lam),  B = cos R - u_y z,
// decided on the squares (s2 A^2 against B^2) so that no square root is taken; un and cos R come with the disc.  (The form with
// sqrt, a normalisation and cos(R) per call was 18 % of the count kernels' instructions: ncu source view, round 2.)
// The ring number passes through an empty volatile asm: without it the compiler hoists the part that depends on the ring alone out
// of the callers' loops and executes it — in double — for every ring, whether or not any pixel falls inside the fp32 margin
// (another 10 % of the instructions); as a __noinline__ call instead, the count kernels lost more to the call's register spills
// than they gained (config 4 tile lists 7.6 -> 8.6 ms).
__host__ __device__ __forceinline__ bool ring_pixel_inside_exact(const RingDisc& D, int N, int i, int g) {
#ifdef __CUDA_ARCH__
  asm volatile("" : "+r"(i));
#endif
  double z, s2;
  int n;
  const double inv3N2 = 1.0 / (3.0 * (double)N * (double)N);
  if (i < N) { n = i; const double w = (double)n * (double)n * inv3N2; z = 1.0 - w; s2 = w * (2.0 - w); }
  else if (i > 3 * N) { n = 4 * N - i; const double w = (double)n * (double)n * inv3N2; z = w - 1.0; s2 = w * (2.0 - w); }
  else { n = N; z = (double)(2 * (2 * N - i)) / (double)(3 * N); s2 = (1.0 - z) * (1.0 + z); }
  const double lam = (kPi / 4) * ((double)g / (double)n);
  double sn, cs;
  sincos(lam, &sn, &cs);
  const double A = D.un[0] * sn + D.un[2] * cs, B = D.cosR - D.un[1] * z;
  const double lhs = s2 * A * A, rhs = B * B;
  if (B <= 0.0) return A >= 0.0 || lhs <= rhs;
  return A > 0.0 && lhs >= rhs;
}

// Phase 1.  In-disc pixel positions of ring i: the integers g = first, first+2, ..., last (not reduced mod 8 n_r;
// |g - g_c| <= 4 n_r).  Empty: last < first.  Whole ring: first = -kRingFull, last = +kRingFull.
__host__ __device__ __forceinline__ void ring_interval(const RingDisc& D, int N, int i, int& first, int& last) {
  first = 0; last = -1;
  int n;
  float z, s;
  const float invN = 1.0f / (float)N;
  const float inv3N2 = 0.333333343f * invN * invN;
  if (i < N) { n = i; const float fn = (float)n; const float w = fn * fn * inv3N2; z = 1.0f - w; s = sqrtf(w * (2.0f - w)); }
  else if (i > 3 * N) { n = 4 * N - i; const float fn = (float)n; const float w = fn * fn * inv3N2; z = w - 1.0f; s = sqrtf(w * (2.0f - w)); }
  else { n = N; z = (float)(2 * (2 * N - i)) * (0.333333343f * invN); s = sqrtf((1.0f - z) * (1.0f + z)); }
  const float dz = z - D.zc, ds = s - D.sc;
  const float A = dz * dz + ds * ds, B = 4.0f * s * D.sc;      // chord^2(g) = A + B sin^2((lam_g - lam_c)/2) >= A
  if (A > D.T2hi) return;
  const int par = ring_parity(N, i);
  const double gc = (double)D.lq * (double)n;                              // exact product: g_c reaches 8 * 8192
  const int g0 = 2 * (int)floor(0.5 * (gc - (double)par) + 0.5) + par;     // pixel position nearest to g_c
  const float frac = (float)(gc - (double)g0);                             // in [-1, 1]
  const float k = 0.39269908169872414f / (float)n;                         // (pi/8) / n_r: half the longitude step per unit g
  auto inside = [&](int g) -> bool {
    float t = fabsf((float)(g - g0) - frac) * k;
    if (t > 1.5707963267948966f) t = 3.14159265358979f - t;
    const float sn = sin_poly(t);
    const float c2 = A + B * sn * sn;
    if (c2 < D.T2lo) return true;
    if (c2 > D.T2hi) return false;
    return ring_pixel_inside_exact(D, N, i, g);
  };
  if (!inside(g0)) return;
  // estimated half width in g units from sin^2(dlam/2) <= (T^2 - A)/B (Eq.5 PAPER.md:106 in chord form)
  const float y = (D.T2 - A) / B;
  float hw;
  if (!(y < 1.0f)) hw = 4.0f * (float)n;
  else if (!(y > 0.0f)) hw = 0.0f;
  else hw = asinf(sqrtf(y)) * (2.5464790894703255f * (float)n);          // (8/pi) n_r
  const int fmin = g0 - 4 * n, lmax = g0 + 4 * n;
  int f = g0 - 2 * (int)floorf(fmaxf(0.0f, 0.5f * (hw - frac)));
  int l = g0 + 2 * (int)floorf(fmaxf(0.0f, 0.5f * (hw + frac)));
  f = max(f, fmin); l = min(l, lmax);
  if (inside(f)) { while (f > fmin && inside(f - 2)) f -= 2; }
  else { do f += 2; while (f < g0 && !inside(f)); }
  if (inside(l)) { while (l < lmax && inside(l + 2)) l += 2; }
  else { do l -= 2; while (l > g0 && !inside(l)); }
  if (((l - f) >> 1) + 1 >= 4 * n) { first = -kRingFull; last = kRingFull; }
  else { first = f; last = l; }
}

// Tile rows of face f that the ring range [i_lo, i_hi] can touch: S in [S_lo, S_hi] (empty if S_lo > S_hi).
__host__ __device__ __forceinline__ void face_row_range(const RingDisc& D, int kq, int kt, int f, int& S_lo, int& S_hi) {
  const int N = 1 << kq, Nt = 1 << kt, ref = kq - kt, m = 1 << ref;
  const int top = ((f >> 2) + 2) * N - 1;                                   // x + y = top - ring
  const int cmin = max(0, top - D.i_hi), cmax = min(2 * N - 2, top - D.i_lo);
  if (cmin > cmax) { S_lo = 0; S_hi = -1; return; }
  S_lo = max(0, (cmin - m + 1) >> ref);
  S_hi = min(2 * Nt - 2, cmax >> ref);
}

// Phase 2.  Tiles of row (face f, S = X + Y) are H = X - Y = -Hm + 2j, j = 0..Hm, Hm = min(S, 2 Nt - 2 - S).
// Returns the membership mask of candidates j = jbase .. jbase + 63.  `tab(i)` yields the (first, last) of ring i in [i_lo, i_hi].
template <class Tab>
__host__ __device__ __forceinline__ unsigned long long tile_row_mask(const RingDisc& D, int kq, int kt, int f, int S, int jbase, const Tab& tab) {
  const int N = 1 << kq, Nt = 1 << kt, ref = kq - kt, m = 1 << ref;
  const int r = f >> 2, c = f & 3;
  const int top = (r + 2) * N - 1, F2 = 2 * c + 1 - (r & 1);
  const int Hm = min(S, 2 * Nt - 2 - S);
  const int jtop = min(Hm, jbase + 63);
  unsigned long long mask = 0;
  // rings of this tile row inside the disc's ring range only: i = top - (m S + d) in [i_lo, i_hi]
  const int d_lo = max(0, top - m * S - D.i_hi), d_hi = min(2 * m - 2, top - m * S - D.i_lo);
  for (int d = d_lo; d <= d_hi; ++d) {
    const int i = top - (m * S + d);
    int first, last;
    tab(i, first, last);
    if (last < first) continue;
    const int n = ring_n(N, i), a = F2 * n, w = min(d, 2 * m - 2 - d);
    // the run of this tile on ring i is [a + mH - w, a + mH + w]; it must meet [first, last] + 8 n k for some k.  The copy
    // whose middle is nearest to the face (|mid + 8 n k - a| <= 4 n) is the only one that can reach the face's pixels
    // (|g - a| < n) unless the interval is wider than 6 n; then its two neighbours are tried as well.
    int k0 = 0, kw = 0;
    if (first != -kRingFull) {
      const int mid = (first + last) >> 1;
      k0 = a - mid > 4 * n ? 1 : (mid - a > 4 * n ? -1 : 0);
      kw = last - first >= 6 * n ? 1 : 0;
    }
    for (int k = k0 - kw; k <= k0 + kw; ++k) {
      const int P = first + 8 * n * k - a - w, Q = last + 8 * n * k - a + w;     // P <= m H <= Q
      const int Hlo = (P + m - 1) >> ref, Hhi = Q >> ref;
      const int jlo = max(jbase, (Hlo + Hm + 1) >> 1), jhi = min(jtop, (Hhi + Hm) >> 1);
      if (jlo <= jhi) {
        const int cnt = jhi - jlo + 1;
        mask |= (cnt >= 64 ? ~0ull : ((1ull << cnt) - 1ull)) << (jlo - jbase);
      }
    }
  }
  return mask;
}

__host__ __device__ __forceinline__ uint32_t spread_bits16_hd(uint32_t v) {          // 16 bits -> even bit positions
  v &= 0xffffu;
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}

__host__ __device__ __forceinline__ uint32_t row_tile_index(int kt, int f, int S, int j) {
  const int Nt = 1 << kt;
  const int Hm = min(S, 2 * Nt - 2 - S), H = -Hm + 2 * j;
  const uint32_t X = (uint32_t)((S + H) >> 1), Y = (uint32_t)((S - H) >> 1);
  return ((uint32_t)f << (2 * kt)) | spread_bits16_hd(X) | (spread_bits16_hd(Y) << 1);
}

}  // namespace uts
