// uts_window_query.cuh — tile set of a SMALL disc from a window of tiles around the disc's centre (F2; Alg.1 l.9-14
// PAPER.md:548-559; the set is reading A6's / Alg.3's, see uts_ring_query.cuh).
//
// The set to compute is  T = { q >> 2(k_q - k_t) : q an order-k_q pixel, u . centre(q) >= cos R }.  A pixel centre lies inside its
// tile, so every tile of T meets the geodesic ball B(u, R).  Leaving the w-ring of tiles around the tile that holds u means
// crossing w tiles from one edge (or vertex) to a non-incident edge, and no HEALPix pixel of order o is narrower than
// h_min(o) = 0.69 / 2^o between opposite edges (measured numerically, orders 0-5: 0.841, 0.755, 0.728, 0.713, 0.704, 0.698 times
// 2^-o, decreasing towards about 0.69; kWindowWidth = 0.6 leaves 13 %).  So for R <= 0.6 w / N_t the (2w+1)^2 window of cells
// around tile(u), taken in the extended (x, y) frame of u's base face and carried into the neighbouring faces by the gluing rules
// below, holds every candidate; each candidate is settled by one fp32 chord test of its centre (all of it inside / outside the
// disc) and, on the rim, by the defining predicate on its 4^(k_q-k_t) query pixels (fp32 chord with a margin, double inside the
// margin).  A candidate outside the FoV mask costs one table read, where the ring path pays for rings and rows before it filters:
// measured (B200, tile-lists call, round 2 after the ring path's exact test became cheap) config 5 (frustum mask = 6 % of the
// tiles, N_t = 128) 4.5 -> 3.7 ms with windows up to 7 x 7; config 3 (cap mask, 55 %) 0.68 -> 0.78 ms, config 2 (no mask) 0.24 ->
// 0.33 ms, config 4 (no mask) unchanged: the work per disc grows with the window AREA times the 4^(k_q-k_t) rim tests.  So the
// caller (uts_tile_query.cu) takes this path by default only under a mask that keeps at most a quarter of the tiles.
// (The gluing table must be `static`: as a plain constexpr local it was copied to each thread's stack, and config 4 went from 8.5
// to 12.3 ms.  Also measured: classifying all cells first and then walking the rim tiles' query pixels in ONE flattened loop per
// lane, so that lanes whose tile was settled by the centre test do not idle through the others' pixel loops — no gain; not kept.)
// Everything is __host__ __device__: tests/hostlogic drives the same code on the CPU against the oracle's sets.
#pragma once
#include "uts_internal.cuh"

namespace uts {

constexpr double kWindowWidth = 0.6;      // lower bound of (pixel width between opposite edges) * N_side, with margin
constexpr int kWindowMax = 3;             // largest window half-width handled here (7 x 7 cells)
constexpr float kWinDelta = 4e-6f;        // fp32 chord margin (the fp32 centres are good to 1e-6)

#ifdef __CUDA_ARCH__
#define UTS_WIN_SINCOSF(x, s, c) __sincosf((x), (s), (c))
#else
#define UTS_WIN_SINCOSF(x, s, c) (*(s) = sinf(x), *(c) = cosf(x))
#endif

// ---------------------------------------------------------------------------------------------- face gluing
// Faces f = 4 r + c: r = 0 north, 1 equatorial, 2 south; in-face axes +x north-east, +y north-west (uts_internal.cuh, pix_geom).
// A cell (X, Y) outside [0, N)^2 of face f lies in another face; direction o = (ox, oy) in {-1, 0, +1}^2:
//   kind 1  translation by N (every edge of an equatorial face, the lower edges of a north face, the upper edges of a south
//           face, and the 4-face vertices);
//   kind 2 / 4  quarter turn (the upper edges of a north face are meridians glued to the next / previous north face; mirror image
//           for the lower edges of a south face);  kind 3  two quarter turns (over the pole);
//   kind 0  the quadrant beyond a vertex shared by only 3 faces does not exist.
// Packed as kind | row << 4 | dcol << 8 per (r, oy + 1, ox + 1).  Derived from the layout of the 12 base faces (the same rules
// as uts_hssim.cu's apron; restated here as host + device code).
__host__ __device__ __forceinline__ int face_step(int r, int oy, int ox) {
#define FS(k, row, dc) ((k) | ((row) << 4) | ((dc) << 8))
  static constexpr int tab[3][3][3] = {
      {{FS(1, 2, 0), FS(1, 1, 1), FS(0, 0, 0)}, {FS(1, 1, 0), FS(1, 0, 0), FS(2, 0, 1)}, {FS(0, 0, 0), FS(4, 0, 3), FS(3, 0, 2)}},
      {{FS(0, 0, 0), FS(1, 2, 0), FS(1, 1, 1)}, {FS(1, 2, 3), FS(1, 1, 0), FS(1, 0, 0)}, {FS(1, 1, 3), FS(1, 0, 3), FS(0, 0, 0)}},
      {{FS(3, 2, 2), FS(4, 2, 1), FS(0, 0, 0)}, {FS(2, 2, 3), FS(1, 2, 0), FS(1, 1, 1)}, {FS(0, 0, 0), FS(1, 1, 0), FS(1, 0, 0)}}};
#undef FS
  return tab[r][oy + 1][ox + 1];
}

// Cell (X, Y), -N <= X, Y < 2N, of the extended frame of face f at order o  ->  (face, x, y) of the pixel it is; false: no such cell.
__host__ __device__ __forceinline__ bool extended_cell(int o, int f, int X, int Y, int& g, int& x, int& y) {
  const int N = 1 << o;
  const int ox = X < 0 ? -1 : (X >= N ? 1 : 0), oy = Y < 0 ? -1 : (Y >= N ? 1 : 0);
  const int s = face_step(f >> 2, oy, ox), kind = s & 15;
  if (kind == 0) return false;
  const int pole = (f >> 2) == 0 ? 2 * N - 1 : -1;      // north: the glued edges are x = N, y = N; south: x = -1, y = -1
  switch (kind) {
    case 1: x = X - ox * N; y = Y - oy * N; break;
    case 2: x = Y; y = pole - X; break;
    case 4: x = pole - Y; y = X; break;
    default: x = pole - X; y = pole - Y; break;
  }
  g = 4 * ((s >> 4) & 15) + ((f + (s >> 8)) & 3);
  return true;
}

// ---------------------------------------------------------------------------------------------- geometry
// Base face and in-face cell (x, y) at order o of the unit vector u (camera frame: polar axis +y, longitude atan2(u_x, u_z)),
// in double: the HEALPix angle -> pixel map (Gorski et al. as cited at PAPER.md:23) written for the (r, c, x, y) conventions of
// pix_geom.  Belt (|z| <= 2/3): the two families of pixel edges are the lines  N (1/2 + tt) -+ (3/4) N z = integer  (tt = longitude
// in quarter turns), which number the ascending (jp) and descending (jm) edges; caps: the same with N sqrt(3 (1 - |z|)) in
// place of the linear term.  A point within rounding of a pixel edge may land on either side: callers keep a margin.
__host__ __device__ __forceinline__ void vec_to_cell(int o, const double u[3], int& f, int& x, int& y) {
  const int N = 1 << o;
  const double z = u[1], za = fabs(z);
  double tt = atan2(u[0], u[2]) * (2.0 / kPi);
  if (tt < 0.0) tt += 4.0;
  if (!(tt < 4.0)) tt = 0.0;
  if (za <= 2.0 / 3.0) {
    const double t1 = (double)N * (0.5 + tt), t2 = (double)N * z * 0.75;
    const int jp = (int)floor(t1 - t2), jm = (int)floor(t1 + t2);
    const int ifp = jp >> o, ifm = jm >> o;
    f = ifp == ifm ? ((ifp & 3) | 4) : (ifp < ifm ? (ifp & 3) : (ifm & 3) + 8);
    x = jm & (N - 1);
    y = N - (jp & (N - 1)) - 1;
  } else {
    int ntt = (int)tt;
    if (ntt > 3) ntt = 3;
    const double tp = tt - (double)ntt;
    const double s2 = u[0] * u[0] + u[2] * u[2];                       // sin^2(colatitude): 1 - |z| = s2 / (1 + |z|), exact near the pole
    const double tmp = (double)N * sqrt(3.0 * s2 / (1.0 + za));
    int jp = (int)(tp * tmp), jm = (int)((1.0 - tp) * tmp);
    if (jp > N - 1) jp = N - 1;
    if (jm > N - 1) jm = N - 1;
    if (z >= 0.0) { f = ntt; x = N - jm - 1; y = N - jp - 1; }
    else { f = ntt + 8; x = jp; y = jm; }
  }
}

// Centre of cell (f, x, y) at order o as a camera-frame unit vector, fp32 (absolute error about 1e-6 per component; the same
// formulas as pix_center_cam_f32 without the bit de-interleave) and double (pix_geom's arithmetic).
__host__ __device__ __forceinline__ void cell_center_f32(int o, int f, int x, int y, float& vx, float& vy, float& vz) {
  const int N = 1 << o;
  const int r = f >> 2, c = f & 3;
  const int i = (r + 2) * N - 1 - (x + y);
  const int h = x - y;
  const float invN = 1.0f / (float)N;
  const float inv3N2 = 0.333333343f * invN * invN;
  float z, sth, q;
  if (i < N) { const float fn = (float)i; const float w = fn * fn * inv3N2; z = 1.0f - w; sth = sqrtf(w * (2.0f - w)); q = (float)h / fn; }
  else if (i > 3 * N) { const float fn = (float)(4 * N - i); const float w = fn * fn * inv3N2; z = w - 1.0f; sth = sqrtf(w * (2.0f - w)); q = (float)h / fn; }
  else { z = (float)(2 * (2 * N - i)) * (0.333333343f * invN); sth = sqrtf((1.0f - z) * (1.0f + z)); q = (float)h * invN; }
  q += (float)(2 * c + 1 - (r & 1));
  if (q > 4.0f) q -= 8.0f;                                             // |longitude| <= pi for the fast sincos
  float s, cs;
  UTS_WIN_SINCOSF(q * 0.78539816339744831f, &s, &cs);
  vx = sth * s; vy = z; vz = sth * cs;
}
__host__ __device__ __forceinline__ void cell_center_f64(int o, int f, int x, int y, double& vx, double& vy, double& vz) {
  const int64_t N = (int64_t)1 << o;
  const int r = f >> 2, c = f & 3;
  const int64_t i = (int64_t)(r + 2) * N - 1 - (x + y), h = x - y;
  double z, sth;
  int64_t n;
  const double inv3N2 = 1.0 / (3.0 * (double)N * (double)N);
  if (i < N) { n = i; const double w = (double)(n * n) * inv3N2; z = 1.0 - w; sth = sqrt(w * (2.0 - w)); }
  else if (i > 3 * N) { n = 4 * N - i; const double w = (double)(n * n) * inv3N2; z = w - 1.0; sth = sqrt(w * (2.0 - w)); }
  else { n = N; z = (double)(2 * (2 * N - i)) / (double)(3 * N); sth = sqrt((1.0 - z) * (1.0 + z)); }
  const double lam = (kPi / 4) * ((double)(2 * c + 1 - (r & 1)) + (double)h / (double)n);
  vx = sth * sin(lam); vy = z; vz = sth * cos(lam);
}

__host__ __device__ __forceinline__ uint32_t win_spread16(uint32_t v) {          // 16 bits -> even bit positions
  v &= 0xffffu;
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}

// ---------------------------------------------------------------------------------------------- the query
struct WindowDisc {
  double u[3], cosR;                      // unit direction (normalised in double from the fp32 record), cos R
  float uf[3];
  float T, Tin, Tout;                     // chord thresholds 2 sin(R/2); 2 sin((R - rho_t)/2) - delta (or -1); 2 sin((R + rho_t)/2) + delta
  int w;                                  // window half-width: R <= 0.98 * kWindowWidth * w / N_t
};

// half-width needed for radius R at tile order kt (may exceed kWindowMax: then the disc is not for this path)
__host__ __device__ __forceinline__ int window_half_width(int kt, double R) {
  return (int)ceil(R * (double)(1 << kt) / (0.98 * kWindowWidth));
}

// rho_t = rho_max(k_t): no point of a tile is farther from its centre
__host__ __device__ __forceinline__ void make_window_disc(int kt, const float dir[3], double R, double rho_t, WindowDisc& D) {
  D.u[0] = (double)dir[0]; D.u[1] = (double)dir[1]; D.u[2] = (double)dir[2];
  const double nrm = sqrt(D.u[0] * D.u[0] + D.u[1] * D.u[1] + D.u[2] * D.u[2]);
  D.u[0] /= nrm; D.u[1] /= nrm; D.u[2] /= nrm;
  D.uf[0] = (float)D.u[0]; D.uf[1] = (float)D.u[1]; D.uf[2] = (float)D.u[2];
  D.cosR = cos(R);
  D.T = (float)(2.0 * sin(0.5 * R));
  D.Tin = R - rho_t > 1e-4 ? (float)(2.0 * sin(0.5 * (R - rho_t))) - kWinDelta : -1.0f;
  D.Tout = (float)(2.0 * sin(0.5 * (R + rho_t))) + kWinDelta;
  D.w = max(1, window_half_width(kt, R));
}

// Does tile (g, tx, ty) of order kt own an order-kq pixel whose centre satisfies the defining predicate?
__host__ __device__ __forceinline__ bool window_tile_inside(const WindowDisc& D, int kt, int kq, int g, int tx, int ty) {
  float cx, cy, cz;
  cell_center_f32(kt, g, tx, ty, cx, cy, cz);
  const float ex = D.uf[0] - cx, ey = D.uf[1] - cy, ez = D.uf[2] - cz;
  const float chord = sqrtf(ex * ex + ey * ey + ez * ez);
  if (chord > D.Tout) return false;                                    // the whole tile is outside
  if (chord < D.Tin) return true;                                      // the whole tile is inside
  const int ref = kq - kt, m = 1 << ref;
  const int x0 = tx << ref, y0 = ty << ref;
  for (int dy = 0; dy < m; ++dy)
    for (int dx = 0; dx < m; ++dx) {
      float px, py, pz;
      cell_center_f32(kq, g, x0 + dx, y0 + dy, px, py, pz);
      const float fx = D.uf[0] - px, fy = D.uf[1] - py, fz = D.uf[2] - pz;
      const float ch = sqrtf(fx * fx + fy * fy + fz * fz);
      if (ch < D.T - kWinDelta) return true;
      if (ch <= D.T + kWinDelta) {                                     // inside the fp32 margin: the exact predicate decides
        double qx, qy, qz;
        cell_center_f64(kq, g, x0 + dx, y0 + dy, qx, qy, qz);
        if (D.u[0] * qx + D.u[1] * qy + D.u[2] * qz >= D.cosR) return true;
      }
    }
  return false;
}

// Calls fn(tile) for every ACTIVE tile of the disc's set (each once, in window order); returns their number.
template <class Fn>
__host__ __device__ __forceinline__ int window_query(const WindowDisc& D, int kt, int kq, const int32_t* __restrict__ slot_of_tile, Fn&& fn) {
  int f, X, Y;
  vec_to_cell(kt, D.u, f, X, Y);
  int n = 0;
  for (int dy = -D.w; dy <= D.w; ++dy)
    for (int dx = -D.w; dx <= D.w; ++dx) {
      int g, tx, ty;
      if (!extended_cell(kt, f, X + dx, Y + dy, g, tx, ty)) continue;
      const uint32_t tile = ((uint32_t)g << (2 * kt)) | win_spread16((uint32_t)tx) | (win_spread16((uint32_t)ty) << 1);
      if (slot_of_tile && slot_of_tile[tile] < 0) continue;
      if (!window_tile_inside(D, kt, kq, g, tx, ty)) continue;
      fn(tile);
      ++n;
    }
  return n;
}

}  // namespace uts
