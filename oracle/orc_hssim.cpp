// ORACLE — TEST INFRASTRUCTURE ONLY (see orc_hssim.hpp for the readings A30-A35 this file follows).
#include "orc_hssim.hpp"

#include <cmath>
#include <vector>

#include "orc_healpix.hpp"

namespace orc {

// A30.  Faces 0..3 touch the north pole, 4..7 straddle the equator, 8..11 touch the south pole.  In the HEALPix plane
// (definition D1 of orc_healpix.hpp) +x runs north-east and +y north-west, and all twelve diamonds have the same
// orientation, so a step across an edge that two faces share IN THE PLANE is a translation by Nside.  The two upper edges
// of a north face and the two lower edges of a south face are not shared in the plane: on the sphere they are glued to the
// next face around the pole along a meridian, which turns the axes by a quarter.
int64_t hssim_neighbor(int order, int64_t p, int dx, int dy, int* rot) {
  const int64_t N = (int64_t)1 << order;
  const XYF c = nest2xyf(order, p);
  const int64_t X = c.x + dx, Y = c.y + dy;
  const int ox = X < 0 ? -1 : (X >= N ? 1 : 0), oy = Y < 0 ? -1 : (Y >= N ? 1 : 0);
  const int row = c.f / 4, col = c.f % 4;
  const int nxt = (col + 1) % 4, prv = (col + 3) % 4, opp = (col + 2) % 4;
  int r = 0;
  XYF q{X, Y, c.f};
  bool ok = true;
  if (ox == 0 && oy == 0) {
    // same face
  } else if (row == 1) {                                   // equatorial face 4 + col
    if (ox == 1 && oy == 0) q = XYF{X - N, Y, col};                    // north-east: north face col
    else if (ox == 0 && oy == 1) q = XYF{X, Y - N, prv};               // north-west: north face col - 1
    else if (ox == -1 && oy == 0) q = XYF{X + N, Y, 8 + prv};          // south-west: south face col - 1
    else if (ox == 0 && oy == -1) q = XYF{X, Y + N, 8 + col};          // south-east: south face col
    else if (ox == 1 && oy == -1) q = XYF{X - N, Y + N, 4 + nxt};      // east vertex (4 faces): next equatorial face
    else if (ox == -1 && oy == 1) q = XYF{X + N, Y - N, 4 + prv};      // west vertex (4 faces)
    else ok = false;                                                   // north / south vertex: only 3 faces meet
  } else if (row == 0) {                                   // north face col
    if (ox == -1 && oy == 0) q = XYF{X + N, Y, 4 + col};               // south-west: equatorial face col
    else if (ox == 0 && oy == -1) q = XYF{X, Y + N, 4 + nxt};          // south-east: equatorial face col + 1
    else if (ox == -1 && oy == -1) q = XYF{X + N, Y + N, 8 + col};     // south vertex (4 faces): south face col
    else if (ox == 1 && oy == 0) { q = XYF{Y, 2 * N - 1 - X, nxt}; r = 1; }        // north-east edge = meridian: next north face
    else if (ox == 0 && oy == 1) { q = XYF{2 * N - 1 - Y, X, prv}; r = 3; }        // north-west edge: previous north face
    else if (ox == 1 && oy == 1) { q = XYF{2 * N - 1 - X, 2 * N - 1 - Y, opp}; r = 2; }   // over the pole
    else ok = false;                                                   // east / west vertex: only 3 faces meet
  } else {                                                 // south face 8 + col
    if (ox == 1 && oy == 0) q = XYF{X - N, Y, 4 + nxt};                // north-east: equatorial face col + 1
    else if (ox == 0 && oy == 1) q = XYF{X, Y - N, 4 + col};           // north-west: equatorial face col
    else if (ox == 1 && oy == 1) q = XYF{X - N, Y - N, col};           // north vertex (4 faces): north face col
    else if (ox == 0 && oy == -1) { q = XYF{-1 - Y, X, 8 + nxt}; r = 3; }          // south-east edge = meridian: next south face
    else if (ox == -1 && oy == 0) { q = XYF{Y, -1 - X, 8 + prv}; r = 1; }          // south-west edge: previous south face
    else if (ox == -1 && oy == -1) { q = XYF{-1 - X, -1 - Y, 8 + opp}; r = 2; }    // over the pole
    else ok = false;
  }
  if (rot) *rot = r;
  if (!ok || q.x < 0 || q.x >= N || q.y < 0 || q.y >= N) return -1;   // (a window wider than a face is not supported)
  return xyf2nest(order, q);
}

// A31
double hssim_weight(int face, int dx, int dy, double sigma) {
  const double pi = 3.14159265358979323846;
  if (face >= 4 && face < 8) return std::exp(-(double)(dx * dx + dy * dy) / (2.0 * sigma * sigma));
  const double u = dx - dy, v = dx + dy;
  return std::exp(-((pi / 4.0) * u * u + (4.0 / pi) * v * v) / (4.0 * sigma * sigma));
}

namespace {
struct Image {
  int order; const int32_t* slot_of_tile; const uint32_t* bits;
  // storage index of NESTED pixel p in the slot layout, or -1 when the pixel is masked out / its tile inactive
  int64_t index(int64_t p) const {
    if (bits && !((bits[p >> 5] >> (p & 31)) & 1u)) return -1;
    const int64_t tile = p >> 8;
    const int64_t slot = slot_of_tile ? slot_of_tile[tile] : tile;
    if (slot < 0) return -1;
    return slot * 256 + (p & 255);
  }
};
}  // namespace

HssimOut hssim_loss(int order, const int32_t* slot_of_tile, const uint32_t* pixel_mask_bits, int64_t n_slot, const float* X,
                    const float* G, double lambda, double sigma, double* h_map, double* dL_dX, const int64_t* q_list, int64_t n_q) {
  const int R = kHssimR, Wn = 2 * R + 1, CH = 3;
  const double C1 = 0.01 * 0.01, C2 = 0.03 * 0.03;       // A33
  const int64_t npix = npix_of_order(order);
  const Image im{order, slot_of_tile, pixel_mask_bits};
  const int64_t n_store = n_slot * 256;
  if (h_map) for (int64_t i = 0; i < n_store; ++i) h_map[i] = 0.0;
  if (dL_dX) for (int64_t i = 0; i < n_store * CH; ++i) dL_dX[i] = 0.0;
  // pass 1: count the valid pixels (Eq.10's denominator)
  int64_t n_valid = 0;
  for (int64_t p = 0; p < npix; ++p) if (im.index(p) >= 0) ++n_valid;
  HssimOut out{0.0, 0.0, 0.0};
  if (n_valid == 0) return out;
  const double inv_n = 1.0 / (double)n_valid;
  double sum_h = 0.0, sum_l1 = 0.0;
  std::vector<int64_t> tap(Wn * Wn);
  std::vector<double> wt(Wn * Wn);
  // q_list (test sampling at sizes where the whole sphere is too slow): only the listed centre pixels are evaluated, against
  // the whole image and with Eq.10's denominator of the whole image; the sums and the gradient then hold their terms only.
  const int64_t n_centres = q_list ? n_q : npix;
  for (int64_t qi = 0; qi < n_centres; ++qi) {
    const int64_t q = q_list ? q_list[qi] : qi;
    const int64_t iq = im.index(q);
    if (iq < 0) continue;
    const int face = (int)(q >> (2 * order));
    // the window of q: taps, weights renormalised over the taps that exist (A30, A32)
    double wsum = 0.0;
    for (int dy = -R; dy <= R; ++dy)
      for (int dx = -R; dx <= R; ++dx) {
        const int t = (dy + R) * Wn + (dx + R);
        const int64_t pn = hssim_neighbor(order, q, dx, dy, nullptr);
        const int64_t ip = pn >= 0 ? im.index(pn) : -1;
        tap[t] = ip;
        wt[t] = ip >= 0 ? hssim_weight(face, dx, dy, sigma) : 0.0;
        wsum += wt[t];
      }
    for (auto& w : wt) w /= wsum;
    double hq = 0.0;
    for (int ch = 0; ch < CH; ++ch) {
      double m1 = 0, m2 = 0, e11 = 0, e22 = 0, e12 = 0;
      for (int t = 0; t < Wn * Wn; ++t) {
        if (tap[t] < 0) continue;
        const double x = X[tap[t] * CH + ch], g = G[tap[t] * CH + ch], w = wt[t];
        m1 += w * x; m2 += w * g; e11 += w * x * x; e22 += w * g * g; e12 += w * x * g;
      }
      const double s11 = e11 - m1 * m1, s22 = e22 - m2 * m2, s12 = e12 - m1 * m2;
      const double a1 = 2 * m1 * m2 + C1, a2 = 2 * s12 + C2, b1 = m1 * m1 + m2 * m2 + C1, b2 = s11 + s22 + C2;
      const double ssim = (a1 * a2) / (b1 * b2);                     // A33
      hq += ssim / CH;
      if (dL_dX) {
        // L contains -lambda * inv_n * ssim / CH.  Derivatives of ssim w.r.t. the window statistics that depend on X:
        // m1, e11, e12 (s11 = e11 - m1^2, s12 = e12 - m1 m2).
        const double d_a1 = a2 / (b1 * b2), d_a2 = a1 / (b1 * b2), d_b1 = -ssim / b1, d_b2 = -ssim / b2;
        const double d_s12 = 2 * d_a2, d_s11 = d_b2;
        const double d_m1 = d_a1 * 2 * m2 + d_b1 * 2 * m1 + d_s11 * (-2 * m1) + d_s12 * (-m2);
        const double d_e11 = d_s11, d_e12 = d_s12;
        const double scale = -lambda * inv_n / CH;
        for (int t = 0; t < Wn * Wn; ++t) {
          if (tap[t] < 0) continue;
          const double x = X[tap[t] * CH + ch], g = G[tap[t] * CH + ch];
          dL_dX[tap[t] * CH + ch] += scale * wt[t] * (d_m1 + 2 * x * d_e11 + g * d_e12);
        }
      }
    }
    sum_h += hq;
    if (h_map) h_map[iq] = hq;
    for (int ch = 0; ch < CH; ++ch) {
      const double d = (double)X[iq * CH + ch] - (double)G[iq * CH + ch];
      sum_l1 += std::fabs(d);
      if (dL_dX) dL_dX[iq * CH + ch] += (1.0 - lambda) * inv_n / CH * (d > 0 ? 1.0 : (d < 0 ? -1.0 : 0.0));
    }
  }
  out.hssim = sum_h * inv_n;                               // Eq.10
  out.l1 = sum_l1 * inv_n / CH;                            // A34
  out.loss = (1.0 - lambda) * out.l1 + lambda * (1.0 - out.hssim);
  return out;
}

}  // namespace orc
