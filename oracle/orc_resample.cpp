// ORACLE — TEST INFRASTRUCTURE ONLY.  See orc_resample.hpp for scope, citations and readings A26-A28.
#include "orc_resample.hpp"
#include "orc_healpix.hpp"
#include <cmath>
#include <vector>

namespace orc {

static const double kPi = 3.14159265358979323846;

// ---------------------------------------------------------------- camera models
bool cam_pixel_dir(const Camera& c, double u, double v, double d[3]) {
  const double W = c.width, H = c.height, cx = W / 2, cy = H / 2;          // principal point (W/2, H/2)
  if (c.model == kPinhole) {
    // f_x = W / (2 tan(FoV_x/2)); x = (u - c_x)/f_x; d = (x,y,1)/|(x,y,1)|
    const double fx = W / (2 * std::tan(c.p0 / 2)), fy = H / (2 * std::tan(c.p1 / 2));
    const double x = (u - cx) / fx, y = (v - cy) / fy, n = std::sqrt(x * x + y * y + 1);
    d[0] = x / n; d[1] = y / n; d[2] = 1 / n;
    return u >= 0 && u < W && v >= 0 && v < H;
  }
  if (c.model == kFisheye) {
    // f_x = W/pi, f_y = H/pi; m = ((u-c_x)/f_x, (v-c_y)/f_y); r_m = |m|; gamma = atan2(m_y, m_x)
    const double fx = W / kPi, fy = H / kPi;
    const double mx = (u - cx) / fx, my = (v - cy) / fy, rm = std::sqrt(mx * mx + my * my), g = std::atan2(my, mx);
    const double weff = std::sqrt(std::pow(c.p0 * std::cos(g), 2) + std::pow(c.p1 * std::sin(g), 2));   // Eq.12
    const double psi = rm * weff;                                                                   // incident angle
    d[0] = std::sin(psi) * std::cos(g); d[1] = std::sin(psi) * std::sin(g); d[2] = std::cos(psi);
    const double a = fx * kPi / 2, b = fy * kPi / 2;                                                // Eq.15
    return (u - cx) * (u - cx) / (a * a) + (v - cy) * (v - cy) / (b * b) <= 1;                      // Eq.14
  }
  // omnidirectional: omega = 2 pi u / W - pi, phi = pi/2 - pi v / H
  const double om = 2 * kPi * u / W - kPi, ph = kPi / 2 - kPi * v / H;
  d[0] = std::cos(ph) * std::sin(om); d[1] = std::sin(ph); d[2] = std::cos(ph) * std::cos(om);
  return u >= 0 && u < W && v >= 0 && v < H;
}

bool cam_project(const Camera& c, const double d[3], double& u, double& v) {
  const double W = c.width, H = c.height, cx = W / 2, cy = H / 2;
  if (c.model == kPinhole) {
    if (!(d[2] > 0)) return false;
    const double fx = W / (2 * std::tan(c.p0 / 2)), fy = H / (2 * std::tan(c.p1 / 2));
    u = cx + fx * d[0] / d[2]; v = cy + fy * d[1] / d[2];
    return u >= 0 && u < W && v >= 0 && v < H;
  }
  if (c.model == kFisheye) {
    const double fx = W / kPi, fy = H / kPi;
    const double psi = std::atan2(std::sqrt(d[0] * d[0] + d[1] * d[1]), d[2]);      // angle from the optical axis
    const double g = std::atan2(d[1], d[0]);
    const double weff = std::sqrt(std::pow(c.p0 * std::cos(g), 2) + std::pow(c.p1 * std::sin(g), 2));
    const double rm = psi / weff;
    u = cx + fx * rm * std::cos(g); v = cy + fy * rm * std::sin(g);
    const double a = fx * kPi / 2, b = fy * kPi / 2;
    return (u - cx) * (u - cx) / (a * a) + (v - cy) * (v - cy) / (b * b) <= 1;
  }
  const double om = std::atan2(d[0], d[2]), ph = std::asin(std::fmax(-1.0, std::fmin(1.0, d[1])));   // Eq.11/13
  u = (om + kPi) * W / (2 * kPi); v = (kPi / 2 - ph) * H / kPi;
  if (u >= W) u -= W;
  return true;
}

// ---------------------------------------------------------------- Interp_H (reading A26)
static double ring_theta(int order, int64_t i) {
  const RingInfo ri = ring_info(order, i);
  return std::atan2(std::sqrt((1 - ri.z) * (1 + ri.z)), ri.z);
}

// the two pixels of ring i nearest in longitude to lam, with linear weights
static void ring_pair(int order, int64_t i, double lam, int64_t pix[2], double w[2]) {
  const RingInfo ri = ring_info(order, i);
  const double step = 2 * kPi / (double)ri.npix;
  const double t = (lam - ri.lam0) / step;               // pixel j of the ring has its centre at lam0 + j step
  const double fl = std::floor(t);
  const double frac = t - fl;
  int64_t j1 = (int64_t)fl % ri.npix; if (j1 < 0) j1 += ri.npix;
  const int64_t j2 = (j1 + 1) % ri.npix;
  pix[0] = ring2nest(order, ri.first + j1); pix[1] = ring2nest(order, ri.first + j2);
  w[0] = 1 - frac; w[1] = frac;
}

int interp_weights(int order, double theta, double lam, int64_t pix[8], double w[8]) {
  const int64_t n = (int64_t)1 << order, last = 4 * n - 1;
  // ring just north of (or at) the point: the largest i with theta_i <= theta; 0 when the point is north of ring 1
  int64_t i1 = 0;
  for (int64_t lo = 1, hi = last; lo <= hi;) { const int64_t mid = (lo + hi) / 2; if (ring_theta(order, mid) <= theta) { i1 = mid; lo = mid + 1; } else hi = mid - 1; }
  const int64_t i2 = i1 + 1;
  int cnt = 0;
  if (i1 == 0) {                                          // between the north pole and ring 1
    const double t2 = ring_theta(order, 1), wt = theta / t2;
    int64_t p[2]; double a[2];
    ring_pair(order, 1, lam, p, a);
    for (int k = 0; k < 2; ++k) { pix[cnt] = p[k]; w[cnt++] = a[k] * wt; }
    const RingInfo ri = ring_info(order, 1);              // pole value = mean of the 4 pixels of ring 1
    for (int j = 0; j < 4; ++j) { pix[cnt] = ring2nest(order, ri.first + j); w[cnt++] = (1 - wt) / 4; }
    return cnt;
  }
  if (i2 > last) {                                        // between the last ring and the south pole
    const double t1 = ring_theta(order, last), wt = (theta - t1) / (kPi - t1);
    int64_t p[2]; double a[2];
    ring_pair(order, last, lam, p, a);
    for (int k = 0; k < 2; ++k) { pix[cnt] = p[k]; w[cnt++] = a[k] * (1 - wt); }
    const RingInfo ri = ring_info(order, last);
    for (int j = 0; j < 4; ++j) { pix[cnt] = ring2nest(order, ri.first + j); w[cnt++] = wt / 4; }
    return cnt;
  }
  const double t1 = ring_theta(order, i1), t2 = ring_theta(order, i2), wt = (theta - t1) / (t2 - t1);
  int64_t p[2]; double a[2];
  ring_pair(order, i1, lam, p, a);
  for (int k = 0; k < 2; ++k) { pix[cnt] = p[k]; w[cnt++] = a[k] * (1 - wt); }
  ring_pair(order, i2, lam, p, a);
  for (int k = 0; k < 2; ++k) { pix[cnt] = p[k]; w[cnt++] = a[k] * wt; }
  return cnt;
}

// ---------------------------------------------------------------- resampling, Eq.7, and its adjoint
static inline bool pix_on(const uint32_t* bits, int64_t p) { return !bits || ((bits[p >> 5] >> (p & 31)) & 1u); }

// support of image pixel (i,j): valid HEALPix pixels (as slot-layout indices) with renormalised weights (reading A27)
static int pixel_support(int order, const Camera& c, const int32_t* slot_of_tile, const uint32_t* bits, int i, int j,
                         int64_t idx[8], double w[8], bool& in_domain) {
  double d[3];
  in_domain = cam_pixel_dir(c, i + 0.5, j + 0.5, d);     // reading A28
  if (!in_domain) return 0;
  // HEALPix frame (reading A1): polar axis = camera +y, longitude = omega = atan2(d_x, d_z)
  const double theta = std::atan2(std::sqrt(d[0] * d[0] + d[2] * d[2]), d[1]);
  double lam = std::atan2(d[0], d[2]);
  if (lam < 0) lam += 2 * kPi;
  int64_t pix[8]; double ww[8];
  const int n = interp_weights(order, theta, lam, pix, ww);
  int cnt = 0; double sum = 0;
  for (int k = 0; k < n; ++k) {
    if (!pix_on(bits, pix[k])) continue;
    const int64_t tile = pix[k] >> 8;
    const int64_t slot = slot_of_tile ? slot_of_tile[tile] : tile;
    if (slot < 0) continue;
    idx[cnt] = slot * 256 + (pix[k] & 255); w[cnt] = ww[k]; sum += ww[k]; ++cnt;
  }
  if (!(sum > 0)) return 0;
  for (int k = 0; k < cnt; ++k) w[k] /= sum;
  return cnt;
}

void resample_fwd(int order, const Camera& c, const int32_t* slot_of_tile, const uint32_t* bits, const float* image,
                  int channels, double* out, uint8_t* valid) {
  for (int j = 0; j < c.height; ++j)
    for (int i = 0; i < c.width; ++i) {
      int64_t idx[8]; double w[8]; bool in;
      const int n = pixel_support(order, c, slot_of_tile, bits, i, j, idx, w, in);
      double* o = out + ((size_t)j * c.width + i) * channels;
      for (int ch = 0; ch < channels; ++ch) o[ch] = 0;
      for (int k = 0; k < n; ++k)
        for (int ch = 0; ch < channels; ++ch) o[ch] += w[k] * (double)image[idx[k] * channels + ch];
      if (valid) valid[(size_t)j * c.width + i] = in ? 1 : 0;
    }
}

void resample_bwd(int order, const Camera& c, const int32_t* slot_of_tile, const uint32_t* bits, int64_t n_slot,
                  const double* dL_dout, int channels, double* dL_dimage) {
  for (int64_t k = 0; k < n_slot * 256 * channels; ++k) dL_dimage[k] = 0;
  for (int j = 0; j < c.height; ++j)
    for (int i = 0; i < c.width; ++i) {
      int64_t idx[8]; double w[8]; bool in;
      const int n = pixel_support(order, c, slot_of_tile, bits, i, j, idx, w, in);
      const double* g = dL_dout + ((size_t)j * c.width + i) * channels;
      for (int k = 0; k < n; ++k)
        for (int ch = 0; ch < channels; ++ch) dL_dimage[idx[k] * channels + ch] += w[k] * g[ch];
    }
}

void camera_mask(int order, const Camera& c, uint32_t* bits) {
  const int64_t np = npix_of_order(order);
  for (int64_t wd = 0; wd < np / 32; ++wd) bits[wd] = 0;
  for (int64_t p = 0; p < np; ++p) {
    double d[3], u, v;
    to_cam_vec(pix_center_D2(order, p), d);
    if (cam_project(c, d, u, v)) bits[p >> 5] |= 1u << (p & 31);
  }
}

}  // namespace orc
