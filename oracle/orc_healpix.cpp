// ORACLE — TEST INFRASTRUCTURE ONLY (see orc_healpix.hpp).  Shares no code with the CUDA path.
#include "orc_healpix.hpp"
#include <cmath>
#include <algorithm>

namespace orc {

static const double kPi = 3.14159265358979323846264338327950288;

int64_t npix_of_order(int order) { return (int64_t)12 << (2 * order); }

// --- NESTED <-> (x,y,f): plain bit loops ("NESTED indexing with (x,y,f) parameterization") ---
XYF nest2xyf(int order, int64_t p) {
  int64_t per_face = (int64_t)1 << (2 * order);
  XYF c; c.f = (int)(p / per_face);
  int64_t m = p % per_face;
  c.x = 0; c.y = 0;
  for (int b = 0; b < order; ++b) {
    c.x |= ((m >> (2 * b)) & 1) << b;        // x lives in the even bits
    c.y |= ((m >> (2 * b + 1)) & 1) << b;    // y lives in the odd bits
  }
  return c;
}

int64_t xyf2nest(int order, XYF c) {
  int64_t m = 0;
  for (int b = 0; b < order; ++b) {
    m |= ((c.x >> b) & 1) << (2 * b);
    m |= ((c.y >> b) & 1) << (2 * b + 1);
  }
  return (int64_t)c.f * ((int64_t)1 << (2 * order)) + m;
}

// --- D1: the HEALPix plane, in units of pi/4 ---
// Face f: row rf = f/4, column cf = f%4; face centre (U_f,V_f) = (1+2cf, +1), (2cf, 0), (1+2cf, -1).
// u = U_f + (x'-y'), v = V_f + (x'+y'-1).  |v|<=1: z = 2v/3, lam = u*pi/4.
// |v|>1 (polar cap): sigma=|v|, 1-|z| = (2-sigma)^2/3, lam = (u + (sigma-1)(u_t-1)/(2-sigma))*pi/4, u_t = u mod 2.
static void face_uv_center(int f, double& U, double& V) {
  int rf = f / 4, cf = f % 4;
  if (rf == 0) { U = 1 + 2 * cf; V = 1; }
  else if (rf == 1) { U = 2 * cf; V = 0; }
  else { U = 1 + 2 * cf; V = -1; }
}

static ZPhi plane_to_sphere(double u, double v) {
  ZPhi r;
  double av = std::fabs(v);
  if (av <= 1.0) {
    r.z = 2.0 * v / 3.0;
    r.sth = std::sqrt((1.0 - r.z) * (1.0 + r.z));
    r.lam = u * (kPi / 4);
  } else {
    double sigma = av;
    double w = (2.0 - sigma) * (2.0 - sigma) / 3.0;      // 1-|z|
    r.z = (v > 0 ? 1.0 : -1.0) * (1.0 - w);
    r.sth = std::sqrt(w * (2.0 - w));
    double ut = u - 2.0 * std::floor(u / 2.0);           // u mod 2 in [0,2)
    double shift = (2.0 - sigma > 0) ? (sigma - 1.0) * (ut - 1.0) / (2.0 - sigma) : 0.0;
    r.lam = (u + shift) * (kPi / 4);
  }
  r.lam = r.lam - 2 * kPi * std::floor(r.lam / (2 * kPi));
  if (r.lam >= 2 * kPi) r.lam = 0;
  return r;
}

ZPhi face_point_D1(int f, double xp, double yp) {
  double U, V; face_uv_center(f, U, V);
  return plane_to_sphere(U + (xp - yp), V + (xp + yp - 1.0));
}

ZPhi pix_center_D1(int order, int64_t p) {
  XYF c = nest2xyf(order, p);
  double n = (double)((int64_t)1 << order);
  return face_point_D1(c.f, (c.x + 0.5) / n, (c.y + 0.5) / n);
}

ZPhi pix_corner_D1(int order, int64_t p, int corner) {
  XYF c = nest2xyf(order, p);
  double n = (double)((int64_t)1 << order);
  return face_point_D1(c.f, (c.x + (corner & 1)) / n, (c.y + ((corner >> 1) & 1)) / n);
}

// --- D2: ring form ---
// F1 = rf+2, F2 = 2cf - (rf mod 2) + 1; ring i = F1*Nside - x - y - 1 (1 = northernmost).
static void xyf_to_ring_coords(int order, XYF c, int64_t& iring, int64_t& nr, int64_t& jp, int& kshift) {
  int64_t n = (int64_t)1 << order;
  int rf = c.f / 4, cf = c.f % 4;
  int64_t F1 = rf + 2, F2 = 2 * cf - (rf % 2) + 1;
  iring = F1 * n - c.x - c.y - 1;
  if (iring < n) { nr = iring; kshift = 0; }
  else if (iring > 3 * n) { nr = 4 * n - iring; kshift = 0; }
  else { nr = n; kshift = (int)((iring - n) & 1); }
  jp = (F2 * nr + c.x - c.y + 1 + kshift) / 2;
  if (jp > 4 * nr) jp -= 4 * nr;
  if (jp < 1) jp += 4 * nr;
}

static ZPhi ring_coords_to_zphi(int order, int64_t iring, int64_t nr, int64_t jp, int kshift) {
  double n = (double)((int64_t)1 << order);
  ZPhi r;
  if (iring < (int64_t)n) {
    double w = (double)nr * (double)nr / (3.0 * n * n);
    r.z = 1.0 - w; r.sth = std::sqrt(w * (2.0 - w));
  } else if (iring > 3 * (int64_t)n) {
    double w = (double)nr * (double)nr / (3.0 * n * n);
    r.z = -1.0 + w; r.sth = std::sqrt(w * (2.0 - w));
  } else {
    r.z = (2.0 * n - (double)iring) * 2.0 / (3.0 * n);
    r.sth = std::sqrt((1.0 - r.z) * (1.0 + r.z));
  }
  r.lam = ((double)jp - (kshift + 1) * 0.5) * kPi / (2.0 * (double)nr);
  return r;
}

ZPhi pix_center_D2(int order, int64_t p) {
  int64_t iring, nr, jp; int kshift;
  xyf_to_ring_coords(order, nest2xyf(order, p), iring, nr, jp, kshift);
  return ring_coords_to_zphi(order, iring, nr, jp, kshift);
}

int64_t nest2ring(int order, int64_t p) {
  int64_t n = (int64_t)1 << order, npix = 12 * n * n;
  int64_t iring, nr, jp; int kshift;
  xyf_to_ring_coords(order, nest2xyf(order, p), iring, nr, jp, kshift);
  if (iring < n) return 2 * iring * (iring - 1) + jp - 1;
  if (iring > 3 * n) return npix - 2 * nr * (nr + 1) + jp - 1;
  return 2 * n * (n - 1) + (iring - n) * 4 * n + jp - 1;
}

int64_t ring_npix_in_ring(int order, int64_t i) {
  int64_t n = (int64_t)1 << order;
  return 4 * std::min(i, std::min(n, 4 * n - i));
}

// RingInfo of Alg.3, from the ring form D2: ring i holds npix = 4*n_r pixels at longitudes
// lam0 + j * 2pi/npix, j = 0..npix-1, lam0 = (1 - (kshift+1)/2) * pi / (2 n_r).
RingInfo ring_info(int order, int64_t i) {
  int64_t n = (int64_t)1 << order, npix = 12 * n * n, ncap = 2 * n * (n - 1);
  int64_t nr; int kshift; int64_t first;
  if (i < n) { nr = i; kshift = 0; first = 2 * i * (i - 1); }
  else if (i > 3 * n) { nr = 4 * n - i; kshift = 0; first = npix - 2 * nr * (nr + 1); }
  else { nr = n; kshift = (int)((i - n) & 1); first = ncap + (i - n) * 4 * n; }
  ZPhi c = ring_coords_to_zphi(order, i, nr, 1, kshift);
  RingInfo r; r.z = c.z; r.npix = 4 * nr; r.lam0 = c.lam; r.first = first;
  return r;
}

static int64_t isqrt64(int64_t v) {
  int64_t r = (int64_t)std::sqrt((double)v);
  while (r * r > v) --r;
  while ((r + 1) * (r + 1) <= v) ++r;
  return r;
}

// Textbook pix2ang in RING order (Gorski et al. [11]): rings counted from the north pole.
ZPhi ring_center(int order, int64_t r) {
  int64_t n = (int64_t)1 << order, npix = 12 * n * n, ncap = 2 * n * (n - 1);
  int64_t iring, nr, jp; int kshift;
  if (r < ncap) {
    iring = (1 + isqrt64(1 + 2 * r)) / 2;
    jp = r + 1 - 2 * iring * (iring - 1);
    nr = iring; kshift = 0;
  } else if (r < npix - ncap) {
    int64_t ip = r - ncap;
    iring = ip / (4 * n) + n;
    jp = ip % (4 * n) + 1;
    nr = n; kshift = (int)((iring + n) & 1);
  } else {
    int64_t ip = npix - r;
    int64_t ir = (1 + isqrt64(2 * ip - 1)) / 2;        // ring counted from the south pole
    jp = 4 * ir + 1 - (ip - 2 * ir * (ir - 1));
    iring = 4 * n - ir; nr = ir; kshift = 0;
  }
  return ring_coords_to_zphi(order, iring, nr, jp, kshift);
}

// --- sphere -> pixel: inverse of D1 ---
int64_t ang2pix_nest(int order, double z, double lam) {
  int64_t n = (int64_t)1 << order;
  lam = lam - 2 * kPi * std::floor(lam / (2 * kPi));
  double u, v;
  double az = std::fabs(z);
  if (az <= 2.0 / 3.0) {
    u = lam / (kPi / 4); v = 1.5 * z;
  } else {
    double sigma = 2.0 - std::sqrt(3.0 * (1.0 - az));
    double lt = lam - (kPi / 2) * std::floor(lam / (kPi / 2));
    u = (lam - (sigma - 1.0) * (lt - kPi / 4)) / (kPi / 4);
    v = (z > 0 ? sigma : -sigma);
  }
  int best_f = -1; double bx = 0, by = 0, best_out = 1e300;
  for (int f = 0; f < 12; ++f) {
    double U, V; face_uv_center(f, U, V);
    for (int wrap = -1; wrap <= 1; ++wrap) {
      double du = u + 8.0 * wrap - U, dv = v - V;
      double xp = (du + dv + 1.0) * 0.5, yp = (dv + 1.0 - du) * 0.5;
      // distance outside the half-open unit square (0 when inside)
      double out = std::max(std::max(-xp, xp - 1.0), std::max(-yp, yp - 1.0));
      if (xp >= 1.0 || yp >= 1.0) out = std::max(out, 1e-300);
      if (out < 0) out = 0;
      if (out < best_out) { best_out = out; best_f = f; bx = xp; by = yp; }
    }
  }
  XYF c; c.f = best_f;
  c.x = std::min<int64_t>(n - 1, std::max<int64_t>(0, (int64_t)std::floor(bx * (double)n)));
  c.y = std::min<int64_t>(n - 1, std::max<int64_t>(0, (int64_t)std::floor(by * (double)n)));
  return xyf2nest(order, c);
}

int64_t ring2nest(int order, int64_t r) {
  ZPhi a = ring_center(order, r);
  return ang2pix_nest(order, a.z, a.lam);
}

void to_cam_vec(const ZPhi& a, double v[3]) {
  double xh = a.sth * std::cos(a.lam), yh = a.sth * std::sin(a.lam), zh = a.z;
  v[0] = yh; v[1] = zh; v[2] = xh;
}

double angle_between(const double a[3], const double b[3]) {
  double cx = a[1] * b[2] - a[2] * b[1], cy = a[2] * b[0] - a[0] * b[2], cz = a[0] * b[1] - a[1] * b[0];
  return std::atan2(std::sqrt(cx * cx + cy * cy + cz * cz), a[0] * b[0] + a[1] * b[1] + a[2] * b[2]);
}

double rho_max_bruteforce(int order) {
  int64_t npix = npix_of_order(order);
  double best = 0;
  for (int64_t p = 0; p < npix; ++p) {
    double c[3]; to_cam_vec(pix_center_D1(order, p), c);
    for (int k = 0; k < 4; ++k) {
      double q[3]; to_cam_vec(pix_corner_D1(order, p, k), q);
      best = std::max(best, angle_between(c, q));
    }
  }
  return best;
}

double rho_max_closed(int order) {
  double n = (double)((int64_t)1 << order);
  ZPhi a; a.z = 2.0 / 3.0; a.sth = std::sqrt(1.0 - a.z * a.z); a.lam = kPi / (4.0 * n);
  double w = (1.0 - 1.0 / n) * (1.0 - 1.0 / n) / 3.0;   // 1-z of the corner
  ZPhi b; b.z = 1.0 - w; b.sth = std::sqrt(w * (2.0 - w)); b.lam = 0.0;
  double va[3], vb[3]; to_cam_vec(a, va); to_cam_vec(b, vb);
  return angle_between(va, vb);
}

}  // namespace orc
