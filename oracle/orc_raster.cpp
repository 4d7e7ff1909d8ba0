// ORACLE — TEST INFRASTRUCTURE ONLY (see orc_raster.hpp).  Shares no code with the CUDA path.
#include "orc_raster.hpp"
#include "orc_healpix.hpp"
#include <cmath>
#include <cstring>
#include <map>
#include <algorithm>

namespace orc {

static const double kPi = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------ small linear algebra (row-major 3x3)
static void mat3_mul(const double A[9], const double B[9], double C[9]) {
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    double s = 0; for (int k = 0; k < 3; ++k) s += A[3 * i + k] * B[3 * k + j]; C[3 * i + j] = s; }
}
static void mat3_T(const double A[9], double B[9]) { for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) B[3 * j + i] = A[3 * i + j]; }
static bool finite3(const double* v, int n) { for (int i = 0; i < n; ++i) if (!std::isfinite(v[i])) return false; return true; }

// QuatToMat (Alg.1 l.4 PAPER.md:537), q = (w,x,y,z) used as given (reading A14).
static void quat_to_mat(const double q[4], double R[9]) {
  double w = q[0], x = q[1], y = q[2], z = q[3];
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

// Jacobian of Eq.1: rows d(omega)/dt and d(phi)/dt.
static void jacobian_eq1(const double t[3], double J[6]) {
  double r2 = t[0] * t[0] + t[2] * t[2], r = std::sqrt(r2), R2 = r2 + t[1] * t[1];
  J[0] = t[2] / r2;                 J[1] = 0;       J[2] = -t[0] / r2;
  J[3] = -t[0] * t[1] / (r * R2);   J[4] = r / R2;  J[5] = -t[2] * t[1] / (r * R2);
}

// ------------------------------------------------------------------ real SH basis, degree <= 3 (reading A13)
void sh_basis(int degree, const double d[3], double* Y) {
  double x = d[0], y = d[1], z = d[2];
  Y[0] = 0.5 * std::sqrt(1.0 / kPi);
  if (degree < 1) return;
  double c1 = std::sqrt(3.0 / (4.0 * kPi));
  Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
  if (degree < 2) return;
  double a = 0.5 * std::sqrt(15.0 / kPi), b = 0.25 * std::sqrt(5.0 / kPi), c = 0.25 * std::sqrt(15.0 / kPi);
  Y[4] = a * x * y; Y[5] = -a * y * z; Y[6] = b * (2 * z * z - x * x - y * y); Y[7] = -a * x * z; Y[8] = c * (x * x - y * y);
  if (degree < 3) return;
  double e = 0.25 * std::sqrt(35.0 / (2.0 * kPi)), f = 0.5 * std::sqrt(105.0 / kPi), g = 0.25 * std::sqrt(21.0 / (2.0 * kPi)),
         h = 0.25 * std::sqrt(7.0 / kPi), k = 0.25 * std::sqrt(105.0 / kPi);
  Y[9]  = -e * y * (3 * x * x - y * y);
  Y[10] =  f * x * y * z;
  Y[11] = -g * y * (4 * z * z - x * x - y * y);
  Y[12] =  h * z * (2 * z * z - 3 * x * x - 3 * y * y);
  Y[13] = -g * x * (4 * z * z - x * x - y * y);
  Y[14] =  k * z * (x * x - y * y);
  Y[15] = -e * x * (x * x - 3 * y * y);
}

// Partial derivatives of the basis polynomials w.r.t. (x,y,z).
void sh_basis_grad(int degree, const double d[3], double* dY) {
  double x = d[0], y = d[1], z = d[2];
  for (int i = 0; i < 48; ++i) dY[i] = 0;
  if (degree < 1) return;
  double c1 = std::sqrt(3.0 / (4.0 * kPi));
  dY[3 * 1 + 1] = -c1; dY[3 * 2 + 2] = c1; dY[3 * 3 + 0] = -c1;
  if (degree < 2) return;
  double a = 0.5 * std::sqrt(15.0 / kPi), b = 0.25 * std::sqrt(5.0 / kPi), c = 0.25 * std::sqrt(15.0 / kPi);
  dY[3 * 4 + 0] = a * y;  dY[3 * 4 + 1] = a * x;
  dY[3 * 5 + 1] = -a * z; dY[3 * 5 + 2] = -a * y;
  dY[3 * 6 + 0] = -2 * b * x; dY[3 * 6 + 1] = -2 * b * y; dY[3 * 6 + 2] = 4 * b * z;
  dY[3 * 7 + 0] = -a * z; dY[3 * 7 + 2] = -a * x;
  dY[3 * 8 + 0] = 2 * c * x; dY[3 * 8 + 1] = -2 * c * y;
  if (degree < 3) return;
  double e = 0.25 * std::sqrt(35.0 / (2.0 * kPi)), f = 0.5 * std::sqrt(105.0 / kPi), g = 0.25 * std::sqrt(21.0 / (2.0 * kPi)),
         h = 0.25 * std::sqrt(7.0 / kPi), k = 0.25 * std::sqrt(105.0 / kPi);
  dY[3 * 9 + 0]  = -e * 6 * x * y;                 dY[3 * 9 + 1]  = -e * (3 * x * x - 3 * y * y);
  dY[3 * 10 + 0] = f * y * z; dY[3 * 10 + 1] = f * x * z; dY[3 * 10 + 2] = f * x * y;
  dY[3 * 11 + 0] = g * 2 * x * y;  dY[3 * 11 + 1] = -g * (4 * z * z - x * x - 3 * y * y); dY[3 * 11 + 2] = -g * 8 * y * z;
  dY[3 * 12 + 0] = -h * 6 * x * z; dY[3 * 12 + 1] = -h * 6 * y * z; dY[3 * 12 + 2] = h * (6 * z * z - 3 * x * x - 3 * y * y);
  dY[3 * 13 + 0] = -g * (4 * z * z - 3 * x * x - y * y); dY[3 * 13 + 1] = g * 2 * x * y; dY[3 * 13 + 2] = -g * 8 * x * z;
  dY[3 * 14 + 0] = k * 2 * x * z; dY[3 * 14 + 1] = -k * 2 * y * z; dY[3 * 14 + 2] = k * (x * x - y * y);
  dY[3 * 15 + 0] = -e * (3 * x * x - 3 * y * y); dY[3 * 15 + 1] = e * 6 * x * y;
}

// ------------------------------------------------------------------ O1 preprocess (Alg.1 l.2-8; Eq.1-2)
static void cull(Proj& out) {
  std::memset(&out, 0, sizeof(Proj));
  out.flags = 1;
}

void preprocess_one(const Config& cfg, const double mu[3], const double s[3], const double q[4], double o,
                    const double* sh, const double W[9], const double b[3], Proj& out, PreSaved* sv) {
  PreSaved local; PreSaved& S = sv ? *sv : local;
  std::memset(&S, 0, sizeof(PreSaved));
  out.flags = 0;
  // l.3: t = W mu + b, (omega,phi) = Pi(t), rho = ||t||
  for (int i = 0; i < 3; ++i) S.t[i] = W[3 * i] * mu[0] + W[3 * i + 1] * mu[1] + W[3 * i + 2] * mu[2] + b[i];
  const double* t = S.t;
  double rho = std::sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
  if (!finite3(mu, 3) || !finite3(s, 3) || !finite3(q, 4) || !std::isfinite(o) || !std::isfinite(rho) ||
      rho <= (double)cfg.r_near) { cull(out); return; }
  double rxz = std::sqrt(t[0] * t[0] + t[2] * t[2]);
  out.rho = rho;
  for (int i = 0; i < 3; ++i) out.dir[i] = t[i] / rho;
  out.lon = std::atan2(t[0], t[2]);                      // Eq.1
  out.lat = std::atan2(t[1], rxz);
  // l.4: Sigma_3D = R diag(s^2) R^T
  quat_to_mat(q, S.R);
  double RS[9];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) RS[3 * i + j] = S.R[3 * i + j] * s[j] * s[j];
  double RT[9]; mat3_T(S.R, RT);
  mat3_mul(RS, RT, S.Sigma3);
  // M = W Sigma_3D W^T
  double WS[9], WT[9]; mat3_mul(W, S.Sigma3, WS); mat3_T(W, WT); mat3_mul(WS, WT, S.M);
  // l.5-6: J, S_phi, Sigma_arc = S_phi J W Sigma_3D W^T J^T S_phi^T   (Eq.2)
  double h = (double)cfg.cov_dilation_px2 * 4.0 * kPi / (double)npix_of_order(cfg.order);   // reading A3
  S.cosphi = rxz / rho; S.sinphi = t[1] / rho;
  double a, bb, c;
  if (rxz > 0) {
    jacobian_eq1(t, S.J);
    double JM[6];
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 3; ++j) {
      double acc = 0; for (int k = 0; k < 3; ++k) acc += S.J[3 * i + k] * S.M[3 * k + j]; JM[3 * i + j] = acc; }
    S.sig_rad[0] = JM[0] * S.J[0] + JM[1] * S.J[1] + JM[2] * S.J[2];
    S.sig_rad[1] = JM[0] * S.J[3] + JM[1] * S.J[4] + JM[2] * S.J[5];
    S.sig_rad[2] = JM[3] * S.J[3] + JM[4] * S.J[4] + JM[5] * S.J[5];
    a = S.cosphi * S.cosphi * S.sig_rad[0] + h;
    bb = S.cosphi * S.sig_rad[1];
    c = S.sig_rad[2] + h;
  } else {
    // reading A22: Gaussian exactly at a pole; e = (1,0,0), n = u x e, Sigma_arc = [e;n] M [e;n]^T / rho^2
    double e[3] = {1, 0, 0};
    double n[3] = {out.dir[1] * e[2] - out.dir[2] * e[1], out.dir[2] * e[0] - out.dir[0] * e[2], out.dir[0] * e[1] - out.dir[1] * e[0]};
    double Me[3], Mn[3];
    for (int i = 0; i < 3; ++i) { Me[i] = S.M[3 * i] * e[0] + S.M[3 * i + 1] * e[1] + S.M[3 * i + 2] * e[2];
                                  Mn[i] = S.M[3 * i] * n[0] + S.M[3 * i + 1] * n[1] + S.M[3 * i + 2] * n[2]; }
    a = (e[0] * Me[0] + e[1] * Me[1] + e[2] * Me[2]) / (rho * rho) + h;
    bb = (e[0] * Mn[0] + e[1] * Mn[1] + e[2] * Mn[2]) / (rho * rho);
    c = (n[0] * Mn[0] + n[1] * Mn[1] + n[2] * Mn[2]) / (rho * rho) + h;
  }
  S.sig_arc[0] = a; S.sig_arc[1] = bb; S.sig_arc[2] = c;
  double det = a * c - bb * bb;
  S.det = det;
  if (!(det > 0) || !std::isfinite(det)) { cull(out); return; }        // reading A23
  out.conic[0] = c / det; out.conic[1] = -bb / det; out.conic[2] = a / det;   // Sigma_arc^{-1}
  // l.7: r_s = 3 sqrt(lambda_max(Sigma_arc)), clamped to pi (reading A4)
  double lmax = 0.5 * (a + c) + std::sqrt(std::max(0.0, 0.25 * (a - c) * (a - c) + bb * bb));
  out.rs = std::min(kPi, 3.0 * std::sqrt(lmax));
  out.opac = o;
  // colour (reading A13): direction from the camera centre to mu, in world space
  for (int i = 0; i < 3; ++i) S.cam[i] = -(W[i] * b[0] + W[3 + i] * b[1] + W[6 + i] * b[2]);
  double v[3] = {mu[0] - S.cam[0], mu[1] - S.cam[1], mu[2] - S.cam[2]};
  S.vlen = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  for (int i = 0; i < 3; ++i) S.vdir[i] = v[i] / S.vlen;
  double Y[16]; sh_basis(cfg.sh_degree, S.vdir, Y);
  int M = n_sh(cfg);
  for (int ch = 0; ch < 3; ++ch) {
    double acc = 0.5;
    for (int m = 0; m < M; ++m) acc += Y[m] * sh[3 * m + ch];
    if (acc < 0) { acc = 0; out.flags |= (uint8_t)(2u << ch); }
    out.rgb[ch] = acc;
  }
}

void sigma_arc_tangent(const double t[3], const double M[9], double out3[3]) {
  double rho = std::sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
  double rxz = std::sqrt(t[0] * t[0] + t[2] * t[2]);
  double e[3] = {t[2] / rxz, 0, -t[0] / rxz};
  double n[3] = {-t[0] * t[1] / (rxz * rho), rxz / rho, -t[2] * t[1] / (rxz * rho)};
  double Me[3], Mn[3];
  for (int i = 0; i < 3; ++i) { Me[i] = M[3 * i] * e[0] + M[3 * i + 1] * e[1] + M[3 * i + 2] * e[2];
                                Mn[i] = M[3 * i] * n[0] + M[3 * i + 1] * n[1] + M[3 * i + 2] * n[2]; }
  out3[0] = (e[0] * Me[0] + e[1] * Me[1] + e[2] * Me[2]) / (rho * rho);
  out3[1] = (e[0] * Mn[0] + e[1] * Mn[1] + e[2] * Mn[2]) / (rho * rho);
  out3[2] = (n[0] * Mn[0] + n[1] * Mn[1] + n[2] * Mn[2]) / (rho * rho);
}

// ------------------------------------------------------------------ O2 tile query (Alg.2; reading A6)
static double rho_max_cached(int order) {
  static std::map<int, double> cache;
  auto it = cache.find(order);
  if (it != cache.end()) return it->second;
  double v = rho_max_closed(order);
  cache[order] = v; return v;
}

void pixel_dir(int order, int64_t p, double v[3]) { to_cam_vec(pix_center_D2(order, p), v); }

static const std::vector<double>& all_dirs(int order) {
  static std::map<int, std::vector<double>> cache;
  auto it = cache.find(order);
  if (it != cache.end()) return it->second;
  int64_t n = npix_of_order(order);
  std::vector<double> d(3 * n);
  for (int64_t p = 0; p < n; ++p) pixel_dir(order, p, &d[3 * p]);
  return cache[order] = std::move(d);
}

namespace {
struct Descent {
  const Config* cfg; const double* u; double R, cosR; int kt, kq; const int32_t* slot;
  std::vector<uint32_t>* out; QueryStats* st;
  void add_tile(int64_t tile) {
    if (slot && slot[tile] < 0) return;
    if (!out->empty() && out->back() == (uint32_t)tile) return;
    out->push_back((uint32_t)tile);
  }
  void visit(int64_t p, int o) {
    double c[3]; pixel_dir(o, p, c);
    st->node_tests++;
    double ang = angle_between(u, c);
    double pr = rho_max_cached(o);
    if (ang > R + pr) return;                                   // zone 0: prune
    if (o <= kt) {
      if (ang + pr <= R) {                                      // zone 3: every descendant centre is inside
        int sh = 2 * (kt - o);
        for (int64_t tl = p << sh; tl < ((p + 1) << sh); ++tl) add_tile(tl);
        return;
      }
    } else {
      int64_t tile = p >> (2 * (o - kt));
      if (!out->empty() && out->back() == (uint32_t)tile) return;   // tile already in the set
      if (ang + pr <= R && o < kq) { add_tile(tile); return; }
    }
    if (o == kq) {                                              // leaf: the defining predicate
      double dot = u[0] * c[0] + u[1] * c[1] + u[2] * c[2];
      st->min_margin = std::min(st->min_margin, std::fabs(dot - cosR));
      if (dot >= cosR) add_tile(p >> (2 * (kq - kt)));
      return;
    }
    for (int ch = 0; ch < 4; ++ch) visit(4 * p + ch, o + 1);
  }
};
}  // namespace

// Alg.3 QUERYDISCRING (§10.2; Eq.5), step by step at the query
// resolution N_side^q = 2^k_q, results mapped back to tile resolution.  Line numbers are Alg.3's.
// Readings: A17 (z-bounds from l.2-3, not the garbled prose), A18 (l.19-20 = ceil / floor: the pixels whose centres lie in
// the longitude interval), epsilon of l.9 = 1e-12 (unstated).  Output sorted ascending, each tile once (the ABI's order).
static void query_disc_ring(const Config& cfg, const double u[3], double rs, const int32_t* slot, std::vector<uint32_t>& out,
                            QueryStats& st) {
  const int kt = tile_order(cfg), kq = query_order(cfg);
  const int64_t N = (int64_t)1 << kq;                                         // l.1
  const double omega = std::atan2(u[0], u[2]);                                // disc centre (omega, phi), Eq.1
  const double phi = std::atan2(u[1], std::sqrt(u[0] * u[0] + u[2] * u[2]));
  const double zc = std::sin(phi);                                            // l.1
  const double phimin = std::max(-kPi / 2, phi - rs), phimax = std::min(kPi / 2, phi + rs);   // l.2
  const double zmin = std::sin(phimin), zmax = std::sin(phimax);              // l.3
  const double cosrs = std::cos(rs);
  // l.4 ZToRingRange: the rings whose z lies in [zmin, zmax] (z decreases with the ring number)
  static std::map<int, std::vector<double>> ring_z_cache;                     // z of every ring of an order, computed once
  std::vector<double>& ring_z = ring_z_cache[kq];
  if (ring_z.empty()) { ring_z.assign(4 * N, 2.0); for (int64_t i = 1; i <= 4 * N - 1; ++i) ring_z[i] = ring_info(kq, i).z; }
  int64_t ir_min = 4 * N, ir_max = 0;
  for (int64_t i = 1; i <= 4 * N - 1; ++i)
    if (ring_z[i] >= zmin && ring_z[i] <= zmax) { ir_min = std::min(ir_min, i); ir_max = std::max(ir_max, i); }
  std::vector<uint32_t> found;
  auto add = [&](const RingInfo& ri, int64_t j) {                             // Ring2Nest(i_r, j), then the ancestor tile
    int64_t p = ring2nest(kq, ri.first + j);
    int64_t tile = p >> (2 * (kq - kt));
    if (slot && slot[tile] < 0) return;
    found.push_back((uint32_t)tile);
  };
  auto margin = [&](const RingInfo& ri, int64_t j) {                          // instrumentation only: distance of a centre to the disc edge
    j = ((j % ri.npix) + ri.npix) % ri.npix;
    double c[3]; to_cam_vec(ring_center(kq, ri.first + j), c);
    st.min_margin = std::min(st.min_margin, std::fabs(u[0] * c[0] + u[1] * c[1] + u[2] * c[2] - cosrs));
  };
  for (int64_t ir = ir_min; ir <= ir_max; ++ir) {                             // l.5
    const RingInfo ri = ring_info(kq, ir);                                    // l.7 (z_r, n_r, omega_0)
    st.node_tests++;
    const double delta = std::sqrt(std::max(0.0, 1 - zc * zc)) * std::sqrt(std::max(0.0, 1 - ri.z * ri.z));   // l.8
    if (delta < 1e-12) {                                                      // l.9 disc centre or ring at a pole
      if (zc * ri.z >= cosrs) for (int64_t j = 0; j < ri.npix; ++j) add(ri, j);   // l.10-11
      continue;                                                               // l.13
    }
    const double cw = (cosrs - zc * ri.z) / delta;                            // l.15, Eq.5
    if (cw <= -1) { for (int64_t j = 0; j < ri.npix; ++j) add(ri, j); }       // l.16-17 full ring
    else if (cw < 1) {                                                        // l.18
      const double dw = std::acos(std::min(1.0, std::max(-1.0, cw)));
      const double a = (omega - dw - ri.lam0) * (double)ri.npix / (2 * kPi);  // l.19
      const double b = (omega + dw - ri.lam0) * (double)ri.npix / (2 * kPi);  // l.20
      const int64_t ipmin = (int64_t)std::ceil(a), ipmax = (int64_t)std::floor(b);
      margin(ri, ipmin); margin(ri, ipmin - 1); margin(ri, ipmax); margin(ri, ipmax + 1);
      if (ipmax - ipmin + 1 >= ri.npix) { for (int64_t j = 0; j < ri.npix; ++j) add(ri, j); }
      else for (int64_t ip = ipmin; ip <= ipmax; ++ip) add(ri, ((ip % ri.npix) + ri.npix) % ri.npix);   // l.21-22
    }
  }
  std::sort(found.begin(), found.end());
  found.erase(std::unique(found.begin(), found.end()), found.end());
  out = found;                                                                // l.26
}

void tile_query_one(const Config& cfg, const double dir_in[3], double rs, const int32_t* slot_of_tile, bool brute,
                    std::vector<uint32_t>& tiles_out, QueryStats& st) {
  int kt = tile_order(cfg), kq = query_order(cfg);
  double nrm = std::sqrt(dir_in[0] * dir_in[0] + dir_in[1] * dir_in[1] + dir_in[2] * dir_in[2]);
  double u[3] = {dir_in[0] / nrm, dir_in[1] / nrm, dir_in[2] / nrm};
  // NESTED (Alg.2, reading A6): centres within r_s + PixRad(k_q).  RING (Alg.3): centres within r_s itself.
  double R = cfg.query_mode == 1 ? std::min(kPi, rs) : std::min(kPi, rs + rho_max_cached(kq));
  double cosR = std::cos(R);
  tiles_out.clear();
  if (brute) {
    const std::vector<double>& d = all_dirs(kq);
    int64_t nq = npix_of_order(kq);
    int sh = 2 * (kq - kt);
    for (int64_t qp = 0; qp < nq; ++qp) {
      double dot = u[0] * d[3 * qp] + u[1] * d[3 * qp + 1] + u[2] * d[3 * qp + 2];
      st.node_tests++;
      st.min_margin = std::min(st.min_margin, std::fabs(dot - cosR));
      if (dot >= cosR) {
        int64_t tile = qp >> sh;
        if (slot_of_tile && slot_of_tile[tile] < 0) continue;
        if (tiles_out.empty() || tiles_out.back() != (uint32_t)tile) tiles_out.push_back((uint32_t)tile);
      }
    }
    return;
  }
  if (cfg.query_mode == 1) { query_disc_ring(cfg, u, R, slot_of_tile, tiles_out, st); return; }
  Descent D{&cfg, u, R, cosR, kt, kq, slot_of_tile, &tiles_out, &st};
  for (int64_t f = 0; f < 12; ++f) D.visit(f, 0);
}

// ------------------------------------------------------------------ O5 blend forward (Alg.1 l.17-30; Eq.6)
namespace {
struct Frame { double u[3], e[3], n[3]; };
// unit direction and its (east,north) tangent basis (pole guard A22)
Frame make_frame(const double dir[3]) {
  Frame F;
  double nrm = std::sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
  for (int i = 0; i < 3; ++i) F.u[i] = dir[i] / nrm;
  double rxz = std::sqrt(F.u[0] * F.u[0] + F.u[2] * F.u[2]);
  if (rxz > 0) { F.e[0] = F.u[2] / rxz; F.e[1] = 0; F.e[2] = -F.u[0] / rxz; }
  else { F.e[0] = 1; F.e[1] = 0; F.e[2] = 0; }
  F.n[0] = F.u[1] * F.e[2] - F.u[2] * F.e[1];
  F.n[1] = F.u[2] * F.e[0] - F.u[0] * F.e[2];
  F.n[2] = F.u[0] * F.e[1] - F.u[1] * F.e[0];
  return F;
}
struct Offset { double a, b, c, s, g, k, dx, dy; };
// SphericalOffset (Alg.1 l.22): great-circle distance g (haversine-equivalent atan2 form) decomposed along the bearing
// taken at the Gaussian centre towards the pixel, in the Gaussian's (east,north) basis (reading A11).
Offset spherical_offset(const Frame& F, const double up[3]) {
  Offset o;
  o.a = F.e[0] * up[0] + F.e[1] * up[1] + F.e[2] * up[2];
  o.b = F.n[0] * up[0] + F.n[1] * up[1] + F.n[2] * up[2];
  o.c = F.u[0] * up[0] + F.u[1] * up[1] + F.u[2] * up[2];
  o.s = std::sqrt(o.a * o.a + o.b * o.b);
  o.g = std::atan2(o.s, o.c);
  o.k = (o.s > 0) ? o.g / o.s : 1.0;
  o.dx = o.k * o.a; o.dy = o.k * o.b;
  return o;
}
}  // namespace

void blend_pixel_fwd(const Config& cfg, const double up[3], const Proj* recs, const uint32_t* vals, uint64_t start,
                     uint64_t end, PixelOut& out, BlendCounters* ctr) {
  double T = 1.0, C[3] = {0, 0, 0};
  uint32_t n_last = 0;
  double margin = 1e300;
  const double amin = cfg.alpha_min, amax = cfg.alpha_max, eps = cfg.t_eps;
  for (uint64_t j = start; j < end; ++j) {
    const Proj& G = recs[vals[j]];
    Frame F = make_frame(G.dir);
    Offset d = spherical_offset(F, up);
    double power = -0.5 * (G.conic[0] * d.dx * d.dx + G.conic[2] * d.dy * d.dy) - G.conic[1] * d.dx * d.dy;
    if (ctr) ctr->evaluated++;
    if (power > 0) continue;
    double raw = G.opac * std::exp(power);
    double alpha = std::min(amax, raw);
    if (amin > 0) margin = std::min(margin, std::fabs(alpha - amin) / amin);
    if (amax > 0) margin = std::min(margin, std::fabs(raw - amax) / amax);
    if (alpha < amin) continue;
    if (ctr) ctr->contributing++;
    for (int ch = 0; ch < 3; ++ch) C[ch] += T * alpha * G.rgb[ch];
    T = T * (1.0 - alpha);
    n_last = (uint32_t)(j - start + 1);
    if (eps > 0) margin = std::min(margin, std::fabs(T - eps) / eps);
    if (T < eps) { if (ctr) ctr->early_exit_pixels++; break; }
  }
  for (int ch = 0; ch < 3; ++ch) out.color[ch] = C[ch] + T * (double)cfg.bg[ch];
  out.alpha = 1.0 - T;
  out.n_last = n_last;
  out.margin = margin;
}

// ------------------------------------------------------------------ O7 blend backward
void blend_pixel_bwd(const Config& cfg, const double up[3], const Proj* recs, const uint32_t* vals, uint64_t start,
                     uint32_t n_last, const double gcol[3], double galpha, RecGrad* grads) {
  const double amin = cfg.alpha_min, amax = cfg.alpha_max;
  // forward replay to get the final transmittance (only entries < n_last matter)
  std::vector<double> alphas(n_last, 0.0), pows(n_last, 0.0);
  std::vector<char> used(n_last, 0), clamped(n_last, 0);
  double T = 1.0;
  for (uint32_t m = 0; m < n_last; ++m) {
    const Proj& G = recs[vals[start + m]];
    Frame F = make_frame(G.dir);
    Offset d = spherical_offset(F, up);
    double power = -0.5 * (G.conic[0] * d.dx * d.dx + G.conic[2] * d.dy * d.dy) - G.conic[1] * d.dx * d.dy;
    if (power > 0) continue;
    double raw = G.opac * std::exp(power);
    double alpha = std::min(amax, raw);
    if (alpha < amin) continue;
    used[m] = 1; clamped[m] = raw > amax; alphas[m] = alpha; pows[m] = power;
    T *= (1.0 - alpha);
  }
  const double Tfinal = T;
  double S[3] = {Tfinal * cfg.bg[0], Tfinal * cfg.bg[1], Tfinal * cfg.bg[2]};   // colour accumulated behind j
  for (int64_t m = (int64_t)n_last - 1; m >= 0; --m) {
    if (!used[m]) continue;
    uint32_t id = vals[start + m];
    const Proj& G = recs[id];
    RecGrad& g = grads[id];
    double alpha = alphas[m];
    T = T / (1.0 - alpha);                                   // transmittance before entry m
    double dL_dalpha = 0;
    for (int ch = 0; ch < 3; ++ch) {
      g.rgb[ch] += T * alpha * gcol[ch];
      dL_dalpha += gcol[ch] * (T * G.rgb[ch] - S[ch] / (1.0 - alpha));
    }
    dL_dalpha += galpha * Tfinal / (1.0 - alpha);            // alpha_out = 1 - prod(1-alpha)
    for (int ch = 0; ch < 3; ++ch) S[ch] += T * alpha * G.rgb[ch];
    if (clamped[m]) continue;                                // gradient through a clamped alpha is zero (A7)
    double ep = std::exp(pows[m]);
    g.opac += ep * dL_dalpha;
    double gp = alpha * dL_dalpha;                           // dL/dpower
    Frame F = make_frame(G.dir);
    Offset d = spherical_offset(F, up);
    g.conic[0] += -0.5 * d.dx * d.dx * gp;
    g.conic[1] += -d.dx * d.dy * gp;
    g.conic[2] += -0.5 * d.dy * d.dy * gp;
    double gdx = -(G.conic[0] * d.dx + G.conic[1] * d.dy) * gp;
    double gdy = -(G.conic[1] * d.dx + G.conic[2] * d.dy) * gp;
    // (dx,dy) = k(s,c) (a,b), k = atan2(s,c)/s
    double ga, gb, gc;
    if (d.s > 0) {
      double den = d.s * d.s + d.c * d.c;
      double dg_ds = d.c / den, dg_dc = -d.s / den;
      double dk_ds = (dg_ds - d.k) / d.s, dk_dc = dg_dc / d.s;
      double gk = gdx * d.a + gdy * d.b;
      ga = d.k * gdx + gk * dk_ds * d.a / d.s;
      gb = d.k * gdy + gk * dk_ds * d.b / d.s;
      gc = gk * dk_dc;
    } else { ga = gdx; gb = gdy; gc = 0; }
    // a = e.up, b = n.up, c = u.up with e(lon), n(lon,lat), u(lon,lat):
    //   de/dlon = (-sin lon,0,-cos lon) ; dn/dlon = (-sin lat cos lon, 0, sin lat sin lon) ; du/dlon = cos lat * e
    //   de/dlat = 0                     ; dn/dlat = -u                                     ; du/dlat = n
    double sl = F.u[1];                                      // sin lat
    double cl = std::sqrt(F.u[0] * F.u[0] + F.u[2] * F.u[2]);// cos lat
    double slon = (cl > 0) ? F.u[0] / cl : 0.0, clon = (cl > 0) ? F.u[2] / cl : 1.0;
    double de_dlon[3] = {-slon, 0, -clon};
    double dn_dlon[3] = {-sl * clon, 0, sl * slon};
    double du_dlon[3] = {cl * F.e[0], cl * F.e[1], cl * F.e[2]};
    double da_dlon = de_dlon[0] * up[0] + de_dlon[1] * up[1] + de_dlon[2] * up[2];
    double db_dlon = dn_dlon[0] * up[0] + dn_dlon[1] * up[1] + dn_dlon[2] * up[2];
    double dc_dlon = du_dlon[0] * up[0] + du_dlon[1] * up[1] + du_dlon[2] * up[2];
    double db_dlat = -d.c, dc_dlat = d.b;
    g.mu2[0] += ga * da_dlon + gb * db_dlon + gc * dc_dlon;
    g.mu2[1] += gb * db_dlat + gc * dc_dlat;
  }
}

// ------------------------------------------------------------------ O8 preprocess backward (Eq.3-4)
void preprocess_bwd_one(const Config& cfg, const double mu[3], const double s[3], const double q[4],
                        const double* sh, const double W[9], const double b[3], const RecGrad& g,
                        ParamGrad& pg, double* dsh, double* dbg) {
  Proj P; PreSaved S;
  // opacity is not needed for the geometry chain; pass 0.5
  preprocess_one(cfg, mu, s, q, 0.5, sh, W, b, P, &S);
  if (dbg) for (int i = 0; i < 8; ++i) dbg[i] = 0;
  if (P.flags & 1) return;
  const double* t = S.t;
  double dL_dt[3] = {0, 0, 0};
  double dL_dmu_world[3] = {0, 0, 0};
  int M = n_sh(cfg);
  // ---- colour: rgb_ch = max(0, 0.5 + sum_m Y_m(vdir) sh[m,ch])
  {
    double Y[16], dY[48];
    sh_basis(cfg.sh_degree, S.vdir, Y);
    sh_basis_grad(cfg.sh_degree, S.vdir, dY);
    double dL_dv[3] = {0, 0, 0};
    for (int ch = 0; ch < 3; ++ch) {
      if (P.flags & (2u << ch)) continue;                    // clamped channel: zero gradient
      for (int m = 0; m < M; ++m) {
        dsh[3 * m + ch] += Y[m] * g.rgb[ch];
        for (int k = 0; k < 3; ++k) dL_dv[k] += dY[3 * m + k] * sh[3 * m + ch] * g.rgb[ch];
      }
    }
    // vdir = v/|v|: d vdir / d v = (I - vdir vdir^T)/|v|
    double dot = dL_dv[0] * S.vdir[0] + dL_dv[1] * S.vdir[1] + dL_dv[2] * S.vdir[2];
    for (int k = 0; k < 3; ++k) dL_dmu_world[k] += (dL_dv[k] - dot * S.vdir[k]) / S.vlen;
  }
  double rxz2 = t[0] * t[0] + t[2] * t[2], rxz = std::sqrt(rxz2), R2 = rxz2 + t[1] * t[1];
  if (!(rxz > 0)) {
    // pole (A22): gradients there are untested; only the colour path is propagated
    for (int k = 0; k < 3; ++k) pg.mu[k] += dL_dmu_world[k];
    return;
  }
  // ---- conic -> Sigma_arc (a,b,c), off-diagonal stored once (A15)
  double a = S.sig_arc[0], bb = S.sig_arc[1], c = S.sig_arc[2], det = S.det, d2 = det * det;
  double gA = g.conic[0], gB = g.conic[1], gC = g.conic[2];
  // A = c/det, B = -b/det, C = a/det
  double L_a = gA * (-c * c / d2) + gB * (bb * c / d2) + gC * (-bb * bb / d2);
  double L_b = gA * (2 * bb * c / d2) + gB * (-(a * c + bb * bb) / d2) + gC * (2 * a * bb / d2);
  double L_c = gA * (-bb * bb / d2) + gB * (a * bb / d2) + gC * (-a * a / d2);
  // ---- Eq.3: Sigma_arc = S_phi Sigma_rad S_phi^T
  double cp = S.cosphi, sp = S.sinphi;
  double L_ww = cp * cp * L_a, L_wp = cp * L_b, L_pp = L_c;          // L_Sigma_rad = S^T L_Sigma_arc S
  double L_phi_S = -sp * (2 * cp * S.sig_rad[0] * L_a + S.sig_rad[1] * L_b);   // literal Eq.3
  if (dbg) { dbg[0] = L_phi_S; dbg[1] = L_a; dbg[2] = L_b; dbg[3] = L_c; dbg[4] = S.sig_rad[0]; dbg[5] = S.sig_rad[1];
             dbg[6] = S.sig_rad[2]; dbg[7] = std::atan2(t[1], rxz); }
  // ---- Sigma_rad = J M J^T.  Full symmetric gradient matrix G (off-diagonal halves).
  double G2[4] = {L_ww, 0.5 * L_wp, 0.5 * L_wp, L_pp};
  const double* J = S.J;
  // dL/dJ = 2 G J M
  double JM[6];
  for (int i = 0; i < 2; ++i) for (int j = 0; j < 3; ++j) {
    double acc = 0; for (int k = 0; k < 3; ++k) acc += J[3 * i + k] * S.M[3 * k + j]; JM[3 * i + j] = acc; }
  double dL_dJ[6];
  for (int i = 0; i < 2; ++i) for (int j = 0; j < 3; ++j)
    dL_dJ[3 * i + j] = 2 * (G2[2 * i] * JM[j] + G2[2 * i + 1] * JM[3 + j]);
  // dL/dM = J^T G J ; dL/dSigma3 = W^T dL/dM W
  double dL_dM[9];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    double acc = 0;
    for (int p = 0; p < 2; ++p) for (int r = 0; r < 2; ++r) acc += J[3 * p + i] * G2[2 * p + r] * J[3 * r + j];
    dL_dM[3 * i + j] = acc;
  }
  double WT[9], tmp[9], dL_dS3[9];
  mat3_T(W, WT); mat3_mul(WT, dL_dM, tmp); mat3_mul(tmp, W, dL_dS3);
  // Sigma3 = R diag(s^2) R^T : dL/ds_k = 2 s_k (R^T G R)_kk ; dL/dR = 2 G R diag(s^2)
  const double* R = S.R;
  double RT[9], GR[9], RtGR[9];
  mat3_T(R, RT); mat3_mul(dL_dS3, R, GR); mat3_mul(RT, GR, RtGR);
  for (int k = 0; k < 3; ++k) pg.s[k] += 2 * s[k] * RtGR[4 * k];
  double dL_dR[9];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) dL_dR[3 * i + j] = 2 * GR[3 * i + j] * s[j] * s[j];
  // R(q) polynomial derivative
  {
    double w = q[0], x = q[1], y = q[2], z = q[3];
    const double* D = dL_dR;
    pg.q[0] += 2 * (-z * D[1] + y * D[2] + z * D[3] - x * D[5] - y * D[6] + x * D[7]);
    pg.q[1] += 2 * (y * D[1] + z * D[2] + y * D[3] - 2 * x * D[4] - w * D[5] + z * D[6] + w * D[7] - 2 * x * D[8]);
    pg.q[2] += 2 * (-2 * y * D[0] + x * D[1] + w * D[2] + x * D[3] + z * D[5] - w * D[6] + z * D[7] - 2 * y * D[8]);
    pg.q[3] += 2 * (-2 * z * D[0] - w * D[1] + x * D[2] + w * D[3] - 2 * z * D[4] + y * D[5] + x * D[6] + y * D[7]);
  }
  // ---- Eq.4, J path: dL/dt|_J = sum_ij dL/dJ_ij dJ_ij/dt
  {
    double tx = t[0], ty = t[1], tz = t[2], r = rxz, r2 = rxz2, r4 = r2 * r2;
    double D = r * R2;
    double dD[3] = {tx * (R2 / r + 2 * r), 2 * r * ty, tz * (R2 / r + 2 * r)};
    double dJ[6][3];
    dJ[0][0] = -2 * tx * tz / r4;        dJ[0][1] = 0; dJ[0][2] = (tx * tx - tz * tz) / r4;
    dJ[1][0] = 0; dJ[1][1] = 0; dJ[1][2] = 0;
    dJ[2][0] = (tx * tx - tz * tz) / r4; dJ[2][1] = 0; dJ[2][2] = 2 * tx * tz / r4;
    dJ[3][0] = -ty / D + tx * ty * dD[0] / (D * D);
    dJ[3][1] = -tx / D + tx * ty * dD[1] / (D * D);
    dJ[3][2] = tx * ty * dD[2] / (D * D);
    dJ[4][0] = (tx / r) / R2 - 2 * r * tx / (R2 * R2);
    dJ[4][1] = -2 * r * ty / (R2 * R2);
    dJ[4][2] = (tz / r) / R2 - 2 * r * tz / (R2 * R2);
    dJ[5][0] = tz * ty * dD[0] / (D * D);
    dJ[5][1] = -tz / D + tz * ty * dD[1] / (D * D);
    dJ[5][2] = -ty / D + tz * ty * dD[2] / (D * D);
    for (int ij = 0; ij < 6; ++ij) for (int k = 0; k < 3; ++k) dL_dt[k] += dL_dJ[ij] * dJ[ij][k];
  }
  // ---- Eq.4, S_phi path: dL/dt|_S = L_phi|S * dphi/dt (second row of J)
  for (int k = 0; k < 3; ++k) dL_dt[k] += L_phi_S * J[3 + k];
  // ---- mu' path: dL/dmu' J
  for (int k = 0; k < 3; ++k) dL_dt[k] += g.mu2[0] * J[k] + g.mu2[1] * J[3 + k];
  // ---- world space: dL/dmu = W^T dL/dt
  for (int k = 0; k < 3; ++k)
    pg.mu[k] += W[k] * dL_dt[0] + W[3 + k] * dL_dt[1] + W[6 + k] * dL_dt[2] + dL_dmu_world[k];
}

}  // namespace orc
