// ORACLE — TEST INFRASTRUCTURE ONLY.  C entry points for the ctypes wrapper (oracle/__init__.py).
// Stage functions take the same fp32/u64/u32 arrays the library's ABI stores between stages (DESIGN.md
// "Readings" P1: inter-stage records are fp32; every stage converts its inputs to double and computes in double).
// The *_f64 functions run preprocess -> blend without any fp32 rounding, for finite-difference pins.
#include "orc_healpix.hpp"
#include "orc_raster.hpp"
#include "orc_resample.hpp"
#include "orc_hssim.hpp"
#include <cmath>
#include <cstring>
#include <vector>
#include <algorithm>

using namespace orc;

namespace {
std::vector<uint64_t> g_keys;
std::vector<uint32_t> g_vals;

inline uint32_t f32_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

void load_proj(const Config& cfg, int v, const float* dir, const float* conic_opac, const float* rgb,
               const uint8_t* flags, std::vector<Proj>& recs) {
  int P = cfg.n_gauss;
  recs.resize(P);
  for (int i = 0; i < P; ++i) {
    size_t k = (size_t)v * P + i;
    Proj& r = recs[i];
    std::memset(&r, 0, sizeof(Proj));
    for (int c = 0; c < 3; ++c) { r.dir[c] = dir[3 * k + c]; r.rgb[c] = rgb[3 * k + c]; r.conic[c] = conic_opac[4 * k + c]; }
    r.opac = conic_opac[4 * k + 3];
    r.flags = flags ? flags[k] : 0;
  }
}

inline bool pixel_on(const uint32_t* bits, int64_t p) { return !bits || ((bits[p >> 5] >> (p & 31)) & 1u); }
}  // namespace

extern "C" {

// ---------------------------------------------------------------- HEALPix
int64_t orc_npix(int order) { return npix_of_order(order); }
void orc_nest2xyf(int order, int64_t p, int64_t* xyf) { XYF c = nest2xyf(order, p); xyf[0] = c.x; xyf[1] = c.y; xyf[2] = c.f; }
int64_t orc_xyf2nest(int order, int64_t x, int64_t y, int f) { XYF c{x, y, f}; return xyf2nest(order, c); }
// which: 1 = D1 (plane), 2 = D2 (ring form of the nested pixel), 3 = textbook RING-order centre (p is a RING index)
void orc_centers(int order, int which, int64_t first, int64_t n, double* z, double* lam, double* vec_cam) {
  for (int64_t i = 0; i < n; ++i) {
    ZPhi a = which == 1 ? pix_center_D1(order, first + i) : which == 2 ? pix_center_D2(order, first + i) : ring_center(order, first + i);
    if (z) z[i] = a.z;
    if (lam) lam[i] = a.lam;
    if (vec_cam) to_cam_vec(a, vec_cam + 3 * i);
  }
}
void orc_corner(int order, int64_t p, int corner, double* vec_cam) { to_cam_vec(pix_corner_D1(order, p, corner), vec_cam); }
void orc_nest2ring(int order, int64_t first, int64_t n, int64_t* out) { for (int64_t i = 0; i < n; ++i) out[i] = nest2ring(order, first + i); }
void orc_ring2nest(int order, int64_t first, int64_t n, int64_t* out) { for (int64_t i = 0; i < n; ++i) out[i] = ring2nest(order, first + i); }
void orc_ang2pix(int order, int64_t n, const double* z, const double* lam, int64_t* out) { for (int64_t i = 0; i < n; ++i) out[i] = ang2pix_nest(order, z[i], lam[i]); }
// camera-frame unit vectors -> NESTED pixel
void orc_vec2pix(int order, int64_t n, const double* v, int64_t* out) {
  for (int64_t i = 0; i < n; ++i) {
    double x = v[3 * i], y = v[3 * i + 1], zc = v[3 * i + 2];
    double nrm = std::sqrt(x * x + y * y + zc * zc);
    out[i] = ang2pix_nest(order, y / nrm, std::atan2(x, zc));
  }
}
int64_t orc_ring_npix_in_ring(int order, int64_t i) { return ring_npix_in_ring(order, i); }
double orc_rho_max_bruteforce(int order) { return rho_max_bruteforce(order); }
double orc_rho_max_closed(int order) { return rho_max_closed(order); }

// ---------------------------------------------------------------- masks (PAPER.md:62 M_C; built on the host, mask is an INPUT of the path)
// kind 0: cap  u_p . axis >= cos(half_angle)           params = axis[3], half_angle
// kind 1: pinhole frustum in the frame (right,up,fwd):  params = right[3], up[3], fwd[3], tan_x, tan_y
void orc_mask(int order, int kind, const double* prm, uint32_t* bits /*N_pix/32 words*/) {
  int64_t n = npix_of_order(order);
  std::memset(bits, 0, (size_t)((n + 31) / 32) * 4);
  for (int64_t p = 0; p < n; ++p) {
    double v[3]; pixel_dir(order, p, v);
    bool on;
    if (kind == 0) on = (v[0] * prm[0] + v[1] * prm[1] + v[2] * prm[2]) >= std::cos(prm[3]);
    else {
      double x = v[0] * prm[0] + v[1] * prm[1] + v[2] * prm[2];
      double y = v[0] * prm[3] + v[1] * prm[4] + v[2] * prm[5];
      double z = v[0] * prm[6] + v[1] * prm[7] + v[2] * prm[8];
      on = z > 0 && std::fabs(x) <= prm[9] * z && std::fabs(y) <= prm[10] * z;
    }
    if (on) bits[p >> 5] |= 1u << (p & 31);
  }
}

// ---------------------------------------------------------------- image synthesis (orc_resample.hpp; Eq.7, Eq.9, Eq.11-15)
int orc_cam_pixel_dir(int model, int W, int H, double p0, double p1, double u, double v, double* d) {
  Camera c{model, W, H, p0, p1};
  return cam_pixel_dir(c, u, v, d) ? 1 : 0;
}
int orc_cam_project(int model, int W, int H, double p0, double p1, const double* d, double* uv) {
  Camera c{model, W, H, p0, p1};
  return cam_project(c, d, uv[0], uv[1]) ? 1 : 0;
}
int orc_interp_weights(int order, double theta, double lam, int64_t* pix, double* w) { return interp_weights(order, theta, lam, pix, w); }
void orc_resample_fwd(int order, int model, int W, int H, double p0, double p1, const int32_t* slot_of_tile, const uint32_t* bits,
                      const float* image, int channels, double* out, uint8_t* valid) {
  Camera c{model, W, H, p0, p1};
  resample_fwd(order, c, slot_of_tile, bits, image, channels, out, valid);
}
void orc_resample_bwd(int order, int model, int W, int H, double p0, double p1, const int32_t* slot_of_tile, const uint32_t* bits,
                      int64_t n_slot, const double* dL_dout, int channels, double* dL_dimage) {
  Camera c{model, W, H, p0, p1};
  resample_bwd(order, c, slot_of_tile, bits, n_slot, dL_dout, channels, dL_dimage);
}
void orc_camera_mask(int order, int model, int W, int H, double p0, double p1, uint32_t* bits) {
  Camera c{model, W, H, p0, p1};
  camera_mask(order, c, bits);
}

// ---------------------------------------------------------------- O1 preprocess, fp32 ABI
void orc_preprocess(const Config* cfg, const float* means, const float* scales, const float* quats, const float* opac,
                    const float* sh, const float* Wv, const float* bv,
                    float* dir, float* lonlat, float* rho, float* conic_opac, float* rs, float* rgb, uint8_t* flags) {
  int P = cfg->n_gauss, M = n_sh(*cfg);
  std::vector<double> shd(3 * M);
  for (int v = 0; v < cfg->n_views; ++v) {
    double W[9], b[3];
    for (int i = 0; i < 9; ++i) W[i] = Wv[9 * v + i];
    for (int i = 0; i < 3; ++i) b[i] = bv[3 * v + i];
    for (int i = 0; i < P; ++i) {
      double mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
      double s[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
      double q[4] = {quats[4 * i], quats[4 * i + 1], quats[4 * i + 2], quats[4 * i + 3]};
      for (int m = 0; m < 3 * M; ++m) shd[m] = sh[(size_t)i * 3 * M + m];
      Proj r;
      preprocess_one(*cfg, mu, s, q, opac[i], shd.data(), W, b, r, nullptr);
      size_t k = (size_t)v * P + i;
      for (int c = 0; c < 3; ++c) { dir[3 * k + c] = (float)r.dir[c]; rgb[3 * k + c] = (float)r.rgb[c]; conic_opac[4 * k + c] = (float)r.conic[c]; }
      conic_opac[4 * k + 3] = (float)r.opac;
      lonlat[2 * k] = (float)r.lon; lonlat[2 * k + 1] = (float)r.lat;
      rho[k] = (float)r.rho; rs[k] = (float)r.rs; flags[k] = r.flags;
    }
  }
}

// Sigma_arc of one Gaussian two ways (pin): literal Eq.2 (incl. dilation h) and tangent-basis form (without h).
void orc_sigma_arc_both(const Config* cfg, const double* mu, const double* s, const double* q, const double* W, const double* b,
                        double* literal3, double* tangent3, double* J6, double* t3) {
  Proj r; PreSaved sv; double sh[48] = {0};
  preprocess_one(*cfg, mu, s, q, 0.5, sh, W, b, r, &sv);
  for (int i = 0; i < 3; ++i) { literal3[i] = sv.sig_arc[i]; t3[i] = sv.t[i]; }
  for (int i = 0; i < 6; ++i) J6[i] = sv.J[i];
  sigma_arc_tangent(sv.t, sv.M, tangent3);
}
void orc_sh_basis(int degree, const double* d, double* Y16) { sh_basis(degree, d, Y16); }
void orc_sh_basis_grad(int degree, const double* d, double* dY48) { sh_basis_grad(degree, d, dY48); }

// ---------------------------------------------------------------- O2 tile query, fp32 ABI
// Fills offsets[V*P+1]; pairs are kept in a static buffer and copied out by orc_tile_query_fetch.
// gauss_subset (may be null): only these Gaussian ids are queried (others get zero tiles) — for sampled brute-force pins.
int64_t orc_tile_query(const Config* cfg, const float* dir, const float* rho, const float* rs, const uint8_t* flags,
                       const int32_t* slot_of_tile, int brute, const int32_t* gauss_subset, int n_subset,
                       uint64_t* offsets, double* min_margin, int64_t* node_tests) {
  int P = cfg->n_gauss; int64_t NT = n_tiles(*cfg);
  g_keys.clear(); g_vals.clear();
  QueryStats st; st.min_margin = 1e300; st.node_tests = 0;
  std::vector<char> sel;
  if (gauss_subset) { sel.assign(P, 0); for (int i = 0; i < n_subset; ++i) sel[gauss_subset[i]] = 1; }
  std::vector<uint32_t> tiles;
  for (int v = 0; v < cfg->n_views; ++v)
    for (int i = 0; i < P; ++i) {
      size_t k = (size_t)v * P + i;
      offsets[k] = g_keys.size();
      if ((flags[k] & 1) || (gauss_subset && !sel[i])) continue;
      double d[3] = {dir[3 * k], dir[3 * k + 1], dir[3 * k + 2]};
      tile_query_one(*cfg, d, (double)rs[k], slot_of_tile, brute != 0, tiles, st);
      uint32_t depth = f32_bits(rho[k]);                                     // reading A10
      for (uint32_t tl : tiles) {
        g_keys.push_back((((uint64_t)v * (uint64_t)NT + tl) << 32) | depth);  // Alg.1 l.12: ((t, rho), i)
        g_vals.push_back((uint32_t)i);
      }
    }
  offsets[(size_t)cfg->n_views * P] = g_keys.size();
  if (min_margin) *min_margin = st.min_margin;
  if (node_tests) *node_tests = st.node_tests;
  return (int64_t)g_keys.size();
}
void orc_tile_query_fetch(uint64_t* keys, uint32_t* vals) {
  if (!g_keys.empty()) { std::memcpy(keys, g_keys.data(), g_keys.size() * 8); std::memcpy(vals, g_vals.data(), g_vals.size() * 4); }
  g_keys.clear(); g_keys.shrink_to_fit(); g_vals.clear(); g_vals.shrink_to_fit();
}

// ---------------------------------------------------------------- O3 sort (Alg.1 l.15): std::stable_sort on the key alone
void orc_sort(uint64_t n, uint64_t* keys, uint32_t* vals) {
  std::vector<uint64_t> idx(n);
  for (uint64_t i = 0; i < n; ++i) idx[i] = i;
  std::stable_sort(idx.begin(), idx.end(), [&](uint64_t a, uint64_t b) { return keys[a] < keys[b]; });
  std::vector<uint64_t> k2(n); std::vector<uint32_t> v2(n);
  for (uint64_t i = 0; i < n; ++i) { k2[i] = keys[idx[i]]; v2[i] = vals[idx[i]]; }
  if (n) { std::memcpy(keys, k2.data(), n * 8); std::memcpy(vals, v2.data(), n * 4); }
}

// ---------------------------------------------------------------- O4 ranges (Alg.1 l.16): linear scan; empty -> (0,0)
void orc_tile_ranges(const Config* cfg, uint64_t n, const uint64_t* keys, uint64_t* ranges) {
  int64_t NT = n_tiles(*cfg) * cfg->n_views;
  for (int64_t t = 0; t < 2 * NT; ++t) ranges[t] = 0;
  for (uint64_t j = 0; j < n; ++j) {
    uint64_t id = keys[j] >> 32;
    if (j == 0 || (keys[j - 1] >> 32) != id) ranges[2 * id] = j;
    if (j + 1 == n || (keys[j + 1] >> 32) != id) ranges[2 * id + 1] = j + 1;
  }
}

// ---------------------------------------------------------------- O5/O6 blend forward + mask, fp32 ABI
// active_tiles null => full sphere, slot = tile.  slots_todo null => all slots, else only those (others untouched).
void orc_render_fwd(const Config* cfg, const float* dir, const float* conic_opac, const float* rgb,
                    const uint32_t* active_tiles, int n_active, const uint32_t* pixel_mask_bits,
                    const uint64_t* ranges, const uint32_t* vals, const int32_t* slots_todo, int n_todo,
                    float* color, float* alpha, uint32_t* n_last, double* margin, int64_t* counters /*[3]*/) {
  int64_t NT = n_tiles(*cfg);
  int64_t S = active_tiles ? n_active : NT;
  int ppt = 1 << (2 * cfg->tile_log2);
  BlendCounters ctr{0, 0, 0};
  std::vector<Proj> recs;
  for (int v = 0; v < cfg->n_views; ++v) {
    load_proj(*cfg, v, dir, conic_opac, rgb, nullptr, recs);
    int64_t ns = slots_todo ? n_todo : S;
    for (int64_t si = 0; si < ns; ++si) {
      int64_t slot = slots_todo ? slots_todo[si] : si;
      int64_t tile = active_tiles ? active_tiles[slot] : slot;
      uint64_t start = ranges[2 * (v * NT + tile)], end = ranges[2 * (v * NT + tile) + 1];
      for (int i = 0; i < ppt; ++i) {
        int64_t p = tile * ppt + i;
        size_t o = ((size_t)v * S + slot) * ppt + i;
        if (!pixel_on(pixel_mask_bits, p)) {
          color[3 * o] = color[3 * o + 1] = color[3 * o + 2] = 0; alpha[o] = 0; n_last[o] = 0;
          if (margin) margin[o] = 1e300;
          continue;
        }
        double up[3]; pixel_dir(cfg->order, p, up);
        PixelOut po;
        blend_pixel_fwd(*cfg, up, recs.data(), vals, start, end, po, &ctr);
        for (int c = 0; c < 3; ++c) color[3 * o + c] = (float)po.color[c];
        alpha[o] = (float)po.alpha; n_last[o] = po.n_last;
        if (margin) margin[o] = po.margin;
      }
    }
  }
  if (counters) { counters[0] = ctr.evaluated; counters[1] = ctr.contributing; counters[2] = ctr.early_exit_pixels; }
}

// ---------------------------------------------------------------- O7 blend backward, fp32 ABI inputs, double outputs
void orc_render_bwd(const Config* cfg, const float* dir, const float* conic_opac, const float* rgb,
                    const uint32_t* active_tiles, int n_active, const uint32_t* pixel_mask_bits,
                    const uint64_t* ranges, const uint32_t* vals, const uint32_t* n_last,
                    const float* dL_dcolor, const float* dL_dalpha,
                    double* dL_drgb, double* dL_dconic, double* dL_dmu2, double* dL_dopac) {
  int P = cfg->n_gauss; int64_t NT = n_tiles(*cfg);
  int64_t S = active_tiles ? n_active : NT;
  int ppt = 1 << (2 * cfg->tile_log2);
  for (int i = 0; i < P; ++i) dL_dopac[i] = 0;
  std::vector<Proj> recs;
  std::vector<RecGrad> grads(P);
  for (int v = 0; v < cfg->n_views; ++v) {
    load_proj(*cfg, v, dir, conic_opac, rgb, nullptr, recs);
    std::memset(grads.data(), 0, sizeof(RecGrad) * P);
    for (int64_t slot = 0; slot < S; ++slot) {
      int64_t tile = active_tiles ? active_tiles[slot] : slot;
      uint64_t start = ranges[2 * (v * NT + tile)];
      for (int i = 0; i < ppt; ++i) {
        int64_t p = tile * ppt + i;
        size_t o = ((size_t)v * S + slot) * ppt + i;
        if (!pixel_on(pixel_mask_bits, p) || n_last[o] == 0) continue;
        double up[3]; pixel_dir(cfg->order, p, up);
        double gc[3] = {dL_dcolor[3 * o], dL_dcolor[3 * o + 1], dL_dcolor[3 * o + 2]};
        blend_pixel_bwd(*cfg, up, recs.data(), vals, start, n_last[o], gc, dL_dalpha ? (double)dL_dalpha[o] : 0.0, grads.data());
      }
    }
    for (int i = 0; i < P; ++i) {
      size_t k = (size_t)v * P + i;
      for (int c = 0; c < 3; ++c) { dL_drgb[3 * k + c] = grads[i].rgb[c]; dL_dconic[3 * k + c] = grads[i].conic[c]; }
      dL_dmu2[2 * k] = grads[i].mu2[0]; dL_dmu2[2 * k + 1] = grads[i].mu2[1];
      dL_dopac[i] += grads[i].opac;
    }
  }
}

// ---------------------------------------------------------------- O8 preprocess backward, fp32 parameter inputs
void orc_preprocess_bwd(const Config* cfg, const float* means, const float* scales, const float* quats, const float* sh,
                        const float* Wv, const float* bv, const double* dL_drgb, const double* dL_dconic, const double* dL_dmu2,
                        double* dL_dmeans, double* dL_dscales, double* dL_dquats, double* dL_dsh) {
  int P = cfg->n_gauss, M = n_sh(*cfg);
  std::vector<double> shd(3 * M);
  for (size_t i = 0; i < (size_t)3 * P; ++i) { dL_dmeans[i] = 0; dL_dscales[i] = 0; }
  for (size_t i = 0; i < (size_t)4 * P; ++i) dL_dquats[i] = 0;
  for (size_t i = 0; i < (size_t)3 * M * P; ++i) dL_dsh[i] = 0;
  for (int v = 0; v < cfg->n_views; ++v) {
    double W[9], b[3];
    for (int i = 0; i < 9; ++i) W[i] = Wv[9 * v + i];
    for (int i = 0; i < 3; ++i) b[i] = bv[3 * v + i];
    for (int i = 0; i < P; ++i) {
      size_t k = (size_t)v * P + i;
      double mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
      double s[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
      double q[4] = {quats[4 * i], quats[4 * i + 1], quats[4 * i + 2], quats[4 * i + 3]};
      for (int m = 0; m < 3 * M; ++m) shd[m] = sh[(size_t)i * 3 * M + m];
      RecGrad g; std::memset(&g, 0, sizeof(g));
      for (int c = 0; c < 3; ++c) { g.rgb[c] = dL_drgb[3 * k + c]; g.conic[c] = dL_dconic[3 * k + c]; }
      g.mu2[0] = dL_dmu2[2 * k]; g.mu2[1] = dL_dmu2[2 * k + 1];
      ParamGrad pg; std::memset(&pg, 0, sizeof(pg));
      preprocess_bwd_one(*cfg, mu, s, q, shd.data(), W, b, g, pg, dL_dsh + (size_t)i * 3 * M, nullptr);
      for (int c = 0; c < 3; ++c) { dL_dmeans[3 * i + c] += pg.mu[c]; dL_dscales[3 * i + c] += pg.s[c]; }
      for (int c = 0; c < 4; ++c) dL_dquats[4 * i + c] += pg.q[c];
    }
  }
}

// ---------------------------------------------------------------- fp64 end-to-end (preprocess -> blend) with FIXED lists, for FD pins
// loss = sum_pixels <G_color, color> + <G_alpha, alpha>.  All parameter arrays are double.  want_grad=0: loss only.
double orc_e2e_f64(const Config* cfg, const double* means, const double* scales, const double* quats, const double* opac,
                   const double* sh, const double* Wv, const double* bv,
                   const uint32_t* active_tiles, int n_active, const uint32_t* pixel_mask_bits,
                   const uint64_t* ranges, const uint32_t* vals, const double* G_color, const double* G_alpha,
                   int want_grad, double* dL_dmeans, double* dL_dscales, double* dL_dquats, double* dL_dopac, double* dL_dsh,
                   double* dbg8 /*optional: preprocess_bwd debug terms of Gaussian 0, view 0*/) {
  int P = cfg->n_gauss, M = n_sh(*cfg); int64_t NT = n_tiles(*cfg);
  int64_t S = active_tiles ? n_active : NT;
  int ppt = 1 << (2 * cfg->tile_log2);
  double loss = 0;
  if (want_grad) {
    for (size_t i = 0; i < (size_t)3 * P; ++i) { dL_dmeans[i] = 0; dL_dscales[i] = 0; }
    for (size_t i = 0; i < (size_t)4 * P; ++i) dL_dquats[i] = 0;
    for (size_t i = 0; i < (size_t)P; ++i) dL_dopac[i] = 0;
    for (size_t i = 0; i < (size_t)3 * M * P; ++i) dL_dsh[i] = 0;
  }
  std::vector<Proj> recs(P);
  std::vector<RecGrad> grads(P);
  for (int v = 0; v < cfg->n_views; ++v) {
    const double* W = Wv + 9 * v; const double* b = bv + 3 * v;
    for (int i = 0; i < P; ++i)
      preprocess_one(*cfg, means + 3 * i, scales + 3 * i, quats + 4 * i, opac[i], sh + (size_t)i * 3 * M, W, b, recs[i], nullptr);
    if (want_grad) std::memset(grads.data(), 0, sizeof(RecGrad) * P);
    for (int64_t slot = 0; slot < S; ++slot) {
      int64_t tile = active_tiles ? active_tiles[slot] : slot;
      uint64_t start = ranges[2 * (v * NT + tile)], end = ranges[2 * (v * NT + tile) + 1];
      for (int i = 0; i < ppt; ++i) {
        int64_t p = tile * ppt + i;
        size_t o = ((size_t)v * S + slot) * ppt + i;
        if (!pixel_on(pixel_mask_bits, p)) continue;
        double up[3]; pixel_dir(cfg->order, p, up);
        PixelOut po;
        blend_pixel_fwd(*cfg, up, recs.data(), vals, start, end, po, nullptr);
        for (int c = 0; c < 3; ++c) loss += G_color[3 * o + c] * po.color[c];
        if (G_alpha) loss += G_alpha[o] * po.alpha;
        if (want_grad && po.n_last > 0)
          blend_pixel_bwd(*cfg, up, recs.data(), vals, start, po.n_last, G_color + 3 * o, G_alpha ? G_alpha[o] : 0.0, grads.data());
      }
    }
    if (want_grad)
      for (int i = 0; i < P; ++i) {
        ParamGrad pg; std::memset(&pg, 0, sizeof(pg));
        preprocess_bwd_one(*cfg, means + 3 * i, scales + 3 * i, quats + 4 * i, sh + (size_t)i * 3 * M, W, b, grads[i], pg,
                           dL_dsh + (size_t)i * 3 * M, (dbg8 && v == 0 && i == 0) ? dbg8 : nullptr);
        for (int c = 0; c < 3; ++c) { dL_dmeans[3 * i + c] += pg.mu[c]; dL_dscales[3 * i + c] += pg.s[c]; }
        for (int c = 0; c < 4; ++c) dL_dquats[4 * i + c] += pg.q[c];
        dL_dopac[i] += grads[i].opac;
      }
  }
  return loss;
}


// ---- NEXT-3: L1 + HEALPix-SSIM loss (orc_hssim.cpp)
int64_t orc_hssim_neighbor(int order, int64_t p, int dx, int dy, int* rot) { return hssim_neighbor(order, p, dx, dy, rot); }
double orc_hssim_weight(int face, int dx, int dy, double sigma) { return hssim_weight(face, dx, dy, sigma); }
void orc_hssim_loss(int order, const int32_t* slot_of_tile, const uint32_t* bits, int64_t n_slot, const float* X, const float* G,
                    double lambda, double sigma, double* h_map, double* dL_dX, double* out3, const int64_t* q_list, int64_t n_q) {
  const HssimOut o = hssim_loss(order, slot_of_tile, bits, n_slot, X, G, lambda, sigma, h_map, dL_dX, q_list, n_q);
  out3[0] = o.loss; out3[1] = o.l1; out3[2] = o.hssim;
}
}  // extern "C"
