// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, double precision.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
// It shares no code with the CUDA path (paper_2606_29794_b200/csrc); its own structs are defined here.
//
// UniTriSplat HEALPix rasteriser, Alg.1 step by step, and its backward
// (Eq.3-4).  Readings of silent / garbled passages are DESIGN.md "Readings" A1-A25.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   preprocess      : isotropic closed form, literal Eq.2 == tangent-basis form, J == finite differences of Eq.1,
//                     degree-0 colour, SH orthonormality by quadrature on the HEALPix grid
//   tile query      : brute force every-Gaussian x every-order-k_q-pixel == descent; superset property; r_s>=pi
//   RING tile query : Alg.3 == brute force "order-k_q centres within r_s" (every Gaussian x every pixel); subset of the
//                     NESTED set; z-range / full-ring / pole branches exercised by discs over the poles
//   sort / ranges   : permutation + order properties
//   blend forward   : single isotropic Gaussian closed form (independent haversine), two-Gaussian closed form,
//                     permutation invariance, 4-fold rotation symmetry
//   backward        : central finite differences of the fp64 forward for every parameter group; Eq.3 literal term
//   Image-level parity against the authors' implementation: PARITY UNPINNED (the paper prints no values).
#pragma once
#include <cstdint>
#include <vector>

namespace orc {

struct Config {                 // oracle's own definition (same meaning as the ABI's config, no shared header)
  int   order;                  // k; Nside = 1<<k
  int   tile_log2;              // l; B = 1<<l (16 => 4)                              Table 6
  int   query_refine_log2;      // log2 f (x4 => 2)
  int   sh_degree;              // 0..3
  int   n_gauss;                // P
  int   n_views;                // V
  float r_near;                 // cull rho <= r_near                                 reading A5
  float cov_dilation_px2;       // h = value * Omega_pix added to diag(Sigma_arc)     reading A3
  float alpha_min, alpha_max, t_eps;   //                                             reading A7
  float bg[3];                  //                                                    reading A8
  int   query_mode;             // 0: NESTED descent, Alg.2 (reading A6); 1: RING scan, Alg.3 (readings A17, A18)
};

inline int  tile_order(const Config& c) { return c.order - c.tile_log2; }            // k_t, Table 6
inline int  query_order(const Config& c) { return tile_order(c) + c.query_refine_log2; }  // k_q
inline int64_t n_tiles(const Config& c) { return (int64_t)12 << (2 * tile_order(c)); }
inline int  n_sh(const Config& c) { return (c.sh_degree + 1) * (c.sh_degree + 1); }

// Projected Gaussian record in double (what Alg.1 l.2-8 produces).
struct Proj {
  double dir[3];      // unit direction u = t/rho (camera frame)
  double lon, lat;    // (omega, phi) of Eq.1
  double rho;         // radial depth ||t||
  double conic[3];    // (A,B,C) = Sigma_arc^{-1}: A dx^2 + 2B dx dy + C dy^2
  double opac;
  double rs;          // min(pi, 3 sqrt(lambda_max))
  double rgb[3];
  uint8_t flags;      // bit0 culled; bits1-3 colour channel clamped at 0
};

// Intermediates of one preprocess call, kept for the backward.
struct PreSaved {
  double t[3], R[9], Sigma3[9], M[9], J[6], cosphi, sinphi;
  double sig_rad[3];   // (s_ww, s_wp, s_pp) of Sigma_rad = J M J^T
  double sig_arc[3];   // (a,b,c) of Sigma_arc incl. dilation
  double det;
  double vdir[3], vlen; // world-space view direction and |mu - cam|
  double cam[3];
};

void preprocess_one(const Config& cfg, const double mu[3], const double s[3], const double q[4], double o,
                    const double* sh /*[M,3]*/, const double W[9], const double b[3], Proj& out, PreSaved* sv);

// Sigma_arc through the tangent-basis identity S_phi J = [e; n]/rho — used only as a pin.
void sigma_arc_tangent(const double t[3], const double M[9], double out3[3]);
void sh_basis(int degree, const double d[3], double* Y /*[16]*/);
void sh_basis_grad(int degree, const double d[3], double* dY /*[16][3]*/);

struct QueryStats { double min_margin; int64_t node_tests; };

// Tile set of one Gaussian.  brute=true: literal loop over every order-k_q pixel.
// cfg.query_mode 0: the NESTED set (centres within r_s + rho_max(k_q), reading A6) by a safe descent;
// cfg.query_mode 1: Alg.3 QueryDiscRing step by step (centres within r_s).
void tile_query_one(const Config& cfg, const double dir[3], double rs, const int32_t* slot_of_tile /*may be null*/,
                    bool brute, std::vector<uint32_t>& tiles_out, QueryStats& st);

struct BlendCounters { int64_t evaluated, contributing, early_exit_pixels; };

// Per-pixel forward: returns colour[3], alpha, n_last; margin = smallest relative distance of any decision to its threshold.
struct PixelOut { double color[3]; double alpha; uint32_t n_last; double margin; };
void pixel_dir(int order, int64_t p, double v[3]);
void blend_pixel_fwd(const Config& cfg, const double up[3], const Proj* recs, const uint32_t* vals, uint64_t start,
                     uint64_t end, PixelOut& out, BlendCounters* ctr);

// Gradient of the blend w.r.t. each record: rgb[3], conic[3], opac, and the projected mean mu' = (lon,lat).
struct RecGrad { double rgb[3], conic[3], opac, mu2[2]; };
void blend_pixel_bwd(const Config& cfg, const double up[3], const Proj* recs, const uint32_t* vals, uint64_t start,
                     uint32_t n_last, const double gcol[3], double galpha, RecGrad* grads /*indexed by vals[j]*/);

struct ParamGrad { double mu[3], s[3], q[4]; };
// Backward of preprocess_one for one (view,Gaussian): adds into pg and dsh [M,3].
void preprocess_bwd_one(const Config& cfg, const double mu[3], const double s[3], const double q[4],
                        const double* sh, const double W[9], const double b[3], const RecGrad& g,
                        ParamGrad& pg, double* dsh,
                        double* dbg /*optional [8]: L_phi|S_phi (literal Eq.3), L_arc(a,b,c), Sigma_rad(ww,wp,pp), phi*/);

}  // namespace orc
