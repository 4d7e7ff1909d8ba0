// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, double precision.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
// It shares no code with the CUDA path (paper_2606_29794_b200/csrc).
//
// Training loss on the HEALPix grid: L = (1 - lambda) L1^H + lambda L_HSSIM, with the
// HEALPix-SSIM of §4.1 and its masked average (Eq.10), forward and backward.
//
// The paper describes HSSIM in words only and prints no kernel weight, window size or constant.  Readings (A30-A35):
//  A30  Neighbourhood N_H(q): the (2R+1)^2 window around q in the (x,y) grid of q's base face ("the NESTED (x,y,f)
//       parameterization approximates a local 2D grid"), R = 5 (the 11 x 11 window of the SSIM that 3DGS uses,
//       on which the paper builds).  Outside [0,Nside)^2 the window continues into the neighbouring face
//       ("cross-face padding"): across one edge into the edge-adjacent face (the polar faces meet each other
//       with a quarter turn of the axes), across two edges into the face diagonally opposite at that vertex.  At the 8
//       vertices where only 3 faces meet (z = +-2/3) there is no such face: those taps do not exist ("some corner pixels have
//       only 7 neighbors").
//  A31  Weights: equatorial faces (4..7) use the isotropic Gaussian w = exp(-(dx^2 + dy^2) / (2 sigma^2)), sigma = 1.5
//       ("isotropic for the equatorial zone where pixels are roughly square").  Polar faces (0..3, 8..11) use
//       w = exp(-[(pi/4)(dx - dy)^2 + (4/pi)(dx + dy)^2] / (4 sigma^2)): the same angular Gaussian written for a polar-cap
//       pixel, whose east-west diagonal is shorter than its north-south one by pi/4 : 4/pi at equal area ("anisotropic for
//       polar zones where pixel geometry is longitudinally compressed").  The zone is that of the centre pixel's face.
//  A32  Missing taps (A30's vertices, pixels with M_C = 0) get weight 0 and the remaining weights are renormalised to sum 1
//       ("we detect such cases and renormalize kernel weights accordingly").
//  A33  SSIM index per pixel and channel with the standard constants C1 = 0.01^2, C2 = 0.03^2 (data range 1) from the weighted
//       local means, variances and covariance; h_q = mean over the channels.
//  A34  L_HSSIM = 1 - sum_q M(q) h_q / sum_q M(q) (Eq.10);  L1^H = sum_q M(q) sum_ch |X - G| / (channels * sum_q M(q)).
//  A35  lambda = 0.2 (3DGS default; the paper does not print its value).
// PARITY UNPINNED against the authors' implementation for A30-A35.  The oracle itself is pinned in tests/test_oracle_hssim.py:
// the neighbour map against shared-corner geometry (8 neighbours everywhere except 24 pixels with 7), closed forms (X = G,
// G = a X + b on constant-weight windows), the separable form of the isotropic kernel, and finite differences of the loss.
#pragma once
#include <cstdint>

namespace orc {

constexpr int kHssimR = 5;                       // window radius (A30)

// The pixel at offset (dx,dy) from NESTED pixel p in p's own face frame (A30), or -1 when it does not exist.
// rot: quarter turns (counter-clockwise, 0..3) that take p's face axes to the found pixel's face axes.
int64_t hssim_neighbor(int order, int64_t p, int dx, int dy, int* rot);
// Unnormalised tap weight of offset (dx,dy) for a centre pixel on `face` (A31).
double hssim_weight(int face, int dx, int dy, double sigma);

struct HssimOut { double loss, l1, hssim; };     // L, L1^H, mean h (so L_HSSIM = 1 - hssim)

// X, G: [n_slot*256][3] fp32 in the rasteriser's slot layout (slot_of_tile NULL: slot = tile; bits NULL: all pixels valid).
// h_map (may be NULL): [n_slot*256] per-pixel h_q (0 where masked out).  dL_dX (may be NULL): [n_slot*256][3] gradient of L.
// q_list (may be NULL = every pixel): centre pixels q to evaluate; with a list, h_map / the sums / dL_dX hold the listed centres'
// terms only (Eq.10's denominator stays the whole image's), which lets a test check sampled outputs of a full-size image.
HssimOut hssim_loss(int order, const int32_t* slot_of_tile, const uint32_t* pixel_mask_bits, int64_t n_slot, const float* X,
                    const float* G, double lambda, double sigma, double* h_map, double* dL_dX, const int64_t* q_list = nullptr,
                    int64_t n_q = 0);

}  // namespace orc
