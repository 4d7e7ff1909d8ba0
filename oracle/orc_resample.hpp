// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, double precision.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
// It shares no code with the CUDA path (paper_2606_29794_b200/csrc).
//
// Image synthesis from the HEALPix image: camera models P_C and valid domains D_C
// (§10.1, Eq.11-15), the visibility mask M_C (Eq.9) and
// I_C(u,v) = Interp_H(I_H, P_C(u,v)) (Eq.7) with its adjoint.
//
// Readings (A26-A28):
//  A26  Interp_H is not defined by the paper ("interpolating neighboring HEALPix samples").  Taken as the
//       HEALPix scheme's own bilinear interpolation (Gorski et al. [11], "get_interpol"): linear in longitude between the two
//       nearest pixel centres on each of the two iso-latitude rings that bracket the point, then linear in colatitude
//       between the rings; beyond the first / last ring the pole value is the mean of that ring's 4 pixels.
//  A27  HEALPix pixels with M_C = 0 hold no rendered value; their weights are dropped and the remaining
//       weights renormalised (an image pixel with no valid neighbour gets 0).
//  A28  Image pixel (i,j) is sampled at its centre (u,v) = (i + 1/2, j + 1/2); D_C = [0,W) x [0,H) (pinhole, equirect) or
//       the ellipse of Eq.14 (fisheye).
// PARITY UNPINNED against the authors' implementation for A26/A27 (the paper prints no value); the oracle itself is pinned
// by the closed forms and brute-force checks in tests/test_oracle_resample.py.
#pragma once
#include <cstdint>

namespace orc {

enum CameraModel { kPinhole = 0, kFisheye = 1, kEquirect = 2 };

// p0, p1: pinhole FoV_x, FoV_y in radians; fisheye w_x, w_y (= FoV/180deg, Eq.12); equirect: unused.
struct Camera { int model; int width, height; double p0, p1; };

// P_C: continuous image position (u,v) -> unit direction in the camera frame.  Returns false outside D_C.
bool cam_pixel_dir(const Camera& c, double u, double v, double d[3]);
// Pi_C^{-1}: unit direction -> continuous image position.  Returns false when the direction is not imaged (Eq.9).
bool cam_project(const Camera& c, const double d[3], double& u, double& v);

// Interp_H support of a direction given as (z, lam) in the HEALPix frame with colatitude theta: up to 8 (NESTED pixel, weight)
// entries, weights >= 0 summing to 1 (a pixel may appear twice).  Returns the number of entries.
int interp_weights(int order, double theta, double lam, int64_t pix[8], double w[8]);

// I_C = Interp_H(I_H, P_C): image [n_slot*256][C] fp32 in the rasteriser's slot layout (slot_of_tile NULL: slot = tile),
// pixel_mask_bits NULL: every pixel valid.  out [H][W][C] (0 outside D_C), valid [H][W] (may be NULL).
void resample_fwd(int order, const Camera& c, const int32_t* slot_of_tile, const uint32_t* pixel_mask_bits,
                  const float* image, int channels, double* out, uint8_t* valid);
// adjoint: dL_dimage [n_slot*256][C] (double, zeroed here) += w * dL_dout
void resample_bwd(int order, const Camera& c, const int32_t* slot_of_tile, const uint32_t* pixel_mask_bits,
                  int64_t n_slot, const double* dL_dout, int channels, double* dL_dimage);
// M_C(q) = 1[Pi_C^{-1}(s_q) in D_C]  (Eq.9): N_pix/32 words, NESTED order
void camera_mask(int order, const Camera& c, uint32_t* bits);

}  // namespace orc
