// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, double precision.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
// It shares no code with the CUDA path (paper_2606_29794_b200/csrc).
//
// HEALPix geometry as used by UniTriSplat (§3.1; Table 6):
// N_pix = 12*Nside^2 equal-area pixels, NESTED indexing with the (x,y,f) parameterisation,
// RING indexing along iso-latitude rings.  The paper cites HEALPix [11] for the scheme and prints no
// formula; the definitions D1 (plane form) and D2 (ring form) are the readings of SURVEY.md §8c c.1
// (DESIGN.md "Readings" A1, A12).  D1 and D2 are implemented independently here and tests assert
// they agree; the invariants that pin them are listed in tests/test_oracle_healpix.py.
#pragma once
#include <cstdint>

namespace orc {

struct XYF { int64_t x, y; int f; };

// A point of the sphere in the HEALPix frame: z = cos(colatitude), lam = longitude,
// sth = sin(colatitude) computed without cancellation near the poles.
struct ZPhi { double z, lam, sth; };

int64_t npix_of_order(int order);                    // 12 * 4^order
XYF     nest2xyf(int order, int64_t p);              // p = f*4^k + interleave(x even bits, y odd bits)
int64_t xyf2nest(int order, XYF c);

// D1: HEALPix plane -> sphere, continuous face coordinates (xp,yp) in [0,1]^2 of face f.
ZPhi face_point_D1(int f, double xp, double yp);
ZPhi pix_center_D1(int order, int64_t p);            // Nest2Lonlat(p,k) of Alg.1 l.18, plane form
ZPhi pix_corner_D1(int order, int64_t p, int corner);// corner in {0,1,2,3}: (x+{0,1}, y+{0,1})/Nside
// D2: ring form of the same centre.
ZPhi pix_center_D2(int order, int64_t p);
// RING scheme.
int64_t nest2ring(int order, int64_t p);
ZPhi    ring_center(int order, int64_t r);           // textbook pix2ang in RING order
int64_t ring2nest(int order, int64_t r);             // = ang2pix_nest(ring_center(r))
int64_t ring_npix_in_ring(int order, int64_t i);     // ring i in [1,4Nside-1] has 4*min(i,Nside,4Nside-i) pixels
// RingInfo(i_r) of Alg.3 l.7: z of the ring, its pixel count, the longitude of its first pixel, and the
// RING index of that first pixel (so that Ring2Nest(i_r, j) = ring2nest(first + j)).
struct RingInfo { double z; int64_t npix; double lam0; int64_t first; };
RingInfo ring_info(int order, int64_t i);
// sphere -> pixel (inverse of D1)
int64_t ang2pix_nest(int order, double z, double lam);

// camera-frame unit vector of a HEALPix-frame point: (x,y,z)_cam = (y_hp, z_hp, x_hp)   (reading A1)
void to_cam_vec(const ZPhi& a, double v[3]);
double angle_between(const double a[3], const double b[3]);  // atan2(|a x b|, a.b), accurate at all angles

// PixRad(o) of Alg.2: largest centre-to-own-corner great-circle distance at order o.
double rho_max_bruteforce(int order);                // loops over all pixels x 4 corners
double rho_max_closed(int order);                    // closed form of SURVEY.md §8c c.1

}  // namespace orc
