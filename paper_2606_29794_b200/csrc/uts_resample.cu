// uts_resample.cu — image synthesis from the HEALPix image:
//   I_C(u,v) = Interp_H(I_H, P_C(u,v)), (u,v) in D_C                       Eq.7
// for the paper's three camera models (pinhole PAPER.md:477-484 Eq.11; anisotropic equidistant fisheye PAPER.md:486-507
// Eq.12-15; omnidirectional PAPER.md:511), its adjoint (the gradient the blend backward consumes), and the visibility mask
// M_C(q) = 1[Pi_C^{-1}(s_q) in D_C] of Eq.9 built on the device from the camera intrinsics.
//
// Interp_H (reading A26): the HEALPix scheme's ring-bilinear interpolation — linear in longitude between the two nearest
// pixel centres on each of the two iso-latitude rings bracketing the direction, linear in colatitude between the rings, the
// pole standing for the mean of the 4 pixels of the first / last ring.  Weights of pixels with M_C = 0 are dropped and the
// rest renormalised (reading A27); image pixel (i,j) is sampled at (i + 1/2, j + 1/2) (reading A28).
//
// One thread per image pixel; all geometry in double (the longitude weight at Nside 2048 needs ~1e-9 rad to keep the
// interpolated colour within 1e-4 of the oracle; the kernel is bound by its gathers and stores, not by this arithmetic).
// A ring's pixels are addressed by the integer position g of uts_ring_query.cuh (longitude = (pi/4) g / n_r, centres at
// g = parity (mod 2)); (ring, g) -> NESTED goes through x + y = (r+2) N - 1 - ring, x - y = g - F2 n_r on the face that
// holds the pixel.  HBM: 4 C bytes written per image pixel + each HEALPix sample read about once (neighbouring image pixels
// share their four samples through L1/L2).
#include "uts_internal.cuh"

namespace uts {

struct CamParams {
  int model, W, H;
  double a, b;        // pinhole: 1/f_x, 1/f_y; fisheye: 1/f_x = pi/W, 1/f_y = pi/H; equirect: 2 pi / W, pi / H
  double wx, wy;      // fisheye FoV factors (Eq.12)
  double fx, fy;      // focal lengths (projection)
};

__device__ __forceinline__ bool cam_pixel_dir(const CamParams& c, double u, double v, double& dx, double& dy, double& dz) {
  const double cx = 0.5 * c.W, cy = 0.5 * c.H;
  if (c.model == UTS_CAM_PINHOLE) {
    const double x = (u - cx) * c.a, y = (v - cy) * c.b;
    const double inv = rsqrt(x * x + y * y + 1.0);
    dx = x * inv; dy = y * inv; dz = inv;
    return u >= 0.0 && u < (double)c.W && v >= 0.0 && v < (double)c.H;
  }
  if (c.model == UTS_CAM_FISHEYE) {
    const double mx = (u - cx) * c.a, my = (v - cy) * c.b;
    const double rm2 = mx * mx + my * my, rm = sqrt(rm2);
    double cg = 1.0, sg = 0.0;                                   // cos / sin of the azimuth gamma (gamma = 0 at the centre)
    if (rm > 0.0) { cg = mx / rm; sg = my / rm; }
    const double weff = sqrt(c.wx * c.wx * cg * cg + c.wy * c.wy * sg * sg);     // Eq.12
    double sp, cp;
    sincos(rm * weff, &sp, &cp);                                 // incident angle psi = r_m w_eff
    dx = sp * cg; dy = sp * sg; dz = cp;
    return rm2 <= 0.25 * kPi * kPi;                              // Eq.14-15: ((u-c_x)/a)^2 + ((v-c_y)/b)^2 <= 1, a = f_x pi/2
  }
  const double om = u * c.a - kPi, ph = 0.5 * kPi - v * c.b;
  double so, co, sp, cp;
  sincos(om, &so, &co); sincos(ph, &sp, &cp);
  dx = cp * so; dy = sp; dz = cp * co;
  return u >= 0.0 && u < (double)c.W && v >= 0.0 && v < (double)c.H;
}

// Pi_C^{-1}: is the direction imaged (Eq.9)?
__device__ __forceinline__ bool cam_sees(const CamParams& c, double dx, double dy, double dz) {
  if (c.model == UTS_CAM_PINHOLE) {
    if (!(dz > 0.0)) return false;
    const double u = 0.5 * c.W + c.fx * dx / dz, v = 0.5 * c.H + c.fy * dy / dz;
    return u >= 0.0 && u < (double)c.W && v >= 0.0 && v < (double)c.H;
  }
  if (c.model == UTS_CAM_FISHEYE) {
    const double rho = sqrt(dx * dx + dy * dy);
    const double psi = atan2(rho, dz);
    double cg = 1.0, sg = 0.0;
    if (rho > 0.0) { cg = dx / rho; sg = dy / rho; }
    const double weff = sqrt(c.wx * c.wx * cg * cg + c.wy * c.wy * sg * sg);
    const double rm = psi / weff;
    // image position (c_x + f_x r_m cos(gamma), c_y + f_y r_m sin(gamma)) against the ellipse of Eq.14, a = f_x pi/2, b = f_y pi/2
    const double ex = rm * cg / (0.5 * kPi), ey = rm * sg / (0.5 * kPi);
    return ex * ex + ey * ey <= 1.0;
  }
  return true;
}

// ring i of an order with N = 2^order: z of the ring and sin(colatitude)
__device__ __forceinline__ void ring_z(int N, int i, double& z, double& sth) {
  const double inv3N2 = 1.0 / (3.0 * (double)N * (double)N);
  if (i < N) { const double w = (double)i * (double)i * inv3N2; z = 1.0 - w; sth = sqrt(w * (2.0 - w)); }
  else if (i > 3 * N) { const double n = (double)(4 * N - i); const double w = n * n * inv3N2; z = w - 1.0; sth = sqrt(w * (2.0 - w)); }
  else { z = (double)(2 * (2 * N - i)) / (double)(3 * N); sth = sqrt((1.0 - z) * (1.0 + z)); }
}

// NESTED index of the pixel at position g of ring i (g already reduced to [0, 8 n_r) with the ring's parity).  A ring crosses at
// most two face rows; on a face of row r the pixel's x - y = g - F2 n_r lies within (-n_r, n_r), which fixes the face column.
__device__ __forceinline__ uint32_t spread_bits16(uint32_t v) {   // 16 bits -> even bit positions
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}
__device__ __forceinline__ uint64_t ring_pos_to_nest(int order, int i, int g) {
  const int N = 1 << order;
  const int n = min(i, min(N, 4 * N - i));
  for (int r = 0; r < 3; ++r) {
    const int s = (r + 2) * N - 1 - i;                          // x + y on a face of row r
    if (s < 0 || s > 2 * N - 2) continue;
    const int hm = min(s, 2 * N - 2 - s);
    const int t = r & 1;
    const int c = ((g + t * n) / (2 * n)) & 3;                  // the column whose centre F2 n is within n of g
    int h = g - (2 * c + 1 - t) * n;                            // x - y, modulo the ring length 8 n
    if (h > 4 * n) h -= 8 * n;
    if (h <= -4 * n) h += 8 * n;
    if (h < -hm || h > hm || ((s + h) & 1)) continue;
    const uint32_t x = (uint32_t)((s + h) >> 1), y = (uint32_t)((s - h) >> 1);
    const uint64_t f = (uint64_t)(4 * r + c);
    return (f << (2 * order)) | (uint64_t)(spread_bits16(x) | (spread_bits16(y) << 1));
  }
  return 0;                                                     // unreachable: every (ring, position) is a pixel
}

// the two pixels of ring i nearest in longitude to lam in [0, 2 pi), with their linear weights
__device__ __forceinline__ void ring_pair(int order, int i, double lam, uint64_t pix[2], double w[2]) {
  const int N = 1 << order;
  const int n = min(i, min(N, 4 * N - i));
  const int par = (i < N || i > 3 * N) ? 1 : ((N + 1 + i) & 1);
  const double t = lam * (4.0 * (double)n / kPi);               // real-valued position; centres at par, par + 2, ...
  const double q = floor(0.5 * (t - (double)par));
  int g1 = par + 2 * (int)q;
  const double frac = 0.5 * (t - (double)g1);
  int g2 = g1 + 2;
  const int L = 8 * n;
  g1 %= L; if (g1 < 0) g1 += L;
  g2 %= L; if (g2 < 0) g2 += L;
  pix[0] = ring_pos_to_nest(order, i, g1); pix[1] = ring_pos_to_nest(order, i, g2);
  w[0] = 1.0 - frac; w[1] = frac;
}

// Interp_H support of direction (dx,dy,dz) (camera frame; polar axis +y, longitude atan2(dx,dz): reading A1).
// (the direction as longitude lam in [0, 2 pi), z = cos(colatitude) and sth = sin(colatitude), up to a common positive factor of z, sth)
__device__ __forceinline__ int interp_support_lzs(int order, double lam, double z, double sth, uint64_t pix[8], double w[8]) {
  const int N = 1 << order, last = 4 * N - 1;
  double theta = 0.0;                                 // colatitude: only the two polar caps below need the angle itself
  // largest ring whose colatitude is <= theta (0: north of ring 1): closed-form estimate, then settled on ring colatitudes
  int i1;
  if (z > 2.0 / 3.0) i1 = (int)floor((double)N * sqrt(3.0 * (1.0 - z)));
  else if (z < -2.0 / 3.0) i1 = 4 * N - (int)ceil((double)N * sqrt(3.0 * (1.0 + z)));
  else i1 = (int)floor((double)N * (2.0 - 1.5 * z));
  i1 = max(0, min(last, i1));
  auto theta_of = [&](int i) { double zz, ss; ring_z(N, i, zz, ss); return atan2(ss, zz); };
  // settled on the rings' z (colatitude <= theta  <=>  z_ring >= cos theta): no inverse trigonometry in the search; at a tie either
  // ring gives the same interpolated value (the weight of the other ring is then 0)
  auto z_of = [&](int i) { double zz, ss; ring_z(N, i, zz, ss); return zz; };
  const double zn = z / sqrt(z * z + sth * sth);
  while (i1 < last && z_of(i1 + 1) >= zn) ++i1;
  while (i1 >= 1 && z_of(i1) < zn) --i1;
  int cnt = 0;
  uint64_t p2[2]; double a2[2];
  if (i1 == 0) {
    theta = atan2(sth, z);
    const double wt = theta / theta_of(1);
    ring_pair(order, 1, lam, p2, a2);
    pix[0] = p2[0]; w[0] = a2[0] * wt; pix[1] = p2[1]; w[1] = a2[1] * wt; cnt = 2;
    for (int j = 0; j < 4; ++j) { pix[cnt] = ring_pos_to_nest(order, 1, 2 * j + 1); w[cnt++] = 0.25 * (1.0 - wt); }
    return cnt;
  }
  if (i1 == last) {
    theta = atan2(sth, z);
    const double t1 = theta_of(last), wt = (theta - t1) / (kPi - t1);
    ring_pair(order, last, lam, p2, a2);
    pix[0] = p2[0]; w[0] = a2[0] * (1.0 - wt); pix[1] = p2[1]; w[1] = a2[1] * (1.0 - wt); cnt = 2;
    for (int j = 0; j < 4; ++j) { pix[cnt] = ring_pos_to_nest(order, last, 2 * j + 1); w[cnt++] = 0.25 * wt; }
    return cnt;
  }
  // wt = (theta - t1) / (t2 - t1) from the sines of the two differences (no colatitude is formed): with (z, s) = (cos, sin),
  // sin(theta - t1) = s z1 - z s1 and sin(t2 - t1) = s2 z1 - z2 s1; the rings are at most a few hundredths of a radian apart, where
  // asin x = x + x^3/6 + 3 x^5/40 + 15 x^7/336 is exact to 1e-10 relative; wider gaps (orders below 4) take atan2.
  double wt;
  {
    double z1, s1, z2, s2;
    ring_z(N, i1, z1, s1); ring_z(N, i1 + 1, z2, s2);
    const double inv_n = 1.0 / sqrt(z * z + sth * sth), zc = z * inv_n, sc = sth * inv_n;
    const double d1 = sc * z1 - zc * s1, d21 = s2 * z1 - z2 * s1;
    if (d21 < 0.15) {
      auto asin_small = [](double x) { const double x2 = x * x; return x * (1.0 + x2 * (1.0 / 6.0 + x2 * (3.0 / 40.0 + x2 * (15.0 / 336.0 + x2 * (105.0 / 3456.0))))); };
      wt = asin_small(d1) / asin_small(d21);
    } else {
      theta = atan2(sth, z);
      const double t1 = atan2(s1, z1), t2 = atan2(s2, z2);
      wt = (theta - t1) / (t2 - t1);
    }
  }
  ring_pair(order, i1, lam, p2, a2);
  pix[0] = p2[0]; w[0] = a2[0] * (1.0 - wt); pix[1] = p2[1]; w[1] = a2[1] * (1.0 - wt);
  ring_pair(order, i1 + 1, lam, p2, a2);
  pix[2] = p2[0]; w[2] = a2[0] * wt; pix[3] = p2[1]; w[3] = a2[1] * wt;
  return 4;
}

__device__ __forceinline__ int interp_support(int order, double dx, double dy, double dz, uint64_t pix[8], double w[8]) {
  double lam = atan2(dx, dz);
  if (lam < 0.0) lam += 2.0 * kPi;
  return interp_support_lzs(order, lam, dy, sqrt(dx * dx + dz * dz), pix, w);
}

// valid HEALPix samples of image pixel (i,j) as slot-layout indices with renormalised weights (reading A27)
__device__ __forceinline__ int pixel_support(int order, const CamParams& c, const int32_t* __restrict__ slot_of_tile,
                                             const uint32_t* __restrict__ mask_bits, int i, int j, int64_t idx[8], float w[8], bool& in_domain) {
  uint64_t pix[8]; double ww[8];
  int n;
  if (c.model == UTS_CAM_EQUIRECT) {
    // the image's own coordinates are longitude and latitude (cam_pixel_dir's last branch): lam = om mod 2 pi, (z, sth) = (sin, cos)(ph),
    // without the detour through the direction and its atan2
    const double u = (double)i + 0.5, v = (double)j + 0.5;
    in_domain = u >= 0.0 && u < (double)c.W && v >= 0.0 && v < (double)c.H;
    if (!in_domain) return 0;
    double lam = u * c.a - kPi, sp, cp;
    if (lam < 0.0) lam += 2.0 * kPi;
    sincos(0.5 * kPi - v * c.b, &sp, &cp);
    n = interp_support_lzs(order, lam, sp, fabs(cp), pix, ww);
  } else {
    double dx, dy, dz;
    in_domain = cam_pixel_dir(c, (double)i + 0.5, (double)j + 0.5, dx, dy, dz);
    if (!in_domain) return 0;
    n = interp_support(order, dx, dy, dz, pix, ww);
  }
  int cnt = 0; double sum = 0.0;
  for (int k = 0; k < n; ++k) {
    const uint64_t p = pix[k];
    if (mask_bits && !((__ldg(mask_bits + (p >> 5)) >> (p & 31)) & 1u)) continue;
    const int64_t tile = (int64_t)(p >> 8);
    const int64_t slot = slot_of_tile ? (int64_t)__ldg(slot_of_tile + tile) : tile;
    if (slot < 0) continue;
    idx[cnt] = slot * kTilePix + (int64_t)(p & 255); ww[cnt] = ww[k]; sum += ww[k]; ++cnt;
  }
  if (!(sum > 0.0)) return 0;
  const double inv = 1.0 / sum;
  for (int k = 0; k < cnt; ++k) w[k] = (float)(ww[k] * inv);
  return cnt;
}

__global__ void __launch_bounds__(256)
resample_fwd_kernel(int order, CamParams c, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ mask_bits,
                    const float* __restrict__ image, int channels, float* __restrict__ out, uint8_t* __restrict__ valid) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)c.W * c.H) return;
  const int i = (int)(t % c.W), j = (int)(t / c.W);
  int64_t idx[8]; float w[8]; bool in;
  const int n = pixel_support(order, c, slot_of_tile, mask_bits, i, j, idx, w, in);
  for (int ch = 0; ch < channels; ++ch) {
    float acc = 0.f;
    for (int k = 0; k < n; ++k) acc = fmaf(w[k], __ldg(image + idx[k] * channels + ch), acc);
    out[t * channels + ch] = acc;
  }
  if (valid) valid[t] = in ? 1 : 0;
}

__global__ void __launch_bounds__(256)
resample_bwd_kernel(int order, CamParams c, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ mask_bits,
                    const float* __restrict__ dL_dout, int channels, float* __restrict__ dL_dimage) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)c.W * c.H) return;
  const int i = (int)(t % c.W), j = (int)(t / c.W);
  int64_t idx[8]; float w[8]; bool in;
  const int n = pixel_support(order, c, slot_of_tile, mask_bits, i, j, idx, w, in);
  for (int ch = 0; ch < channels; ++ch) {
    const float g = __ldg(dL_dout + t * channels + ch);
    for (int k = 0; k < n; ++k) atomicAdd(dL_dimage + idx[k] * channels + ch, w[k] * g);
  }
}

// One thread per 32-pixel word of M_C (Eq.9)
__global__ void camera_mask_kernel(int order, CamParams c, uint32_t* __restrict__ bits, uint64_t n_words) {
  const uint64_t wd = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (wd >= n_words) return;
  uint32_t word = 0;
  for (int b = 0; b < 32; ++b) {
    double vx, vy, vz;
    pix_center_cam(order, wd * 32 + b, vx, vy, vz);
    if (cam_sees(c, vx, vy, vz)) word |= 1u << b;
  }
  bits[wd] = word;
}

static int make_cam(const uts_camera& cam, CamParams& c) {
  if (cam.width <= 0 || cam.height <= 0) return UTS_ERR_INVALID_ARG;
  c.model = cam.model; c.W = cam.width; c.H = cam.height; c.wx = c.wy = 0.0; c.fx = c.fy = 0.0;
  if (cam.model == UTS_CAM_PINHOLE) {
    if (!(cam.p0 > 0.0 && cam.p0 < kPi && cam.p1 > 0.0 && cam.p1 < kPi)) return UTS_ERR_INVALID_ARG;
    c.fx = cam.width / (2.0 * tan(0.5 * cam.p0)); c.fy = cam.height / (2.0 * tan(0.5 * cam.p1));
    c.a = 1.0 / c.fx; c.b = 1.0 / c.fy;
  } else if (cam.model == UTS_CAM_FISHEYE) {
    if (!(cam.p0 > 0.0 && cam.p0 <= 2.0 && cam.p1 > 0.0 && cam.p1 <= 2.0)) return UTS_ERR_INVALID_ARG;  // FoV <= 360 deg
    c.fx = cam.width / kPi; c.fy = cam.height / kPi;
    c.a = 1.0 / c.fx; c.b = 1.0 / c.fy; c.wx = cam.p0; c.wy = cam.p1;
  } else if (cam.model == UTS_CAM_EQUIRECT) {
    c.a = 2.0 * kPi / cam.width; c.b = kPi / cam.height;
  } else return UTS_ERR_INVALID_ARG;
  return UTS_OK;
}

int build_mask_tiles(const Dims& d, uint32_t* pixel_mask_bits, int32_t* slot_of_tile, uint32_t* active_tiles, int* h_n_active, cudaStream_t s);

}  // namespace uts

using namespace uts;

extern "C" {

int uts_resample_fwd(const uts_config* cfg, uts_camera cam, uts_mask mask, const float* image, int channels, float* out,
                     uint8_t* valid, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  CamParams c;
  if ((st = make_cam(cam, c))) return st;
  if (!image || !out || channels < 1 || channels > 16) return UTS_ERR_INVALID_ARG;
  const int64_t n = (int64_t)c.W * c.H;
  resample_fwd_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(cfg->order, c, mask.slot_of_tile, mask.pixel_mask_bits,
                                                                                   image, channels, out, valid);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_resample_bwd(const uts_config* cfg, uts_camera cam, uts_mask mask, const float* dL_dout, int channels, float* dL_dimage,
                     void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  CamParams c;
  if ((st = make_cam(cam, c))) return st;
  if (!dL_dout || !dL_dimage || channels < 1 || channels > 16) return UTS_ERR_INVALID_ARG;
  const Dims d = dims_of(cfg, &mask);
  cudaStream_t s = (cudaStream_t)stream;
  UTS_CUDA(cudaMemsetAsync(dL_dimage, 0, (size_t)d.n_slot * kTilePix * channels * sizeof(float), s));
  const int64_t n = (int64_t)c.W * c.H;
  resample_bwd_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(cfg->order, c, mask.slot_of_tile, mask.pixel_mask_bits, dL_dout, channels,
                                                                  dL_dimage);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_build_camera_mask(const uts_config* cfg, uts_camera cam, uint32_t* pixel_mask_bits, int32_t* slot_of_tile,
                          uint32_t* active_tiles, int* h_n_active, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  CamParams c;
  if ((st = make_cam(cam, c))) return st;
  if (!pixel_mask_bits || !slot_of_tile || !active_tiles || !h_n_active) return UTS_ERR_INVALID_ARG;
  const Dims d = dims_of(cfg, nullptr);
  cudaStream_t s = (cudaStream_t)stream;
  const uint64_t n_words = (uint64_t)d.n_pix / 32;
  camera_mask_kernel<<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(d.k, c, pixel_mask_bits, n_words);
  UTS_LAUNCH_CHECK();
  return build_mask_tiles(d, pixel_mask_bits, slot_of_tile, active_tiles, h_n_active, s);
}

}  // extern "C"
