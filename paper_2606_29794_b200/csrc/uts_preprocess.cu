// uts_preprocess.cu — F1 (Alg.1 l.2-8, Eq.1-2) and B2 (Eq.3-4).
//
// One thread per (view, Gaussian) forward, one thread per Gaussian backward (two kernels: geometry chain, colour path; views
// summed in registers, so the parameter gradients are written once, no atomics).  Both kernels are streaming: 236 B in + 57 B out per Gaussian
// forward at SH degree 3.  The geometry chain runs in double precision: it is ~1.5 k instructions per Gaussian, below
// the HBM time of the 48 SH floats, and it makes the stored fp32 records (dir, rho, r_s) the correctly rounded
// values, so that the integer stages downstream (tile query, sort key) see the same bits as a double reference.
//
// Sigma_arc uses the tangent-basis identity S_phi J = [e; n]/rho: Alg.1 l.6's
// S_phi J W Sigma3D W^T J^T S_phi^T equals [e;n] (W Sigma3D W^T) [e;n]^T / rho^2 with e = d u/d omega / cos(phi),
// n = d u/d phi the local east / north unit vectors; this form has no 1/cos(phi) pole factor.
#include "uts_internal.cuh"

namespace uts {

struct ViewConst { double W[9]; double b[3]; double cam[3]; };   // cam = -W^T b (camera centre in world space)

__device__ __forceinline__ void load_view(const float* __restrict__ Wv, const float* __restrict__ bv, int v, ViewConst& vc) {
#pragma unroll
  for (int i = 0; i < 9; ++i) vc.W[i] = (double)__ldg(Wv + 9 * v + i);
#pragma unroll
  for (int i = 0; i < 3; ++i) vc.b[i] = (double)__ldg(bv + 3 * v + i);
#pragma unroll
  for (int i = 0; i < 3; ++i) vc.cam[i] = -(vc.W[i] * vc.b[0] + vc.W[3 + i] * vc.b[1] + vc.W[6 + i] * vc.b[2]);
}

// Real spherical-harmonic basis to degree 3 at unit direction (x,y,z), sign convention of standard 3DGS (reading A13).
template <typename T>
__device__ __forceinline__ void sh_basis_eval(int deg, T x, T y, T z, T* Y) {
  Y[0] = (T)0.28209479177387814;
  if (deg < 1) return;
  const T k1 = (T)0.4886025119029199;
  Y[1] = -k1 * y; Y[2] = k1 * z; Y[3] = -k1 * x;
  if (deg < 2) return;
  const T xx = x * x, yy = y * y, zz = z * z;
  const T k2a = (T)1.0925484305920792, k2b = (T)0.31539156525252005, k2c = (T)0.5462742152960396;
  Y[4] = k2a * x * y; Y[5] = -k2a * y * z; Y[6] = k2b * (2 * zz - xx - yy); Y[7] = -k2a * x * z; Y[8] = k2c * (xx - yy);
  if (deg < 3) return;
  const T k3a = (T)0.5900435899266435, k3b = (T)2.890611442640554, k3c = (T)0.4570457994644658,
          k3d = (T)0.3731763325901154, k3e = (T)1.445305721320277;
  Y[9]  = -k3a * y * (3 * xx - yy);
  Y[10] =  k3b * x * y * z;
  Y[11] = -k3c * y * (4 * zz - xx - yy);
  Y[12] =  k3d * z * (2 * zz - 3 * xx - 3 * yy);
  Y[13] = -k3c * x * (4 * zz - xx - yy);
  Y[14] =  k3e * z * (xx - yy);
  Y[15] = -k3a * x * (xx - 3 * yy);
}

// sum_m sh_m * grad(Y_m): gradient of sum_m Y_m(d) c_m w.r.t. the (unconstrained) direction components.
__device__ __forceinline__ void sh_dir_grad(int deg, float x, float y, float z, const float* c /*[16]*/, float& gx, float& gy, float& gz) {
  gx = gy = gz = 0.f;
  if (deg < 1) return;
  const float k1 = 0.4886025119029199f;
  gy += -k1 * c[1]; gz += k1 * c[2]; gx += -k1 * c[3];
  if (deg < 2) return;
  const float k2a = 1.0925484305920792f, k2b = 0.31539156525252005f, k2c = 0.5462742152960396f;
  gx += k2a * y * c[4] - 2 * k2b * x * c[6] - k2a * z * c[7] + 2 * k2c * x * c[8];
  gy += k2a * x * c[4] - k2a * z * c[5] - 2 * k2b * y * c[6] - 2 * k2c * y * c[8];
  gz += -k2a * y * c[5] + 4 * k2b * z * c[6] - k2a * x * c[7];
  if (deg < 3) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  const float k3a = 0.5900435899266435f, k3b = 2.890611442640554f, k3c = 0.4570457994644658f,
              k3d = 0.3731763325901154f, k3e = 1.445305721320277f;
  gx += -k3a * 6 * x * y * c[9] + k3b * y * z * c[10] + k3c * 2 * x * y * c[11] - k3d * 6 * x * z * c[12]
        - k3c * (4 * zz - 3 * xx - yy) * c[13] + k3e * 2 * x * z * c[14] - k3a * 3 * (xx - yy) * c[15];
  gy += -k3a * 3 * (xx - yy) * c[9] + k3b * x * z * c[10] - k3c * (4 * zz - xx - 3 * yy) * c[11] - k3d * 6 * y * z * c[12]
        + k3c * 2 * x * y * c[13] - k3e * 2 * y * z * c[14] + k3a * 6 * x * y * c[15];
  gz += k3b * x * y * c[10] - k3c * 8 * y * z * c[11] + k3d * 3 * (2 * zz - xx - yy) * c[12] - k3c * 8 * x * z * c[13]
        + k3e * (xx - yy) * c[14];
}

// R(q), q = (w,x,y,z) used as given (reading A14; Alg.1 l.4 QuatToMat PAPER.md:537).
__device__ __forceinline__ void quat_rot(const double q[4], double R[9]) {
  const double w = q[0], x = q[1], y = q[2], z = q[3];
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z); R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z); R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y); R[7] = 2 * (y * z + w * x); R[8] = 1 - 2 * (x * x + y * y);
}

// Geometry shared by forward and backward: everything that depends on (mu, s, q, view).
struct Geo {
  double t[3], rho, rxz, u[3], e[3], n[3];
  double R[9];
  double Mc[6];          // M = W Sigma3D W^T, symmetric: (00,01,02,11,12,22)
  double a, b, c, det;   // Sigma_arc incl. dilation
  bool culled, pole;
};

__device__ __forceinline__ void sym_mul_vec(const double S[6], const double v[3], double out[3]) {
  out[0] = S[0] * v[0] + S[1] * v[1] + S[2] * v[2];
  out[1] = S[1] * v[0] + S[3] * v[1] + S[4] * v[2];
  out[2] = S[2] * v[0] + S[4] * v[1] + S[5] * v[2];
}

__device__ __forceinline__ void geometry(const ViewConst& vc, const double mu[3], const double s[3], const double q[4],
                                         double r_near, double h, Geo& g) {
  g.culled = false; g.pole = false;
#pragma unroll
  for (int i = 0; i < 3; ++i) g.t[i] = vc.W[3 * i] * mu[0] + vc.W[3 * i + 1] * mu[1] + vc.W[3 * i + 2] * mu[2] + vc.b[i];
  const double r2 = g.t[0] * g.t[0] + g.t[1] * g.t[1] + g.t[2] * g.t[2];
  g.rho = sqrt(r2);
  const bool fin = isfinite(mu[0]) && isfinite(mu[1]) && isfinite(mu[2]) && isfinite(s[0]) && isfinite(s[1]) && isfinite(s[2]) &&
                   isfinite(q[0]) && isfinite(q[1]) && isfinite(q[2]) && isfinite(q[3]) && isfinite(g.rho);
  if (!fin || !(g.rho > r_near)) { g.culled = true; return; }
  const double ir = 1.0 / g.rho;
  g.u[0] = g.t[0] / g.rho; g.u[1] = g.t[1] / g.rho; g.u[2] = g.t[2] / g.rho;
  g.rxz = sqrt(g.t[0] * g.t[0] + g.t[2] * g.t[2]);
  if (g.rxz > 0) { g.e[0] = g.t[2] / g.rxz; g.e[1] = 0; g.e[2] = -g.t[0] / g.rxz; }
  else { g.pole = true; g.e[0] = 1; g.e[1] = 0; g.e[2] = 0; }              // reading A22
  g.n[0] = g.u[1] * g.e[2] - g.u[2] * g.e[1];
  g.n[1] = g.u[2] * g.e[0] - g.u[0] * g.e[2];
  g.n[2] = g.u[0] * g.e[1] - g.u[1] * g.e[0];
  // Sigma3D = R diag(s^2) R^T  (Alg.1 l.4), M = W Sigma3D W^T  =  (W R) diag(s^2) (W R)^T
  quat_rot(q, g.R);
  double A[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) A[3 * i + j] = vc.W[3 * i] * g.R[j] + vc.W[3 * i + 1] * g.R[3 + j] + vc.W[3 * i + 2] * g.R[6 + j];
  const double s2[3] = {s[0] * s[0], s[1] * s[1], s[2] * s[2]};
  int k = 0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j)
      g.Mc[k++] = A[3 * i] * s2[0] * A[3 * j] + A[3 * i + 1] * s2[1] * A[3 * j + 1] + A[3 * i + 2] * s2[2] * A[3 * j + 2];
  double Me[3], Mn[3];
  sym_mul_vec(g.Mc, g.e, Me); sym_mul_vec(g.Mc, g.n, Mn);
  const double ir2 = ir * ir;
  g.a = (g.e[0] * Me[0] + g.e[1] * Me[1] + g.e[2] * Me[2]) * ir2 + h;      // Eq.2 + dilation (reading A3)
  g.b = (g.e[0] * Mn[0] + g.e[1] * Mn[1] + g.e[2] * Mn[2]) * ir2;
  g.c = (g.n[0] * Mn[0] + g.n[1] * Mn[1] + g.n[2] * Mn[2]) * ir2 + h;
  g.det = g.a * g.c - g.b * g.b;
  if (!(g.det > 0) || !isfinite(g.det)) g.culled = true;                   // reading A23
}

// PARTS: 1 = geometry records only (everything but rgb; needs no SH), 2 = colour only (rgb and the clamp bits of flags, on records
// whose geometry part has run), 3 = both in one pass (uts_preprocess).  1 then 2 writes exactly what 3 writes.
template <int PARTS>
__global__ void __launch_bounds__(128, 8)
preprocess_fwd_kernel(uts_config cfg, const float* __restrict__ means, const float* __restrict__ scales,
                      const float* __restrict__ quats, const float* __restrict__ opac, const float* __restrict__ sh,
                      const float* __restrict__ Wv, const float* __restrict__ bv, uts_proj out, double h) {
  const int P = cfg.n_gauss;
  const int v = blockIdx.y;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P) return;
  ViewConst vc; load_view(Wv, bv, v, vc);
  const double mu[3] = {(double)__ldg(means + 3 * i), (double)__ldg(means + 3 * i + 1), (double)__ldg(means + 3 * i + 2)};
  double s[3] = {0, 0, 0}, q[4] = {0, 0, 0, 0};
  float o = 0.f;
  if (PARTS & 1) {
    s[0] = (double)__ldg(scales + 3 * i); s[1] = (double)__ldg(scales + 3 * i + 1); s[2] = (double)__ldg(scales + 3 * i + 2);
    const float4 qf = __ldg(reinterpret_cast<const float4*>(quats) + i);
    q[0] = (double)qf.x; q[1] = (double)qf.y; q[2] = (double)qf.z; q[3] = (double)qf.w;
    o = __ldg(opac + i);
  }
  const size_t k = (size_t)v * P + i;
  Geo g;
  if (PARTS & 1) {
    geometry(vc, mu, s, q, (double)cfg.r_near, h, g);
    if (!isfinite(o)) g.culled = true;
  } else {
    g.culled = (out.flags[k] & 1) != 0;
  }
  if (g.culled) {
    if (PARTS & 1) {
      out.dir[3 * k] = out.dir[3 * k + 1] = out.dir[3 * k + 2] = 0.f;
      out.lonlat[2 * k] = out.lonlat[2 * k + 1] = 0.f;
      out.rho[k] = 0.f; out.rs[k] = 0.f;
      reinterpret_cast<float4*>(out.conic_opac)[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      out.flags[k] = 1;
    }
    if (PARTS & 2) out.rgb[3 * k] = out.rgb[3 * k + 1] = out.rgb[3 * k + 2] = 0.f;
    return;
  }
  if (PARTS & 1) {
    // l.7: r_s = 3 sqrt(lambda_max), clamped to pi (reading A4)
    const double hd = 0.5 * (g.a - g.c);
    const double lmax = 0.5 * (g.a + g.c) + sqrt(fmax(0.0, hd * hd + g.b * g.b));
    const double rs = fmin(kPi, 3.0 * sqrt(lmax));
    const double idet = 1.0 / g.det;
    out.dir[3 * k] = (float)g.u[0]; out.dir[3 * k + 1] = (float)g.u[1]; out.dir[3 * k + 2] = (float)g.u[2];
    out.lonlat[2 * k] = (float)atan2(g.t[0], g.t[2]);                         // Eq.1
    out.lonlat[2 * k + 1] = (float)atan2(g.t[1], g.rxz);
    out.rho[k] = (float)g.rho;
    out.rs[k] = (float)rs;
    reinterpret_cast<float4*>(out.conic_opac)[k] =
        make_float4((float)(g.c * idet), (float)(-g.b * idet), (float)(g.a * idet), o);   // Sigma_arc^{-1}
    if (!(PARTS & 2)) { out.flags[k] = 0; return; }
  }
  // colour (reading A13): direction from the camera centre to mu in world space
  double vd[3] = {mu[0] - vc.cam[0], mu[1] - vc.cam[1], mu[2] - vc.cam[2]};
  const double vl = sqrt(vd[0] * vd[0] + vd[1] * vd[1] + vd[2] * vd[2]);
  vd[0] /= vl; vd[1] /= vl; vd[2] /= vl;
  const int M = (cfg.sh_degree + 1) * (cfg.sh_degree + 1);
  float Y[16];
  sh_basis_eval<float>(cfg.sh_degree, (float)vd[0], (float)vd[1], (float)vd[2], Y);
  float acc[3] = {0.5f, 0.5f, 0.5f};
  const float* shp = sh + (size_t)i * 3 * M;
  if ((M & 3) == 0) {                      // degree 1 or 3: 3M floats = whole float4s, rows are 16-byte aligned
    const float4* s4 = reinterpret_cast<const float4*>(shp);
    for (int j = 0; j < 3 * M / 4; ++j) {
      const float4 c4 = __ldg(s4 + j);
      const float cc[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
      for (int l = 0; l < 4; ++l) { const int idx = 4 * j + l; acc[idx % 3] += Y[idx / 3] * cc[l]; }
    }
  } else {
    for (int m = 0; m < M; ++m)
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) acc[ch] += Y[m] * __ldg(shp + 3 * m + ch);
  }
  // The clamp decision (flag bits 1-3) is taken in double when the fp32 sum is within rounding reach of zero.
  bool near0 = fabsf(acc[0]) < 1e-4f || fabsf(acc[1]) < 1e-4f || fabsf(acc[2]) < 1e-4f;
  if (near0) {
    double Yd[16];
    sh_basis_eval<double>(cfg.sh_degree, vd[0], vd[1], vd[2], Yd);
    double ad[3] = {0.5, 0.5, 0.5};
    for (int m = 0; m < M; ++m)
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) ad[ch] += Yd[m] * (double)__ldg(shp + 3 * m + ch);
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) acc[ch] = (ad[ch] < 0) ? -1.f : (float)ad[ch];
  }
  uint8_t fl = 0;
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) if (acc[ch] < 0.f) { acc[ch] = 0.f; fl |= (uint8_t)(2u << ch); }

  out.rgb[3 * k] = acc[0]; out.rgb[3 * k + 1] = acc[1]; out.rgb[3 * k + 2] = acc[2];
  out.flags[k] = fl;                     // (a record that reaches this line is not culled: bit0 = 0)
}

// ------------------------------------------------------------------------------------------- backward
// Chain used (own derivation): with E = [e; n] (2x3), Sigma' = E M E^T / rho^2 + h I,
//   X  = dL/dSigma'  = -K Gk K                 (K = conic as a matrix, Gk = conic gradient with halved off-diagonal)
//   dL/dM = E^T X E / rho^2 ;  dL/dSigma3D = W^T dL/dM W ;  dL/ds_k = 2 s_k (R^T . R)_kk ;  dL/dR = 2 . R diag(s^2)
//   dL/dE = 2 X E M / rho^2  (rows g_e, g_n) ;  dL/drho|_Sigma = -(2/rho) <X, Sigma' - h I>
//   e = e(omega), n = n(omega,phi), u = u(omega,phi):  de/domega = -hh, dn/domega = -sin(phi) e, dn/dphi = -u,
//   with hh = cos(phi) u - sin(phi) n the horizontal unit vector;  d omega/dt = e / rxz,  d phi/dt = n / rho,  d rho/dt = u.
// The three paths of PAPER.md:91-96 (mu' path, J path, S_phi path) are this single chain written in the (e,n,u) frame.
// Two kernels, one thread per Gaussian each, views summed in registers (no atomics, the sums are deterministic):
//   preprocess_bwd_geo_kernel    the geometry chain (double precision, no SH): writes dL_dmeans (geometry part), dL_dscales, dL_dquats;
//   preprocess_bwd_color_kernel  the colour path: dL_dsh accumulated over the views in registers and written once (48 floats at
//                                degree 3, as float4), and the view-direction term added to dL_dmeans.
// As one kernel the 128-register cap spilt 0.5 KB per thread and every further view read-modified-wrote the 192 B of dL_dsh
// (config 5, 4 views: 2.2 ms for 1 M Gaussians); split, neither kernel spills.
// (four resident blocks per SM: 128 registers with 0.3 KB of spills beat 192 registers without: 0.21 -> 0.16 ms on config 4)
__global__ void __launch_bounds__(128, 4)
preprocess_bwd_geo_kernel(uts_config cfg, const float* __restrict__ means, const float* __restrict__ scales,
                          const float* __restrict__ quats, const float* __restrict__ Wv, const float* __restrict__ bv,
                          const uint8_t* __restrict__ flags, const float* __restrict__ dL_dconic, const float* __restrict__ dL_dmu2,
                          float* __restrict__ dL_dmeans, float* __restrict__ dL_dscales, float* __restrict__ dL_dquats, double h) {
  const int P = cfg.n_gauss;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P) return;
  const double mu[3] = {(double)__ldg(means + 3 * i), (double)__ldg(means + 3 * i + 1), (double)__ldg(means + 3 * i + 2)};
  const double s[3] = {(double)__ldg(scales + 3 * i), (double)__ldg(scales + 3 * i + 1), (double)__ldg(scales + 3 * i + 2)};
  const float4 qf = __ldg(reinterpret_cast<const float4*>(quats) + i);
  const double q[4] = {(double)qf.x, (double)qf.y, (double)qf.z, (double)qf.w};
  double g_mu[3] = {0, 0, 0}, g_s[3] = {0, 0, 0}, g_q[4] = {0, 0, 0, 0};
  for (int v = 0; v < cfg.n_views; ++v) {
    const size_t k = (size_t)v * P + i;
    if (__ldg(flags + k) & 1) continue;                  // culled in this view: contributes nothing
    ViewConst vc; load_view(Wv, bv, v, vc);
    Geo g;
    geometry(vc, mu, s, q, (double)cfg.r_near, h, g);
    if (g.culled || g.pole) continue;                    // A22: only the colour path at an exact pole
    const double idet = 1.0 / g.det;
    const double KA = g.c * idet, KB = -g.b * idet, KC = g.a * idet;
    const double gA = (double)__ldg(dL_dconic + 3 * k), gB = 0.5 * (double)__ldg(dL_dconic + 3 * k + 1), gC = (double)__ldg(dL_dconic + 3 * k + 2);
    // X = -K Gk K
    const double T00 = KA * gA + KB * gB, T01 = KA * gB + KB * gC, T10 = KB * gA + KC * gB, T11 = KB * gB + KC * gC;
    const double X00 = -(T00 * KA + T01 * KB), X01 = -(T00 * KB + T01 * KC), X11 = -(T10 * KB + T11 * KC);
    const double ir = 1.0 / g.rho, ir2 = ir * ir;
    // dL/dM = E^T X E / rho^2, symmetric (00,01,02,11,12,22)
    const double Xe[3] = {X00 * g.e[0] + X01 * g.n[0], X00 * g.e[1] + X01 * g.n[1], X00 * g.e[2] + X01 * g.n[2]};   // row 0 of X E
    const double Xn[3] = {X01 * g.e[0] + X11 * g.n[0], X01 * g.e[1] + X11 * g.n[1], X01 * g.e[2] + X11 * g.n[2]};   // row 1 of X E
    double dM[9];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c2 = 0; c2 < 3; ++c2) dM[3 * r + c2] = (g.e[r] * Xe[c2] + g.n[r] * Xn[c2]) * ir2;
    // Sigma3D = R S2 R^T, M = (W R) S2 (W R)^T with A = W R:  dL/dA = 2 dM A S2 ;  dL/ds_k = 2 s_k (A^T dM A)_kk ; dL/dR = W^T dL/dA
    double A[9];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c2 = 0; c2 < 3; ++c2) A[3 * r + c2] = vc.W[3 * r] * g.R[c2] + vc.W[3 * r + 1] * g.R[3 + c2] + vc.W[3 * r + 2] * g.R[6 + c2];
    double dMA[9];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c2 = 0; c2 < 3; ++c2) dMA[3 * r + c2] = dM[3 * r] * A[c2] + dM[3 * r + 1] * A[3 + c2] + dM[3 * r + 2] * A[6 + c2];
    const double s2[3] = {s[0] * s[0], s[1] * s[1], s[2] * s[2]};
#pragma unroll
    for (int c2 = 0; c2 < 3; ++c2) g_s[c2] += 2.0 * s[c2] * (A[c2] * dMA[c2] + A[3 + c2] * dMA[3 + c2] + A[6 + c2] * dMA[6 + c2]);
    double D[9];                                         // dL/dR = W^T (2 dM A S2)
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c2 = 0; c2 < 3; ++c2)
        D[3 * r + c2] = 2.0 * s2[c2] * (vc.W[r] * dMA[c2] + vc.W[3 + r] * dMA[3 + c2] + vc.W[6 + r] * dMA[6 + c2]);
    {
      const double w = q[0], x = q[1], y = q[2], z = q[3];
      g_q[0] += 2 * (z * (D[3] - D[1]) + y * (D[2] - D[6]) + x * (D[7] - D[5]));
      g_q[1] += 2 * (y * (D[1] + D[3]) + z * (D[2] + D[6]) + w * (D[7] - D[5]) - 2 * x * (D[4] + D[8]));
      g_q[2] += 2 * (x * (D[1] + D[3]) + z * (D[5] + D[7]) + w * (D[2] - D[6]) - 2 * y * (D[0] + D[8]));
      g_q[3] += 2 * (x * (D[2] + D[6]) + y * (D[5] + D[7]) + w * (D[3] - D[1]) - 2 * z * (D[0] + D[4]));
    }
    // dL/dE = 2 X E M / rho^2
    double ge[3], gn[3];
    sym_mul_vec(g.Mc, Xe, ge); sym_mul_vec(g.Mc, Xn, gn);
#pragma unroll
    for (int r = 0; r < 3; ++r) { ge[r] *= 2.0 * ir2; gn[r] *= 2.0 * ir2; }
    const double g_rho = -2.0 * ir * (X00 * (g.a - h) + 2.0 * X01 * g.b + X11 * (g.c - h));
    const double sphi = g.u[1], cphi = g.rxz * ir;
    const double hh[3] = {cphi * g.u[0] - sphi * g.n[0], cphi * g.u[1] - sphi * g.n[1], cphi * g.u[2] - sphi * g.n[2]};
    const double ge_h = ge[0] * hh[0] + ge[1] * hh[1] + ge[2] * hh[2];
    const double gn_e = gn[0] * g.e[0] + gn[1] * g.e[1] + gn[2] * g.e[2];
    const double gn_u = gn[0] * g.u[0] + gn[1] * g.u[1] + gn[2] * g.u[2];
    const double c_om = (-ge_h - sphi * gn_e + (double)__ldg(dL_dmu2 + 2 * k)) / g.rxz;       // coefficient of e
    const double c_ph = (-gn_u + (double)__ldg(dL_dmu2 + 2 * k + 1)) * ir;                     // coefficient of n
    const double gt[3] = {c_om * g.e[0] + c_ph * g.n[0] + g_rho * g.u[0], c_om * g.e[1] + c_ph * g.n[1] + g_rho * g.u[1],
                          c_om * g.e[2] + c_ph * g.n[2] + g_rho * g.u[2]};
#pragma unroll
    for (int r = 0; r < 3; ++r) g_mu[r] += vc.W[r] * gt[0] + vc.W[3 + r] * gt[1] + vc.W[6 + r] * gt[2];   // W^T dL/dt
  }
#pragma unroll
  for (int r = 0; r < 3; ++r) { dL_dmeans[3 * i + r] = (float)g_mu[r]; dL_dscales[3 * i + r] = (float)g_s[r]; }
  reinterpret_cast<float4*>(dL_dquats)[i] = make_float4((float)g_q[0], (float)g_q[1], (float)g_q[2], (float)g_q[3]);
}

// Colour path: rgb_ch = max(0, 1/2 + sum_m Y_m(vdir) sh[m,ch]) (reading A13).  dL_dmeans must hold the geometry part already.
template <int DEG>
__global__ void __launch_bounds__(128, 4)
preprocess_bwd_color_kernel(uts_config cfg, const float* __restrict__ means, const float* __restrict__ sh, const float* __restrict__ Wv,
                            const float* __restrict__ bv, const uint8_t* __restrict__ flags, const float* __restrict__ dL_drgb,
                            float* __restrict__ dL_dmeans, float* __restrict__ dL_dsh) {
  constexpr int M = (DEG + 1) * (DEG + 1), NF = 3 * M;
  const int P = cfg.n_gauss;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P) return;
  const double mu[3] = {(double)__ldg(means + 3 * i), (double)__ldg(means + 3 * i + 1), (double)__ldg(means + 3 * i + 2)};
  const float* shp = sh + (size_t)i * NF;
  float* gsh = dL_dsh + (size_t)i * NF;
  float acc[NF];                                         // dL_dsh of this Gaussian, [m][ch], summed over the views
#pragma unroll
  for (int j = 0; j < NF; ++j) acc[j] = 0.f;
  double g_mu[3] = {0, 0, 0};
  for (int v = 0; v < cfg.n_views; ++v) {
    const size_t k = (size_t)v * P + i;
    const uint8_t fl = __ldg(flags + k);
    if (fl & 1) continue;
    const float gr[3] = {(fl & 2) ? 0.f : __ldg(dL_drgb + 3 * k), (fl & 4) ? 0.f : __ldg(dL_drgb + 3 * k + 1),
                         (fl & 8) ? 0.f : __ldg(dL_drgb + 3 * k + 2)};
    // camera centre -W^T b of this view
    double cam[3];
#pragma unroll
    for (int r = 0; r < 3; ++r)
      cam[r] = -((double)__ldg(Wv + 9 * v + r) * (double)__ldg(bv + 3 * v) + (double)__ldg(Wv + 9 * v + 3 + r) * (double)__ldg(bv + 3 * v + 1) +
                 (double)__ldg(Wv + 9 * v + 6 + r) * (double)__ldg(bv + 3 * v + 2));
    double vd[3] = {mu[0] - cam[0], mu[1] - cam[1], mu[2] - cam[2]};
    const double vl = sqrt(vd[0] * vd[0] + vd[1] * vd[1] + vd[2] * vd[2]);
    vd[0] /= vl; vd[1] /= vl; vd[2] /= vl;
    const float dx = (float)vd[0], dy = (float)vd[1], dz = (float)vd[2];
    float Y[16];
    sh_basis_eval<float>(DEG, dx, dy, dz, Y);
    float cmix[16];                                      // sum_ch g_ch sh[m,ch]; the coefficients are re-read per view (L1 / L2 hits)
#pragma unroll
    for (int m = 0; m < M; ++m) cmix[m] = 0.f;
    if (DEG == 3) {                                      // 48 floats = 12 aligned float4
#pragma unroll
      for (int j = 0; j < NF / 4; ++j) {
        const float4 c4 = __ldg(reinterpret_cast<const float4*>(shp) + j);
        const float cc[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
        for (int l = 0; l < 4; ++l) {
          const int idx = 4 * j + l;                     // = 3 m + ch, compile-time after unrolling
          cmix[idx / 3] = fmaf(gr[idx % 3], cc[l], cmix[idx / 3]);
          acc[idx] = fmaf(Y[idx / 3], gr[idx % 3], acc[idx]);
        }
      }
    } else {
#pragma unroll
      for (int idx = 0; idx < NF; ++idx) {
        cmix[idx / 3] = fmaf(gr[idx % 3], __ldg(shp + idx), cmix[idx / 3]);
        acc[idx] = fmaf(Y[idx / 3], gr[idx % 3], acc[idx]);
      }
    }
    float gvx, gvy, gvz;
    sh_dir_grad(DEG, dx, dy, dz, cmix, gvx, gvy, gvz);
    // vdir = v/|v|  =>  d vdir/d mu = (I - vdir vdir^T)/|v|
    const double dot = gvx * vd[0] + gvy * vd[1] + gvz * vd[2];
    g_mu[0] += (gvx - dot * vd[0]) / vl; g_mu[1] += (gvy - dot * vd[1]) / vl; g_mu[2] += (gvz - dot * vd[2]) / vl;
  }
  if (DEG == 3) {
#pragma unroll
    for (int j = 0; j < NF / 4; ++j) reinterpret_cast<float4*>(gsh)[j] = make_float4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < NF; ++j) gsh[j] = acc[j];
  }
#pragma unroll
  for (int r = 0; r < 3; ++r) dL_dmeans[3 * i + r] = (float)((double)dL_dmeans[3 * i + r] + g_mu[r]);
}

}  // namespace uts

using namespace uts;

extern "C" {

int uts_preprocess(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (!g.means || !g.scales || !g.quats || !g.opac || !g.sh || !views.W || !views.b) return UTS_ERR_INVALID_ARG;
  if (!out.dir || !out.lonlat || !out.rho || !out.conic_opac || !out.rs || !out.rgb || !out.flags) return UTS_ERR_INVALID_ARG;
  if (cfg->n_gauss == 0) return UTS_OK;
  const double h = (double)cfg->cov_dilation_px2 * 4.0 * kPi / (double)((int64_t)12 << (2 * cfg->order));
  dim3 grid((cfg->n_gauss + 127) / 128, cfg->n_views);
  preprocess_fwd_kernel<3><<<grid, 128, 0, (cudaStream_t)stream>>>(*cfg, g.means, g.scales, g.quats, g.opac, g.sh, views.W, views.b, out, h);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_preprocess_geometry(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (!g.means || !g.scales || !g.quats || !g.opac || !views.W || !views.b) return UTS_ERR_INVALID_ARG;
  if (!out.dir || !out.lonlat || !out.rho || !out.conic_opac || !out.rs || !out.flags) return UTS_ERR_INVALID_ARG;
  if (cfg->n_gauss == 0) return UTS_OK;
  const double h = (double)cfg->cov_dilation_px2 * 4.0 * kPi / (double)((int64_t)12 << (2 * cfg->order));
  dim3 grid((cfg->n_gauss + 127) / 128, cfg->n_views);
  preprocess_fwd_kernel<1><<<grid, 128, 0, (cudaStream_t)stream>>>(*cfg, g.means, g.scales, g.quats, g.opac, nullptr, views.W, views.b, out, h);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_preprocess_color(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (!g.means || !g.sh || !views.W || !views.b || !out.rgb || !out.flags) return UTS_ERR_INVALID_ARG;
  if (cfg->n_gauss == 0) return UTS_OK;
  dim3 grid((cfg->n_gauss + 127) / 128, cfg->n_views);
  preprocess_fwd_kernel<2><<<grid, 128, 0, (cudaStream_t)stream>>>(*cfg, g.means, nullptr, nullptr, nullptr, g.sh, views.W, views.b, out, 0.0);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_preprocess_bwd(const uts_config* cfg, uts_gaussians g, uts_views views, const uint8_t* flags,
                       const float* dL_drgb, const float* dL_dconic, const float* dL_dmu2, float* dL_dmeans,
                       float* dL_dscales, float* dL_dquats, float* dL_dsh, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (!g.means || !g.scales || !g.quats || !g.sh || !views.W || !views.b || !flags) return UTS_ERR_INVALID_ARG;
  if (!dL_drgb || !dL_dconic || !dL_dmu2 || !dL_dmeans || !dL_dscales || !dL_dquats || !dL_dsh) return UTS_ERR_INVALID_ARG;
  if (cfg->n_gauss == 0) return UTS_OK;
  const double h = (double)cfg->cov_dilation_px2 * 4.0 * kPi / (double)((int64_t)12 << (2 * cfg->order));
  const unsigned grid = (unsigned)((cfg->n_gauss + 127) / 128);
  cudaStream_t s = (cudaStream_t)stream;
  preprocess_bwd_geo_kernel<<<grid, 128, 0, s>>>(*cfg, g.means, g.scales, g.quats, views.W, views.b, flags, dL_dconic, dL_dmu2, dL_dmeans,
                                                 dL_dscales, dL_dquats, h);
  UTS_LAUNCH_CHECK();
  switch (cfg->sh_degree) {
    case 0: preprocess_bwd_color_kernel<0><<<grid, 128, 0, s>>>(*cfg, g.means, g.sh, views.W, views.b, flags, dL_drgb, dL_dmeans, dL_dsh); break;
    case 1: preprocess_bwd_color_kernel<1><<<grid, 128, 0, s>>>(*cfg, g.means, g.sh, views.W, views.b, flags, dL_drgb, dL_dmeans, dL_dsh); break;
    case 2: preprocess_bwd_color_kernel<2><<<grid, 128, 0, s>>>(*cfg, g.means, g.sh, views.W, views.b, flags, dL_drgb, dL_dmeans, dL_dsh); break;
    default: preprocess_bwd_color_kernel<3><<<grid, 128, 0, s>>>(*cfg, g.means, g.sh, views.W, views.b, flags, dL_drgb, dL_dmeans, dL_dsh); break;
  }
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // extern "C"
