// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, double precision; shares no code with the CUDA path.
//
// the inverse radial depth channel used for depth supervision ("we use inverse radial depth
// r^-1, whose gradient is d r^-1 / dt = -t / r^3") and the per-Gaussian r_s,max buffer of the radian-space density control
// ("r_s,max <- max(r_s,max, r_s) whenever the Gaussian is visible").
//
// Reading A29: the depth image is the blend of Eq.6 with the colour c_i replaced by r_i^-1,  D(p) = sum_i r_i^-1 alpha_i(p)
// prod_{j<i}(1 - alpha_j(p))  (no background term, not normalised by alpha): the same compositing the paper defines for colour,
// so the oracle forms the per-Gaussian channel (r^-1, 0, 0) here and runs its ordinary blend on it.  "Visible" is
// read as "not culled by the preprocess" (flags bit 0 clear), in any view of the call.
// Pins (tests/test_oracle_depth.py): equal-radius scene => D = alpha / r exactly; the gradient against central differences of
// r^-1 = 1/||W mu + b||; r_s,max is monotone, idempotent and ignores culled Gaussians.
#include <cmath>
#include <cstdint>

extern "C" {

// chan [V,P,3] = (1/rho, 0, 0); culled Gaussians (flags bit 0) get 0.  rho is the fp32 record of the preprocess (reading P1).
void orc_inv_depth_channel(int n_views, int n_gauss, const float* rho, const uint8_t* flags, float* chan) {
  for (int64_t k = 0; k < (int64_t)n_views * n_gauss; ++k) {
    const bool culled = flags && (flags[k] & 1);
    chan[3 * k] = culled ? 0.0f : (float)(1.0 / (double)rho[k]);
    chan[3 * k + 1] = 0.0f; chan[3 * k + 2] = 0.0f;
  }
}

// dL_dmeans [P,3] (double, overwritten) = sum_v W_v^T ( -t / r^3 ) dL_dinv[v,i],  t = W_v mu_i + b_v
void orc_inv_depth_bwd(int n_views, int n_gauss, const float* means, const float* Wv, const float* bv, const uint8_t* flags,
                       const double* dL_dinv /*[V,P]*/, double* dL_dmeans) {
  for (int64_t i = 0; i < (int64_t)3 * n_gauss; ++i) dL_dmeans[i] = 0;
  for (int v = 0; v < n_views; ++v) {
    const float* W = Wv + 9 * v; const float* b = bv + 3 * v;
    for (int i = 0; i < n_gauss; ++i) {
      const int64_t k = (int64_t)v * n_gauss + i;
      if (flags && (flags[k] & 1)) continue;
      double t[3];
      for (int r = 0; r < 3; ++r)
        t[r] = (double)W[3 * r] * means[3 * i] + (double)W[3 * r + 1] * means[3 * i + 1] + (double)W[3 * r + 2] * means[3 * i + 2] + (double)b[r];
      const double rr = std::sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
      const double s = -dL_dinv[k] / (rr * rr * rr);
      for (int c = 0; c < 3; ++c)                       // dL/dmu = W^T dL/dt
        dL_dmeans[3 * i + c] += s * ((double)W[c] * t[0] + (double)W[3 + c] * t[1] + (double)W[6 + c] * t[2]);
    }
  }
}

// rs_max[i] <- max(rs_max[i], rs[v,i]) over the views in which Gaussian i is visible
void orc_rs_max_update(int n_views, int n_gauss, const float* rs, const uint8_t* flags, float* rs_max) {
  for (int v = 0; v < n_views; ++v)
    for (int i = 0; i < n_gauss; ++i) {
      const int64_t k = (int64_t)v * n_gauss + i;
      if (flags && (flags[k] & 1)) continue;
      if (rs[k] > rs_max[i]) rs_max[i] = rs[k];
    }
}

}  // extern "C"
