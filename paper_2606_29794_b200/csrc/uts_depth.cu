// uts_depth.cu — inverse radial depth channel and the r_s,max buffer.
//   "For depth supervision, we use inverse radial depth r^-1, whose gradient is d r^-1/dt = -t / r^3"
//   "r_s,max <- max(r_s,max, r_s) whenever the Gaussian is visible"
// Reading A29: the depth image is Eq.6 with the colour c_i replaced by r_i^-1.  The blend kernels take the per-Gaussian value to
// composite from `uts_proj.rgb`, so the depth image is uts_render_fwd on a record whose rgb is the channel (r^-1, 0, 0) built
// here, and uts_render_bwd on the same record returns dL/d(r_i^-1) in dL_drgb[..., 0] together with the alpha-path terms of the
// depth loss (dL_dconic, dL_dmu2, dL_dopac), which add to those of the colour loss.  uts_inv_depth_bwd then carries dL/d(r^-1)
// to the means.  That form costs a second blend pass; uts_render_fwd_depth / uts_render_bwd_depth (uts_render.cu) blend 1 / rho as a
// FOURTH CHANNEL of the colour pass instead (+2 % forward, +7 % backward on config 4) and return dL/d(r^-1) as dL_dinvr [V,P],
// which uts_inv_depth_bwd takes with chan_stride = 1.  Streaming kernels, one thread per (view, Gaussian) or per Gaussian.
#include "uts_internal.cuh"

namespace uts {

__global__ void inv_depth_channel_kernel(int64_t n, const float* __restrict__ rho, const uint8_t* __restrict__ flags, float* __restrict__ chan) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const bool culled = (__ldg(flags + k) & 1) != 0;
  chan[3 * k] = culled ? 0.f : __fdiv_rn(1.0f, __ldg(rho + k));
  chan[3 * k + 1] = 0.f; chan[3 * k + 2] = 0.f;
}

// one thread per Gaussian, views summed in registers; double like the geometry chain of the preprocess
__global__ void inv_depth_bwd_kernel(int P, int V, const float* __restrict__ means, const float* __restrict__ Wv, const float* __restrict__ bv,
                                     const uint8_t* __restrict__ flags, const float* __restrict__ dL_dchan, int chan_stride, int accumulate,
                                     float* __restrict__ dL_dmeans) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P) return;
  const double mx = __ldg(means + 3 * i), my = __ldg(means + 3 * i + 1), mz = __ldg(means + 3 * i + 2);
  double gx = 0.0, gy = 0.0, gz = 0.0;
  for (int v = 0; v < V; ++v) {
    const int64_t k = (int64_t)v * P + i;
    if (__ldg(flags + k) & 1) continue;
    const float* W = Wv + 9 * v; const float* b = bv + 3 * v;
    const double tx = (double)W[0] * mx + (double)W[1] * my + (double)W[2] * mz + (double)b[0];
    const double ty = (double)W[3] * mx + (double)W[4] * my + (double)W[5] * mz + (double)b[1];
    const double tz = (double)W[6] * mx + (double)W[7] * my + (double)W[8] * mz + (double)b[2];
    const double r2 = tx * tx + ty * ty + tz * tz;
    const double s = -(double)__ldg(dL_dchan + (size_t)chan_stride * k) / (r2 * sqrt(r2));      // dL/d(r^-1) * (-1/r^3)
    gx += s * ((double)W[0] * tx + (double)W[3] * ty + (double)W[6] * tz);    // W^T (s t)
    gy += s * ((double)W[1] * tx + (double)W[4] * ty + (double)W[7] * tz);
    gz += s * ((double)W[2] * tx + (double)W[5] * ty + (double)W[8] * tz);
  }
  if (accumulate) { dL_dmeans[3 * i] += (float)gx; dL_dmeans[3 * i + 1] += (float)gy; dL_dmeans[3 * i + 2] += (float)gz; }
  else { dL_dmeans[3 * i] = (float)gx; dL_dmeans[3 * i + 1] = (float)gy; dL_dmeans[3 * i + 2] = (float)gz; }
}

__global__ void rs_max_kernel(int P, int V, const float* __restrict__ rs, const uint8_t* __restrict__ flags, float* __restrict__ rs_max) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P) return;
  float m = rs_max[i];
  for (int v = 0; v < V; ++v) {
    const int64_t k = (int64_t)v * P + i;
    if (!(__ldg(flags + k) & 1)) m = fmaxf(m, __ldg(rs + k));
  }
  rs_max[i] = m;
}

// ---- occlusion-bounded lists: helpers, the orchestration is the caller's
__global__ void depth_prefix_flags_kernel(int P, int64_t n, const uint8_t* __restrict__ flags, const uint32_t* __restrict__ emit_rank, uint32_t keep,
                                          uint8_t* __restrict__ out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const uint32_t v = (uint32_t)(k / P);
  const uint32_t rank_in_view = __ldg(emit_rank + k) - v * (uint32_t)P;       // emit_rank orders by (view, depth, id)
  out[k] = (uint8_t)(__ldg(flags + k) | (rank_in_view >= keep ? 1u : 0u));
}

__global__ void count_unsaturated_kernel(int64_t n, int64_t n_slot, const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ bits,
                                         const float* __restrict__ trans, float t_eps, unsigned long long* __restrict__ count) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool open = false;
  if (idx < n) {
    const int64_t slot = (idx >> 8) % n_slot;
    const int64_t tile = active_tiles ? (int64_t)__ldg(active_tiles + slot) : slot;
    const int64_t p = tile * 256 + (idx & 255);
    const bool on = bits ? ((__ldg(bits + (p >> 5)) >> (p & 31)) & 1u) != 0 : true;
    open = on && !(__ldg(trans + idx) < t_eps);
  }
  const unsigned m = __ballot_sync(0xffffffffu, open);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(count, (unsigned long long)__popc(m));
}

}  // namespace uts

using namespace uts;

extern "C" {

int uts_inv_depth_channel(const uts_config* cfg, const float* rho, const uint8_t* flags, float* chan, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  const int64_t n = (int64_t)cfg->n_gauss * cfg->n_views;
  if (n == 0) return UTS_OK;
  if (!rho || !flags || !chan) return UTS_ERR_INVALID_ARG;
  inv_depth_channel_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n, rho, flags, chan);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_inv_depth_bwd(const uts_config* cfg, const float* means, uts_views views, const uint8_t* flags, const float* dL_dchan,
                      int chan_stride, int accumulate, float* dL_dmeans, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (cfg->n_gauss == 0) return UTS_OK;
  if (!means || !views.W || !views.b || !flags || !dL_dchan || !dL_dmeans || chan_stride < 1) return UTS_ERR_INVALID_ARG;
  inv_depth_bwd_kernel<<<(unsigned)((cfg->n_gauss + 255) / 256), 256, 0, (cudaStream_t)stream>>>(cfg->n_gauss, cfg->n_views, means, views.W, views.b,
                                                                                               flags, dL_dchan, chan_stride, accumulate, dL_dmeans);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_rs_max_update(const uts_config* cfg, const float* rs, const uint8_t* flags, float* rs_max, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if (cfg->n_gauss == 0) return UTS_OK;
  if (!rs || !flags || !rs_max) return UTS_ERR_INVALID_ARG;
  rs_max_kernel<<<(unsigned)((cfg->n_gauss + 255) / 256), 256, 0, (cudaStream_t)stream>>>(cfg->n_gauss, cfg->n_views, rs, flags, rs_max);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_depth_prefix_flags(const uts_config* cfg, const uint8_t* flags, const uint32_t* emit_rank, uint32_t keep, uint8_t* flags_out, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  const int64_t n = (int64_t)cfg->n_gauss * cfg->n_views;
  if (n == 0) return UTS_OK;
  if (!flags || !emit_rank || !flags_out) return UTS_ERR_INVALID_ARG;
  depth_prefix_flags_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(cfg->n_gauss, n, flags, emit_rank, keep, flags_out);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

int uts_count_unsaturated(const uts_config* cfg, uts_mask mask, const float* trans, uint64_t* h_count, void* scratch, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!h_count || !scratch || ((uintptr_t)scratch & 7)) return UTS_ERR_INVALID_ARG;
  const Dims d = dims_of(cfg, &mask);
  const int64_t n = (int64_t)d.V * d.n_slot * kTilePix;
  cudaStream_t s = (cudaStream_t)stream;
  UTS_CUDA(cudaMemsetAsync(scratch, 0, 8, s));
  if (n > 0) {
    if (!trans) return UTS_ERR_INVALID_ARG;
    count_unsaturated_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, d.n_slot, mask.active_tiles, mask.pixel_mask_bits, trans, cfg->t_eps,
                                                                         (unsigned long long*)scratch);
    UTS_LAUNCH_CHECK();
  }
  UTS_CUDA(cudaMemcpyAsync(h_count, scratch, 8, cudaMemcpyDeviceToHost, s));
  UTS_CUDA(cudaStreamSynchronize(s));
  return UTS_OK;
}

}  // extern "C"
