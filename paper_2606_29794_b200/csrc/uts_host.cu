// uts_host.cu — the whole hot path behind one call that takes HOST buffers (bench.py's end-to-end leg and the
// simplest way to use the library): H2D copies, the seven stages in Alg.1's order followed by the
// backward, D2H copies.  All device memory comes from the caller's workspace.
#include "uts_internal.cuh"

namespace uts {

struct Bump {
  char* base; size_t off;
  template <typename T> T* take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

struct HostLayout {
  float *means, *scales, *quats, *opac, *sh, *W, *b;
  uts_proj proj;
  uint64_t *offsets, *keys, *keys_tmp, *ranges;
  uint32_t *vals, *vals_tmp, *n_last, *marks;
  size_t marks_bytes;
  void *tq_scratch, *sort_scratch, *do_scratch;
  size_t tq_bytes, sort_bytes, do_bytes;
  uint32_t* emit_rank;
  float *color, *alpha, *trans, *g_color;
  float *g_rgb, *g_conic, *g_mu2, *g_opac, *g_means, *g_scales, *g_quats, *g_sh;
  size_t total;
};

static HostLayout layout(const uts_config* cfg, int64_t n_slot, uint64_t cap, char* base) {
  HostLayout L;
  Bump B{base, 0};
  const size_t P = cfg->n_gauss, V = cfg->n_views, M = (size_t)(cfg->sh_degree + 1) * (cfg->sh_degree + 1);
  const size_t VP = V * P, npx = V * (size_t)n_slot * kTilePix;
  const size_t ids = ((size_t)12 << (2 * (cfg->order - cfg->tile_log2))) * V;
  L.means = B.take<float>(3 * P); L.scales = B.take<float>(3 * P); L.quats = B.take<float>(4 * P);
  L.opac = B.take<float>(P); L.sh = B.take<float>(3 * M * P); L.W = B.take<float>(9 * V); L.b = B.take<float>(3 * V);
  L.proj.dir = B.take<float>(3 * VP); L.proj.lonlat = B.take<float>(2 * VP); L.proj.rho = B.take<float>(VP);
  L.proj.conic_opac = B.take<float>(4 * VP); L.proj.rs = B.take<float>(VP); L.proj.rgb = B.take<float>(3 * VP);
  L.proj.flags = B.take<uint8_t>(VP);
  L.offsets = B.take<uint64_t>(VP + 1);
  L.tq_bytes = uts_tile_lists_scratch_bytes(cfg); L.tq_scratch = B.take<char>(L.tq_bytes);
  L.do_bytes = uts_depth_order_scratch_bytes(cfg); L.do_scratch = B.take<char>(L.do_bytes);
  L.emit_rank = B.take<uint32_t>(VP);
  L.keys = B.take<uint64_t>(cap); L.keys_tmp = B.take<uint64_t>(cap);
  L.vals = B.take<uint32_t>(cap); L.vals_tmp = B.take<uint32_t>(cap);
  L.sort_bytes = uts_sort_scratch_bytes(cap); L.sort_scratch = B.take<char>(L.sort_bytes);
  L.ranges = B.take<uint64_t>(2 * ids);
  L.color = B.take<float>(3 * npx); L.alpha = B.take<float>(npx); L.trans = B.take<float>(npx); L.n_last = B.take<uint32_t>(npx);
  L.g_color = B.take<float>(3 * npx);
  L.marks_bytes = uts_render_marks_bytes(cfg, cap); L.marks = B.take<uint32_t>(L.marks_bytes / 4);
  L.g_rgb = B.take<float>(3 * VP); L.g_conic = B.take<float>(3 * VP); L.g_mu2 = B.take<float>(2 * VP); L.g_opac = B.take<float>(P);
  L.g_means = B.take<float>(3 * P); L.g_scales = B.take<float>(3 * P); L.g_quats = B.take<float>(4 * P); L.g_sh = B.take<float>(3 * M * P);
  L.total = B.off + 256;
  return L;
}

}  // namespace uts

using namespace uts;

extern "C" {

size_t uts_host_workspace_bytes(const uts_config* cfg, int n_active, uint64_t pair_capacity) {
  if (check_config(cfg) != UTS_OK) return 0;
  const int64_t n_tile = (int64_t)12 << (2 * (cfg->order - cfg->tile_log2));
  return layout(cfg, n_active >= 0 ? n_active : n_tile, pair_capacity, nullptr).total;
}

int uts_host_forward_backward(const uts_config* cfg, const float* h_means, const float* h_scales, const float* h_quats,
                              const float* h_opac, const float* h_sh, const float* h_W, const float* h_b, uts_mask mask,
                              const float* h_dL_dcolor, float* h_color, float* h_alpha, float* h_dL_dmeans,
                              float* h_dL_dscales, float* h_dL_dquats, float* h_dL_dopac, float* h_dL_dsh,
                              uint64_t pair_capacity, uint64_t* h_n_pairs, void* workspace, size_t workspace_bytes,
                              void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!h_means || !h_scales || !h_quats || !h_opac || !h_sh || !h_W || !h_b || !h_color || !h_n_pairs || !workspace)
    return UTS_ERR_INVALID_ARG;
  const bool bwd = h_dL_dcolor != nullptr;
  if (bwd && (!h_dL_dmeans || !h_dL_dscales || !h_dL_dquats || !h_dL_dopac || !h_dL_dsh)) return UTS_ERR_INVALID_ARG;
  if ((uintptr_t)workspace & 255) return UTS_ERR_INVALID_ARG;
  Dims d = dims_of(cfg, &mask);
  HostLayout L = layout(cfg, d.n_slot, pair_capacity, reinterpret_cast<char*>(workspace));
  if (L.total > workspace_bytes) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t P = d.P, V = d.V, M = d.M, npx = V * (size_t)d.n_slot * kTilePix;
  const size_t f = sizeof(float);
  UTS_CUDA(cudaMemcpyAsync(L.means, h_means, 3 * P * f, cudaMemcpyHostToDevice, s));
  UTS_CUDA(cudaMemcpyAsync(L.scales, h_scales, 3 * P * f, cudaMemcpyHostToDevice, s));
  UTS_CUDA(cudaMemcpyAsync(L.quats, h_quats, 4 * P * f, cudaMemcpyHostToDevice, s));
  UTS_CUDA(cudaMemcpyAsync(L.opac, h_opac, P * f, cudaMemcpyHostToDevice, s));
  UTS_CUDA(cudaMemcpyAsync(L.W, h_W, 9 * V * f, cudaMemcpyHostToDevice, s));
  UTS_CUDA(cudaMemcpyAsync(L.b, h_b, 3 * V * f, cudaMemcpyHostToDevice, s));
  // A second, library-private stream carries the copies that are not on the critical path: the SH coefficients (4/5 of the
  // Gaussian bytes at degree 3) and the upstream gradient go up while the geometry is projected and the tile lists are built —
  // only the colour pass, just before the blend, needs the SH — and the image comes down while the backward runs (effective
  // with pinned host buffers).
  // The stream and its four events belong to the device context (created once per device); ctx->mu is held for the whole call,
  // which ends with both streams synchronised, so the events are never shared between two calls in flight.
  DeviceCtx* ctx = device_ctx();
  if (!ctx) return UTS_ERR_CUDA;
  std::lock_guard<std::recursive_mutex> lock(ctx->mu);
  cudaStream_t s2 = ctx->copy;
  cudaEvent_t ev_up = ctx->ev[0], ev_fwd = ctx->ev[1], ev_start = ctx->ev[2], ev_sh = ctx->ev[3];
  struct Drain { cudaStream_t s2; ~Drain() { cudaStreamSynchronize(s2); } } drain{s2};      // on every exit path
  UTS_CUDA(cudaEventRecord(ev_start, s));                 // s2 must not run ahead of work already queued on the caller's stream
  UTS_CUDA(cudaStreamWaitEvent(s2, ev_start, 0));
  UTS_CUDA(cudaMemcpyAsync(L.sh, h_sh, 3 * M * P * f, cudaMemcpyHostToDevice, s2));
  UTS_CUDA(cudaEventRecord(ev_sh, s2));
  if (bwd) {
    UTS_CUDA(cudaMemcpyAsync(L.g_color, h_dL_dcolor, 3 * npx * f, cudaMemcpyHostToDevice, s2));
    UTS_CUDA(cudaEventRecord(ev_up, s2));
  }

  uts_gaussians g{L.means, L.scales, L.quats, L.opac, L.sh};
  uts_views vw{L.W, L.b};
  if ((st = uts_preprocess_geometry(cfg, g, vw, L.proj, stream))) return st;
  if ((st = uts_depth_order(cfg, L.proj.rho, L.emit_rank, L.do_scratch, L.do_bytes, stream))) return st;
  // Alg.1 l.9-16 in one call: sorted pairs + tile ranges (large discs through the bit matrix, the rest through emit + radix sort)
  if ((st = uts_tile_lists(cfg, L.proj, mask, L.emit_rank, L.keys, L.vals, L.keys_tmp, L.vals_tmp, pair_capacity, L.ranges, h_n_pairs,
                           L.tq_scratch, L.tq_bytes, L.sort_scratch, L.sort_bytes, nullptr, stream)))
    return st;
  UTS_CUDA(cudaStreamWaitEvent(s, ev_sh, 0));
  if ((st = uts_preprocess_color(cfg, g, vw, L.proj, stream))) return st;
  if ((st = uts_render_fwd_marked(cfg, L.proj, mask, L.ranges, L.vals, pair_capacity, L.color, L.alpha, L.trans, L.n_last, L.marks, L.marks_bytes,
                                  stream)))
    return st;
  UTS_CUDA(cudaEventRecord(ev_fwd, s));
  UTS_CUDA(cudaStreamWaitEvent(s2, ev_fwd, 0));
  UTS_CUDA(cudaMemcpyAsync(h_color, L.color, 3 * npx * f, cudaMemcpyDeviceToHost, s2));
  if (h_alpha) UTS_CUDA(cudaMemcpyAsync(h_alpha, L.alpha, npx * f, cudaMemcpyDeviceToHost, s2));
  if (bwd) {
    UTS_CUDA(cudaStreamWaitEvent(s, ev_up, 0));
    if ((st = uts_render_bwd_marked(cfg, L.proj, mask, L.ranges, L.vals, pair_capacity, L.trans, L.n_last, L.marks, L.g_color, nullptr, L.g_rgb,
                                    L.g_conic, L.g_mu2, L.g_opac, stream)))
      return st;
    if ((st = uts_preprocess_bwd(cfg, g, vw, L.proj.flags, L.g_rgb, L.g_conic, L.g_mu2, L.g_means, L.g_scales, L.g_quats, L.g_sh, stream)))
      return st;
    UTS_CUDA(cudaMemcpyAsync(h_dL_dmeans, L.g_means, 3 * P * f, cudaMemcpyDeviceToHost, s));
    UTS_CUDA(cudaMemcpyAsync(h_dL_dscales, L.g_scales, 3 * P * f, cudaMemcpyDeviceToHost, s));
    UTS_CUDA(cudaMemcpyAsync(h_dL_dquats, L.g_quats, 4 * P * f, cudaMemcpyDeviceToHost, s));
    UTS_CUDA(cudaMemcpyAsync(h_dL_dopac, L.g_opac, P * f, cudaMemcpyDeviceToHost, s));
    UTS_CUDA(cudaMemcpyAsync(h_dL_dsh, L.g_sh, 3 * M * P * f, cudaMemcpyDeviceToHost, s));
  }
  UTS_CUDA(cudaStreamSynchronize(s2));
  UTS_CUDA(cudaStreamSynchronize(s));
  return UTS_OK;
}

}  // extern "C"
