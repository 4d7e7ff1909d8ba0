// uts_tile_query.cu — F2: NESTED-scheme tile query and pair emission (Alg.1 l.9-14 PAPER.md:548-559; Alg.2
// PAPER.md:599-620; §3.3; reading A6 for the garbled parts of Alg.2).
//
// Tile set of one projected Gaussian (direction u, radius r_s):
//     T = { q >> 2(k_q - k_t) : q an order-k_q pixel,  u . centre(q) >= cos R },   R = min(pi, r_s + rho_max(k_q)),
// intersected with the active tiles of the mask.  The predicate is evaluated in double precision.
//
// Differences from the paper's kernel (written for sm_89):
//   * The paper's DFS keeps an explicit O(log Nside) stack per thread.  Here the traversal is
//     STACKLESS: a NESTED index IS its own path (child c of p is 4p+c), so "next node in depth-first order" is
//     `while ((p & 3) == 3) p >>= 2, --o;  ++p` — two registers, no local memory.
//   * Zone tests compare the dot product with per-level cosine thresholds cos(R +- rho_max(o)) obtained from one
//     sincos(R) and a constant table of cos/sin rho_max(o) — no inverse trigonometry per node.
//   * count -> exclusive scan -> emit, so the pair arrays are written once, densely, in (view, Gaussian, tile) order;
//     depth-first order over NESTED indices is ascending tile order, so no per-Gaussian sort is needed.
#include "uts_internal.cuh"
#include "uts_scan.cuh"

namespace uts {

struct QueryParams {
  int kt, kq, P, V;
  int64_t n_tile;
  double rho_q;                         // rho_max(k_q)
  double cos_rho[kMaxOrder + 1], sin_rho[kMaxOrder + 1];
};

constexpr double kSlack = 1e-12;        // zone decisions are conservative by this much; the leaf test alone defines T

template <bool EMIT>
struct Sink {
  uint64_t* keys; uint32_t* vals; uint64_t base; uint64_t key_hi_base; uint32_t depth_bits; uint32_t gid;
  const int32_t* slot_of_tile;
  uint32_t count;
  int64_t last_tile;
  __device__ __forceinline__ void add(int64_t tile) {
    if (tile == last_tile) return;
    if (slot_of_tile && __ldg(slot_of_tile + tile) < 0) return;
    if (EMIT) {
      keys[base + count] = ((key_hi_base + (uint64_t)tile) << 32) | depth_bits;   // Alg.1 l.12: ((t, rho), i)
      vals[base + count] = gid;
    }
    ++count;
    last_tile = tile;
  }
};

// Depth-first walk over the NESTED quadtree from the 12 base pixels down to order k_q.
template <bool EMIT>
__device__ __forceinline__ void walk(const QueryParams& qp, const double u[3], double R, Sink<EMIT>& sink) {
  const int kt = qp.kt, kq = qp.kq;
  if (R >= kPi) {                       // reading A24: the disc is the whole sphere
    for (int64_t t = 0; t < qp.n_tile; ++t) sink.add(t);
    return;
  }
  double sR, cR;
  sincos(R, &sR, &cR);
  int o = 0;
  uint64_t p = 0;
  while (true) {
    double cx, cy, cz;
    pix_center_cam(o, p, cx, cy, cz);
    const double dot = u[0] * cx + u[1] * cy + u[2] * cz;
    const double cr = qp.cos_rho[o], sr = qp.sin_rho[o];
    // cos(R + rho_o) is a valid "outside" threshold only while R + rho_o < pi, cos(R - rho_o) a valid "inside" one only
    // while R - rho_o >= 0; encoded by the host as sin/cos of rho_o and checked here through the sign of sin(R +- rho_o).
    const double cos_sum = cR * cr - sR * sr, sin_sum = sR * cr + cR * sr;     // R + rho_o in (0, 2pi)
    const double cos_dif = cR * cr + sR * sr, sin_dif = sR * cr - cR * sr;     // R - rho_o in (-pi/2, pi)
    const bool outside = (sin_sum > 0.0) && (dot < cos_sum - kSlack);
    const bool inside = (sin_dif >= 0.0) && (dot >= cos_dif + kSlack);
    bool descend = false;
    if (!outside) {
      if (o <= kt) {
        if (inside) {
          const int sh = 2 * (kt - o);
          const int64_t t0 = (int64_t)(p << sh), t1 = (int64_t)((p + 1) << sh);
          for (int64_t t = t0; t < t1; ++t) sink.add(t);
        } else descend = true;
      } else {
        const int64_t tile = (int64_t)(p >> (2 * (o - kt)));
        if (tile != sink.last_tile) {
          if (inside && o < kq) sink.add(tile);
          else descend = true;
        }
      }
      if (descend && o == kq) {          // leaf: the defining predicate
        if (dot >= cR) sink.add((int64_t)(p >> (2 * (kq - kt))));
        descend = false;
      }
    }
    if (descend) { p <<= 2; ++o; continue; }
    while (o > 0 && (p & 3) == 3) { p >>= 2; --o; }
    ++p;
    if (o == 0 && p == 12) break;
  }
}

template <bool EMIT>
__global__ void __launch_bounds__(128)
tile_query_kernel(QueryParams qp, const float* __restrict__ dir, const float* __restrict__ rho, const float* __restrict__ rs,
                  const uint8_t* __restrict__ flags, const int32_t* __restrict__ slot_of_tile, uint32_t* __restrict__ counts,
                  const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const int64_t n = (int64_t)qp.P * qp.V;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  if (__ldg(flags + k) & 1) { if (!EMIT) counts[k] = 0; return; }
  if (EMIT && offsets[k + 1] == offsets[k]) return;
  const int v = (int)(k / qp.P);
  const uint32_t i = (uint32_t)(k - (int64_t)v * qp.P);
  double u[3] = {(double)__ldg(dir + 3 * k), (double)__ldg(dir + 3 * k + 1), (double)__ldg(dir + 3 * k + 2)};
  const double nrm = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
  u[0] /= nrm; u[1] /= nrm; u[2] /= nrm;
  const double R = fmin(kPi, (double)__ldg(rs + k) + qp.rho_q);
  Sink<EMIT> sink;
  sink.keys = keys; sink.vals = vals; sink.base = EMIT ? offsets[k] : 0;
  sink.key_hi_base = (uint64_t)v * (uint64_t)qp.n_tile;
  sink.depth_bits = __float_as_uint(__ldg(rho + k));                         // reading A10
  sink.gid = i; sink.slot_of_tile = slot_of_tile; sink.count = 0; sink.last_tile = -1;
  walk<EMIT>(qp, u, R, sink);
  if (!EMIT) counts[k] = sink.count;
}

}  // namespace uts

using namespace uts;

extern "C" {

size_t uts_tile_query_scratch_bytes(const uts_config* cfg) {
  if (check_config(cfg) != UTS_OK) return 0;
  const int64_t n = (int64_t)cfg->n_gauss * cfg->n_views;
  return (size_t)(((n * 4 + 255) / 256) * 256) + scan_scratch_bytes(n);
}

int uts_tile_query(const uts_config* cfg, uts_proj in, uts_mask mask, uint64_t* offsets, uint64_t* keys, uint32_t* vals,
                   uint64_t capacity, uint64_t* h_n_pairs, void* scratch, size_t scratch_bytes, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!offsets || !h_n_pairs) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  Dims d = dims_of(cfg, &mask);
  const int64_t n = (int64_t)d.P * d.V;
  if (n == 0) {                         // empty Gaussian set: no pairs, nothing else is read
    UTS_CUDA(cudaMemsetAsync(offsets, 0, sizeof(uint64_t), s));
    UTS_CUDA(cudaStreamSynchronize(s));
    *h_n_pairs = 0;
    return UTS_OK;
  }
  if (!in.dir || !in.rho || !in.rs || !in.flags || !scratch) return UTS_ERR_INVALID_ARG;
  if (keys && !vals) return UTS_ERR_INVALID_ARG;
  if (scratch_bytes < uts_tile_query_scratch_bytes(cfg) || ((uintptr_t)scratch & 255)) return UTS_ERR_INVALID_ARG;
  QueryParams qp;
  qp.kt = d.kt; qp.kq = d.kq; qp.P = d.P; qp.V = d.V; qp.n_tile = d.n_tile;
  const double* rm = rho_max_table_host();
  qp.rho_q = rm[d.kq];
  for (int o = 0; o <= kMaxOrder; ++o) { qp.cos_rho[o] = cos(rm[o]); qp.sin_rho[o] = sin(rm[o]); }
  uint32_t* counts = reinterpret_cast<uint32_t*>(scratch);
  uint64_t* block_sums = reinterpret_cast<uint64_t*>(reinterpret_cast<char*>(scratch) + ((n * 4 + 255) / 256) * 256);
  const unsigned qgrid = (unsigned)((n + 127) / 128);
  tile_query_kernel<false><<<qgrid, 128, 0, s>>>(qp, in.dir, in.rho, in.rs, in.flags, mask.slot_of_tile, counts, nullptr, nullptr, nullptr);
  UTS_LAUNCH_CHECK();
  if ((st = exclusive_scan_u32(counts, n, offsets, block_sums, s))) return st;
  UTS_CUDA(cudaMemcpyAsync(h_n_pairs, offsets + n, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
  UTS_CUDA(cudaStreamSynchronize(s));
  if (!keys) return UTS_OK;
  if (*h_n_pairs > capacity) return UTS_ERR_CAPACITY;
  if (*h_n_pairs == 0) return UTS_OK;
  tile_query_kernel<true><<<qgrid, 128, 0, s>>>(qp, in.dir, in.rho, in.rs, in.flags, mask.slot_of_tile, nullptr, offsets, keys, vals);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // extern "C"
