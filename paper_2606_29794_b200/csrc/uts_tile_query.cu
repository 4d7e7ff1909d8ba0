// uts_tile_query.cu — F2: NESTED-scheme tile query and pair emission (Alg.1 l.9-14 PAPER.md:548-559; Alg.2
// PAPER.md:599-620; §3.3; reading A6 for the garbled parts of Alg.2).
//
// Tile set of one projected Gaussian (direction u, radius r_s):
//     T = { q >> 2(k_q - k_t) : q an order-k_q pixel,  u . centre(q) >= cos R },   R = min(pi, r_s + rho_max(k_q)),
// intersected with the active tiles of the mask.  The defining predicate is evaluated in double precision.
//
// Differences from the paper's kernel (written for sm_89), see DESIGN.md "Kernels/F2":
//   * STACKLESS traversal.  The paper's DFS keeps an O(log Nside) stack per thread.  A NESTED index
//     IS its own path (child c of p is 4p+c), so "next node in depth-first order" is
//     `while ((p & 3) == 3) p >>= 2, --o;  ++p` — two registers, no local memory.
//   * Zone tests (Alg.2's Classify) run in single precision on CHORD lengths |u - c| against 2 sin((R +- rho_o)/2), with a
//     margin far above the fp32 error, and only prune / accept whole subtrees; the leaf test falls back to the double
//     precision dot product whenever it is within the margin, so the emitted set is exactly T.
//   * Two work shapes.  Small discs: one thread per Gaussian walks the tree.  Large discs (tens of thousands of tiles;
//     config 4's outliers own most of the pairs): one thread BLOCK per Gaussian classifies every order-o_s node in
//     parallel, walks the boundary subtrees from a shared work list, and records tiles in a shared-memory BITMAP over all
//     tiles.  The bitmap makes the result independent of visiting order, removes duplicates for free, and turns emission
//     into a rank query, so pairs come out in ascending tile order with fully coalesced stores.
//   * count -> exclusive scan -> emit: the pair arrays are written once, densely, in (view, Gaussian, tile) order.
#include "uts_internal.cuh"
#include "uts_scan.cuh"
#include "uts_ring_query.cuh"
#include "uts_window_query.cuh"
#include <cstring>

namespace uts {

constexpr float kDelta = 4e-6f;         // fp32 chord margin (chord error of the fp32 centres is below 1e-6)
constexpr int kLargeThreads = 256;
constexpr size_t kMaxLargeSmem = 200 * 1024;
constexpr int kTileCacheK = 16;         // tiles of a small disc remembered by the count pass (64 B per Gaussian)

struct QueryParams {
  int kt, kq, P, V;
  int os;                               // split order of the block-per-Gaussian path
  int n_words;                          // bitmap words = n_tile / 32 (0: block path disabled)
  int wl_cap;                           // capacity of each of the two block work lists
  int64_t n_tile;
  double rho_q;                         // rho_max(k_q) (NESTED set) or 0 (RING set): R = min(pi, r_s + rho_q)
  double rho_t;                         // rho_max(k_t)
  int w_max;                            // window class: largest half-width
  float r_large;                        // discs with R above this go to the block path
  uint32_t* tile_cache;                 // [V*P][kTileCacheK] tiles found by the count pass (thread path), reused by the emit pass
  uint32_t* bitmap_cache;               // [bitmap_cache_cap][n_words] bitmaps of the count pass (block path)
  uint32_t bitmap_cache_cap;
  float rho[kMaxOrder + 1], sin_hrho[kMaxOrder + 1], cos_hrho[kMaxOrder + 1];   // rho_max(o), sin/cos(rho_max(o)/2)
  // ring-interval path (uts_ring_query.cuh): discs are split by radius bucket into block / warp / thread work
  int b_block, b_warp;                  // buckets <= b_block: one block per disc; <= b_warp: one warp; others: one thread
  int rc_thread, rc_warp, rc_block;     // ring-table capacities of the three shapes
  const uint32_t* active_tiles; int n_active;   // mask's ascending active-tile list (whole-sphere discs), or null
  // row-mask cache of the block-per-disc shape: the count pass stores every (row, chunk) mask of a disc at
  // mask_cache[mask_base[k] ...], the emit pass replays them (no ring phase); a disc that does not fit is recomputed
  unsigned long long* mask_cache; uint32_t mask_cache_cap; uint32_t* mask_cursor; uint32_t* mask_base;
};

// Per-Gaussian query state.
struct Disc {
  double u[3]; double cosR;
  float uf[3]; float Rf, sh, ch;        // sin(R/2), cos(R/2)
  bool all;                             // R >= pi: every tile (reading A24)
};

__device__ __forceinline__ bool load_disc(const QueryParams& qp, const float* __restrict__ dir, const float* __restrict__ rs,
                                          int64_t k, Disc& D) {
  D.u[0] = (double)__ldg(dir + 3 * k); D.u[1] = (double)__ldg(dir + 3 * k + 1); D.u[2] = (double)__ldg(dir + 3 * k + 2);
  const double nrm = sqrt(D.u[0] * D.u[0] + D.u[1] * D.u[1] + D.u[2] * D.u[2]);
  D.u[0] /= nrm; D.u[1] /= nrm; D.u[2] /= nrm;
  const double R = fmin(kPi, (double)__ldg(rs + k) + qp.rho_q);
  D.all = R >= kPi;
  D.cosR = cos(R);
  double s, c;
  sincos(0.5 * R, &s, &c);
  D.uf[0] = (float)D.u[0]; D.uf[1] = (float)D.u[1]; D.uf[2] = (float)D.u[2];
  D.Rf = (float)R; D.sh = (float)s; D.ch = (float)c;
  return true;
}

enum Zone { kOutside = 0, kInside = 1, kPartial = 2 };

// Alg.2's Classify for node (o,p): kOutside = no descendant centre can be within R, kInside = all are.
__device__ __forceinline__ Zone classify(const QueryParams& qp, const Disc& D, int o, uint32_t p, float& chord) {
  float cx, cy, cz;
  pix_center_cam_f32(o, p, cx, cy, cz);
  const float dx = D.uf[0] - cx, dy = D.uf[1] - cy, dz = D.uf[2] - cz;
  chord = sqrtf(dx * dx + dy * dy + dz * dz);
  const float a = D.sh * qp.cos_hrho[o], b = D.ch * qp.sin_hrho[o];
  const float rho = qp.rho[o];
  if (D.Rf + rho < 3.1415f && chord > 2.0f * (a + b) + kDelta) return kOutside;
  if (D.Rf - rho > 1e-4f && chord < 2.0f * (a - b) - kDelta) return kInside;
  return kPartial;
}

// The defining predicate at a leaf (order k_q).
__device__ __forceinline__ bool leaf_inside(const QueryParams& qp, const Disc& D, uint32_t p, float chord) {
  const float t = 2.0f * D.sh;
  if (chord < t - kDelta) return true;
  if (chord > t + kDelta) return false;
  double cx, cy, cz;
  pix_center_cam(qp.kq, (uint64_t)p, cx, cy, cz);
  return D.u[0] * cx + D.u[1] * cy + D.u[2] * cz >= D.cosR;
}

__device__ __forceinline__ uint32_t spread_bits16(uint32_t v) {          // 16 bits -> even bit positions
  v &= 0xffffu;
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}

// A tile that the zone tests leave undecided: does any of its 4^(k_q-k_t) query pixels satisfy the defining predicate?
// Straight-line loop over the leaves with the face / tile decode shared (about 25 instructions per leaf, early exit), instead
// of walking two more quadtree levels node by node (measured: the leaf levels were most of the walk).
__device__ __forceinline__ bool any_leaf_inside(const QueryParams& qp, const Disc& D, uint32_t tile) {
  const int kt = qp.kt, kq = qp.kq, ref = kq - kt, m = 1 << ref;
  const int f = (int)(tile >> (2 * kt));
  const uint32_t mt = tile & ((1u << (2 * kt)) - 1u);
  const int x0 = (int)squeeze_even_bits32(mt) << ref, y0 = (int)squeeze_even_bits32(mt >> 1) << ref;
  const int N = 1 << kq, r = f >> 2, c = f & 3;
  const int base_i = (r + 2) * N - 1;                                     // ring = base_i - (x + y)
  const float Fc = (float)(2 * c + 1 - (r & 1));
  const float invN = __int_as_float((127 - kq) << 23);
  const float inv3N2 = 0.333333343f * invN * invN;
  const float T = 2.0f * D.sh;
  for (int dy = 0; dy < m; ++dy) {
    for (int dx = 0; dx < m; ++dx) {
      const int x = x0 + dx, y = y0 + dy;
      const int i = base_i - (x + y), h = x - y;
      float z, sth, q;
      if (i < N) { const float fn = (float)i; const float w = fn * fn * inv3N2; z = 1.0f - w; sth = sqrtf(w * (2.0f - w)); q = __fdividef((float)h, fn); }
      else if (i > 3 * N) { const float fn = (float)(4 * N - i); const float w = fn * fn * inv3N2; z = w - 1.0f; sth = sqrtf(w * (2.0f - w)); q = __fdividef((float)h, fn); }
      else { z = (float)(2 * (2 * N - i)) * (0.333333343f * invN); sth = sqrtf((1.0f - z) * (1.0f + z)); q = (float)h * invN; }
      q += Fc;
      if (q > 4.0f) q -= 8.0f;
      float sn, cs;
      __sincosf(q * 0.78539816339744831f, &sn, &cs);
      const float ex = D.uf[0] - sth * sn, ey = D.uf[1] - z, ez = D.uf[2] - sth * cs;
      const float chord = sqrtf(ex * ex + ey * ey + ez * ez);
      if (chord < T - kDelta) return true;
      if (chord <= T + kDelta) {                                          // inside the fp32 margin: the exact predicate decides
        const uint32_t p = ((uint32_t)f << (2 * kq)) | spread_bits16((uint32_t)x) | (spread_bits16((uint32_t)y) << 1);
        double cx, cy, cz;
        pix_center_cam(kq, (uint64_t)p, cx, cy, cz);
        if (D.u[0] * cx + D.u[1] * cy + D.u[2] * cz >= D.cosR) return true;
      }
    }
  }
  return false;
}

// Depth-first walk of the subtrees rooted at the order-ro nodes rp0..rp1 (inclusive), one node per step().
// Sink: add(tile), add_range(t0,t1), has(tile).  The climb after a finished subtree is a count of trailing 11 bit pairs,
// so a step has no data-dependent loop in its control path.  Callers drive step() from a WARP-SYNCHRONOUS loop
// (`while (__any_sync(full, running))`): every lane walks its own tree, and the vote makes the lanes reconverge at every
// node.  (Left to the compiler, the walk loop's reconvergence point was the loop exit: 2 of 32 lanes active, measured.)
struct Walker {
  int o, ro;
  uint32_t p, rp1;               // a NESTED index at order <= 13 fits 32 bits
  __device__ __forceinline__ void start(int ro_, uint32_t rp0, uint32_t rp1_) { o = ro = ro_; p = rp0; rp1 = rp1_; }
  // returns true when the walk is finished
  // LEAF_LOOP: undecided tiles are settled by any_leaf_inside (pays off in the block path, where idle lanes refill
  // themselves; in the thread-per-Gaussian path the long inner loop costs more in divergence than it saves: measured)
  template <bool LEAF_LOOP, class Sink>
  __device__ __forceinline__ bool step(const QueryParams& qp, const Disc& D, Sink& sink) {
    const int kt = qp.kt, kq = qp.kq;
    float chord;
    const Zone z = classify(qp, D, o, p, chord);
    bool descend = false;
    if (z != kOutside) {
      if (o <= kt) {
        if (z == kInside) { const int sh = 2 * (kt - o); sink.add_range((int64_t)p << sh, (int64_t)(p + 1) << sh); }
        else if (LEAF_LOOP && o == kt && kq > kt) { if (any_leaf_inside(qp, D, p)) sink.add((int64_t)p); }      // undecided tile: test its leaves
        else descend = true;
      } else {
        const int64_t tile = (int64_t)(p >> (2 * (o - kt)));
        if (!sink.has(tile)) {
          if (z == kInside && o < kq) sink.add(tile);
          else descend = true;
        }
      }
      if (descend && o == kq) {
        if (leaf_inside(qp, D, p, chord)) sink.add((int64_t)(p >> (2 * (kq - kt))));
        descend = false;
      }
    }
    bool finished = false;
    if (descend) { p <<= 2; ++o; }
    else {
      const int ones = __ffs((int)~p) - 1;              // trailing one bits of p
      const int up = min(ones >> 1, o - ro);                    // finished last children to climb over
      p >>= 2 * up; o -= up;
      if (o == ro && p == rp1) finished = true; else ++p;
    }
    return finished;
  }
};

// ------------------------------------------------------------------------------------- thread-per-Gaussian path
template <bool EMIT>
struct ThreadSink {
  uint64_t* keys; uint32_t* vals; uint64_t base; uint64_t key_hi_base; uint32_t depth_bits; uint32_t gid;
  const int32_t* slot_of_tile;
  uint32_t* cache;                       // count pass: this Gaussian's kTileCacheK-entry slot
  uint32_t count;
  int64_t last_tile;
  __device__ __forceinline__ bool has(int64_t tile) const { return tile == last_tile; }
  __device__ __forceinline__ void add(int64_t tile) {
    if (tile == last_tile) return;
    last_tile = tile;
    if (slot_of_tile && __ldg(slot_of_tile + tile) < 0) return;
    if (EMIT) {
      keys[base + count] = ((key_hi_base + (uint64_t)tile) << 32) | depth_bits;   // Alg.1 l.12: ((t, rho), i)
      vals[base + count] = gid;
    } else if (count < (uint32_t)kTileCacheK) cache[count] = (uint32_t)tile;
    ++count;
  }
  __device__ __forceinline__ void add_range(int64_t t0, int64_t t1) { for (int64_t t = t0; t < t1; ++t) add(t); }
};

// Work classes.  A thread-per-Gaussian walk is only efficient when the 32 lanes of a warp have similar amounts of work
// (measured: with Gaussians in input order 1.7 of 32 lanes were active on config 4).  So the count pass first buckets the
// Gaussians by disc radius (4 buckets per octave of R, largest first) into a permutation; thread t then walks perm[t].
constexpr int kBuckets = 64;

__device__ __forceinline__ int radius_bucket(float R32) {      // larger discs -> smaller bucket index
  const int e = (int)(__float_as_uint(R32) >> 21);               // exponent and two mantissa bits; R32 in (0, pi]
  const int top = (int)(__float_as_uint(4.0f) >> 21);
  return min(kBuckets - 1, max(0, top - e));
}

// which = 0: histogram of buckets (+ culled counts, + block-path list); which = 1: scatter into perm.
template <int WHICH>
__global__ void __launch_bounds__(256)
classify_kernel(QueryParams qp, const float* __restrict__ rs, const uint8_t* __restrict__ flags, uint32_t* __restrict__ counts,
                uint32_t* __restrict__ large_list, uint32_t* __restrict__ n_large, uint32_t* __restrict__ hist /*[64] counts, then cursors*/,
                uint32_t* __restrict__ perm, const uint32_t* __restrict__ emit_rank) {
  __shared__ uint32_t s_hist[kBuckets];
  if (threadIdx.x < kBuckets) s_hist[threadIdx.x] = 0;
  __syncthreads();
  const int64_t n = (int64_t)qp.P * qp.V;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int b = -1;
  if (k < n) {
    if (__ldg(flags + k) & 1) { if (WHICH == 0) counts[emit_rank ? emit_rank[k] : k] = 0; }
    else {
      const float R32 = fminf(3.14159274f, __ldg(rs + k) + (float)qp.rho_q);
      if (qp.n_words > 0 && R32 > qp.r_large) { if (WHICH == 0) large_list[atomicAdd(n_large, 1u)] = (uint32_t)k; }
      else b = radius_bucket(R32);
    }
  }
  uint32_t local = 0;
  if (b >= 0) local = atomicAdd(&s_hist[b], 1u);
  __syncthreads();
  if (WHICH == 0) {
    if (threadIdx.x < kBuckets && s_hist[threadIdx.x]) atomicAdd(hist + threadIdx.x, s_hist[threadIdx.x]);
  } else {
    __shared__ uint32_t s_base[kBuckets];
    if (threadIdx.x < kBuckets) s_base[threadIdx.x] = s_hist[threadIdx.x] ? atomicAdd(hist + threadIdx.x, s_hist[threadIdx.x]) : 0u;
    __syncthreads();
    if (b >= 0) perm[s_base[b] + local] = (uint32_t)k;
  }
}

// hist[64] counts -> exclusive start offsets (in place); n_small = total
// n_small[1], n_small[2]: ends of the block-per-disc and warp-per-disc parts of perm (ring-interval path)
// n_small[3]: end of the matrix class (uts_tile_lists): whole buckets <= b_mat while they fit cap_rows rows; 0 when b_mat < 0 or
// when the pairs those discs own (estimated from the bucket radii) would not pay for the per-(view, tile) bookkeeping of the
// matrix path (about 256 B per (view, tile) against about 90 B per pair saved)
// n_small[4]: start of the window class (uts_window_query.cuh): buckets >= b_fast, the smallest discs
__global__ void bucket_scan_kernel(uint32_t* __restrict__ hist, uint32_t* __restrict__ n_small, int b_block, int b_warp, int b_mat, int b_fast,
                                   uint32_t cap_rows, double n_tile, double nvt) {
  if (threadIdx.x == 0) {
    uint32_t run = 0, e_block = 0, e_warp = 0, e_mat = 0, e_fast = 0;
    double est_pairs = 0.0, est_at_mat = 0.0;
    const int top = (int)(__float_as_uint(4.0f) >> 21);
    for (int b = 0; b < kBuckets; ++b) {
      const uint32_t c = hist[b]; hist[b] = run; run += c;
      const float r_lo = fminf(3.14159274f, __uint_as_float((uint32_t)(top - b) << 21));     // smallest radius of bucket b
      est_pairs += (double)c * fmin(n_tile, 0.5 * n_tile * (1.0 - cos((double)r_lo)));
      if (b <= b_block) e_block = run;
      if (b <= b_warp) e_warp = run;
      if (b < b_fast) e_fast = run;
      if (b <= b_mat && run <= cap_rows) { e_mat = run; est_at_mat = est_pairs; }
    }
    if (est_at_mat * 90.0 < nvt * 256.0) e_mat = 0;
    n_small[0] = run; n_small[1] = e_block; n_small[2] = e_warp; n_small[3] = e_mat; n_small[4] = e_fast;
  }
}

template <bool EMIT>
__device__ __forceinline__ void
small_body(int64_t block, const QueryParams& qp, const float* __restrict__ dir, const float* __restrict__ rho, const float* __restrict__ rs,
                        const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small,
           const uint32_t* __restrict__ emit_rank,
                        uint32_t* __restrict__ counts, const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys,
                        uint32_t* __restrict__ vals) {
  const int64_t t = block * blockDim.x + threadIdx.x;
  bool running = t < (int64_t)*n_small;
  const int64_t k = running ? (int64_t)perm[t] : 0;
  const int64_t slot = emit_rank ? (int64_t)emit_rank[k] : k;     // position of this Gaussian in the emission order
  if (EMIT && running) {
    // the count pass left the tiles of discs with at most kTileCacheK tiles in tile_cache: emit them without walking
    const uint64_t b0 = offsets[slot], cnt = offsets[slot + 1] - b0;
    if (cnt <= (uint64_t)kTileCacheK) {
      const int v = (int)(k / qp.P);
      const uint64_t hi = (uint64_t)v * (uint64_t)qp.n_tile;
      const uint32_t depth = __float_as_uint(__ldg(rho + k)), gid = (uint32_t)(k - (int64_t)v * qp.P);
      const uint32_t* c = qp.tile_cache + (size_t)k * kTileCacheK;
      for (uint32_t j = 0; j < (uint32_t)cnt; ++j) { keys[b0 + j] = ((hi + c[j]) << 32) | depth; vals[b0 + j] = gid; }
      running = false;
    }
  }
  Disc D;
  ThreadSink<EMIT> sink;
  sink.cache = qp.tile_cache + (size_t)k * kTileCacheK;
  sink.count = 0; sink.last_tile = -1; sink.slot_of_tile = slot_of_tile; sink.keys = keys; sink.vals = vals;
  sink.base = 0; sink.key_hi_base = 0; sink.depth_bits = 0; sink.gid = 0;
  const bool valid = running;
  if (running) {
    load_disc(qp, dir, rs, k, D);
    const int v = (int)(k / qp.P);
    sink.base = EMIT ? offsets[slot] : 0;
    sink.key_hi_base = (uint64_t)v * (uint64_t)qp.n_tile;
    sink.depth_bits = __float_as_uint(__ldg(rho + k));                       // reading A10
    sink.gid = (uint32_t)(k - (int64_t)v * qp.P);
    if (D.all) { sink.add_range(0, qp.n_tile); running = false; }
  }
  Walker w;
  w.start(0, 0, 11);
  while (__any_sync(0xffffffffu, running)) {
    if (running) running = !w.step<false>(qp, D, sink);
  }
  if (!EMIT && valid) counts[slot] = sink.count;
}

// -------------------------------------------------------------------------------------- block-per-Gaussian path
struct BitmapSink {
  uint32_t* bits;
  __device__ __forceinline__ bool has(int64_t tile) const { return (bits[tile >> 5] >> (tile & 31)) & 1u; }
  __device__ __forceinline__ void add(int64_t tile) { atomicOr(bits + (tile >> 5), 1u << (tile & 31)); }
  __device__ __forceinline__ void add_range(int64_t t0, int64_t t1) {       // [t0,t1) is an aligned block of 4^j tiles
    if (t1 - t0 >= 32) { for (int64_t w = t0 >> 5; w < (t1 >> 5); ++w) bits[w] = 0xffffffffu; }
    else atomicOr(bits + (t0 >> 5), (uint32_t)((((uint64_t)1 << (t1 - t0)) - 1) << (t0 & 31)));
  }
};

__device__ __forceinline__ uint32_t block_sum_u32(uint32_t x, uint32_t* s_w /*[8]*/, uint32_t& before) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
  __syncthreads();
  if (lane == 31) s_w[wid] = incl;
  __syncthreads();
  uint32_t b = 0, total = 0;
#pragma unroll
  for (int w = 0; w < kLargeThreads / 32; ++w) { const uint32_t s = s_w[w]; if (w < wid) b += s; total += s; }
  before = b + incl - x;
  return total;
}

// active_words[w]: bit t set <=> tile 32w+t is active (built once per call from slot_of_tile)
__global__ void active_words_kernel(const int32_t* __restrict__ slot_of_tile, int n_words, uint32_t* __restrict__ active_words) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_words) return;
  uint32_t m = 0;
  for (int t = 0; t < 32; ++t) if (__ldg(slot_of_tile + 32 * (int64_t)w + t) >= 0) m |= 1u << t;
  active_words[w] = m;
}

template <bool EMIT>
__device__ __forceinline__ void
large_body(int n_blocks, const QueryParams& qp, const float* __restrict__ dir, const float* __restrict__ rho, const float* __restrict__ rs,
                        const uint32_t* __restrict__ active_words, const uint32_t* __restrict__ emit_rank, const uint32_t* __restrict__ large_list,
                        const uint32_t* __restrict__ n_large, uint32_t* __restrict__ counts, const uint64_t* __restrict__ offsets,
                        uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  extern __shared__ uint32_t smem[];
  uint32_t* bits = smem;                         // [n_words]
  uint32_t* pref = smem + qp.n_words;            // [n_words]  exclusive popcount prefix (emit only)
  uint32_t* work = smem + 2 * qp.n_words;        // [2][wl_cap] boundary nodes, ping-pong
  __shared__ Disc s_disc;
  __shared__ uint32_t s_count, s_next, s_w[kLargeThreads / 32];
  const int n_split = 12 << (2 * qp.os);
  const uint32_t nl = *n_large;
  for (uint32_t li = blockIdx.x; li < nl; li += (uint32_t)n_blocks) {
    const int64_t k = (int64_t)large_list[li];
    const bool cached = li < qp.bitmap_cache_cap;                 // the count pass kept this disc's (masked) bitmap
    uint32_t* cache_row = qp.bitmap_cache + (size_t)li * qp.n_words;
    __syncthreads();
    if (threadIdx.x == 0) { if (!(EMIT && cached)) load_disc(qp, dir, rs, k, s_disc); s_count = 0; s_next = 0; }
    for (int w = threadIdx.x; w < qp.n_words; w += kLargeThreads) bits[w] = (EMIT && cached) ? cache_row[w] : 0u;
    __syncthreads();
    const Disc D = s_disc;
    BitmapSink sink{bits};
    if (EMIT && cached) {
      // nothing to walk
    } else if (D.all) {
      for (int w = threadIdx.x; w < qp.n_words; w += kLargeThreads) bits[w] = 0xffffffffu;
    } else {
      for (int node = threadIdx.x; node < n_split; node += kLargeThreads) {
        float chord;
        const Zone z = classify(qp, D, qp.os, (uint32_t)node, chord);
        if (z == kInside) { const int sh = 2 * (qp.kt - qp.os); sink.add_range((int64_t)node << sh, (int64_t)(node + 1) << sh); }
        else if (z == kPartial) work[atomicAdd(&s_count, 1u)] = (uint32_t)node;
      }
      __syncthreads();
      // breadth-first refinement of the boundary nodes down to tile order while the next level fits the work list: turns a
      // few large subtrees into many small ones, so that all 256 lanes have walks of a few nodes each
      uint32_t* cur = work; uint32_t* nxt = work + qp.wl_cap;
      int level = qp.os;
      uint32_t nw = s_count;
      while (level < qp.kt && 4u * nw <= (uint32_t)qp.wl_cap && nw > 0) {
        __syncthreads();
        if (threadIdx.x == 0) s_count = 0;
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < 4u * nw; i += kLargeThreads) {
          const uint32_t child = 4u * cur[i >> 2] + (i & 3u);
          float chord;
          const Zone z = classify(qp, D, level + 1, child, chord);
          if (z == kInside) { const int sh = 2 * (qp.kt - level - 1); sink.add_range((int64_t)child << sh, (int64_t)(child + 1) << sh); }
          else if (z == kPartial) nxt[atomicAdd(&s_count, 1u)] = child;
        }
        __syncthreads();
        nw = s_count; ++level;
        uint32_t* t = cur; cur = nxt; nxt = t;
      }
      Walker w;
      bool active = false, exhausted = false;
      while (true) {                                  // every lane does one node per iteration and refills itself when idle
        if (!active && !exhausted) {
          const uint32_t i = atomicAdd(&s_next, 1u);
          if (i < nw) { w.start(level, cur[i], cur[i]); active = true; }
          else exhausted = true;
        }
        if (!__any_sync(0xffffffffu, active)) break;
        if (active) active = !w.step<true>(qp, D, sink);
      }
    }
    __syncthreads();
    // mask, then count / prefix: each thread owns a contiguous chunk of words
    const int chunk = (qp.n_words + kLargeThreads - 1) / kLargeThreads;
    const int w0 = min(qp.n_words, (int)threadIdx.x * chunk), w1 = min(qp.n_words, w0 + chunk);
    uint32_t mine = 0;
    for (int w = w0; w < w1; ++w) {
      uint32_t b = bits[w];
      if (active_words && !(EMIT && cached)) { b &= __ldg(active_words + w); bits[w] = b; }
      if (!EMIT && cached) cache_row[w] = b;
      mine += __popc(b);
    }
    uint32_t before;
    const uint32_t total = block_sum_u32(mine, s_w, before);
    const int64_t slot = emit_rank ? (int64_t)emit_rank[k] : k;
    if (!EMIT) { if (threadIdx.x == 0) counts[slot] = total; continue; }
    for (int w = w0; w < w1; ++w) { pref[w] = before; before += __popc(bits[w]); }
    __syncthreads();
    const int v = (int)(k / qp.P);
    const uint32_t gid = (uint32_t)(k - (int64_t)v * qp.P);
    const uint64_t base = offsets[slot], hi = (uint64_t)v * (uint64_t)qp.n_tile;
    const uint32_t depth = __float_as_uint(__ldg(rho + k));
    for (uint32_t r = threadIdx.x; r < total; r += kLargeThreads) {
      int lo = 0, hi_w = qp.n_words - 1;                       // largest w with pref[w] <= r
      while (lo < hi_w) { const int mid = (lo + hi_w + 1) >> 1; if (pref[mid] <= r) lo = mid; else hi_w = mid - 1; }
      const uint32_t bit = __fns(bits[lo], 0, (int)(r - pref[lo]) + 1);
      keys[base + r] = ((hi + (uint64_t)lo * 32 + bit) << 32) | depth;
      vals[base + r] = gid;
    }
  }
}

// One launch for both work shapes: the first n_large_blocks blocks run the block-per-Gaussian path (long, few), the others
// the thread-per-Gaussian path, so the two overlap instead of running back to back.
template <bool EMIT>
__global__ void __launch_bounds__(kLargeThreads)
tile_query_kernel(QueryParams qp, int n_large_blocks, const float* __restrict__ dir, const float* __restrict__ rho,
                  const float* __restrict__ rs, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ active_words,
                  const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small, const uint32_t* __restrict__ large_list,
                  const uint32_t* __restrict__ n_large, const uint32_t* __restrict__ emit_rank, uint32_t* __restrict__ counts,
                  const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  if ((int)blockIdx.x < n_large_blocks)
    large_body<EMIT>(n_large_blocks, qp, dir, rho, rs, active_words, emit_rank, large_list, n_large, counts, offsets, keys, vals);
  else
    small_body<EMIT>((int64_t)blockIdx.x - n_large_blocks, qp, dir, rho, rs, slot_of_tile, perm, n_small, emit_rank, counts, offsets, keys, vals);
}

// ================================================================================== ring-interval path
// (uts_ring_query.cuh)  Two work shapes over the radius-bucketed permutation `perm` (largest discs first):
//   perm[0, e_block)         one thread block per disc (ring table: every ring of the order);
//   perm[e_block, e_warp)    batches of kBatchB discs of up to rc_warp rings   } one block per batch; the rings of all discs of the
//   perm[e_warp, n_small)    batches of kBatchA discs of up to rc_thread rings } batch, then their tile rows, are FLATTENED over the
//                                                                                block's lanes, so that no lane waits for a longer disc.
// Phase 1 fills the ring tables in shared memory, phase 2 walks the (face, tile diagonal) rows, a lane per row.  A row's tiles
// are placed with a shared-memory cursor per disc, so the pairs of one Gaussian are contiguous but their order inside the
// segment is not fixed; the sort's result does not depend on it (a Gaussian's tiles are distinct: no two of its keys tie).

struct GroupTab {
  const int2* base; int i_lo;
  __device__ __forceinline__ void operator()(int i, int& f, int& l) const { const int2 v = base[i - i_lo]; f = v.x; l = v.y; }
};

__device__ __forceinline__ void load_ring_disc(const QueryParams& qp, const float* __restrict__ dir, const float* __restrict__ lonlat,
                                               const float* __restrict__ rs, int64_t k, RingDisc& D) {
  const float d[3] = {__ldg(dir + 3 * k), __ldg(dir + 3 * k + 1), __ldg(dir + 3 * k + 2)};
  make_ring_disc(qp.kq, d, __ldg(lonlat + 2 * k), __ldg(lonlat + 2 * k + 1), fmin(kPi, (double)__ldg(rs + k) + qp.rho_q), D);
}

// Tiles of one 64-candidate chunk of a row.  Returns how many are active; with VISIT, fn(tile) is called for each.
// X = (S - Hm)/2 + j, Y = (S + Hm)/2 - j: the interleaved bits are stepped along the row, not recomputed.
template <bool VISIT, class Fn>
__device__ __forceinline__ uint32_t visit_row_chunk(int kt, int f, int S, int jbase, unsigned long long mask, const int32_t* __restrict__ slot_of_tile, Fn&& fn) {
  if (!VISIT && !slot_of_tile) return (uint32_t)__popcll(mask);
  const int Nt = 1 << kt, Hm = min(S, 2 * Nt - 2 - S);
  const uint32_t fbase = (uint32_t)f << (2 * kt);
  const int j0 = __ffsll((long long)mask) - 1, j1 = 63 - __clzll((long long)mask);
  uint32_t sX = spread_bits16_hd((uint32_t)(((S - Hm) >> 1) + jbase + j0));
  uint32_t sY = spread_bits16_hd((uint32_t)(((S + Hm) >> 1) - jbase - j0)) << 1;
  uint32_t cnt = 0;
  for (int j = j0; j <= j1; ++j) {
    if ((mask >> j) & 1ull) {
      const uint32_t tile = fbase | sX | sY;
      if (!slot_of_tile || __ldg(slot_of_tile + tile) >= 0) { if (VISIT) fn(tile); ++cnt; }
    }
    sX = ((sX | 0xAAAAAAAAu) + 1u) & 0x55555555u;
    sY = (sY - 2u) & 0xAAAAAAAAu;
  }
  return cnt;
}

// the chunk's mask restricted to active tiles
__device__ __forceinline__ unsigned long long filter_row_chunk(int kt, int f, int S, int jbase, unsigned long long mask, const int32_t* __restrict__ slot_of_tile) {
  if (!slot_of_tile || !mask) return mask;
  unsigned long long out = 0;
  int j = __ffsll((long long)mask) - 1;
  visit_row_chunk<true>(kt, f, S, jbase, mask, nullptr, [&](uint32_t tile) {
    while (!((mask >> j) & 1ull)) ++j;
    if (__ldg(slot_of_tile + tile) >= 0) out |= 1ull << j;
    ++j;
  });
  return out;
}

// position of the r-th (0-based) set bit of mask
__device__ __forceinline__ int nth_set_bit(unsigned long long mask, int r) {
  const int j0 = __ffsll((long long)mask) - 1;
  const unsigned long long run = mask >> j0;
  if ((run & (run + 1ull)) == 0ull) return j0 + r;                      // one contiguous run (the usual case)
  const uint32_t lo = (uint32_t)mask, hi = (uint32_t)(mask >> 32);
  const int nlo = __popc(lo);
  return r < nlo ? (int)__fns(lo, 0, r + 1) : 32 + (int)__fns(hi, 0, r - nlo + 1);
}

// rows of a disc: face f owns rows [pre[f], pre[f+1]) of the flat enumeration, S = S_lo(f) + (row - pre[f])
__device__ __forceinline__ int disc_face_rows(const QueryParams& qp, const RingDisc& D, uint16_t* pre /*[13]*/) {
  int run = 0;
  for (int f = 0; f < 12; ++f) {
    pre[f] = (uint16_t)run;
    if (!face_in_extent(D, f)) continue;
    int S_lo, S_hi;
    face_row_range(D, qp.kq, qp.kt, f, S_lo, S_hi);
    if (S_hi >= S_lo) run += S_hi - S_lo + 1;
  }
  pre[12] = (uint16_t)run;
  return run;
}

// ---------------------------------------------------------------------------------------------- batch of small discs
struct BatchRec {
  RingDisc D;
  uint64_t hi, base;          // key high part of the view; first pair of the Gaussian (emit)
  uint32_t depth, gid, slot, k;
  uint32_t cached;            // emit: the count pass left the tiles in tile_cache
  uint32_t mbase;             // first row mask of this disc in mask_cache, or 0xffffffff
  uint32_t skip;              // no rows to walk (no tiles, replayed from tile_cache, or a whole-sphere disc)
};

template <int G, bool EMIT>
__global__ void __launch_bounds__(kLargeThreads, 4)
ring_query_batch_kernel(QueryParams qp, int which /*0: rc_warp class, 1: rc_thread class*/, const float* __restrict__ dir, const float* __restrict__ lonlat,
                        const float* __restrict__ rho, const float* __restrict__ rs, const int32_t* __restrict__ slot_of_tile,
                        const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small, const uint32_t* __restrict__ emit_rank,
                        uint32_t* __restrict__ counts, const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ uint32_t s_w[kLargeThreads / 32];
  __shared__ int ring_off[G + 1], row_off[G + 1];
  __shared__ uint32_t cursor[G];
  __shared__ uint32_t s_bbase;
  __shared__ uint16_t rowpre[G][13];
  BatchRec* rec = reinterpret_cast<BatchRec*>(smem_raw);
  int2* tab = reinterpret_cast<int2*>(smem_raw + sizeof(BatchRec) * G);
  const int rc = which == 0 ? qp.rc_warp : qp.rc_thread;
  const uint32_t begin = which == 0 ? n_small[1] : n_small[2], end = which == 0 ? n_small[2] : n_small[4];      // [n_small[4], n_small[0]): window class
  const int N = 1 << qp.kq, tid = threadIdx.x;
  for (uint32_t b0 = begin + blockIdx.x * G; b0 < end; b0 += gridDim.x * G) {
    const int ng = min((uint32_t)G, end - b0);
    __syncthreads();                                   // the previous batch is done with shared memory
    // ---- records
    uint32_t my_rings = 0;
    if (tid < ng) {
      BatchRec& r = rec[tid];
      const int64_t k = (int64_t)perm[b0 + tid];
      const int64_t slot = emit_rank ? (int64_t)emit_rank[k] : k;
      const int v = (int)(k / qp.P);
      r.k = (uint32_t)k; r.slot = (uint32_t)slot;
      r.hi = (uint64_t)v * (uint64_t)qp.n_tile;
      r.depth = __float_as_uint(__ldg(rho + k)); r.gid = (uint32_t)(k - (int64_t)v * qp.P);           // reading A10
      r.cached = 0; r.base = 0;
      cursor[tid] = 0;
      bool skip = false;
      if (EMIT) {
        r.base = offsets[slot];
        const uint64_t cnt = offsets[slot + 1] - r.base;
        if (cnt == 0) skip = true;
        else if (cnt <= (uint64_t)kTileCacheK) { r.cached = (uint32_t)cnt; skip = true; }
      }
      if (EMIT && skip) r.D.all = false;               // no pairs, or replayed from tile_cache: the disc itself is not needed
      else {
        load_ring_disc(qp, dir, lonlat, rs, k, r.D);
        if (r.D.all) skip = true;                      // handled after the row loop
        r.D.i_hi = min(r.D.i_hi, r.D.i_lo + rc - 1);
      }
      r.skip = skip ? 1u : 0u;
      r.mbase = (EMIT && !skip) ? qp.mask_base[k] : 0xffffffffu;          // emit: the count pass kept this disc's row masks
      if (!skip && r.mbase == 0xffffffffu) my_rings = (uint32_t)(r.D.i_hi - r.D.i_lo + 1);
    }
    uint32_t before;
    const uint32_t n_rings = block_sum_u32(my_rings, s_w, before);
    if (tid < ng) ring_off[tid] = (int)before;
    if (tid == 0) ring_off[ng] = (int)n_rings;
    __syncthreads();
    // ---- phase 1, flattened over (disc, ring)
    for (uint32_t it = tid; it < n_rings; it += kLargeThreads) {
      int lo = 0, hi = ng;                             // largest g with ring_off[g] <= it
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if ((uint32_t)ring_off[mid] <= it) lo = mid; else hi = mid; }
      const RingDisc& D = rec[lo].D;
      int2 fl;
      ring_interval(D, N, D.i_lo + (int)(it - (uint32_t)ring_off[lo]), fl.x, fl.y);
      tab[it] = fl;
    }
    // ---- rows of every disc
    uint32_t my_rows = 0;
    if (tid < ng && !rec[tid].skip) my_rows = (uint32_t)disc_face_rows(qp, rec[tid].D, rowpre[tid]);
    const uint32_t n_rows = block_sum_u32(my_rows, s_w, before);
    const int n_chunks = ((1 << qp.kt) + 63) >> 6;     // 64-candidate chunks per row
    if (tid < ng) row_off[tid] = (int)before;
    if (tid == 0) {
      row_off[ng] = (int)n_rows;
      if (!EMIT) {                                     // claim room for the batch's row masks
        const uint32_t n_it = n_rows * (uint32_t)n_chunks;
        uint32_t at = atomicAdd(qp.mask_cursor, n_it);
        if (at > qp.mask_cache_cap || n_it > qp.mask_cache_cap - at) at = 0xffffffffu;
        s_bbase = at;
      }
    }
    __syncthreads();
    if (!EMIT && tid < ng && !rec[tid].skip) {
      rec[tid].mbase = s_bbase == 0xffffffffu ? 0xffffffffu : s_bbase + (uint32_t)row_off[tid] * (uint32_t)n_chunks;
      qp.mask_base[rec[tid].k] = rec[tid].mbase;
    }
    __syncthreads();
    // ---- phase 2, flattened over (disc, row)
    for (uint32_t it = tid; it < n_rows; it += kLargeThreads) {
      int lo = 0, hi = ng;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if ((uint32_t)row_off[mid] <= it) lo = mid; else hi = mid; }
      const BatchRec& r = rec[lo];
      const int row = (int)(it - (uint32_t)row_off[lo]);
      int f = 0;
      while (f < 11 && (int)rowpre[lo][f + 1] <= row) ++f;
      int S_lo, S_hi;
      face_row_range(r.D, qp.kq, qp.kt, f, S_lo, S_hi);
      const int S = S_lo + row - (int)rowpre[lo][f], Hm = min(S, (2 << qp.kt) - 2 - S);
      const GroupTab T{tab + ring_off[lo], r.D.i_lo};
      for (int jbase = 0; jbase <= Hm; jbase += 64) {
        const size_t mi = (size_t)r.mbase + (size_t)row * n_chunks + (size_t)(jbase >> 6);
        unsigned long long mask;
        if (EMIT && r.mbase != 0xffffffffu) mask = qp.mask_cache[mi];
        else {
          mask = filter_row_chunk(qp.kt, f, S, jbase, tile_row_mask(r.D, qp.kq, qp.kt, f, S, jbase, T), slot_of_tile);
          if (!EMIT && r.mbase != 0xffffffffu) qp.mask_cache[mi] = mask;
        }
        if (!mask) continue;
        const uint32_t c = (uint32_t)__popcll(mask);
        if (EMIT) {
          uint64_t pos = r.base + atomicAdd(&cursor[lo], c);
          visit_row_chunk<true>(qp.kt, f, S, jbase, mask, nullptr, [&](uint32_t tile) {
            keys[pos] = ((r.hi + tile) << 32) | r.depth; vals[pos] = r.gid; ++pos;            // Alg.1 l.12: ((t, rho), i)
          });
        } else {
          uint32_t pos = atomicAdd(&cursor[lo], c);
          if (pos < (uint32_t)kTileCacheK) {           // remember the first tiles: the emit pass replays discs of <= kTileCacheK tiles
            uint32_t* cache = qp.tile_cache + (size_t)r.k * kTileCacheK;
            visit_row_chunk<true>(qp.kt, f, S, jbase, mask, nullptr, [&](uint32_t tile) { if (pos < (uint32_t)kTileCacheK) cache[pos] = tile; ++pos; });
          }
        }
      }
    }
    __syncthreads();
    // ---- results, cached discs, whole-sphere discs
    if (tid < ng) {
      const BatchRec& r = rec[tid];
      if (r.D.all) {
        const uint32_t total = qp.active_tiles ? (uint32_t)qp.n_active : (uint32_t)qp.n_tile;
        if (!EMIT) counts[r.slot] = total;
        else if (!r.cached && offsets[r.slot + 1] != r.base)
          for (uint32_t j = 0; j < total; ++j) { const uint32_t tile = qp.active_tiles ? __ldg(qp.active_tiles + j) : j; keys[r.base + j] = ((r.hi + tile) << 32) | r.depth; vals[r.base + j] = r.gid; }
        if (!EMIT && total <= (uint32_t)kTileCacheK) {
          uint32_t* cache = qp.tile_cache + (size_t)r.k * kTileCacheK;
          for (uint32_t j = 0; j < total; ++j) cache[j] = qp.active_tiles ? __ldg(qp.active_tiles + j) : j;
        }
      } else if (!EMIT) counts[r.slot] = cursor[tid];
      if (EMIT && r.cached) {
        const uint32_t* cache = qp.tile_cache + (size_t)r.k * kTileCacheK;
        for (uint32_t j = 0; j < r.cached; ++j) { keys[r.base + j] = ((r.hi + cache[j]) << 32) | r.depth; vals[r.base + j] = r.gid; }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- one block per large disc
template <bool EMIT>
__global__ void __launch_bounds__(kLargeThreads, 4)
ring_query_block_kernel(QueryParams qp, const float* __restrict__ dir, const float* __restrict__ lonlat, const float* __restrict__ rho,
                        const float* __restrict__ rs, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ perm,
                        const uint32_t* __restrict__ n_small, const uint32_t* __restrict__ emit_rank, uint32_t* __restrict__ counts,
                        const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  extern __shared__ int2 ring_tab[];                 // [rc_block]
  __shared__ RingDisc s_disc;
  __shared__ uint16_t s_pre[13];
  __shared__ int s_Slo[12];
  __shared__ uint32_t s_cursor, s_mbase;
  __shared__ unsigned long long s_em_mask[kLargeThreads / 32][32];
  __shared__ uint32_t s_em_pre[kLargeThreads / 32][33], s_em_row[kLargeThreads / 32][32];
  const uint32_t end = n_small[1];
  const int N = 1 << qp.kq, tid = threadIdx.x;
  for (uint32_t idx = n_small[3] + blockIdx.x; idx < end; idx += gridDim.x) {        // discs before n_small[3] are uts_tile_lists' matrix rows
    const int64_t k = (int64_t)perm[idx];
    const int64_t slot = emit_rank ? (int64_t)emit_rank[k] : k;
    uint64_t b0 = 0;
    if (EMIT) { b0 = offsets[slot]; if (offsets[slot + 1] == b0) continue; }
    const int v = (int)(k / qp.P);
    const uint64_t hi = (uint64_t)v * (uint64_t)qp.n_tile;
    const uint32_t depth = __float_as_uint(__ldg(rho + k)), gid = (uint32_t)(k - (int64_t)v * qp.P);
    __syncthreads();                                   // the previous disc is done with shared memory
    if (tid == 0) {
      load_ring_disc(qp, dir, lonlat, rs, k, s_disc);
      s_disc.i_hi = min(s_disc.i_hi, s_disc.i_lo + qp.rc_block - 1);
      disc_face_rows(qp, s_disc, s_pre);
      for (int f = 0; f < 12; ++f) { int S_lo, S_hi; face_row_range(s_disc, qp.kq, qp.kt, f, S_lo, S_hi); s_Slo[f] = S_lo; }
      s_cursor = 0;
      const uint32_t n_it = (uint32_t)s_pre[12] * (uint32_t)(((1 << qp.kt) + 63) >> 6);
      if (s_disc.all) s_mbase = 0xffffffffu;
      else if (!EMIT) {                                // claim room for this disc's row masks
        uint32_t at = atomicAdd(qp.mask_cursor, n_it);
        if (at > qp.mask_cache_cap || n_it > qp.mask_cache_cap - at) at = 0xffffffffu;
        qp.mask_base[k] = at; s_mbase = at;
      } else s_mbase = qp.mask_base[k];
    }
    __syncthreads();
    const RingDisc& D = s_disc;
    if (D.all) {                                       // reading A24: every active tile
      const uint32_t total = qp.active_tiles ? (uint32_t)qp.n_active : (uint32_t)qp.n_tile;
      if (!EMIT) { if (tid == 0) counts[slot] = total; }
      else for (uint32_t j = tid; j < total; j += kLargeThreads) {
        const uint32_t tile = qp.active_tiles ? __ldg(qp.active_tiles + j) : j;
        keys[b0 + j] = ((hi + tile) << 32) | depth; vals[b0 + j] = gid;
      }
      continue;
    }
    const bool cached = s_mbase != 0xffffffffu;
    unsigned long long* mcache = qp.mask_cache + (cached ? (size_t)s_mbase : 0);
    if (!(EMIT && cached)) {                           // phase 1 (the emit pass skips it when the masks were kept)
      for (int e = tid; e <= D.i_hi - D.i_lo; e += kLargeThreads) { int2 fl; ring_interval(D, N, D.i_lo + e, fl.x, fl.y); ring_tab[e] = fl; }
      __syncthreads();
    }
    const GroupTab T{ring_tab, D.i_lo};
    const int n_rows = (int)s_pre[12];
    const int n_chunks = ((1 << qp.kt) + 63) >> 6;                         // chunks per row (a row has at most 2^kt tiles)
    const int n_items = n_rows * n_chunks;
    // the active-tile mask of item = (row, 64-candidate chunk)
    auto item_mask = [&](int item, int& f, int& S, int& jbase) -> unsigned long long {
      const int row = item / n_chunks;
      jbase = (item - row * n_chunks) << 6;
      f = 0;
      while (f < 11 && (int)s_pre[f + 1] <= row) ++f;
      S = s_Slo[f] + row - (int)s_pre[f];
      if (EMIT && cached) return mcache[item];
      if (jbase > min(S, (2 << qp.kt) - 2 - S)) return 0ull;
      return filter_row_chunk(qp.kt, f, S, jbase, tile_row_mask(D, qp.kq, qp.kt, f, S, jbase, T), slot_of_tile);
    };
    if (!EMIT) {
      uint32_t mine = 0;
      for (int item = tid; item < n_items; item += kLargeThreads) {
        int f, S, jbase;
        const unsigned long long mask = item_mask(item, f, S, jbase);
        if (cached) mcache[item] = mask;
        mine += (uint32_t)__popcll(mask);
      }
      if (mine) atomicAdd(&s_cursor, mine);
    } else {
      // Each lane settles one (row, chunk); the warp then writes the tiles of its 32 chunks as ONE contiguous run of pairs
      // (lane p takes the p-th tile of the run), so the stores are coalesced.
      const int lane = tid & 31, wid = tid >> 5;
      const int n_rounds = (n_items + kLargeThreads - 1) / kLargeThreads;
      for (int round = 0; round < n_rounds; ++round) {
        const int item = round * kLargeThreads + tid;
        unsigned long long mask = 0;
        int f = 0, S = 0, jbase = 0;
        if (item < n_items) mask = item_mask(item, f, S, jbase);
        const uint32_t c = (uint32_t)__popcll(mask);
        uint32_t incl = c;
#pragma unroll
        for (int dd = 1; dd < 32; dd <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, dd); if (lane >= dd) incl += y; }
        const uint32_t wtotal = __shfl_sync(0xffffffffu, incl, 31);
        if (wtotal == 0) continue;
        uint32_t wbase = 0;
        if (lane == 0) wbase = atomicAdd(&s_cursor, wtotal);
        wbase = __shfl_sync(0xffffffffu, wbase, 0);
        __syncwarp();
        {
          const int Hm = min(S, (2 << qp.kt) - 2 - S);
          s_em_mask[wid][lane] = mask;
          s_em_pre[wid][lane] = incl - c;
          if (lane == 31) s_em_pre[wid][32] = wtotal;
          s_em_row[wid][lane] = ((uint32_t)f << 24) | ((uint32_t)(((S - Hm) >> 1) + jbase) << 12) | (uint32_t)(((S + Hm) >> 1) - jbase);   // f, X0, Y0
        }
        __syncwarp();
        int lo = 0, hi2 = 32;                                              // owner of pair `lane`: last chunk whose exclusive prefix is <= it
        while (hi2 - lo > 1) { const int mid = (lo + hi2) >> 1; if (s_em_pre[wid][mid] <= (uint32_t)lane) lo = mid; else hi2 = mid; }
        for (uint32_t pp = lane; pp < wtotal; pp += 32) {
          while (s_em_pre[wid][lo + 1] <= pp) ++lo;                        // owners are monotone in pp; skips empty chunks
          const unsigned long long mk = s_em_mask[wid][lo];
          const uint32_t rw = s_em_row[wid][lo];
          const int j = nth_set_bit(mk, (int)(pp - s_em_pre[wid][lo]));
          const uint32_t tile = ((rw >> 24) << (2 * qp.kt)) | spread_bits16_hd(((rw >> 12) & 0xfffu) + (uint32_t)j) |
                                (spread_bits16_hd((rw & 0xfffu) - (uint32_t)j) << 1);
          keys[b0 + wbase + pp] = ((hi + tile) << 32) | depth;            // Alg.1 l.12: ((t, rho), i)
          vals[b0 + wbase + pp] = gid;
        }
      }
    }
    __syncthreads();
    if (!EMIT && tid == 0) counts[slot] = s_cursor;
  }
}

// ---------------------------------------------------------------------------------------------- window class: the smallest discs
// perm[n_small[4], n_small[0]): one thread per disc (uts_window_query.cuh); neighbouring threads hold discs of the same radius
// bucket, so their windows have the same size.  The count pass remembers up to kTileCacheK tiles per disc, the emit pass replays
// them (a 7 x 7 window can hold more: such a disc is queried again).
constexpr int kWindowThreads = 128;
template <bool EMIT>
__global__ void __launch_bounds__(kWindowThreads)
window_query_kernel(QueryParams qp, const float* __restrict__ dir, const float* __restrict__ rho, const float* __restrict__ rs,
                    const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small,
                    const uint32_t* __restrict__ emit_rank, uint32_t* __restrict__ counts, const uint64_t* __restrict__ offsets,
                    uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const uint64_t idx = (uint64_t)n_small[4] + (uint64_t)blockIdx.x * kWindowThreads + threadIdx.x;
  if (idx >= (uint64_t)n_small[0]) return;
  const int64_t k = (int64_t)perm[idx];
  const int64_t slot = emit_rank ? (int64_t)emit_rank[k] : k;
  const int v = (int)(k / qp.P);
  const uint64_t hi = (uint64_t)v * (uint64_t)qp.n_tile;
  const uint32_t depth = __float_as_uint(__ldg(rho + k)), gid = (uint32_t)(k - (int64_t)v * qp.P);           // reading A10
  uint32_t* cache = qp.tile_cache + (size_t)k * kTileCacheK;
  uint64_t b0 = 0;
  if (EMIT) {
    b0 = offsets[slot];
    const uint64_t cnt = offsets[slot + 1] - b0;
    if (cnt == 0) return;
    if (cnt <= (uint64_t)kTileCacheK) {
      for (uint32_t j = 0; j < (uint32_t)cnt; ++j) { keys[b0 + j] = ((hi + cache[j]) << 32) | depth; vals[b0 + j] = gid; }   // Alg.1 l.12: ((t, rho), i)
      return;
    }
  }
  const float d[3] = {__ldg(dir + 3 * k), __ldg(dir + 3 * k + 1), __ldg(dir + 3 * k + 2)};
  WindowDisc D;
  make_window_disc(qp.kt, d, fmin(kPi, (double)__ldg(rs + k) + qp.rho_q), qp.rho_t, D);
  D.w = min(D.w, qp.w_max);               // the class holds R <= 0.98 (1 - 1e-6) kWindowWidth w_max / N_t: a last-ulp excess stays inside the margin
  uint32_t pos = 0;
  window_query(D, qp.kt, qp.kq, slot_of_tile, [&](uint32_t tile) {
    if (EMIT) { keys[b0 + pos] = ((hi + tile) << 32) | depth; vals[b0 + pos] = gid; }
    else if (pos < (uint32_t)kTileCacheK) cache[pos] = tile;
    ++pos;
  });
  if (!EMIT) counts[slot] = pos;
}

}  // namespace uts

#include "uts_tile_matrix.cuh"

using namespace uts;

namespace {
inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int radius_bucket_host(float R32) {                    // host replica of radius_bucket()
  uint32_t u, t; const float four = 4.0f;
  memcpy(&u, &R32, 4); memcpy(&t, &four, 4);
  const int b = (int)(t >> 21) - (int)(u >> 21);
  return b < 0 ? 0 : (b > kBuckets - 1 ? kBuckets - 1 : b);
}
// The three shapes of the ring path are independent: they run side by side on the device context's two auxiliary streams, forked
// from and joined back to the caller's stream with events, so the caller still sees one ordered stream.  ctx->mu is held from
// the fork to the join (QueryRun::count / emit), so two callers never interleave their records of the shared events.
#ifndef UTS_RING_WARP_RINGS
#define UTS_RING_WARP_RINGS 128
#endif
constexpr int kRingThreadRings = 24, kRingWarpRings = UTS_RING_WARP_RINGS, kRingBlockRingsMax = 24575;   // ring-table capacities (8 B per ring)

struct QueryLayout { size_t counts, list, perm, nlarge, active, scan, tcache, bcache, bcache_bytes, total; uint32_t bcache_cap; };
QueryLayout query_layout(const uts_config* cfg) {
  const size_t n = (size_t)cfg->n_gauss * cfg->n_views;
  const size_t n_tile = (size_t)12 << (2 * (cfg->order - cfg->tile_log2));
  QueryLayout L;
  size_t off = 0;
  L.counts = off; off += align256(n * 4);
  L.list = off;   off += align256(n * 4);
  L.perm = off;   off += align256(n * 4);
  L.nlarge = off; off += 512;      // n_large, n_small, 64 bucket counters
  L.active = off; off += align256((n_tile / 32 + 1) * 4);
  L.scan = off;   off += scan_scratch_bytes((int64_t)n);
  L.tcache = off; off += align256(n * kTileCacheK * 4);
  // bitmap cache of the block path: as many discs as fit 384 MB (config 4: 65 536 bitmaps of 6 KB)
  const size_t row = (n_tile / 32) * 4;
  size_t cap = row ? (size_t)(384u << 20) / row : 0;
  if (cap > n) cap = n;
  if (n_tile < 192 || row * 2 + 4096 * 8 > kMaxLargeSmem) cap = 0;
  L.bcache_cap = (uint32_t)cap;
  // at least 64 B per (view, Gaussian), at most 384 MB: the ring path keeps its row masks here
  size_t bytes = cap * row;
  const size_t want = n * 64 < (size_t)(384u << 20) ? n * 64 : (size_t)(384u << 20);
  if (bytes < want) bytes = want;
  L.bcache_bytes = bytes;
  L.bcache = off; off += align256(bytes);
  L.total = off + 256;
  return L;
}
// Scratch of the matrix path (uts_tile_lists), appended after the query's own scratch.
struct MatLayout { size_t flag, rank_scan, scan, M, MT, row_key, views, large, loff, total, start, sranges, offsets, misc, total_bytes; uint32_t cap_rows; size_t mt_words; };
MatLayout mat_layout(const uts_config* cfg, size_t base) {
  const size_t n = (size_t)cfg->n_gauss * cfg->n_views;
  const size_t n_tile = (size_t)12 << (2 * (cfg->order - cfg->tile_log2));
  const size_t nvt = n_tile * (size_t)cfg->n_views;
  const size_t n_words = n_tile / 32;
  MatLayout L;
  size_t cap = n_words ? ((size_t)1 << 30) / (n_words * 4) : 0;         // bitmap rows that fit 1 GB
  if (cap > n) cap = n;
  if (cap > 0xfffffff0u) cap = 0xfffffff0u;
  L.cap_rows = (uint32_t)cap;
  L.mt_words = n_tile * (((cap + 255) / 256 + (size_t)cfg->n_views) * 8);  // sum over views of n_tile * W_v
  size_t off = base;
  L.flag = off;      off += align256(n * 4);
  L.rank_scan = off; off += align256((n + 1) * 8);
  L.scan = off;      off += scan_scratch_bytes((int64_t)(n > nvt ? n : nvt));
  L.M = off;         off += align256(cap * n_words * 4);
  L.MT = off;        off += align256(L.mt_words * 4);
  L.row_key = off;   off += align256((cap + 1024) * 8);
  L.views = off;     off += align256((size_t)cfg->n_views * sizeof(MatView));
  L.large = off;     off += align256(nvt * 4);
  L.loff = off;      off += align256((nvt + 1) * 8);
  L.total = off;     off += align256(nvt * 4);
  L.start = off;     off += align256((nvt + 1) * 8);
  L.sranges = off;   off += align256(nvt * 16);
  L.offsets = off;   off += align256((n + 1) * 8);
  L.misc = off;      off += 256;
  L.total_bytes = off + 256;
  return L;
}

// three device words -> three consecutive words (a null source reads as 0)
__global__ void gather3_kernel(const uint64_t* a, const uint64_t* b, const uint64_t* c, unsigned long long* out) {
  out[0] = a ? *a : 0ull; out[1] = b ? *b : 0ull; out[2] = c ? *c : 0ull;
}

// One tile query on the ring-interval path (or the quadtree descent): host-side parameters, then count() and emit().
struct QueryRun {
  const uts_config* cfg; uts_proj in; uts_mask mask; const uint32_t* emit_rank; cudaStream_t s;
  Dims d; int64_t n;
  QueryParams qp;
  bool ring_impl, use_large;
  bool side_forked = false;          // count() put the matrix class on ctx->side: the caller joins
  uint32_t *counts, *list, *n_large, *n_small, *hist, *perm, *active;
  uint64_t* block_sums;
  const uint32_t* active_arg;
  unsigned qgrid; int lgrid; size_t dyn_smem;
  size_t smem_a, smem_b, smem_block;
  unsigned agrid, wgrid, bgrid, agrid_e, wgrid_e, bgrid_e;
  static constexpr int kBatchA = 128, kBatchB = 32;          // discs per batch: rc_thread class, rc_warp class
  int b_mat; uint32_t cap_rows;                              // matrix class of uts_tile_lists (b_mat < 0: none)
  int b_fast;                                                // window class: radius buckets >= b_fast (kBuckets: none)
  DeviceCtx* ctx;
  enum { kOccBlock0 = 1, kOccBlock1, kOccB0, kOccB1, kOccA0, kOccA1, kOccMat };

  int setup(const uts_config* cfg_, uts_proj in_, uts_mask mask_, const uint32_t* emit_rank_, void* scratch, const uts_tuning* tuning, cudaStream_t s_) {
    cfg = cfg_; in = in_; mask = mask_; emit_rank = emit_rank_; s = s_;
    ctx = device_ctx();
    if (!ctx) return UTS_ERR_CUDA;
    const uts_tuning tn = tuning ? *tuning : uts_tuning{0, 0.f, 0, 0, 0.f, 0};
    d = dims_of(cfg, &mask);
    n = (int64_t)d.P * d.V;
    b_mat = -1; cap_rows = 0;
    qp.kt = d.kt; qp.kq = d.kq; qp.P = d.P; qp.V = d.V; qp.n_tile = d.n_tile;
    const double* rm = rho_max_table_host();
    qp.rho_q = cfg->query_mode == UTS_QUERY_RING ? 0.0 : rm[d.kq];      // Alg.3's set has no PixRad margin
    qp.rho_t = rm[d.kt];
    for (int o = 0; o <= kMaxOrder; ++o) { qp.rho[o] = (float)rm[o]; qp.sin_hrho[o] = (float)sin(0.5 * rm[o]); qp.cos_hrho[o] = (float)cos(0.5 * rm[o]); }
    // Implementation choice: the ring-interval path (uts_ring_query.cuh) whenever a block's ring table fits shared memory
    // (k_q <= 12); the quadtree descent (Alg.2's depth-first form) otherwise, or when uts_tuning.query_impl = 1 asks for it.
    const int Nq = 1 << d.kq;
    ring_impl = 4 * Nq - 1 <= kRingBlockRingsMax && tn.query_impl != 1;
    qp.rc_thread = kRingThreadRings; qp.rc_warp = 4 * Nq - 1 < kRingWarpRings ? 4 * Nq - 1 : kRingWarpRings; qp.rc_block = 4 * Nq - 1;
    // a disc of radius R reaches at most 3 R N + 4 rings (ring spacing >= 2/(3N) in colatitude, +-1 ring of padding at each end)
    qp.b_warp = radius_bucket_host((float)((qp.rc_thread - 6) / (3.0 * Nq)));
    qp.b_block = radius_bucket_host((float)((qp.rc_warp - 6) / (3.0 * Nq)));
    if (qp.b_block > qp.b_warp) qp.b_block = qp.b_warp;
    // window class (uts_window_query.cuh): discs of the thread class with R <= 0.98 kWindowWidth w_max / N_t, i.e. the
    // radius buckets strictly below the one that holds that radius; needs N_t >= 2 kWindowMax + 1 so that the window's cells are distinct
    b_fast = kBuckets;
    // When: measured after the ring path's exact test became cheap (round 2), the window wins only where most candidates fall
    // outside the mask (config 5, frustum = 6 % of the tiles: tile lists 4.5 -> 3.7 ms; config 3, cap = 55 %: 0.68 -> 0.78;
    // no mask: config 2 0.24 -> 0.33, config 4 unchanged) — so by default it is taken when the mask keeps at most a quarter of
    // the tiles; uts_tuning.window_mode forces it on (tests) or off.
    qp.w_max = kWindowMax;
    const bool window_auto = mask.slot_of_tile && (int64_t)mask.n_active * 4 <= d.n_tile;
    const bool window_on = tn.window_mode == 2 || (tn.window_mode == 0 && window_auto);
    if (ring_impl && window_on && (1 << d.kt) >= 2 * kWindowMax + 1) {
      b_fast = radius_bucket_host((float)(0.98 * (1.0 - 1e-6) * kWindowWidth * qp.w_max / (double)(1 << d.kt))) + 1;
      if (b_fast <= qp.b_warp) b_fast = qp.b_warp + 1;
    }
    qp.active_tiles = mask.active_tiles; qp.n_active = mask.active_tiles ? mask.n_active : -1;
    qp.os = d.kt < 4 ? d.kt : 4;
    const size_t n_split = (size_t)12 << (2 * qp.os);
    qp.wl_cap = (int)(n_split > 4096 ? n_split : 4096);
    const size_t large_smem = (2 * (size_t)(d.n_tile / 32) + 2 * (size_t)qp.wl_cap) * 4;
    use_large = !ring_impl && d.kt >= 2 && large_smem <= kMaxLargeSmem;
    qp.n_words = use_large ? (int)(d.n_tile / 32) : 0;
    qp.r_large = (float)((tn.descent_block_radius > 0.f ? (double)tn.descent_block_radius : 36.0) / sqrt((double)d.n_tile));      // ~320 tiles (pi R^2 / (4 pi / n_tile)); measured crossover on config 4

    const QueryLayout L = query_layout(cfg);
    char* sp = reinterpret_cast<char*>(scratch);
    counts = reinterpret_cast<uint32_t*>(sp + L.counts);
    list = reinterpret_cast<uint32_t*>(sp + L.list);
    n_large = reinterpret_cast<uint32_t*>(sp + L.nlarge);
    n_small = n_large + 1;
    hist = n_large + 32;
    perm = reinterpret_cast<uint32_t*>(sp + L.perm);
    active = reinterpret_cast<uint32_t*>(sp + L.active);
    block_sums = reinterpret_cast<uint64_t*>(sp + L.scan);
    qp.tile_cache = reinterpret_cast<uint32_t*>(sp + L.tcache);
    qp.bitmap_cache = reinterpret_cast<uint32_t*>(sp + L.bcache);
    qp.bitmap_cache_cap = L.bcache_cap;
    // the ring path reuses two scratch regions of the descent: the bitmap cache holds the row masks, `list` their bases
    qp.mask_cache = reinterpret_cast<unsigned long long*>(sp + L.bcache);
    qp.mask_cache_cap = (uint32_t)(L.bcache_bytes / 8);
    qp.mask_cursor = n_large + 8;                                              // zeroed with the header in count()
    qp.mask_base = list;
    active_arg = nullptr;
    qgrid = (unsigned)((n + kLargeThreads - 1) / kLargeThreads);
    lgrid = use_large ? ctx->sms * (tn.descent_blocks_per_sm > 0 ? tn.descent_blocks_per_sm : 2) : 0;
    dyn_smem = use_large ? large_smem : 0;
    smem_a = sizeof(BatchRec) * kBatchA + (size_t)kBatchA * qp.rc_thread * sizeof(int2);
    smem_b = sizeof(BatchRec) * kBatchB + (size_t)kBatchB * qp.rc_warp * sizeof(int2);
    smem_block = (size_t)qp.rc_block * sizeof(int2);
    agrid = wgrid = bgrid = agrid_e = wgrid_e = bgrid_e = 0;     // persistent grids: exactly the resident blocks
    std::lock_guard<std::recursive_mutex> lock(ctx->mu);
    if (!ctx->attrs_set[0]) {                                    // once per device
      UTS_CUDA(cudaFuncSetAttribute(tile_query_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxLargeSmem));
      UTS_CUDA(cudaFuncSetAttribute(tile_query_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxLargeSmem));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_block_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingBlockRingsMax * 8 + 8));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_block_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingBlockRingsMax * 8 + 8));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_batch_kernel<kBatchA, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_batch_kernel<kBatchA, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_batch_kernel<kBatchB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
      UTS_CUDA(cudaFuncSetAttribute(ring_query_batch_kernel<kBatchB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
      UTS_CUDA(cudaFuncSetAttribute(matrix_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
      ctx->attrs_set[0] = true;
    }
    if (ring_impl) {                                             // occupancy numbers are cached per (kernel, shared-memory size)
      const unsigned sms = (unsigned)ctx->sms;
      bgrid = sms * (unsigned)cached_occupancy(ctx, kOccBlock0, ring_query_block_kernel<false>, kLargeThreads, smem_block);
      bgrid_e = sms * (unsigned)cached_occupancy(ctx, kOccBlock1, ring_query_block_kernel<true>, kLargeThreads, smem_block);
      wgrid = sms * (unsigned)cached_occupancy(ctx, kOccB0, ring_query_batch_kernel<kBatchB, false>, kLargeThreads, smem_b);
      wgrid_e = sms * (unsigned)cached_occupancy(ctx, kOccB1, ring_query_batch_kernel<kBatchB, true>, kLargeThreads, smem_b);
      agrid = sms * (unsigned)cached_occupancy(ctx, kOccA0, ring_query_batch_kernel<kBatchA, false>, kLargeThreads, smem_a);
      agrid_e = sms * (unsigned)cached_occupancy(ctx, kOccA1, ring_query_batch_kernel<kBatchA, true>, kLargeThreads, smem_a);
    }
    return UTS_OK;
  }

  // classification + count pass + exclusive scan of the per-slot counts into offsets[n + 1].  mp != nullptr: the discs of the
  // matrix class write bitmap rows instead (and count 0).  Enqueues only.
  // the aux streams wait for everything queued on s so far
  int fork() {
    UTS_CUDA(cudaEventRecord(ctx->fork, s));
    UTS_CUDA(cudaStreamWaitEvent(ctx->aux[0], ctx->fork, 0));
    UTS_CUDA(cudaStreamWaitEvent(ctx->aux[1], ctx->fork, 0));
    return UTS_OK;
  }
  // s waits for the aux streams; called on every exit path after fork() so that no work is left unjoined
  int join() {
    for (int i = 0; i < 2; ++i) { UTS_CUDA(cudaEventRecord(ctx->join[i], ctx->aux[i])); UTS_CUDA(cudaStreamWaitEvent(s, ctx->join[i], 0)); }
    return UTS_OK;
  }

  int count(uint64_t* offsets, MatParams* mp, uint32_t* flag_by_rank, uint64_t* rank_scan, uint64_t* rank_scan_sums) {
    std::lock_guard<std::recursive_mutex> lock(ctx->mu);
    if (use_large && mask.slot_of_tile) {
      active_words_kernel<<<(qp.n_words + 255) / 256, 256, 0, s>>>(mask.slot_of_tile, qp.n_words, active);
      UTS_LAUNCH_CHECK();
      active_arg = active;
    }
    UTS_CUDA(cudaMemsetAsync(n_large, 0, 512, s));
    const unsigned cgrid = (unsigned)((n + 255) / 256);
    classify_kernel<0><<<cgrid, 256, 0, s>>>(qp, in.rs, in.flags, counts, list, n_large, hist, perm, emit_rank);
    UTS_LAUNCH_CHECK();
    bucket_scan_kernel<<<1, 32, 0, s>>>(hist, n_small, qp.b_block, qp.b_warp, mp ? b_mat : -1, ring_impl ? b_fast : kBuckets, cap_rows, (double)d.n_tile, (double)d.n_tile * d.V);
    UTS_LAUNCH_CHECK();
    classify_kernel<1><<<cgrid, 256, 0, s>>>(qp, in.rs, in.flags, counts, list, n_large, hist, perm, emit_rank);
    UTS_LAUNCH_CHECK();
    if (ring_impl) {
      if (mp) {                                       // rows of the bit matrix: rank order of the matrix-class discs
        UTS_CUDA(cudaMemsetAsync(flag_by_rank, 0, (size_t)n * 4, s));
        UTS_CUDA(cudaMemsetAsync(mp->n_L, 0, 8, s));
        mat_flag_kernel<<<ctx->sms * 4, 256, 0, s>>>(perm, n_small, emit_rank, flag_by_rank, counts);
        UTS_LAUNCH_CHECK();
        int st = exclusive_scan_u32(flag_by_rank, n, rank_scan, rank_scan_sums, s);
        if (st) return st;
        mat_view_tab_kernel<<<1, 32, 0, s>>>(*mp, d.P, d.V, d.n_tile);
        UTS_LAUNCH_CHECK();
        if (mask.slot_of_tile) {
          active_words_kernel<<<(mp->n_words + 255) / 256, 256, 0, s>>>(mask.slot_of_tile, mp->n_words, active);
          UTS_LAUNCH_CHECK();
        }
      }
      int st = fork();
      if (st) return st;
      st = [&]() -> int {
        ring_query_block_kernel<false><<<bgrid, kLargeThreads, smem_block, s>>>(qp, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small, emit_rank,
                                                                              counts, nullptr, nullptr, nullptr);
        UTS_LAUNCH_CHECK();
        ring_query_batch_kernel<kBatchB, false><<<wgrid, kLargeThreads, smem_b, ctx->aux[0]>>>(qp, 0, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small,
                                                                                   emit_rank, counts, nullptr, nullptr, nullptr);
        UTS_LAUNCH_CHECK();
        ring_query_batch_kernel<kBatchA, false><<<agrid, kLargeThreads, smem_a, ctx->aux[1]>>>(qp, 1, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small,
                                                                                   emit_rank, counts, nullptr, nullptr, nullptr);
        UTS_LAUNCH_CHECK();
        if (b_fast < kBuckets) {
          window_query_kernel<false><<<(unsigned)((n + kWindowThreads - 1) / kWindowThreads), kWindowThreads, 0, ctx->aux[1]>>>(
              qp, in.dir, in.rho, in.rs, mask.slot_of_tile, perm, n_small, emit_rank, counts, nullptr, nullptr, nullptr);
          UTS_LAUNCH_CHECK();
        }
        return UTS_OK;
      }();
      const int stj = join();
      if (st) return st;
      if (stj) return stj;
      if (mp) {
        // The bitmap rows of the matrix class go to the context's side stream, behind the small discs' count: issue-bound geometry
        // that then runs beside the host's read of the pair count and the small pairs' emit and radix sort (HBM-bound) instead of
        // in front of them.  The caller joins (side_forked).
        UTS_CUDA(cudaEventRecord(ctx->side_fork, s));
        UTS_CUDA(cudaStreamWaitEvent(ctx->side, ctx->side_fork, 0));
        side_forked = true;
        const size_t smem_m = smem_block + (size_t)mp->n_words * 4;
        const int occ = cached_occupancy(ctx, kOccMat, matrix_count_kernel, kMatThreads, smem_m);
        matrix_count_kernel<<<(unsigned)ctx->sms * (unsigned)(occ < kMatSideBlocks ? occ : kMatSideBlocks), kMatThreads, smem_m, ctx->side>>>(
            qp, *mp, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, mask.slot_of_tile ? active : nullptr, perm, n_small, emit_rank);
        UTS_LAUNCH_CHECK();
      }
    } else {
      tile_query_kernel<false><<<qgrid + lgrid, kLargeThreads, dyn_smem, s>>>(qp, lgrid, in.dir, in.rho, in.rs, mask.slot_of_tile, active_arg, perm,
                                                                             n_small, list, n_large, emit_rank, counts, nullptr, nullptr, nullptr);
      UTS_LAUNCH_CHECK();
    }
    return exclusive_scan_u32(counts, n, offsets, block_sums, s);
  }

  // emit pass: the pairs of every slot at keys/vals[offsets[slot] ...).  Enqueues only.
  int emit(const uint64_t* offsets, uint64_t* keys, uint32_t* vals) {
    if (ring_impl) {
      std::lock_guard<std::recursive_mutex> lock(ctx->mu);
      int st = fork();
      if (st) return st;
      st = [&]() -> int {
        ring_query_block_kernel<true><<<bgrid_e, kLargeThreads, smem_block, s>>>(qp, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small, emit_rank,
                                                                             nullptr, offsets, keys, vals);
        UTS_LAUNCH_CHECK();
        ring_query_batch_kernel<kBatchB, true><<<wgrid_e, kLargeThreads, smem_b, ctx->aux[0]>>>(qp, 0, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small,
                                                                                  emit_rank, nullptr, offsets, keys, vals);
        UTS_LAUNCH_CHECK();
        ring_query_batch_kernel<kBatchA, true><<<agrid_e, kLargeThreads, smem_a, ctx->aux[1]>>>(qp, 1, in.dir, in.lonlat, in.rho, in.rs, mask.slot_of_tile, perm, n_small,
                                                                                  emit_rank, nullptr, offsets, keys, vals);
        UTS_LAUNCH_CHECK();
        if (b_fast < kBuckets) {
          window_query_kernel<true><<<(unsigned)((n + kWindowThreads - 1) / kWindowThreads), kWindowThreads, 0, ctx->aux[1]>>>(
              qp, in.dir, in.rho, in.rs, mask.slot_of_tile, perm, n_small, emit_rank, nullptr, offsets, keys, vals);
          UTS_LAUNCH_CHECK();
        }
        return UTS_OK;
      }();
      const int stj = join();
      return st ? st : stj;
    }
    tile_query_kernel<true><<<qgrid + lgrid, kLargeThreads, dyn_smem, s>>>(qp, lgrid, in.dir, in.rho, in.rs, mask.slot_of_tile, active_arg, perm,
                                                                          n_small, list, n_large, emit_rank, nullptr, offsets, keys, vals);
    UTS_LAUNCH_CHECK();
    return UTS_OK;
  }
};
}  // namespace

extern "C" {

size_t uts_tile_query_scratch_bytes(const uts_config* cfg) {
  if (check_config(cfg) != UTS_OK) return 0;
  return query_layout(cfg).total;
}

int uts_tile_query(const uts_config* cfg, uts_proj in, uts_mask mask, const uint32_t* emit_rank, uint64_t* offsets, uint64_t* keys,
                   uint32_t* vals, uint64_t capacity, uint64_t* h_n_pairs, void* scratch, size_t scratch_bytes, const uts_tuning* tuning,
                   void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!offsets || !h_n_pairs) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t n = (int64_t)cfg->n_gauss * cfg->n_views;
  if (n == 0) {                         // empty Gaussian set: no pairs, nothing else is read
    UTS_CUDA(cudaMemsetAsync(offsets, 0, sizeof(uint64_t), s));
    UTS_CUDA(cudaStreamSynchronize(s));
    *h_n_pairs = 0;
    return UTS_OK;
  }
  if (!in.dir || !in.lonlat || !in.rho || !in.rs || !in.flags || !scratch) return UTS_ERR_INVALID_ARG;
  if (keys && !vals) return UTS_ERR_INVALID_ARG;
  if (scratch_bytes < uts_tile_query_scratch_bytes(cfg) || ((uintptr_t)scratch & 255)) return UTS_ERR_INVALID_ARG;
  QueryRun q;
  if ((st = q.setup(cfg, in, mask, emit_rank, scratch, tuning, s))) return st;
  if ((st = q.count(offsets, nullptr, nullptr, nullptr, nullptr))) return st;
  UTS_CUDA(cudaMemcpyAsync(h_n_pairs, offsets + n, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
  UTS_CUDA(cudaStreamSynchronize(s));
  if (!keys) return UTS_OK;
  if (*h_n_pairs > capacity) return UTS_ERR_CAPACITY;
  if (*h_n_pairs == 0) return UTS_OK;
  return q.emit(offsets, keys, vals);
}

size_t uts_tile_lists_scratch_bytes(const uts_config* cfg) {
  if (check_config(cfg) != UTS_OK) return 0;
  return mat_layout(cfg, query_layout(cfg).total).total_bytes;
}

int uts_tile_lists(const uts_config* cfg, uts_proj in, uts_mask mask, const uint32_t* emit_rank, uint64_t* keys, uint32_t* vals,
                   uint64_t* keys_tmp, uint32_t* vals_tmp, uint64_t capacity, uint64_t* ranges, uint64_t* h_n_pairs, void* scratch,
                   size_t scratch_bytes, void* sort_scratch, size_t sort_scratch_bytes, const uts_tuning* tuning, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  if ((st = check_mask(cfg, mask))) return st;
  if (!ranges || !h_n_pairs || !emit_rank) return UTS_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const Dims d = dims_of(cfg, &mask);
  const int64_t n = (int64_t)d.P * d.V, nvt = (int64_t)d.V * d.n_tile;
  if (n == 0) {
    UTS_CUDA(cudaMemsetAsync(ranges, 0, (size_t)nvt * 16, s));
    UTS_CUDA(cudaStreamSynchronize(s));
    *h_n_pairs = 0;
    return UTS_OK;
  }
  if (!in.dir || !in.lonlat || !in.rho || !in.rs || !in.flags || !scratch || !sort_scratch) return UTS_ERR_INVALID_ARG;
  if (!keys || !vals || !keys_tmp || !vals_tmp) return UTS_ERR_INVALID_ARG;
  if (scratch_bytes < uts_tile_lists_scratch_bytes(cfg) || ((uintptr_t)scratch & 255) || ((uintptr_t)sort_scratch & 255)) return UTS_ERR_INVALID_ARG;
  const QueryLayout QL = query_layout(cfg);
  const MatLayout ML = mat_layout(cfg, QL.total);
  char* sp = reinterpret_cast<char*>(scratch);
  uint64_t* offsets = reinterpret_cast<uint64_t*>(sp + ML.offsets);
  QueryRun q;
  if ((st = q.setup(cfg, in, mask, emit_rank, scratch, tuning, s))) return st;
  MatParams mp;
  mp.M = reinterpret_cast<uint32_t*>(sp + ML.M); mp.MT = reinterpret_cast<uint32_t*>(sp + ML.MT);
  mp.row_key = reinterpret_cast<unsigned long long*>(sp + ML.row_key);
  mp.row_of_rank = reinterpret_cast<const uint64_t*>(sp + ML.rank_scan);
  mp.views = reinterpret_cast<MatView*>(sp + ML.views);
  mp.large_count = reinterpret_cast<uint32_t*>(sp + ML.large);
  mp.n_L = reinterpret_cast<unsigned long long*>(sp + ML.misc);
  mp.n_words = (int)(d.n_tile / 32);
  // Matrix class: ring-interval path, tile bitmaps that fit a block's shared memory next to the ring table, and discs large enough
  // that a bitmap row (about 5 passes over n_tile / 8 bytes) is cheaper than the disc's pairs through emit + radix sort + ranges
  // (about 90 B per pair): tiles >= n_tile / 144.
  const size_t smem_m = q.smem_block + (size_t)mp.n_words * 4;
  const bool mat_ok = q.ring_impl && d.kt >= 2 && smem_m <= 220 * 1024 && ML.cap_rows > 0 && !(tuning && tuning->matrix_off);
  if (mat_ok) {
    const double tiles_min = (tuning && tuning->matrix_min_tiles > 0.f) ? (double)tuning->matrix_min_tiles : fmax(48.0, (double)d.n_tile / 144.0);
    const double cosR = 1.0 - 2.0 * tiles_min / (double)d.n_tile;           // cap of tiles_min tiles: n_tile (1 - cos R) / 2
    q.b_mat = cosR <= -1.0 ? -1 : radius_bucket_host((float)acos(cosR));
    if (q.b_mat > q.qp.b_block) q.b_mat = q.qp.b_block;                     // only discs of the block-per-disc class
    q.cap_rows = ML.cap_rows;
  }
  uint32_t* flag_by_rank = reinterpret_cast<uint32_t*>(sp + ML.flag);
  uint64_t* scan_sums = reinterpret_cast<uint64_t*>(sp + ML.scan);
  // The matrix class runs on the context's side stream from its count on (q.count forks it): bitmap rows, transpose, per-tile counts
  // beside the small discs' count, emit, radix sort and ranges; joined back before the totals.  The guard joins on every exit path,
  // so no work is ever left unjoined; the context stays locked for the call (side stream, its events and the pinned words).
  DeviceCtx* ctx = q.ctx;
  std::lock_guard<std::recursive_mutex> side_lock(ctx->mu);
  struct SideJoin {
    DeviceCtx* c; cudaStream_t s; bool forked = false;
    int join() { if (!forked) return UTS_OK; forked = false; UTS_CUDA(cudaEventRecord(c->side_join, c->side)); UTS_CUDA(cudaStreamWaitEvent(s, c->side_join, 0)); return UTS_OK; }
    ~SideJoin() { join(); }
  } side{ctx, s};
  st = q.count(offsets, mat_ok ? &mp : nullptr, flag_by_rank, reinterpret_cast<uint64_t*>(sp + ML.rank_scan), scan_sums);
  side.forked = q.side_forked;
  if (st) return st;
  if (side.forked) {                                  // the matrix pairs' total, read by the host while the small pairs are sorted
    UTS_CUDA(cudaMemcpyAsync(ctx->pin + 4, mp.n_L, 8, cudaMemcpyDeviceToHost, ctx->side));
    UTS_CUDA(cudaEventRecord(ctx->side_mid, ctx->side));
  }
  // host needs now: small pairs and matrix rows — gathered on the device, one copy into the context's pinned words
  uint64_t n_S = 0, n_mat = 0;
  {
    unsigned long long* g3 = reinterpret_cast<unsigned long long*>(sp + ML.misc) + 8;
    gather3_kernel<<<1, 1, 0, s>>>(offsets + n, nullptr, mat_ok ? mp.row_of_rank + n : nullptr, g3);
    UTS_LAUNCH_CHECK();
    UTS_CUDA(cudaMemcpyAsync(ctx->pin, g3, 24, cudaMemcpyDeviceToHost, s));
    UTS_CUDA(cudaStreamSynchronize(s));
    n_S = ctx->pin[0]; n_mat = ctx->pin[2];
  }
  *h_n_pairs = n_S;
  if (n_S > capacity) {                               // report the whole need: wait for the matrix pairs' total as well
    if (side.forked) { UTS_CUDA(cudaEventSynchronize(ctx->side_mid)); *h_n_pairs = n_S + ctx->pin[4]; }
    return UTS_ERR_CAPACITY;
  }
  if (sort_scratch_bytes < uts_sort_scratch_bytes(n_S)) return UTS_ERR_INVALID_ARG;
  if (!side.forked || n_mat == 0) {                   // no large discs: the plain sequence
    if ((st = side.join())) return st;
    if (n_S) {
      if ((st = q.emit(offsets, keys, vals))) return st;
      if ((st = uts_sort(cfg, n_S, keys, vals, keys_tmp, vals_tmp, 1, sort_scratch, sort_scratch_bytes, stream))) return st;
    }
    return uts_tile_ranges(cfg, n_S, keys, ranges, stream);
  }
  {
    dim3 grid((unsigned)((mp.n_words + 31) / 32), (unsigned)(n_mat / 256 + (uint64_t)d.V + 1));
    UTS_CUDA(cudaMemsetAsync(mp.large_count, 0, (size_t)nvt * 4, ctx->side));       // the transpose adds each row block's counts
    matrix_transpose_kernel<<<grid, 256, 0, ctx->side>>>(mp, d.V, d.n_tile);
    UTS_LAUNCH_CHECK();
  }
  // ---- small discs: emit at keys_tmp / vals_tmp, sort there (ping-pong through keys / vals, free until the merge), their ranges
  uint64_t* s_ranges = reinterpret_cast<uint64_t*>(sp + ML.sranges);
  if (n_S) {
    if ((st = q.emit(offsets, keys_tmp, vals_tmp))) return st;
    if ((st = uts_sort(cfg, n_S, keys_tmp, vals_tmp, keys, vals, 1, sort_scratch, sort_scratch_bytes, stream))) return st;
  }
  if ((st = uts_tile_ranges(cfg, n_S, keys_tmp, s_ranges, stream))) return st;
  UTS_CUDA(cudaEventSynchronize(ctx->side_mid));     // the bitmap rows are done (the stream s is still busy with the sort)
  const uint64_t n_L = ctx->pin[4];
  *h_n_pairs = n_S + n_L;
  if (*h_n_pairs > capacity) return UTS_ERR_CAPACITY;
  if ((st = side.join())) return st;
  // ---- final ranges, then one warp per (view, tile) merges its large discs (bit vector) with its small pairs into keys / vals
  uint32_t* total = reinterpret_cast<uint32_t*>(sp + ML.total);
  uint64_t* start = reinterpret_cast<uint64_t*>(sp + ML.start);
  mat_totals_kernel<<<(unsigned)((nvt + 255) / 256), 256, 0, s>>>(nvt, mp.large_count, s_ranges, total);
  UTS_LAUNCH_CHECK();
  if ((st = exclusive_scan_u32(total, nvt, start, scan_sums, s))) return st;
  mat_ranges_kernel<<<(unsigned)((nvt + 255) / 256), 256, 0, s>>>(nvt, start, ranges);
  UTS_LAUNCH_CHECK();
  matrix_emit_merge_kernel<<<(unsigned)sm_count() * 8, 256, 0, s>>>(mp, d.V, d.n_tile, start, s_ranges, keys_tmp, vals_tmp, keys, vals);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // extern "C"
