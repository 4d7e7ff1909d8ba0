// uts_hssim.cu — training loss on the HEALPix grid, forward and backward in one pass.
//   "L = (1 - lambda) L1^H + lambda L_HSSIM"
//   "the NESTED (x,y,f) parameterization approximates a local 2D grid ... some corner pixels have only 7 neighbors;
//    we detect such cases and renormalize kernel weights accordingly ... isotropic for the equatorial zone ...
//    anisotropic for polar zones"
//   "shared memory with cross-face padding ... cached derivatives"
//   HSSIM = sum_q M(q) h_q / sum_q M(q)                                                                   Eq.10
// Readings A30-A35: 11 x 11 window in the face grid of the centre pixel, continued into the neighbouring faces,
// taps that do not exist (3-face vertices, M_C = 0) dropped and the weights renormalised, zone of the centre pixel's face,
// SSIM constants 0.01^2 / 0.03^2, h_q = channel mean.
//
// B200 design.  One block of 64 threads per 16 x 16 tile (the rasteriser's slot).  The block stages the 26 x 26 patch of the
// tile's own face frame — tile plus a 5-pixel apron, the apron resolved through the face-adjacency rules below — in shared
// memory as (x, g) pairs per channel plus a validity plane.  Every thread owns four pixels of one tile column: a patch cell read
// once from shared memory serves up to four windows, which is what keeps the kernel on the FP32 pipe rather than on the
// shared-memory pipe (the first version, one pixel per thread, ran at 99 % of the L1/shared wavefront rate).  The thread walks
// the 11 x 14 cells under its four windows once for the five window sums per pixel and channel (taken about a reference value
// next to the pixel: variances do not lose digits to e11 - m1^2), forms the SSIM index and its derivatives with respect to
// (m1, s11, s12), and — this is the "transposed convolution" with "cached derivatives" — walks the cells a second time adding
// weight * (c0 + K1 dx + K2 dg), summed over its four pixels in registers, into a gradient patch private to its warp (plain
// read-add-write between __syncwarp()s: float atomics on shared memory are compare-and-swap loops on sm_100).  The two warps'
// patches are summed and flushed to dL_dX with one red.global per cell and channel.  The upstream gradient of a loss is 1, so
// forward and backward share the staged patch and X, G are read from HBM once.  Tiles of the equatorial faces whose whole patch is
// visible take a SEPARABLE form of both walks (11 + 11 taps; see `sep` in the kernel): a third of the tiles on a full sphere.  The path is bound by fp32 ALU: about 24 FP32
// instructions per tap and pixel forward and 10 backward, against 36 B of compulsory traffic per pixel.
#include "uts_internal.cuh"

namespace uts {

constexpr int kHR = 5;                       // window radius (A30)
constexpr int kHW = 2 * kHR + 1;             // 11
constexpr int kHTaps = kHW * kHW;            // 121
constexpr int kHP = 16 + 2 * kHR;            // 26: patch side
constexpr int kHCells = kHP * kHP;           // 676

struct HssimWeights { float w[2][kHTaps]; }; // [0] equatorial faces, [1] polar faces; tap t = (dy + R) * 11 + (dx + R)

// ---------------------------------------------------------------------------------------------- face adjacency
// Faces f = 4 r + c: r = 0 north (touching the pole), 1 equatorial, 2 south.  In-face axes: +x points north-east, +y north-west.
// A cell (X, Y) outside [0, N)^2 of face f lies in another face.  Eight directions o = (ox, oy), ox, oy in {-1, 0, +1}:
//   - where the neighbour across that edge / vertex has the same axis orientation the step is a translation by N
//     (every edge of an equatorial face; the two lower edges of a north face; the two upper edges of a south face; the lower
//     vertex of a north face and the upper vertex of a south face, where 4 faces meet);
//   - the two upper edges of a north face are meridians glued to the next / previous north face: the coordinate along the edge
//     becomes the other face's coordinate along ITS glued edge, the depth beyond the edge becomes depth below that edge — a
//     quarter turn; beyond both (over the pole) two quarter turns.  Mirror image for the lower edges of a south face;
//   - the left / right vertex of a polar face and the upper / lower vertex of an equatorial face are shared by 3 faces only:
//     the diagonal quadrant there does not exist.
// One table entry per (r, oy + 1, ox + 1): kind 0 none, 1 translate, 2..4 quarter turn +1 / two / -1; dr, dc: face row, column step.
struct FaceStep { int8_t kind, row, dcol; };
__device__ __constant__ FaceStep kFaceStep[3][3][3] = {
    // north faces                 ox = -1            ox = 0            ox = +1
    {/* oy = -1 */ {{1, 2, 0}, {1, 1, 1}, {0, 0, 0}},
     /* oy =  0 */ {{1, 1, 0}, {1, 0, 0}, {2, 0, 1}},
     /* oy = +1 */ {{0, 0, 0}, {4, 0, 3}, {3, 0, 2}}},
    // equatorial faces
    {/* oy = -1 */ {{0, 0, 0}, {1, 2, 0}, {1, 1, 1}},
     /* oy =  0 */ {{1, 2, 3}, {1, 1, 0}, {1, 0, 0}},
     /* oy = +1 */ {{1, 1, 3}, {1, 0, 3}, {0, 0, 0}}},
    // south faces
    {/* oy = -1 */ {{3, 2, 2}, {4, 2, 1}, {0, 0, 0}},
     /* oy =  0 */ {{2, 2, 3}, {1, 2, 0}, {1, 1, 1}},
     /* oy = +1 */ {{0, 0, 0}, {1, 1, 0}, {1, 0, 0}}},
};

__device__ __forceinline__ uint32_t spread16(uint32_t v) {          // 16 bits -> even bit positions
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}

// NESTED pixel of cell (X, Y) in the extended frame of face f at order k (N = 2^k, -N <= X, Y < 2N), or -1.
__device__ __forceinline__ int64_t cell_to_pixel(int k, int f, int X, int Y) {
  const int N = 1 << k;
  const int ox = X < 0 ? -1 : (X >= N ? 1 : 0), oy = Y < 0 ? -1 : (Y >= N ? 1 : 0);
  const FaceStep s = kFaceStep[f >> 2][oy + 1][ox + 1];
  if (s.kind == 0) return -1;
  const int pole = (f >> 2) == 0 ? 2 * N - 1 : -1;      // north: the glued edges are x = N, y = N; south: x = -1, y = -1
  int x, y;
  switch (s.kind) {
    case 1: x = X - ox * N; y = Y - oy * N; break;       // translation
    case 2: x = Y; y = pole - X; break;                  // quarter turn: along-edge y -> x, depth beyond x-edge -> depth in y
    case 4: x = pole - Y; y = X; break;                  // quarter turn the other way
    default: x = pole - X; y = pole - Y; break;          // over the pole
  }
  const int g = 4 * s.row + ((f + s.dcol) & 3);
  return ((int64_t)g << (2 * k)) | spread16((uint32_t)x) | (spread16((uint32_t)y) << 1);
}

// storage index (slot layout) of pixel p, or -1 when masked out
__device__ __forceinline__ int64_t store_index(int64_t p, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ bits) {
  if (p < 0) return -1;
  if (bits && !((__ldg(bits + (p >> 5)) >> (p & 31)) & 1u)) return -1;
  const int64_t tile = p >> 8;
  const int64_t slot = slot_of_tile ? (int64_t)__ldg(slot_of_tile + tile) : tile;
  return slot < 0 ? -1 : slot * 256 + (p & 255);
}

// ------------------------------------------------------------------------------------------------- count
// acc[2] = number of valid pixels (Eq.10's denominator): one warp per slot, 8 mask words each.
__global__ void hssim_count_kernel(int64_t n_slot, const uint32_t* __restrict__ active_tiles, const uint32_t* __restrict__ bits, double* acc) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 3;   // 8 lanes per slot
  const int j = threadIdx.x & 7;
  int c = 0;
  if (w < n_slot) {
    const int64_t tile = active_tiles ? (int64_t)__ldg(active_tiles + w) : w;
    c = __popc(__ldg(bits + tile * 8 + j));
  }
  for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(acc + 2, (double)c);
}

// -------------------------------------------------------------------------------------------------- main
// 64 threads per tile: thread (lx, strip) owns the four pixels (lx, 4 strip + j), j = 0..3, of one tile column.  A patch cell
// loaded once serves up to four of the thread's windows (14 patch rows instead of 44 per window column), which takes the kernel
// off the shared-memory pipe.  Sums are taken about the value of the thread's second pixel.
constexpr int kHT = 64;                      // threads per block
constexpr int kHJ = 4;                       // pixels per thread (rows)
constexpr int kHRows = kHJ + 2 * kHR;        // 14 patch rows per thread
constexpr int kHS = 28;                      // patch row stride: 4 rows apart = 16 banks apart (the two half warps never collide)
constexpr int kHCellsS = kHP * kHS;
constexpr int kGR = 8 + 2 * kHR;             // 18 rows of a warp's private gradient patch (8 tile rows + apron)

template <int V> struct Int { static constexpr int value = V; };

template <bool GRAD>
__global__ void __launch_bounds__(kHT, 6)
hssim_kernel(int k, int64_t n_pix_full, const uint32_t* __restrict__ active_tiles, const int32_t* __restrict__ slot_of_tile,
             const uint32_t* __restrict__ bits, const float* __restrict__ X, const float* __restrict__ G, float lambda,
             const __grid_constant__ HssimWeights wts, float* __restrict__ h_map, float* __restrict__ dL_dX, double* acc) {
  __shared__ float2 s_xg[3][kHCellsS];       // (x, g) per channel
  __shared__ float s_val[kHCellsS];          // 1 valid, 0 missing
  __shared__ int s_idx[kHCellsS];            // storage index (pixels, < 2^31) or -1
  __shared__ float s_w[kHTaps];
  __shared__ __align__(16) float s_grad[2 * 3 * kGR * kHS];                // [warp][channel][row][col]: no two warps share a cell; scratch of the separable path
  __shared__ float s_red[2][2];

  const int tid = threadIdx.x;
  const int64_t slot = blockIdx.x;
  const int64_t tile = active_tiles ? (int64_t)__ldg(active_tiles + slot) : slot;
  const int kt = k - kTileLog2;
  const int f = (int)(tile >> (2 * kt));
  const uint32_t tm = (uint32_t)(tile & (((int64_t)1 << (2 * kt)) - 1));
  const int x0 = (int)squeeze_even_bits32(tm) << kTileLog2, y0 = (int)squeeze_even_bits32(tm >> 1) << kTileLog2;
  const bool polar = (f >> 2) != 1;

  for (int t = tid; t < kHTaps; t += kHT) s_w[t] = wts.w[polar ? 1 : 0][t];
  bool mine_valid = true;                                     // every patch cell this thread staged exists and is visible
  for (int c = tid; c < kHCells; c += kHT) {
    const int cy = c / kHP, cx = c - cy * kHP;
    const int cell = cy * kHS + cx;
    const int64_t p = cell_to_pixel(k, f, x0 - kHR + cx, y0 - kHR + cy);
    const int64_t i = store_index(p, slot_of_tile, bits);
    s_idx[cell] = (int)i;
    s_val[cell] = i >= 0 ? 1.f : 0.f;
    mine_valid = mine_valid && i >= 0;
    float x[3] = {0.f, 0.f, 0.f}, g[3] = {0.f, 0.f, 0.f};
    if (i >= 0) {
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) { x[ch] = __ldg(X + 3 * i + ch); g[ch] = __ldg(G + 3 * i + ch); }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) s_xg[ch][cell] = make_float2(x[ch], g[ch]);
  }
  if (GRAD) for (int c = tid; c < 2 * 3 * kGR * kHS; c += kHT) s_grad[c] = 0.f;
  // Separable path ("enabling separable convolution"): on an equatorial face the window weights are the isotropic
  // Gaussian g(dx) g(dy) (reading A31), and when every cell of the patch exists and is visible no tap is dropped (A32), so the
  // renormalisation is the constant (sum g)^2: the five window sums are an 11-tap pass along x followed by an 11-tap pass along y,
  // and the transposed window of the gradient is the same two passes on the per-pixel coefficient maps.  Block-uniform decision;
  // polar faces (anisotropic, not separable over the square window) and patches with a missing or masked cell take all 121 taps.
  // (Measured, order 10 full sphere, loss + gradient: all 121 taps everywhere 3.01 ms; this path unblocked 2.96; with four outputs
  // per item in registers 2.73; the two paths as two launches, each with its own register budget, 2.80.)
  const bool sep = __syncthreads_and(mine_valid) && !polar;

  const int lx = tid & 15, r0 = (tid >> 4) * kHJ;             // tile rows r0 .. r0+3; half warp = one strip of 16 x 4 pixels
  const int base = r0 * kHS + lx;                             // patch cell of tap (0,0) of pixel j = 0
  float xr[3], gr[3];
  {
    // reference value of the sums: the thread's second pixel, or its first visible one (a masked cell holds 0, which would
    // leave the sums uncentred)
    int cref = (r0 + 1 + kHR) * kHS + lx + kHR;
    if (sep) cref = (8 + kHR) * kHS + 8 + kHR;                // the intermediate sums are shared: one reference for the block
    else if (s_idx[cref] < 0) {
#pragma unroll
      for (int j = kHJ - 1; j >= 0; --j) { const int cj = (r0 + j + kHR) * kHS + lx + kHR; if (s_idx[cj] >= 0) cref = cj; }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) { const float2 v = s_xg[ch][cref]; xr[ch] = v.x; gr[ch] = v.y; }
  }
  const double n_valid = bits ? acc[2] : (double)n_pix_full;
  const float inv_n = (float)(1.0 / n_valid);

  float wsum[kHJ], S1[kHJ][3], S2[kHJ][3], S11[kHJ][3], S22[kHJ][3], S12[kHJ][3];
#pragma unroll
  for (int j = 0; j < kHJ; ++j) {
    wsum[j] = 0.f;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) S1[j][ch] = S2[j][ch] = S11[j][ch] = S22[j][ch] = S12[j][ch] = 0.f;
  }
  // One patch cell under the windows of pixels J0..J1 (compile-time range): wp points at the weight of pixel j = 0 for this cell,
  // pixel j's weight sits j window rows before it.
  // The 121-tap walk keeps (S1, S2) and (S11, S22) as packed fp32 pairs: per tap, pixel and channel (a, b) = w (dx, dg) is one
  // FMUL2, the two sums one FADD2, the two squares one FFMA2 and the cross term one FFMA — four issue slots instead of seven, the
  // same roundings as the scalar form.
  f2_t P12[kHJ][3], P1122[kHJ][3], nref[3];
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) nref[ch] = f2_pack(-xr[ch], -gr[ch]);
#pragma unroll
  for (int j = 0; j < kHJ; ++j)
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) P12[j][ch] = P1122[j][ch] = 0;
  auto fwd_cell = [&](int c, const float* wp, auto j0, auto j1) {
    const float val = s_val[c];
    f2_t d2[3];                                               // (dx, dg) per channel
    float dg[3];
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      d2[ch] = f2_add(*reinterpret_cast<const f2_t*>(&s_xg[ch][c]), nref[ch]);
      float lo; f2_unpack(d2[ch], lo, dg[ch]);
    }
#pragma unroll
    for (int j = decltype(j0)::value; j <= decltype(j1)::value; ++j) {
      const float wv = wp[-j * kHW] * val;
      wsum[j] += wv;
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) {
        const f2_t ab = f2_mul(f2_bc(wv), d2[ch]);
        float a, b; f2_unpack(ab, a, b);
        P12[j][ch] = f2_add(P12[j][ch], ab);
        P1122[j][ch] = f2_fma(ab, d2[ch], P1122[j][ch]);
        S12[j][ch] = fmaf(a, dg[ch], S12[j][ch]);
      }
    }
  };
  // Patch rows 0..2 and 11..13 lie under fewer than four of the thread's windows (unrolled); rows 3..10 under all four: a real
  // loop, so that the body stays inside the instruction cache (fully unrolled, 14 rows x 4 pixels, it stalled on fetch).
  using I0 = Int<0>; using I1 = Int<1>; using I2 = Int<2>; using I3 = Int<3>;
  if (sep) {
    // g(d) = the window's middle row; pass 1 along x into s_grad as H[row][col][6] (26 x 16 records of 5 floats + 1 of padding), pass 2 along y in registers
    const float* g1 = s_w + kHR * kHW;
    float gsum = 0.f;
#pragma unroll
    for (int t = 0; t < kHW; ++t) gsum += g1[t];
#pragma unroll
    for (int j = 0; j < kHJ; ++j) wsum[j] = gsum * gsum;
    float* H = s_grad;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {                          // unrolled: ch indexes register arrays
      __syncthreads();                                          // the previous channel's H has been consumed
      for (int it = tid; it < kHP * 4; it += kHT) {             // item = (patch row, group of 4 tile columns): 14 cells serve 4 outputs
        const int row = it >> 2, cg = (it & 3) * 4;
        const float2* src = &s_xg[ch][row * kHS + cg];
        f2_t dv[14];                                            // (dx, dg) of the 14 cells, packed
        float dgv[14];
#pragma unroll
        for (int i = 0; i < 14; ++i) { dv[i] = f2_add(*reinterpret_cast<const f2_t*>(src + i), nref[ch]); float lo; f2_unpack(dv[i], lo, dgv[i]); }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          f2_t h12p = 0, h1122 = 0;
          float h12 = 0.f;
#pragma unroll
          for (int t = 0; t < kHW; ++t) {
            const f2_t ab = f2_mul(f2_bc(g1[t]), dv[q + t]);
            float a, b; f2_unpack(ab, a, b);
            h12p = f2_add(h12p, ab); h1122 = f2_fma(ab, dv[q + t], h1122); h12 = fmaf(a, dgv[q + t], h12);
          }
          float* dst = H + (row * 16 + cg + q) * 6;             // records of 6 floats: the two pairs stay 8-byte aligned
          *reinterpret_cast<f2_t*>(dst) = h12p; *reinterpret_cast<f2_t*>(dst + 2) = h1122; dst[4] = h12;
        }
      }
      __syncthreads();
#pragma unroll
      for (int rho = 0; rho < kHRows; ++rho) {                  // patch rows r0 .. r0 + 13 of column lx
        const float* hv = H + ((r0 + rho) * 16 + lx) * 6;
        const f2_t v01 = *reinterpret_cast<const f2_t*>(hv), v23 = *reinterpret_cast<const f2_t*>(hv + 2);
        const float v4 = hv[4];
#pragma unroll
        for (int j = 0; j < kHJ; ++j) {
          const int t = rho - j;                                // window row of pixel j
          if (t >= 0 && t < kHW) {
            const float wv = g1[t];
            P12[j][ch] = f2_fma(f2_bc(wv), v01, P12[j][ch]); P1122[j][ch] = f2_fma(f2_bc(wv), v23, P1122[j][ch]);
            S12[j][ch] = fmaf(wv, v4, S12[j][ch]);
          }
        }
      }
    }
    __syncthreads();
    if (GRAD) for (int c = tid; c < 2 * 3 * kGR * kHS; c += kHT) s_grad[c] = 0.f;      // not used as warp patches on this path, but kept defined
  } else
#pragma unroll 1
  for (int tx = 0; tx < kHW; ++tx) {
    const int c = base + tx;
    const float* wp = s_w + tx;
    fwd_cell(c, wp, I0(), I0());
    fwd_cell(c + kHS, wp + kHW, I0(), I1());
    fwd_cell(c + 2 * kHS, wp + 2 * kHW, I0(), I2());
#pragma unroll 2
    for (int rho = 3; rho < kHW; ++rho) fwd_cell(c + rho * kHS, wp + rho * kHW, I0(), I3());
    fwd_cell(c + 11 * kHS, wp + 11 * kHW, I1(), I3());
    fwd_cell(c + 12 * kHS, wp + 12 * kHW, I2(), I3());
    fwd_cell(c + 13 * kHS, wp + 13 * kHW, I3(), I3());
  }
  {
#pragma unroll
    for (int j = 0; j < kHJ; ++j)
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) { f2_unpack(P12[j][ch], S1[j][ch], S2[j][ch]); f2_unpack(P1122[j][ch], S11[j][ch], S22[j][ch]); }
  }

  // SSIM index and, for the gradient, its derivatives folded into three coefficients per pixel and channel:
  //   d ssim / d(m1 | s11 | s12) with s11 = e11 - m1^2, s12 = e12 - m1 m2 held as independent variables:
  //     d/dm1 = 2 m2 a2 / (b1 b2) - 2 m1 ssim / b1,  d/ds11 = -ssim / b2,  d/ds12 = 2 a1 / (b1 b2);
  //   a tap value x enters m1 with weight w, s11 with 2 w (x - m1), s12 with w (g - m2), so the tap's share of dL/dx is
  //     w [K0 + K1 (x - m1) + K2 (g - m2)] = w [c0 + K1 dx + K2 dg],  dx = x - x_ref,  c0 = K0 - K1 u1 - K2 u2.
  const float C1 = 1e-4f, C2 = 9e-4f;                         // A33
  float hsum = 0.f, l1 = 0.f;
  float c0[kHJ][3], k1[kHJ][3], k2[kHJ][3], gl1[kHJ][3];
#pragma unroll
  for (int j = 0; j < kHJ; ++j) {
    const int cc = base + (j + kHR) * kHS + kHR;              // centre cell of pixel j
    const bool live = s_idx[cc] >= 0;
    const float inv_w = live ? 1.0f / wsum[j] : 0.f;          // the centre tap is valid: wsum >= w(0,0) = 1
    const float sc = -lambda * inv_n * (1.f / 3.f) * inv_w;
    float hq = 0.f;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      const float u1 = S1[j][ch] * inv_w, u2 = S2[j][ch] * inv_w;   // means about the reference value
      const float s11 = S11[j][ch] * inv_w - u1 * u1, s22 = S22[j][ch] * inv_w - u2 * u2, s12 = S12[j][ch] * inv_w - u1 * u2;
      const float m1 = xr[ch] + u1, m2 = gr[ch] + u2;
      const float a1 = 2.f * m1 * m2 + C1, a2 = 2.f * s12 + C2;
      const float b1 = m1 * m1 + m2 * m2 + C1, b2 = s11 + s22 + C2;
      const float ib1 = 1.0f / b1, ib2 = 1.0f / b2;
      const float ssim = a1 * a2 * ib1 * ib2;
      hq += ssim;
      const float K0 = 2.f * (m2 * a2 * ib1 * ib2 - m1 * ssim * ib1), K1 = -2.f * ssim * ib2, K2 = 2.f * a1 * ib1 * ib2;
      c0[j][ch] = sc * (K0 - K1 * u1 - K2 * u2); k1[j][ch] = sc * K1; k2[j][ch] = sc * K2;
      const float2 v = s_xg[ch][cc];
      const float d = v.x - v.y;
      l1 += live ? fabsf(d) : 0.f;
      gl1[j][ch] = live ? (1.f - lambda) * inv_n * (1.f / 3.f) * (d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f)) : 0.f;
    }
    hq = live ? hq * (1.f / 3.f) : 0.f;
    hsum += hq;
    if (h_map) h_map[slot * 256 + (spread16((uint32_t)lx) | (spread16((uint32_t)(r0 + j)) << 1))] = hq;   // Morton position in the slot
  }

  if (GRAD && sep) {
    // Transposed window, separable: the tap's share of dL/dx at a patch cell is  A + B dx_cell + C dg_cell  with A, B, C the window
    // transforms of the per-pixel coefficient maps c0, k1, k2 over the tile — a pass along y (26 x 16 x 3) and a pass along x
    // (26 x 26 x 3) per channel, in s_grad as Cf[16][16][3] and V[26][16][3]; each patch cell's sum goes straight to dL_dX with one
    // atomic (neighbouring tiles add their aprons to the same pixels).
    const float* g1 = s_w + kHR * kHW;
    float* Cf = s_grad;                                         // 768 floats
    float* V = s_grad + 16 * 16 * 3;                            // 1248 floats
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {                          // unrolled: ch indexes register arrays
      __syncthreads();                                          // the previous channel's maps have been consumed
#pragma unroll
      for (int j = 0; j < kHJ; ++j) {
        float* d = Cf + ((r0 + j) * 16 + lx) * 3;
        d[0] = c0[j][ch]; d[1] = k1[j][ch]; d[2] = k2[j][ch];
      }
      __syncthreads();
      for (int it = tid; it < 16 * 7; it += kHT) {              // along y; item = (tile column, group of 4 patch rows): 14 tile rows serve 4 outputs
        const int col = it & 15, p0 = (it >> 4) * 4;
        float cf[14][3];
#pragma unroll
        for (int i = 0; i < 14; ++i) {
          const int tr = p0 - 10 + i;                           // tile row; patch row prow takes tile rows prow - 10 .. prow
          const bool in = tr >= 0 && tr < 16;
          const float* sp = Cf + ((in ? tr : 0) * 16 + col) * 3;
          cf[i][0] = in ? sp[0] : 0.f; cf[i][1] = in ? sp[1] : 0.f; cf[i][2] = in ? sp[2] : 0.f;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (p0 + q >= kHP) break;
          float a = 0.f, b = 0.f, c = 0.f;
#pragma unroll
          for (int t = 0; t < kHW; ++t) { a = fmaf(g1[t], cf[q - t + 10][0], a); b = fmaf(g1[t], cf[q - t + 10][1], b); c = fmaf(g1[t], cf[q - t + 10][2], c); }
          float* d = V + ((p0 + q) * 16 + col) * 3;
          d[0] = a; d[1] = b; d[2] = c;
        }
      }
      __syncthreads();
      for (int it = tid; it < kHP * 7; it += kHT) {             // along x; item = (patch row, group of 4 patch columns), then the cells' values and atomics
        const int prow = it / 7, p0 = (it - prow * 7) * 4;
        float vv[14][3];
#pragma unroll
        for (int i = 0; i < 14; ++i) {
          const int tc = p0 - 10 + i;
          const bool in = tc >= 0 && tc < 16;
          const float* sp = V + (prow * 16 + (in ? tc : 0)) * 3;
          vv[i][0] = in ? sp[0] : 0.f; vv[i][1] = in ? sp[1] : 0.f; vv[i][2] = in ? sp[2] : 0.f;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int pcol = p0 + q;
          if (pcol >= kHP) break;
          float a = 0.f, b = 0.f, c = 0.f;
#pragma unroll
          for (int t = 0; t < kHW; ++t) { a = fmaf(g1[t], vv[q - t + 10][0], a); b = fmaf(g1[t], vv[q - t + 10][1], b); c = fmaf(g1[t], vv[q - t + 10][2], c); }
          const int cell = prow * kHS + pcol;
          const float2 v = s_xg[ch][cell];
          float val = fmaf(b, v.x - xr[ch], fmaf(c, v.y - gr[ch], a));
          if (prow >= kHR && prow < kHR + 16 && pcol >= kHR && pcol < kHR + 16) {     // L1 term at the tile's own pixels
            const float d = v.x - v.y;
            val += (1.f - lambda) * inv_n * (1.f / 3.f) * (d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f));
          }
          if (val != 0.f) atomicAdd(dL_dX + 3 * (int64_t)s_idx[cell] + ch, val);
        }
      }
    }
  } else if (GRAD) {
    // transposed window: every tap scatters into the warp's private patch.  Within one group of four patch rows the 32 lanes
    // touch 32 different cells (the other half warp works 4 rows further down), so plain read-add-write is safe between the
    // __syncwarp()s (after rows 2, 6, 10, 13); sums over the thread's own four pixels are taken in registers first.
    float* gw = s_grad + (tid >> 5) * (3 * kGR * kHS) + (((tid >> 4) & 1) * kHJ) * kHS + lx;
    // the coefficients of pixel pairs (0, 1) and (2, 3) as packed fp32 pairs: a cell under both windows of a pair takes three FFMA2
    // per channel for the two pixels (the pair's halves are added once per cell)
    f2_t c0p[2][3], k1p[2][3], k2p[2][3];
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) {
        c0p[q][ch] = f2_pack(c0[2 * q][ch], c0[2 * q + 1][ch]); k1p[q][ch] = f2_pack(k1[2 * q][ch], k1[2 * q + 1][ch]);
        k2p[q][ch] = f2_pack(k2[2 * q][ch], k2[2 * q + 1][ch]);
      }
    auto bwd_cell = [&](int c, const float* wp, float* gp, auto j0, auto j1) {
      constexpr int J0 = decltype(j0)::value, J1 = decltype(j1)::value;
      const float val = s_val[c];
      float dx[3], dg[3], ac[3] = {0.f, 0.f, 0.f};
      f2_t ac2[3] = {0, 0, 0};
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) { const float2 v = s_xg[ch][c]; dx[ch] = v.x - xr[ch]; dg[ch] = v.y - gr[ch]; }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        if (J0 <= 2 * q && 2 * q + 1 <= J1) {                   // both pixels of the pair see this cell
          const f2_t wv2 = f2_pack(wp[-(2 * q) * kHW] * val, wp[-(2 * q + 1) * kHW] * val);
#pragma unroll
          for (int ch = 0; ch < 3; ++ch)
            ac2[ch] = f2_fma(wv2, f2_fma(k1p[q][ch], f2_bc(dx[ch]), f2_fma(k2p[q][ch], f2_bc(dg[ch]), c0p[q][ch])), ac2[ch]);
        } else {
#pragma unroll
          for (int j = 2 * q; j <= 2 * q + 1; ++j) {
            if (j < J0 || j > J1) continue;
            const float wv = wp[-j * kHW] * val;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) ac[ch] = fmaf(wv, fmaf(k1[j][ch], dx[ch], fmaf(k2[j][ch], dg[ch], c0[j][ch])), ac[ch]);
          }
        }
      }
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) { float lo, hi; f2_unpack(ac2[ch], lo, hi); gp[ch * (kGR * kHS)] += ac[ch] + (lo + hi); }
    };
#pragma unroll 1
    for (int tx = 0; tx < kHW; ++tx) {
      const int c = base + tx;
      const float* wp = s_w + tx;
      float* gp = gw + tx;
      bwd_cell(c, wp, gp, I0(), I0());
      bwd_cell(c + kHS, wp + kHW, gp + kHS, I0(), I1());
      bwd_cell(c + 2 * kHS, wp + 2 * kHW, gp + 2 * kHS, I0(), I2());
      __syncwarp();
#pragma unroll 1
      for (int rho = 3; rho < kHW; rho += 4) {                // rows 3..6, 7..10
#pragma unroll
        for (int d = 0; d < 4; ++d) bwd_cell(c + (rho + d) * kHS, wp + (rho + d) * kHW, gp + (rho + d) * kHS, I0(), I3());
        __syncwarp();
      }
      bwd_cell(c + 11 * kHS, wp + 11 * kHW, gp + 11 * kHS, I1(), I3());
      bwd_cell(c + 12 * kHS, wp + 12 * kHW, gp + 12 * kHS, I2(), I3());
      bwd_cell(c + 13 * kHS, wp + 13 * kHW, gp + 13 * kHS, I3(), I3());
      __syncwarp();
    }
    // L1 term at the thread's own pixels
#pragma unroll
    for (int j = 0; j < kHJ; ++j)
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) gw[ch * (kGR * kHS) + (j + kHR) * kHS + kHR] += gl1[j][ch];
  }

  // block sums of h and |X - G| -> two double atomics per block
  float a = hsum, b = l1;
  for (int o = 16; o; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
  if ((tid & 31) == 0) { s_red[0][tid >> 5] = a; s_red[1][tid >> 5] = b; }
  __syncthreads();                                            // also: both warps' gradient patches are complete
  if (tid < 2) {
    const double s = (double)s_red[tid][0] + (double)s_red[tid][1];
    if (s != 0.0) atomicAdd(acc + tid, s);
  }
  if (GRAD && !sep) {
    for (int c = tid; c < kHCells; c += kHT) {
      const int cy = c / kHP, cx = c - cy * kHP;
      const int i = s_idx[cy * kHS + cx];
      if (i < 0) continue;
      float* o = dL_dX + 3 * (int64_t)i;
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) {
        float v = 0.f;
        if (cy < kGR) v += s_grad[(ch * kGR + cy) * kHS + cx];                          // warp 0: patch rows 0..17
        if (cy >= 8) v += s_grad[((3 + ch) * kGR + (cy - 8)) * kHS + cx];               // warp 1: patch rows 8..25
        if (v != 0.f) atomicAdd(o + ch, v);
      }
    }
  }
}

// loss3 = (L, L1^H, mean h) from acc = (sum h, sum |X - G|, n_valid)
__global__ void hssim_finish_kernel(const double* acc, double n_pix_full, int has_bits, double lambda, double* loss3) {
  const double n = has_bits ? acc[2] : n_pix_full;
  if (n <= 0.0) { loss3[0] = loss3[1] = loss3[2] = 0.0; return; }
  const double h = acc[0] / n, l1 = acc[1] / (3.0 * n);
  loss3[0] = (1.0 - lambda) * l1 + lambda * (1.0 - h); loss3[1] = l1; loss3[2] = h;
}

}  // namespace uts

using namespace uts;

extern "C" {

size_t uts_hssim_scratch_bytes(const uts_config*) { return 256; }

int uts_hssim_loss(const uts_config* cfg, uts_mask mask, const float* X, const float* G, float lambda, float sigma, float* h_map,
                   float* dL_dX, double* loss3, void* scratch, size_t scratch_bytes, void* stream) {
  int st = check_config(cfg);
  if (st) return st;
  st = check_mask(cfg, mask);
  if (st) return st;
  if (!loss3 || !scratch || scratch_bytes < 256 || ((uintptr_t)scratch & 7) || !(sigma > 0.f) || !(lambda >= 0.f && lambda <= 1.f))
    return UTS_ERR_INVALID_ARG;
  const Dims d = dims_of(cfg, &mask);
  cudaStream_t s = (cudaStream_t)stream;
  double* acc = (double*)scratch;
  UTS_CUDA(cudaMemsetAsync(acc, 0, 3 * sizeof(double), s));
  const bool has_bits = mask.pixel_mask_bits != nullptr;
  if (d.n_slot > 0) {
    if (!X || !G) return UTS_ERR_INVALID_ARG;
    if (dL_dX) UTS_CUDA(cudaMemsetAsync(dL_dX, 0, (size_t)d.n_slot * 256 * 3 * sizeof(float), s));
    if (has_bits) {
      hssim_count_kernel<<<(unsigned)((d.n_slot * 8 + 255) / 256), 256, 0, s>>>(d.n_slot, mask.active_tiles, mask.pixel_mask_bits, acc);
      UTS_LAUNCH_CHECK();
    }
    // tap weights (A31), double on the host, rounded once
    HssimWeights w;
    const double sg = (double)sigma, a = kPi / 4.0, b = 4.0 / kPi;
    for (int dy = -kHR; dy <= kHR; ++dy)
      for (int dx = -kHR; dx <= kHR; ++dx) {
        const int t = (dy + kHR) * kHW + (dx + kHR);
        const double ew = (double)(dx - dy), ns = (double)(dx + dy);     // east-west and north-south diagonals of the pixel
        w.w[0][t] = (float)exp(-(double)(dx * dx + dy * dy) / (2.0 * sg * sg));
        w.w[1][t] = (float)exp(-(a * ew * ew + b * ns * ns) / (4.0 * sg * sg));
      }
    if (dL_dX)
      hssim_kernel<true><<<(unsigned)d.n_slot, kHT, 0, s>>>(d.k, d.n_pix, mask.active_tiles, mask.slot_of_tile, mask.pixel_mask_bits, X, G, lambda, w,
                                                            h_map, dL_dX, acc);
    else
      hssim_kernel<false><<<(unsigned)d.n_slot, kHT, 0, s>>>(d.k, d.n_pix, mask.active_tiles, mask.slot_of_tile, mask.pixel_mask_bits, X, G, lambda, w,
                                                             h_map, dL_dX, acc);
    UTS_LAUNCH_CHECK();
  }
  hssim_finish_kernel<<<1, 1, 0, s>>>(acc, (double)d.n_pix, has_bits ? 1 : 0, (double)lambda, loss3);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // extern "C"
