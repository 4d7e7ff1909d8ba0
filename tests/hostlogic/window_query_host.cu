// Host-side driver of the small-disc window query (csrc/uts_window_query.cuh is __host__ __device__): the tile set of ONE disc, the
// angle -> cell map and the face gluing, evaluated on the CPU with exactly the code the kernel runs, so that
// tests/test_window_query_host.py can compare them with the oracle without a GPU.  Test infrastructure only; not part of libuts.so.
#include "uts_window_query.cuh"
#include <algorithm>
#include <vector>

using namespace uts;

// returns the number of tiles (sorted ascending in out), or -1 when the disc needs a wider window than kWindowMax
extern "C" int window_query_host(int kt, int kq, const float* dir, double R, double rho_t, const int32_t* slot_of_tile, uint32_t* out, int cap) {
  WindowDisc D;
  make_window_disc(kt, dir, R, rho_t, D);
  if (D.w > kWindowMax || (1 << kt) < 2 * kWindowMax + 1) return -1;
  std::vector<uint32_t> tiles;
  window_query(D, kt, kq, slot_of_tile, [&](uint32_t t) { tiles.push_back(t); });
  std::sort(tiles.begin(), tiles.end());
  const int n = (int)tiles.size();
  for (int k = 0; k < n && k < cap; ++k) out[k] = tiles[k];
  return n;
}

// NESTED pixel of the unit vectors u[n][3] at `order`
extern "C" void vec_to_pixel_host(int order, int64_t n, const double* u, int64_t* out) {
  for (int64_t i = 0; i < n; ++i) {
    int f, x, y;
    vec_to_cell(order, u + 3 * i, f, x, y);
    out[i] = ((int64_t)f << (2 * order)) | win_spread16((uint32_t)x) | ((int64_t)win_spread16((uint32_t)y) << 1);
  }
}

// NESTED pixel of cell (X, Y) of the extended frame of face f, or -1
extern "C" int64_t extended_cell_host(int order, int f, int X, int Y) {
  int g, x, y;
  if (!extended_cell(order, f, X, Y, g, x, y)) return -1;
  return ((int64_t)g << (2 * order)) | win_spread16((uint32_t)x) | ((int64_t)win_spread16((uint32_t)y) << 1);
}

// fp32 and double centres of NESTED-decoded cell, for the accuracy check
extern "C" void cell_centers_host(int order, int f, int x, int y, float* c32, double* c64) {
  cell_center_f32(order, f, x, y, c32[0], c32[1], c32[2]);
  cell_center_f64(order, f, x, y, c64[0], c64[1], c64[2]);
}
