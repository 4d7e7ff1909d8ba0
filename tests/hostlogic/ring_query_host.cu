// Host-side driver of the ring-interval tile query (csrc/uts_ring_query.cuh is __host__ __device__): evaluates the tile set of
// ONE disc on the CPU with exactly the code the kernels run, so that tests/test_ring_query_host.py can compare it with the
// oracle's sets without a GPU.  Test infrastructure only; not part of libuts.so.
#include "uts_ring_query.cuh"
#include <algorithm>
#include <vector>

using namespace uts;

extern "C" int ring_query_host(int kt, int kq, const float* dir, float lon, float lat, double R, uint32_t* out, int cap, int* n_rings) {
  RingDisc D;
  make_ring_disc(kq, dir, lon, lat, R, D);
  const int N = 1 << kq, Nt = 1 << kt;
  std::vector<uint32_t> tiles;
  if (D.all) {
    const int n = 12 << (2 * kt);
    for (int t = 0; t < n; ++t) tiles.push_back((uint32_t)t);
  } else {
    std::vector<int> first(D.i_hi - D.i_lo + 1), last(D.i_hi - D.i_lo + 1);
    for (int i = D.i_lo; i <= D.i_hi; ++i) ring_interval(D, N, i, first[i - D.i_lo], last[i - D.i_lo]);
    struct Tab {
      const int* first; const int* last; int i_lo;
      __host__ __device__ void operator()(int i, int& f, int& l) const { f = first[i - i_lo]; l = last[i - i_lo]; }
    } tab{first.data(), last.data(), D.i_lo};
    for (int f = 0; f < 12; ++f) {
      if (!face_in_extent(D, f)) continue;
      int S_lo, S_hi;
      face_row_range(D, kq, kt, f, S_lo, S_hi);
      for (int S = S_lo; S <= S_hi; ++S) {
        const int Hm = std::min(S, 2 * Nt - 2 - S);
        for (int jbase = 0; jbase <= Hm; jbase += 64) {
          unsigned long long mask = tile_row_mask(D, kq, kt, f, S, jbase, tab);
          while (mask) {
            const int j = __builtin_ctzll(mask);
            mask &= mask - 1;
            tiles.push_back(row_tile_index(kt, f, S, jbase + j));
          }
        }
      }
    }
  }
  if (n_rings) *n_rings = D.all ? 0 : D.i_hi - D.i_lo + 1;
  std::sort(tiles.begin(), tiles.end());
  const int n = (int)tiles.size();
  for (int k = 0; k < n && k < cap; ++k) out[k] = tiles[k];
  return n;
}
