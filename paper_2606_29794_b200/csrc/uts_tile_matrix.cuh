// uts_tile_matrix.cuh — tile-major emission of the LARGE discs for uts_tile_lists (F2 + F3 + F4 in one call).
//
// Alg.1 l.9-16 emits ((tile, rho), i) pairs per Gaussian, sorts all of them and cuts the tile ranges.  On the
// paper's kind of scene most pairs belong to a few large discs (config 4: 4 % of the Gaussians own 90 % of the 267 M pairs), and
// for those the per-Gaussian view is the wrong way round: a disc that covers thousands of tiles is better described by ONE bit per
// tile.  So the large discs (radius class chosen so that a bitmap row is cheaper than the disc's pairs through the radix sort) are
// taken out of the pair stream:
//   count     each large disc's tile set is written as a bitmap row of a (disc x tile) bit matrix, rows in (view, depth, id) order
//   transpose 32 x 32 bit blocks -> one bit VECTOR over the large discs per (view, tile), and the vectors' population counts
//   emit      a warp per (view, tile) walks its bit vector: set bit r = disc r belongs to this tile's list.  The list comes out
//             already grouped by tile and ordered by depth — no sort — with coalesced writes.
// Only the small discs' pairs go through emit + radix sort; a per-tile merge of the two depth-ordered lists gives the final
// arrays, bit-identical to uts_tile_query + uts_sort + uts_tile_ranges (tests compare both against the oracle).
// Included by uts_tile_query.cu after its ring-query helpers.
#pragma once

namespace uts {

struct MatView { uint32_t row_start, n_rows, W, pad; unsigned long long mt_base; };   // W: words of a tile's bit vector (multiple of 8)

struct MatParams {
  uint32_t* M;                     // [cap_rows][n_words] disc-major bitmaps
  uint32_t* MT;                    // view v: [n_tile][W_v] at views[v].mt_base
  unsigned long long* row_key;     // [cap_rows] (depth bits << 32) | Gaussian id
  const uint64_t* row_of_rank;     // [V*P + 1] exclusive scan of the large-disc flags in (view, depth, id) order
  MatView* views;                  // [V]
  uint32_t* large_count;           // [V * n_tile] large discs per (view, tile)
  unsigned long long* n_L;         // total number of matrix pairs
  int n_words;                     // n_tile / 32
};

// after the call: x[b] bit i == x_in[i] bit b
__device__ __forceinline__ void transpose32(uint32_t (&x)[32]) {
#pragma unroll
  for (int s = 0; s < 5; ++s) {
    const int j = 16 >> s;
    const uint32_t m = j == 16 ? 0x0000ffffu : j == 8 ? 0x00ff00ffu : j == 4 ? 0x0f0f0f0fu : j == 2 ? 0x33333333u : 0x55555555u;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      if ((k & j) == 0) {
        const uint32_t t = ((x[k] >> j) ^ x[k + j]) & m;
        x[k] ^= (t << j); x[k + j] ^= t;
      }
    }
  }
}

// flag_by_rank[emit_rank[k]] = 1 for the large discs perm[0 .. n_mat); they emit no pairs of their own: counts[slot] = 0
__global__ void mat_flag_kernel(const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small, const uint32_t* __restrict__ emit_rank,
                                uint32_t* __restrict__ flag_by_rank, uint32_t* __restrict__ counts) {
  const uint32_t n_mat = n_small[3];
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_mat; i += gridDim.x * blockDim.x) {
    const uint32_t slot = emit_rank[perm[i]];
    flag_by_rank[slot] = 1u; counts[slot] = 0u;
  }
}

// per view: its rows, the width of its bit vectors and where they start
__global__ void mat_view_tab_kernel(MatParams mp, int P, int V, int64_t n_tile) {
  if (threadIdx.x || blockIdx.x) return;
  unsigned long long base = 0;
  for (int v = 0; v < V; ++v) {
    MatView mv;
    mv.row_start = (uint32_t)mp.row_of_rank[(int64_t)v * P];
    mv.n_rows = (uint32_t)mp.row_of_rank[(int64_t)(v + 1) * P] - mv.row_start;
    mv.W = ((mv.n_rows + 255u) >> 8) << 3;
    mv.pad = 0; mv.mt_base = base;
    base += (unsigned long long)n_tile * mv.W;
    mp.views[v] = mv;
  }
}

// ---------------------------------------------------------------------------------------------- count: bitmap rows
// One block per large disc at a time.  A disc costs a chain of dependent phases (load, ring table, rows, row copy) with block-wide
// barriers between them, so what matters is how many discs an SM has in flight: blocks of kMatThreads threads.
#ifndef UTS_MAT_THREADS
#define UTS_MAT_THREADS 64
#endif
#ifndef UTS_MAT_MINB
#define UTS_MAT_MINB 16
#endif
constexpr int kMatThreads = UTS_MAT_THREADS;
// Blocks per SM the kernel is given when it runs on the side stream beside the small pairs' emit and sort (uts_tile_lists): a persistent
// grid that leaves half of the register file to them.  Measured on config 4 (tile lists): 6 -> 7.16 ms, 8 -> 7.00, 10 -> 7.09, 16 -> 7.16.
#ifndef UTS_MAT_SIDE_BLOCKS
#define UTS_MAT_SIDE_BLOCKS 8
#endif
constexpr int kMatSideBlocks = UTS_MAT_SIDE_BLOCKS;
__global__ void __launch_bounds__(kMatThreads, UTS_MAT_MINB)
matrix_count_kernel(QueryParams qp, MatParams mp, const float* __restrict__ dir, const float* __restrict__ lonlat, const float* __restrict__ rho,
                    const float* __restrict__ rs, const int32_t* __restrict__ slot_of_tile, const uint32_t* __restrict__ active_words,
                    const uint32_t* __restrict__ perm, const uint32_t* __restrict__ n_small, const uint32_t* __restrict__ emit_rank) {
  extern __shared__ int2 ring_tab[];                 // [rc_block], then the bitmap [n_words]
  uint32_t* bitmap = reinterpret_cast<uint32_t*>(ring_tab + qp.rc_block);
  __shared__ RingDisc s_disc;
  __shared__ uint16_t s_pre[13];
  __shared__ int s_Slo[12];
  __shared__ uint32_t s_total;
  const uint32_t end = n_small[3];
  const int N = 1 << qp.kq, tid = threadIdx.x;
  for (uint32_t idx = blockIdx.x; idx < end; idx += gridDim.x) {
    const int64_t k = (int64_t)perm[idx];
    const int64_t slot = (int64_t)emit_rank[k];
    const uint32_t row = (uint32_t)mp.row_of_rank[slot];
    const int v = (int)(k / qp.P);
    __syncthreads();                                   // the previous disc is done with shared memory
    if ((mp.n_words & 1) == 0) {                       // 8-byte stores (the bitmap follows an int2 array: 8-byte aligned)
      uint2* b2 = reinterpret_cast<uint2*>(bitmap);
      for (int w = tid; w < (mp.n_words >> 1); w += kMatThreads) b2[w] = make_uint2(0u, 0u);
    } else {
      for (int w = tid; w < mp.n_words; w += kMatThreads) bitmap[w] = 0u;
    }
    if (tid < 32) {                                    // set-up by the first warp: lane 0 the disc, lanes 0..11 one face each
      if (tid == 0) {
        load_ring_disc(qp, dir, lonlat, rs, k, s_disc);
        s_disc.i_hi = min(s_disc.i_hi, s_disc.i_lo + qp.rc_block - 1);
        s_total = 0;
      }
      __syncwarp();
      int nrows = 0, S_lo = 0, S_hi = -1;
      if (tid < 12 && face_in_extent(s_disc, tid)) { face_row_range(s_disc, qp.kq, qp.kt, tid, S_lo, S_hi); if (S_hi >= S_lo) nrows = S_hi - S_lo + 1; }
      int incl = nrows;
#pragma unroll
      for (int dd = 1; dd < 16; dd <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, dd); if (tid >= dd) incl += y; }
      if (tid < 12) { s_pre[tid] = (uint16_t)(incl - nrows); int a, b; face_row_range(s_disc, qp.kq, qp.kt, tid, a, b); s_Slo[tid] = a; }
      if (tid == 11) s_pre[12] = (uint16_t)incl;
    }
    __syncthreads();
    const RingDisc& D = s_disc;
    if (D.all) {                                       // reading A24: every active tile
      for (int w = tid; w < mp.n_words; w += kMatThreads) bitmap[w] = active_words ? __ldg(active_words + w) : 0xffffffffu;
      if (tid == 0) s_total = qp.active_tiles ? (uint32_t)qp.n_active : (uint32_t)qp.n_tile;
    } else {
      for (int e = tid; e <= D.i_hi - D.i_lo; e += kMatThreads) { int2 fl; ring_interval(D, N, D.i_lo + e, fl.x, fl.y); ring_tab[e] = fl; }
      __syncthreads();
      const GroupTab T{ring_tab, D.i_lo};
      const int n_rows = (int)s_pre[12];
      const int n_chunks = ((1 << qp.kt) + 63) >> 6;
      const int n_items = n_rows * n_chunks;
      uint32_t mine = 0;
      for (int item = tid; item < n_items; item += kMatThreads) {
        const int rowi = item / n_chunks, jbase = (item - rowi * n_chunks) << 6;
        int f = 0;
        while (f < 11 && (int)s_pre[f + 1] <= rowi) ++f;
        const int S = s_Slo[f] + rowi - (int)s_pre[f];
        if (jbase > min(S, (2 << qp.kt) - 2 - S)) continue;
        const unsigned long long mask = filter_row_chunk(qp.kt, f, S, jbase, tile_row_mask(D, qp.kq, qp.kt, f, S, jbase, T), slot_of_tile);
        if (!mask) continue;
        mine += (uint32_t)__popcll(mask);
        visit_row_chunk<true>(qp.kt, f, S, jbase, mask, nullptr, [&](uint32_t tile) { atomicOr(&bitmap[tile >> 5], 1u << (tile & 31)); });
      }
      if (mine) atomicAdd(&s_total, mine);
    }
    __syncthreads();
    uint32_t* dst = mp.M + (size_t)row * mp.n_words;
    if ((mp.n_words & 1) == 0) {                       // rows of M are 8-byte aligned when n_words is even
      uint2* d2 = reinterpret_cast<uint2*>(dst);
      const uint2* b2 = reinterpret_cast<const uint2*>(bitmap);
      for (int w = tid; w < (mp.n_words >> 1); w += kMatThreads) d2[w] = b2[w];
    } else {
      for (int w = tid; w < mp.n_words; w += kMatThreads) dst[w] = bitmap[w];
    }
    if (tid == 0) {
      const uint32_t gid = (uint32_t)(k - (int64_t)v * qp.P);
      mp.row_key[row] = ((unsigned long long)__float_as_uint(__ldg(rho + k)) << 32) | gid;        // reading A10
      atomicAdd(mp.n_L, (unsigned long long)s_total);
    }
  }
}

// ---------------------------------------------------------------------------------------------- transpose
// block = 256 local rows of one view x 32 word columns (1024 tiles); warp w transposes rows [32 w, 32 w + 32) in registers
__global__ void __launch_bounds__(256)
matrix_transpose_kernel(MatParams mp, int V, int64_t n_tile) {
  __shared__ uint32_t sT[8][32 * 33];
  // which view does row block blockIdx.y belong to?
  int v = 0; uint32_t rb = blockIdx.y;
  for (; v < V; ++v) { const uint32_t nb = (mp.views[v].n_rows + 255u) >> 8; if (rb < nb) break; rb -= nb; }
  if (v == V) return;
  const MatView mv = mp.views[v];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int c = blockIdx.x * 32 + lane;                        // word column
  uint32_t x[32];
  const uint32_t r0 = rb * 256u + (uint32_t)wid * 32u;         // local row of x[0]
#pragma unroll
  for (int i = 0; i < 32; ++i) {
    const uint32_t lr = r0 + (uint32_t)i;
    x[i] = (lr < mv.n_rows && c < mp.n_words) ? __ldg(mp.M + (size_t)(mv.row_start + lr) * mp.n_words + c) : 0u;
  }
  transpose32(x);                                              // x[b] = bits of tile 32 c + b over the 32 rows
#pragma unroll
  for (int b = 0; b < 32; ++b) sT[wid][lane * 33 + b] = x[b];
  __syncthreads();
  uint32_t* out = mp.MT + mv.mt_base;
  for (int q = 0; q < 4; ++q) {
    const int tl = threadIdx.x + 256 * q;                      // tile inside the slab
    const int cc = tl >> 5, b = tl & 31;
    const int64_t tile = ((int64_t)blockIdx.x * 32 + cc) * 32 + b;
    if (tile >= n_tile) continue;
    uint4 lo, hi;
    lo.x = sT[0][cc * 33 + b]; lo.y = sT[1][cc * 33 + b]; lo.z = sT[2][cc * 33 + b]; lo.w = sT[3][cc * 33 + b];
    hi.x = sT[4][cc * 33 + b]; hi.y = sT[5][cc * 33 + b]; hi.z = sT[6][cc * 33 + b]; hi.w = sT[7][cc * 33 + b];
    uint4* dst = reinterpret_cast<uint4*>(out + (size_t)tile * mv.W + (size_t)rb * 8);
    dst[0] = lo; dst[1] = hi;
    // large_count[(v, tile)] (zeroed by the caller): this block's 256 rows of the tile's bit vector
    const uint32_t c = (uint32_t)(__popc(lo.x) + __popc(lo.y) + __popc(lo.z) + __popc(lo.w) + __popc(hi.x) + __popc(hi.y) + __popc(hi.z) + __popc(hi.w));
    if (c) atomicAdd(mp.large_count + (size_t)v * (size_t)n_tile + (size_t)tile, c);
  }
}

// ---------------------------------------------------------------------------------------------- emit + merge
// Inside one (view, tile) list every key has the same high word, so an entry is ordered by (depth bits, Gaussian id) alone: the
// merge buffers hold that pair packed in one 64-bit word, (depth << 32) | id — the form row_key already has — and one unsigned
// compare orders two entries.
// number of entries of the sorted buffer b[0, n) that are less than x
__device__ __forceinline__ uint32_t buf_lower_bound(const unsigned long long* b, uint32_t n, unsigned long long x) {
  uint32_t lo = 0, hi = n;
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (b[mid] < x) lo = mid + 1; else hi = mid; }
  return lo;
}

// One warp per (view, tile) writes the tile's FINAL list at keys / vals[start[vt] ...): a streaming merge of two depth-ordered
// streams held in shared memory 256 entries at a time —
//   A: the large discs of the tile, generated from its bit vector (set bit r = matrix row r; entry = row_key[r]),
//   B: the tile's small-disc pairs, already radix-sorted (keysS / valsS[s_ranges[vt] ...)).
// Each round refills both buffers, emits everything up to the smaller of the two "last buffered" entries of streams that still
// continue (so nothing that could precede an emitted entry is still unread) and stores every emitted entry straight at its final
// position, own index + rank in the other buffer (the two streams never tie: different Gaussians) — consecutive lanes hit nearly
// consecutive addresses.  Ranks: the B entries (the minority) by binary search in A; the A entries from those — B[j] precedes A[i]
// iff rank_A(B[j]) <= i, so a histogram of the B ranks over the A positions, prefix-summed by the warp, is every A entry's rank at
// once (a binary search per A entry was half of this kernel's instructions).  Then the unconsumed entries shift to the front;
// one buffer is fully consumed per round.
#ifndef UTS_MB
#define UTS_MB 256
#endif
#ifndef UTS_MB_MINB
#define UTS_MB_MINB 4
#endif
constexpr int kMB = UTS_MB;
static_assert(kMB == 256, "the rank scan below gives every lane 8 consecutive A positions");
__global__ void __launch_bounds__(256, UTS_MB_MINB)
matrix_emit_merge_kernel(MatParams mp, int V, int64_t n_tile, const uint64_t* __restrict__ start, const uint64_t* __restrict__ s_ranges,
                         const uint64_t* __restrict__ keysS, const uint32_t* __restrict__ valsS, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  __shared__ unsigned long long sA[8][kMB], sB[8][kMB];
  __shared__ __align__(16) uint32_t sH[8][kMB];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned long long* A = sA[wid]; unsigned long long* Bq = sB[wid];
  uint32_t* H = sH[wid];
  const int64_t n = (int64_t)V * n_tile;
  for (int64_t vt = (int64_t)blockIdx.x * 8 + wid; vt < n; vt += (int64_t)gridDim.x * 8) {
    uint64_t o = start[vt];
    if (start[vt + 1] == o) continue;
    uint64_t b_pos = s_ranges[2 * vt];
    const uint64_t b_end = s_ranges[2 * vt + 1];
    const int v = (int)(vt / n_tile);
    const MatView mv = mp.views[v];
    const uint32_t* bvec = mp.MT + mv.mt_base + (size_t)(vt - (int64_t)v * n_tile) * mv.W;
    const unsigned long long hi = (unsigned long long)vt << 32;
    uint32_t w_next = 0, w_cur = 0, x = 0;               // A stream: next chunk, current chunk, this lane's unread bits of it
    bool a_done = mv.W == 0 || mp.large_count[vt] == 0;
    uint32_t x_pref = (!a_done && (uint32_t)lane < mv.W) ? __ldg(bvec + lane) : 0u;     // the next chunk's word, fetched one chunk ahead
    uint32_t fillA = 0, fillB = 0;
    __syncwarp();
    for (;;) {
      // ---- refill A from the bit vector
      const uint32_t fillA0 = fillA;
      while (fillA < (uint32_t)kMB && !a_done) {
        if (!__any_sync(0xffffffffu, x != 0u)) {
          if (w_next >= mv.W) { a_done = true; break; }
          w_cur = w_next; w_next += 32;
          x = x_pref;
          x_pref = (w_next + lane < mv.W) ? __ldg(bvec + w_next + lane) : 0u;
          if (!__any_sync(0xffffffffu, x != 0u)) continue;
        }
        const uint32_t c = (uint32_t)__popc(x);
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
        const uint32_t tot = __shfl_sync(0xffffffffu, incl, 31);
        const uint32_t room = (uint32_t)kMB - fillA;
        uint32_t r = incl - c;
        const uint32_t row0 = (w_cur + lane) * 32;
        while (x && r < room) {                            // phase 1: matrix rows of the set bits (no memory access)
          const int b = __ffs((int)x) - 1; x &= x - 1;
          A[fillA + r] = row0 + (uint32_t)b; ++r;
        }
        fillA += tot < room ? tot : room;
      }
      __syncwarp();
      // phase 2: the rows' (depth, id) in one batch of independent loads
      {
        const unsigned long long* rk = mp.row_key + mv.row_start;
#pragma unroll
        for (int q = 0; q < kMB / 32; ++q) {
          const uint32_t i = fillA0 + lane + 32 * q;
          if (i < fillA) A[i] = __ldg(rk + (uint32_t)A[i]);
        }
      }
      // ---- refill B from the sorted small pairs
      if (fillB < (uint32_t)kMB && b_pos < b_end) {
        const uint32_t take = (uint32_t)(((uint64_t)kMB - fillB) < (b_end - b_pos) ? ((uint64_t)kMB - fillB) : (b_end - b_pos));
        for (uint32_t j = lane; j < take; j += 32) Bq[fillB + j] = (keysS[b_pos + j] << 32) | valsS[b_pos + j];
        b_pos += take; fillB += take;
      }
      __syncwarp();
      if (fillA == 0 && fillB == 0) break;
      const bool b_done = b_pos == b_end;
      uint32_t na = fillA, nb = fillB;
      if (fillA && fillB && !(a_done && b_done)) {
        const bool lastA_smaller = A[fillA - 1] < Bq[fillB - 1];
        const bool bound_is_A = !a_done && (b_done || lastA_smaller);
        if (bound_is_A) nb = buf_lower_bound(Bq, fillB, A[fillA - 1]);
        else na = buf_lower_bound(A, fillA, Bq[fillB - 1]);
      } else if (fillA && !fillB && !b_done) { na = 0; }      // cannot happen: B is refilled whenever it has entries left
      // ---- rank and store
      if (nb == 0) {
        for (uint32_t i = lane; i < na; i += 32) { const unsigned long long p = A[i]; keys[o + i] = hi | (p >> 32); vals[o + i] = (uint32_t)p; }
      } else {
        if (na) {
#pragma unroll
          for (int q = 0; q < kMB / 32; ++q) H[lane + 32 * q] = 0u;
          __syncwarp();
        }
        for (uint32_t j = lane; j < nb; j += 32) {
          const unsigned long long p = Bq[j];
          const uint32_t rb = buf_lower_bound(A, na, p);
          if (rb < na) atomicAdd(&H[rb], 1u);              // B[j] precedes A[rb], A[rb+1], ...
          const uint64_t pos = o + j + rb;
          keys[pos] = hi | (p >> 32); vals[pos] = (uint32_t)p;
        }
        if (na) {
          __syncwarp();
          // inclusive prefix sum of H over the A positions: lane l owns positions 8l .. 8l+7
          uint4 h0 = reinterpret_cast<uint4*>(H)[2 * lane], h1 = reinterpret_cast<uint4*>(H)[2 * lane + 1];
          h0.y += h0.x; h0.z += h0.y; h0.w += h0.z; h1.x += h0.w; h1.y += h1.x; h1.z += h1.y; h1.w += h1.z;
          uint32_t incl = h1.w;
#pragma unroll
          for (int d = 1; d < 32; d <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
          const uint32_t ex = incl - h1.w;
          h0.x += ex; h0.y += ex; h0.z += ex; h0.w += ex; h1.x += ex; h1.y += ex; h1.z += ex; h1.w += ex;
          reinterpret_cast<uint4*>(H)[2 * lane] = h0; reinterpret_cast<uint4*>(H)[2 * lane + 1] = h1;
          __syncwarp();
          for (uint32_t i = lane; i < na; i += 32) {
            const unsigned long long p = A[i];
            const uint64_t pos = o + i + H[i];
            keys[pos] = hi | (p >> 32); vals[pos] = (uint32_t)p;
          }
        }
      }
      o += na + nb;
      // ---- shift the unconsumed entries to the front
      unsigned long long tk[kMB / 32];
#pragma unroll
      for (int q = 0; q < kMB / 32; ++q) { const uint32_t i = na + lane + 32 * q; if (i < fillA) tk[q] = A[i]; }
      __syncwarp();
#pragma unroll
      for (int q = 0; q < kMB / 32; ++q) { const uint32_t i = na + lane + 32 * q; if (i < fillA) A[i - na] = tk[q]; }
      fillA -= na;
#pragma unroll
      for (int q = 0; q < kMB / 32; ++q) { const uint32_t i = nb + lane + 32 * q; if (i < fillB) tk[q] = Bq[i]; }
      __syncwarp();
#pragma unroll
      for (int q = 0; q < kMB / 32; ++q) { const uint32_t i = nb + lane + 32 * q; if (i < fillB) Bq[i - nb] = tk[q]; }
      fillB -= nb;
      __syncwarp();
    }
  }
}

// ---------------------------------------------------------------------------------------------- totals, ranges
// total[vt] = large discs + small pairs of (view, tile)
__global__ void mat_totals_kernel(int64_t n, const uint32_t* __restrict__ large_count, const uint64_t* __restrict__ s_ranges, uint32_t* __restrict__ total) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) total[i] = large_count[i] + (uint32_t)(s_ranges[2 * i + 1] - s_ranges[2 * i]);
}
// ranges[vt] = [start, end) of the final arrays, (0,0) for an empty tile (as uts_tile_ranges)
__global__ void mat_ranges_kernel(int64_t n, const uint64_t* __restrict__ start, uint64_t* __restrict__ ranges) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint64_t a = start[i], b = start[i + 1];
  ranges[2 * i] = a == b ? 0 : a; ranges[2 * i + 1] = a == b ? 0 : b;
}

}  // namespace uts
