/* uts.h — C ABI of the B200-native HEALPix spherical Gaussian-splat rasteriser (libuts.so).
 *
 * One entry point per stage of UniTriSplat's Alg.1 and of its backward:
 *
 *   uts_preprocess      Alg.1 l.2-8   (Eq.1-2): projection to the unit sphere, Sigma_arc, conic, r_s, colour
 *   uts_depth_order     (optional) radial-depth order of the Gaussians, lets the sort skip its depth passes
 *   uts_tile_query      Alg.1 l.9-14  (Alg.2; Alg.3 PAPER.md:635-684 with query_mode = RING): tile query, emits
 *                       ((tile,rho),i) pairs
 *   uts_sort            Alg.1 l.15: stable radix sort of the pairs by (tile, radial depth)
 *   uts_tile_ranges     Alg.1 l.16: per-tile [start,end)
 *   uts_render_fwd      Alg.1 l.17-30 (Eq.6) + FoV mask
 *   uts_render_bwd      backward of Eq.6
 *   uts_render_fwd_marked / uts_render_bwd_marked   the same pair; the forward records which (warp, entry) pairs blended anything and
 *                       the backward visits only those (same image, same gradient sums)
 *   uts_preprocess_bwd  Eq.3-4: to means, scales, rotations, SH
 *   uts_hssim_loss      L1 + HEALPix-SSIM loss and dL/dI (Eq.10): produces uts_render_bwd's upstream gradient
 *
 * Conventions
 *   - extern "C"; every call returns an int status (UTS_OK = 0).  Nothing throws, aborts, allocates or frees
 *     device memory: THE CALLER OWNS EVERY BUFFER, including scratch (sizes from uts_*_scratch_bytes).
 *   - Every pointer is a DEVICE pointer unless its name starts with h_ (host; pinned where it is written
 *     asynchronously).  uts_config is read on the host.  The only calls taking host data arrays are the
 *     uts_host_* calls at the end.
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*); calls are asynchronous.  Where a host
 *     count is returned (h_n_pairs) the call synchronises the stream before returning, as documented there.
 *   - Library state: the last CUDA error code, the launch counter, and ONE CONTEXT PER DEVICE, created on the first call made with
 *     that device current and kept until the process ends: the SM count, cached occupancy numbers, three auxiliary streams with their
 *     fork / join events (uts_tile_query / uts_tile_lists run independent kernels side by side on them and join back into
 *     `stream` before returning), one copy stream with four events (uts_host_forward_backward) and 64 bytes of pinned host
 *     memory (the pair counts of uts_tile_lists come back in one copy).  A per-device mutex is held while a call enqueues on
 *     those streams (uts_tile_lists: from its count pass to its last launch, its host read of the pair count included), so calls
 *     may be issued from several threads and on several streams; they never read the environment.  No CPU fallback; sm_100 only.
 *   - Inputs are ACTIVATED values: scales > 0, opacity in (0,1), quaternion (w,x,y,z) used as given
 *     (reading A14).  Arrays are dense row-major float32 unless stated.
 *   - Index conventions: NESTED pixel p = f*4^k + interleave(x,y); tile of p = p >> (2*tile_log2); pixel slot
 *     inside a tile = p & (4^tile_log2 - 1)  (Alg.1 l.18 PAPER.md:564).
 */
#ifndef UTS_H_
#define UTS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  UTS_OK = 0,
  UTS_ERR_INVALID_ARG = 1, /* null pointer, out-of-range config field, misaligned buffer */
  UTS_ERR_CAPACITY = 2,    /* a caller buffer is too small; the needed size is written to the documented out-param */
  UTS_ERR_CUDA = 3,        /* a CUDA runtime call failed; uts_last_cuda_error() returns the cudaError_t */
  UTS_ERR_UNSUPPORTED = 4  /* device is not sm_100, or a config combination that is not implemented */
};

/* POD, host memory, passed by const pointer.  Field meaning follows Alg.1's Require line. */
typedef struct {
  int   order;             /* k; Nside = 1<<k; tile_log2 <= k <= 13 */
  int   tile_log2;         /* l; B = 1<<l pixels per tile side; only 4 (16x16) is implemented     Table 6 */
  int   query_refine_log2; /* log2 f; query pixels are at order k_q = k - l + log2 f; 0..l */
  int   sh_degree;         /* 0..3; M = (sh_degree+1)^2 coefficients per channel */
  int   n_gauss;           /* P */
  int   n_views;           /* V >= 1 */
  float r_near;            /* cull rho <= r_near                                                   reading A5 */
  float cov_dilation_px2;  /* h = value * 4pi/N_pix added to diag(Sigma_arc); 0 disables           reading A3 */
  float alpha_min;         /* skip alpha < alpha_min                                               reading A7 */
  float alpha_max;         /* alpha = min(alpha_max, o*exp(power)); gradient zero when clamped     reading A7 */
  float t_eps;             /* stop after the update when T < t_eps                                 Alg.1 l.27 PAPER.md:578 */
  float bg[3];             /* out = C + T*bg                                                       reading A8 */
  int   query_mode;        /* UTS_QUERY_NESTED (0): Alg.2's set, centres within r_s + PixRad(k_q)  PAPER.md:599-620, reading A6
                              UTS_QUERY_RING   (1): Alg.3's set, centres within r_s (the paper's default "R", non-conservative)
                                                                                                   PAPER.md:104-108, 635-684 */
} uts_config;

enum { UTS_QUERY_NESTED = 0, UTS_QUERY_RING = 1 };

/* Gaussian set G = {mu, s, q, o, c} (Alg.1 Require), SoA. */
typedef struct {
  const float* means;  /* [P,3] world space */
  const float* scales; /* [P,3] */
  const float* quats;  /* [P,4] (w,x,y,z) */
  const float* opac;   /* [P]   */
  const float* sh;     /* [P,M,3] */
} uts_gaussians;

/* Views V = [W|b], t = W mu + b. */
typedef struct {
  const float* W; /* [V,9] row-major 3x3 */
  const float* b; /* [V,3] */
} uts_views;

/* Projected Gaussian records written by uts_preprocess, read by every later stage. */
typedef struct {
  float*   dir;        /* [V,P,3] unit direction t/rho in the camera frame                        Eq.1 */
  float*   lonlat;     /* [V,P,2] (omega, phi) = (atan2(tx,tz), atan2(ty, hypot(tx,tz)))          Eq.1 */
  float*   rho;        /* [V,P]   radial depth ||t||; its fp32 bit pattern is the sort depth      PAPER.md:112, reading A10 */
  float*   conic_opac; /* [V,P,4] (A,B,C,o): power = -1/2 (A dx^2 + C dy^2) - B dx dy             Eq.2 inverse, Alg.1 l.23 */
  float*   rs;         /* [V,P]   r_s = min(pi, 3 sqrt(lambda_max(Sigma_arc))) */
  float*   rgb;        /* [V,P,3] max(0, 0.5 + sum_m Y_m sh_m)                                    reading A13 */
  uint8_t* flags;      /* [V,P]   bit0 culled (no tiles, no gradient); bits1-3 R,G,B clamped at 0 */
} uts_proj;

/* FoV mask M_C (reading A19).  All NULL and n_active = -1  =>  full sphere, slot == tile.
 * Otherwise all four are required. */
typedef struct {
  const uint32_t* active_tiles;    /* [n_active] ascending tile ids that contain at least one visible pixel */
  int             n_active;
  const int32_t*  slot_of_tile;    /* [N_tile] index into active_tiles, or -1 */
  const uint32_t* pixel_mask_bits; /* [N_pix/32] bit (p & 31) of word p>>5 is M_C(p), NESTED order */
} uts_mask;

/* Optional steering of the tile query's implementation choices (tests and A/B measurements).  Production passes NULL, which is
 * the same as every field 0.  None of these changes the result: the tile set, the sorted arrays and the ranges are bit-identical
 * for every setting. */
typedef struct {
  int   query_impl;        /* 0: ring intervals (uts_ring_query.cuh) when k_q <= 12, else the quadtree descent;
                              1: always the quadtree descent — Alg.2's depth-first form, stackless */
  float descent_block_radius; /* descent only: discs with R > value / sqrt(N_tile) take the block-per-Gaussian bitmap path; 0 = 36 */
  int   descent_blocks_per_sm;/* descent only: persistent blocks per SM of that path; 0 = 2 */
  int   matrix_off;        /* uts_tile_lists: 1 = never route discs through the (disc x tile) bit matrix */
  float matrix_min_tiles;  /* uts_tile_lists: discs covering at least this many tiles become matrix rows; 0 = max(48, N_tile / 144) */
  int   window_mode;       /* tile window for the smallest discs (uts_window_query.cuh) instead of ring intervals: 0 = when the mask
                              keeps at most a quarter of the tiles (where it was measured to pay), 1 = never, 2 = always */
} uts_tuning;

/* ---------------------------------------------------------------------------------------------- forward */

/* Alg.1 l.2-8.  For each view v and Gaussian i fills every array of `out` at index v*P+i.  Culled records
 * (rho <= r_near, non-finite input, det(Sigma_arc) <= 0) are written as zeros with flags bit0 set. */
int uts_preprocess(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream);
/* uts_preprocess in two calls, for callers that get the SH coefficients later than the geometry (the host call uploads them while the
 * tile lists are built): uts_preprocess_geometry writes every array of `out` except rgb and needs no g.sh (flags: bit0 only);
 * uts_preprocess_color then writes rgb and the clamp bits of flags from g.means, g.sh and the views (it reads flags bit0).
 * geometry followed by color leaves `out` bit-identical to uts_preprocess. */
int uts_preprocess_geometry(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream);
int uts_preprocess_color(const uts_config* cfg, uts_gaussians g, uts_views views, uts_proj out, void* stream);

/* Optional, Alg.1 l.15 moved ahead of the query: emit_rank[v*P+i] = position of (v,i) in the
 * stable order by (view, float_bits(rho), i).  Passing it to uts_tile_query makes the pairs come out already ordered by radial
 * depth, so that uts_sort(depth_presorted = 1) only has to run its (view,tile) passes; the sorted result is bit-identical.
 * scratch: uts_depth_order_scratch_bytes(cfg) bytes, 256-byte aligned. */
int uts_depth_order(const uts_config* cfg, const float* rho /*[V,P]*/, uint32_t* emit_rank /*[V*P]*/, void* scratch,
                    size_t scratch_bytes, void* stream);
size_t uts_depth_order_scratch_bytes(const uts_config* cfg);
/* uts_depth_order for callers that cannot allocate device memory (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same kernels and the same emit_rank, bit for bit, with the scratch in a 7 MiB file-scope device array of the
 * library (held by every GPU that loads the library until the process exits).  Limit: n_gauss * n_views <=
 * UTS_DEPTH_ORDER_STATIC_MAX = uts_depth_order_static_max(); beyond it the call enqueues nothing and returns UTS_ERR_CAPACITY.
 * The call itself allocates and frees nothing; the first call on a device looks the array's address up (cudaGetSymbolAddress) and
 * creates the device context.  ALL calls share the one array, whose contents are those of the last call (nothing in it needs
 * clearing: every region is written before it is read): two calls that overlap on the GPU — different streams, or graph branches
 * without an edge between them — RACE; order them on one stream or with an event. */
#define UTS_DEPTH_ORDER_STATIC_MAX 262144
uint64_t uts_depth_order_static_max(void);
int uts_depth_order_static(const uts_config* cfg, const float* rho /*[V,P]*/, uint32_t* emit_rank /*[V*P]*/, void* stream);

/* Alg.1 l.9-14 with Alg.2 (reading A6) or, with cfg->query_mode = UTS_QUERY_RING, Alg.3.  The tile set of (v,i) is
 *     { q >> 2(k_q-k_t) : q an order-k_q NESTED pixel with  u . centre(q) >= cos R } ∩ active tiles,
 *     R = min(pi, r_s + rho_max(k_q)) (NESTED set)  or  min(pi, r_s) (RING set),
 * the predicate evaluated in double precision wherever single precision cannot decide it.  Reads in.dir, in.lonlat, in.rho,
 * in.rs, in.flags.  Pairs are written Gaussian by Gaussian; the pairs of one (v,i) are contiguous (offsets) and its tiles are
 * distinct, but their ORDER INSIDE THAT SEGMENT IS UNSPECIFIED (no two keys of a segment tie, so uts_sort's result does not
 * depend on it):
 *     keys[j] = ((v*N_tile + tile) << 32) | float_bits(rho[v,i]),   vals[j] = i.
 * emit_rank == NULL: Gaussians in (view, Gaussian id) order (slot of (v,i) = v*P+i).  Otherwise slot = emit_rank[v*P+i]
 * (a permutation of 0..V*P-1, e.g. from uts_depth_order).  offsets[V*P+1] (exclusive scan of the per-slot counts) is always
 * written.  The call synchronises `stream` and writes the pair count to *h_n_pairs (host).  keys == NULL: count only.
 * If the count exceeds `capacity` nothing is emitted and UTS_ERR_CAPACITY is returned (*h_n_pairs = needed capacity).
 * scratch: uts_tile_query_scratch_bytes(cfg) bytes, 256-byte aligned. */
int uts_tile_query(const uts_config* cfg, uts_proj in, uts_mask mask, const uint32_t* emit_rank, uint64_t* offsets,
                   uint64_t* keys, uint32_t* vals, uint64_t capacity, uint64_t* h_n_pairs, void* scratch,
                   size_t scratch_bytes, const uts_tuning* tuning /* may be NULL */, void* stream);

/* F2 + F3 + F4 in one call (Alg.1 l.9-16): the sorted pair arrays and the tile ranges, bit-identical to
 *     uts_tile_query(emit_rank) -> uts_sort(depth_presorted = 1) -> uts_tile_ranges,
 * without sending every pair through the sort.  Discs that cover many tiles (a radius class chosen so that one bitmap row over the
 * tiles is cheaper than the disc's pairs through the radix sort) are recorded as rows of a (disc x tile) bit matrix in depth
 * order; the matrix is transposed and every (view, tile) reads its list of large discs off its own bit vector, already grouped
 * by tile and ordered by depth.  Only the remaining discs' pairs are emitted and radix-sorted; a per-tile merge of the two
 * depth-ordered lists writes keys / vals.
 * emit_rank: uts_depth_order's output (required).  keys, vals, keys_tmp, vals_tmp: `capacity` entries each; ranges [V*N_tile][2].
 * The call synchronises `stream` once (pair counts) and writes the pair count to *h_n_pairs; if it exceeds `capacity` nothing is
 * emitted and UTS_ERR_CAPACITY is returned.  scratch: uts_tile_lists_scratch_bytes(cfg) bytes, sort_scratch:
 * uts_sort_scratch_bytes(capacity) bytes, both 256-byte aligned. */
size_t uts_tile_lists_scratch_bytes(const uts_config* cfg);
int uts_tile_lists(const uts_config* cfg, uts_proj in, uts_mask mask, const uint32_t* emit_rank, uint64_t* keys, uint32_t* vals,
                   uint64_t* keys_tmp, uint32_t* vals_tmp, uint64_t capacity, uint64_t* ranges, uint64_t* h_n_pairs, void* scratch,
                   size_t scratch_bytes, void* sort_scratch, size_t sort_scratch_bytes, const uts_tuning* tuning /* may be NULL */,
                   void* stream);
size_t uts_tile_query_scratch_bytes(const uts_config* cfg);

/* Alg.1 l.15.  Stable ascending LSD radix sort on the 64-bit key (ties keep emission order; with emission in Gaussian-id
 * or depth order that is ascending Gaussian id, reading A9).  depth_presorted != 0: the pairs were emitted through
 * uts_depth_order's emit_rank, only the (view,tile) bytes are sorted.  Result is left in keys/vals; keys_tmp/vals_tmp are
 * ping-pong buffers of the same size.  scratch: uts_sort_scratch_bytes(n_pairs) bytes, 256-byte aligned. */
int uts_sort(const uts_config* cfg, uint64_t n_pairs, uint64_t* keys, uint32_t* vals, uint64_t* keys_tmp,
             uint32_t* vals_tmp, int depth_presorted, void* scratch, size_t scratch_bytes, void* stream);
size_t uts_sort_scratch_bytes(uint64_t n_pairs);

/* Alg.1 l.16.  ranges[(v*N_tile + tile)*2 + {0,1}] = [start,end) in the sorted arrays; empty tiles get (0,0). */
int uts_tile_ranges(const uts_config* cfg, uint64_t n_pairs, const uint64_t* keys, uint64_t* ranges, void* stream);

/* Alg.1 l.17-30 + mask.  S = n_active (or N_tile on the full sphere); pixel index inside a slot is p & 255.
 * color [V,S*256,3], alpha [V,S*256] (= 1 - T), trans [V,S*256] (the final transmittance T itself, kept for the
 * backward because 1 - alpha loses it to rounding when T is small), n_last [V,S*256] (1 + list position of the
 * last contributing entry, 0 if none).  Masked-out pixels get color 0, alpha 0, trans 1, n_last 0.
 * Entry order inside a tile is the order of `vals`. */
int uts_render_fwd(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                   float* color, float* alpha, float* trans, uint32_t* n_last, void* stream);

/* uts_render_fwd that also counts its work (measurement only: bench.py's roofline lines), walking every entry in full, i.e. without
 * the patch cull of the production kernels (its image is the reference of their bit-identity).  Adds to work[0] the
 * (pixel, entry) pairs Alg.1's loop evaluates (every entry a pixel visits before it stops, l.20-28 PAPER.md:568-584), to work[1] those
 * that contribute (alpha >= alpha_min), to work[2] those the production forward evaluates (the entry passes the patch cull) and
 * to work[3] those of work[2] whose patch has an open pixel with q above the alpha_min cut (what a patch-level early out on q alone
 * would leave; informational, the production forward takes no such early out).  work: 4 DEVICE uint64, zeroed by the caller.  Outputs as
 * uts_render_fwd. */
int uts_render_fwd_counted(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                           float* color, float* alpha, float* trans, uint32_t* n_last, uint64_t* work, void* stream);

/* --------------------------------------------------------------------------------------------- backward */

/* Backward of the blend.  trans and n_last are uts_render_fwd's outputs.  dL_dalpha may be NULL.  Outputs are zeroed by the call, then accumulated with
 * warp-reduced atomics (summation order is not deterministic):
 * dL_drgb [V,P,3], dL_dconic [V,P,3] (off-diagonal stored once, reading A15), dL_dmu2 [V,P,2] (gradient
 * w.r.t. the projected mean mu' = (omega, phi)), dL_dopac [P] (summed over views). */
int uts_render_bwd(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                   const float* trans, const uint32_t* n_last, const float* dL_dcolor, const float* dL_dalpha,
                   float* dL_drgb, float* dL_dconic, float* dL_dmu2, float* dL_dopac, void* stream);

/* The blend pair with MARKS: uts_render_fwd_marked also records, per warp of a tile's thread block (8 warps of 32 pixels) and list
 * entry, whether any of the warp's pixels blended the entry; uts_render_bwd_marked visits only the marked (warp, entry) pairs.
 * Outputs are those of uts_render_fwd / uts_render_bwd (same decisions per pixel: the image is bit-identical, the gradients are the
 * same sums in a possibly different order).  marks: uts_render_marks_bytes(cfg, pair_capacity) bytes, 4-byte aligned, written by
 * the forward, read by the backward.  It need not be cleared: the forward writes every word that describes an entry one of the warp's
 * pixels reached, and stale bits beyond cost the backward one vote each, never a wrong sum with the same cfg / ranges / pair_capacity (>= the number of pairs in vals). */
size_t uts_render_marks_bytes(const uts_config* cfg, uint64_t pair_capacity);
int uts_render_fwd_marked(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                          uint64_t pair_capacity, float* color, float* alpha, float* trans, uint32_t* n_last, uint32_t* marks,
                          size_t marks_bytes, void* stream);
int uts_render_bwd_marked(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                          uint64_t pair_capacity, const float* trans, const uint32_t* n_last, const uint32_t* marks,
                          const float* dL_dcolor, const float* dL_dalpha, float* dL_drgb, float* dL_dconic, float* dL_dmu2,
                          float* dL_dopac, void* stream);

/* Eq.3-4 and the rest of the chain: every output is overwritten with the sum over views.
 * dL_dmeans [P,3], dL_dscales [P,3], dL_dquats [P,4] (gradient of the R(q) polynomial), dL_dsh [P,M,3]. */
int uts_preprocess_bwd(const uts_config* cfg, uts_gaussians g, uts_views views, const uint8_t* flags,
                       const float* dL_drgb, const float* dL_dconic, const float* dL_dmu2, float* dL_dmeans,
                       float* dL_dscales, float* dL_dquats, float* dL_dsh, void* stream);

/* ------------------------------------------------------------------------------------------------- mask */

/* Builds M_C on the device: kind 0 = spherical cap, h_params = axis[3], half_angle;
 * kind 1 = pinhole frustum in the frame (right,up,fwd), h_params = right[3], up[3], fwd[3], tan_x, tan_y.
 * pixel_mask_bits [N_pix/32], slot_of_tile [N_tile], active_tiles [N_tile + 1]: the first n_active entries are the list, entry
 * N_tile receives n_active on the device (the call allocates nothing).  Synchronises `stream` and writes n_active to *h_n_active. */
int uts_build_mask(const uts_config* cfg, int kind, const double* h_params, uint32_t* pixel_mask_bits,
                   int32_t* slot_of_tile, uint32_t* active_tiles, int* h_n_active, void* stream);

/* ------------------------------------------------------------------- image synthesis */

/* Camera models of PAPER.md:477-515.  Principal point (W/2, H/2).  UTS_CAM_PINHOLE: p0, p1 = FoV_x, FoV_y in radians,
 * f_x = W / (2 tan(FoV_x / 2)) (Eq.11).  UTS_CAM_FISHEYE: anisotropic equidistant, p0, p1 = w_x, w_y = FoV / 180 deg,
 * f_x = W / pi, f_y = H / pi, valid domain = the ellipse of Eq.14-15 (Eq.12-13).  UTS_CAM_EQUIRECT: omega = 2 pi u / W - pi,
 * phi = pi/2 - pi v / H.  The camera frame is the one of uts_views (t = W mu + b): +z forward, polar axis +y. */
enum { UTS_CAM_PINHOLE = 0, UTS_CAM_FISHEYE = 1, UTS_CAM_EQUIRECT = 2 };
typedef struct { int model; int width, height; double p0, p1; } uts_camera;

/* I_C(u,v) = Interp_H(I_H, P_C(u,v)) for (u,v) in D_C (Eq.7).  image [S*256, channels] fp32 in the slot layout
 * of uts_render_fwd (one view); out [H, W, channels] row-major, 0 outside D_C; valid [H, W] = 1 inside D_C (may be NULL).
 * Interp_H is the HEALPix ring-bilinear interpolation (reading A26); samples with M_C = 0 are dropped and the weights
 * renormalised (A27); pixel (i,j) is sampled at (i + 1/2, j + 1/2) (A28).  1 <= channels <= 16. */
int uts_resample_fwd(const uts_config* cfg, uts_camera cam, uts_mask mask, const float* image, int channels, float* out,
                     uint8_t* valid, void* stream);
/* Adjoint of uts_resample_fwd: dL_dimage [S*256, channels] is zeroed by the call, then accumulated with atomics
 * (summation order is not deterministic).  dL_dout [H, W, channels]. */
int uts_resample_bwd(const uts_config* cfg, uts_camera cam, uts_mask mask, const float* dL_dout, int channels, float* dL_dimage,
                     void* stream);
/* M_C(q) = 1[Pi_C^{-1}(s_q) in D_C] (Eq.9) from the camera intrinsics; outputs as uts_build_mask.
 * Synchronises `stream` and writes n_active to *h_n_active. */
int uts_build_camera_mask(const uts_config* cfg, uts_camera cam, uint32_t* pixel_mask_bits, int32_t* slot_of_tile,
                          uint32_t* active_tiles, int* h_n_active, void* stream);

/* ------------------------------------------------- inverse radial depth, r_s,max */

/* Per-Gaussian channel of the inverse radial depth image (reading A29: D = Eq.6 with c_i = 1 / r_i):
 * chan [V,P,3] = (1 / rho, 0, 0), culled Gaussians 0.  Use it as `uts_proj.rgb` of uts_render_fwd (bg = 0): color[...,0] is the
 * depth image; uts_render_bwd on the same record with dL_dcolor = (dL/dD, 0, 0) returns dL/d(1/r_i) in dL_drgb[...,0] and the
 * depth loss's share of dL_dconic / dL_dmu2 / dL_dopac. */
int uts_inv_depth_channel(const uts_config* cfg, const float* rho, const uint8_t* flags, float* chan, void* stream);
/* The same depth image as a FOURTH CHANNEL of the colour blend (one pass instead of two; the decisions, and so color / alpha /
 * trans / n_last / marks, are those of uts_render_fwd[_marked]): depth [V,S*256] = sum_i T_i alpha_i / rho_i, 0 at masked-out pixels.
 * marks == NULL: the plain pair.  in.rho is read as well.  The backward takes dL_ddepth [V,S*256] next to dL_dcolor and returns, besides
 * uts_render_bwd's outputs (which now hold the colour loss's AND the depth loss's alpha-path terms), dL_dinvr [V,P] = dL/d(1/rho_i)
 * (zeroed by the call; pass it to uts_inv_depth_bwd with chan_stride = 1). */
int uts_render_fwd_depth(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                         uint64_t pair_capacity, float* color, float* alpha, float* trans, uint32_t* n_last, float* depth,
                         uint32_t* marks, size_t marks_bytes, void* stream);
int uts_render_bwd_depth(const uts_config* cfg, uts_proj in, uts_mask mask, const uint64_t* ranges, const uint32_t* vals,
                         uint64_t pair_capacity, const float* trans, const uint32_t* n_last, const uint32_t* marks,
                         const float* dL_dcolor, const float* dL_dalpha, const float* dL_ddepth, float* dL_drgb, float* dL_dconic,
                         float* dL_dmu2, float* dL_dopac, float* dL_dinvr, void* stream);
/* d(1/r)/dt = -t / r^3 carried to the means: dL_dmeans [P,3] (+)= sum_v W_v^T (-t / r^3) dL_dchan[(v*P + i) * chan_stride].
 * chan_stride = 3 for uts_render_bwd's dL_drgb on a depth-channel record, 1 for uts_render_bwd_depth's dL_dinvr.
 * accumulate != 0 adds to dL_dmeans (after uts_preprocess_bwd), 0 overwrites. */
int uts_inv_depth_bwd(const uts_config* cfg, const float* means, uts_views views, const uint8_t* flags, const float* dL_dchan,
                      int chan_stride, int accumulate, float* dL_dmeans, void* stream);
/* Radian-space density control buffer: rs_max[i] <- max(rs_max[i], rs[v,i]) over the views in which Gaussian i
 * is visible (not culled by uts_preprocess).  rs, flags: uts_preprocess's records; rs_max [P], caller-initialised. */
int uts_rs_max_update(const uts_config* cfg, const float* rs, const uint8_t* flags, float* rs_max, void* stream);

/* ------------------------------------------------------- L1 + HEALPix-SSIM loss */

/* L = (1 - lambda) L1^H + lambda (1 - HSSIM), HSSIM = sum_q M(q) h_q / sum_q M(q) (Eq.10), and its
 * gradient with respect to the rendered image, in one pass.  X (rendered) and G (ground truth): [S*256, 3] fp32 in the slot layout
 * of uts_render_fwd, one view.  h_q is the SSIM index (C1 = 0.01^2, C2 = 0.03^2, mean over the 3 channels) of the 11 x 11 window
 * around q in the (x,y) grid of q's base face, continued across face edges into the neighbouring faces ("cross-face padding",
 * PAPER.md:143; reading A30); taps that do not exist (the quadrant beyond a vertex shared by 3 faces) or have
 * M_C = 0 are dropped and the remaining weights renormalised (A32).  Weights: Gaussian of width `sigma` pixels, isotropic on the
 * equatorial faces 4..7, stretched pi/4 : 4/pi along the pixel diagonals on the polar faces (reading A31).
 * Outputs: loss3 [3] DEVICE doubles (L, L1^H, HSSIM); h_map [S*256] h_q, 0 where M_C = 0 (may be NULL); dL_dX [S*256, 3] (may be
 * NULL: forward only), zeroed by the call and accumulated with atomics (summation order is not deterministic).
 * L1^H = sum_q M(q) sum_ch |X - G| / (3 sum_q M(q)) (A34); lambda in [0,1] (0.2 in 3DGS, A35); sigma > 0 (1.5, A31).
 * scratch: uts_hssim_scratch_bytes(cfg) bytes, 8-byte aligned.  Asynchronous on `stream`. */
size_t uts_hssim_scratch_bytes(const uts_config* cfg);
int uts_hssim_loss(const uts_config* cfg, uts_mask mask, const float* X, const float* G, float lambda, float sigma, float* h_map,
                   float* dL_dX, double* loss3, void* scratch, size_t scratch_bytes, void* stream);

/* ----------------------------------------------- occlusion-bounded lists: helpers */

/* A pixel stops reading its tile's list once T < t_eps, so when every visible pixel saturates inside the lists of the `keep` nearest
 * Gaussians of its view, the image and the gradients do not depend on the other Gaussians at all.  These two calls let a caller use
 * that, exactly: build the tile lists from a depth prefix, blend, and check; if a pixel is still open, repeat with a larger prefix (or
 * all Gaussians).  The tile lists of a prefix are the first entries of Alg.1's full lists (same order), so n_last, marks, image and
 * gradients are those of the full lists; only keys / vals / ranges are shorter.
 * uts_depth_prefix_flags: flags_out[v,i] = flags[v,i] | 1 when (v,i) is not among the `keep` first of view v in uts_depth_order's order
 * (emit_rank); pass a uts_proj with flags_out to uts_tile_lists / uts_tile_query (only they read it as "culled"; uts_preprocess_bwd keeps
 * the original flags).  uts_count_unsaturated: *h_count = number of visible pixels (M_C = 1) with trans >= cfg->t_eps; trans is
 * uts_render_fwd's output; scratch: 8 bytes, 8-byte aligned; synchronises `stream`. */
int uts_depth_prefix_flags(const uts_config* cfg, const uint8_t* flags, const uint32_t* emit_rank, uint32_t keep, uint8_t* flags_out, void* stream);
int uts_count_unsaturated(const uts_config* cfg, uts_mask mask, const float* trans, uint64_t* h_count, void* scratch, void* stream);

/* NESTED pixel centres as camera-frame unit vectors, double [n,3], pixels first..first+n-1 at `order`
 * (exposes the library's HEALPix indexing for tests). */
int uts_pixel_centers(int order, uint64_t first, uint64_t n, double* out_xyz, void* stream);
/* rho_max(o), o = 0..13: largest centre-to-corner angle of an order-o pixel (Alg.2's PixRad, reading A6). Host. */
int uts_rho_max_table(double* h_out14);

/* ------------------------------------------------------------------------------------- whole path, host */

/* Device workspace needed by uts_host_forward_backward for at most `pair_capacity` pairs. */
size_t uts_host_workspace_bytes(const uts_config* cfg, int n_active, uint64_t pair_capacity);

/* The whole hot path with HOST buffers: copies the Gaussians, views and upstream gradient to the device,
 * runs preprocess -> tile query -> sort -> ranges -> blend forward -> blend backward -> preprocess backward,
 * and copies image and gradients back.  Host arrays have the shapes of the device calls above; the mask
 * arrays in `mask` are DEVICE pointers (built once by uts_build_mask).  h_dL_dcolor may be NULL (forward only).
 * workspace: device memory of uts_host_workspace_bytes(); returns UTS_ERR_CAPACITY (needed pairs in *h_n_pairs)
 * if it is too small.  Synchronises `stream` before returning. */
int uts_host_forward_backward(const uts_config* cfg, const float* h_means, const float* h_scales, const float* h_quats,
                              const float* h_opac, const float* h_sh, const float* h_W, const float* h_b, uts_mask mask,
                              const float* h_dL_dcolor, float* h_color, float* h_alpha, float* h_dL_dmeans,
                              float* h_dL_dscales, float* h_dL_dquats, float* h_dL_dopac, float* h_dL_dsh,
                              uint64_t pair_capacity, uint64_t* h_n_pairs, void* workspace, size_t workspace_bytes,
                              void* stream);

int         uts_last_cuda_error(void);
/* Kernel launches this library has enqueued since it was loaded (all streams, all calls; memsets and copies not counted).
 * bench.py reports the difference over its timed region as "gpu_launches". */
uint64_t    uts_launch_count(void);
const char* uts_strerror(int status);
const char* uts_version(void);

#ifdef __cplusplus
}
#endif
#endif /* UTS_H_ */
