"""Thin ctypes binding of libuts.so (include/uts.h): same names, argument marshalling only.

torch is used for device memory and streams; every step of the path runs in the library's CUDA kernels.  There is no
CPU fallback: importing works without a GPU (so that the symbol table can be checked), but any compute call needs the
CUDA library and CUDA tensors and fails loudly otherwise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libuts.so")

UTS_OK, UTS_ERR_INVALID_ARG, UTS_ERR_CAPACITY, UTS_ERR_CUDA, UTS_ERR_UNSUPPORTED = 0, 1, 2, 3, 4

# every symbol include/uts.h declares
SYMBOLS = [
    "uts_preprocess", "uts_preprocess_geometry", "uts_preprocess_color", "uts_depth_order", "uts_depth_order_scratch_bytes", "uts_depth_order_static", "uts_depth_order_static_max", "uts_tile_query", "uts_tile_query_scratch_bytes", "uts_tile_lists", "uts_tile_lists_scratch_bytes", "uts_sort", "uts_sort_scratch_bytes",
    "uts_tile_ranges", "uts_render_fwd", "uts_render_fwd_counted", "uts_render_bwd", "uts_render_marks_bytes", "uts_render_fwd_marked", "uts_render_bwd_marked", "uts_preprocess_bwd", "uts_build_mask", "uts_pixel_centers",
    "uts_rho_max_table", "uts_resample_fwd", "uts_resample_bwd", "uts_build_camera_mask", "uts_inv_depth_channel", "uts_inv_depth_bwd", "uts_render_fwd_depth", "uts_render_bwd_depth", "uts_rs_max_update", "uts_depth_prefix_flags", "uts_count_unsaturated", "uts_hssim_loss", "uts_hssim_scratch_bytes",
    "uts_host_workspace_bytes", "uts_host_forward_backward", "uts_last_cuda_error", "uts_launch_count", "uts_strerror",
    "uts_version",
]


class UtsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib().uts_strerror(status).decode()
        extra = f" (cudaError {lib().uts_last_cuda_error()})" if status == UTS_ERR_CUDA else ""
        super().__init__(f"{where}: {msg}{extra}")


class CConfig(C.Structure):
    _fields_ = [("order", C.c_int), ("tile_log2", C.c_int), ("query_refine_log2", C.c_int), ("sh_degree", C.c_int),
                ("n_gauss", C.c_int), ("n_views", C.c_int), ("r_near", C.c_float), ("cov_dilation_px2", C.c_float),
                ("alpha_min", C.c_float), ("alpha_max", C.c_float), ("t_eps", C.c_float), ("bg", C.c_float * 3),
                ("query_mode", C.c_int)]


class CGaussians(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("means", "scales", "quats", "opac", "sh")]


class CViews(C.Structure):
    _fields_ = [("W", C.c_void_p), ("b", C.c_void_p)]


class CProj(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("dir", "lonlat", "rho", "conic_opac", "rs", "rgb", "flags")]


class CCamera(C.Structure):
    _fields_ = [("model", C.c_int), ("width", C.c_int), ("height", C.c_int), ("p0", C.c_double), ("p1", C.c_double)]


class CMask(C.Structure):
    _fields_ = [("active_tiles", C.c_void_p), ("n_active", C.c_int), ("slot_of_tile", C.c_void_p), ("pixel_mask_bits", C.c_void_p)]


class CTuning(C.Structure):
    _fields_ = [("query_impl", C.c_int), ("descent_block_radius", C.c_float), ("descent_blocks_per_sm", C.c_int), ("matrix_off", C.c_int),
                ("matrix_min_tiles", C.c_float), ("window_mode", C.c_int)]


@dataclass
class Tuning:
    """uts_tuning (include/uts.h): steers implementation choices of the tile query, never its result.  None = defaults."""
    query_impl: int = 0                 # 1: the quadtree descent (Alg.2's depth-first form)
    descent_block_radius: float = 0.0
    descent_blocks_per_sm: int = 0
    matrix_off: int = 0
    matrix_min_tiles: float = 0.0
    window_mode: int = 0                # tile-window path for the smallest discs: 0 automatic (sparse masks), 1 never, 2 always

    def c(self):
        return CTuning(self.query_impl, self.descent_block_radius, self.descent_blocks_per_sm, self.matrix_off, self.matrix_min_tiles, self.window_mode)


def _tuning(t):
    return None if t is None else C.byref(t.c())


@dataclass
class Config:
    """uts_config (include/uts.h).  Defaults follow DESIGN.md readings A3, A5, A7, A8."""
    order: int
    n_gauss: int
    n_views: int = 1
    sh_degree: int = 0
    tile_log2: int = 4
    query_refine_log2: int = 2
    r_near: float = 0.2
    cov_dilation_px2: float = 0.3
    alpha_min: float = 1.0 / 255.0
    alpha_max: float = 0.99
    t_eps: float = 1e-4
    bg: tuple = (0.0, 0.0, 0.0)
    query_mode: int = 0          # UTS_QUERY_NESTED (Alg.2) / 1 = UTS_QUERY_RING (Alg.3)

    @property
    def n_pix(self): return 12 << (2 * self.order)
    @property
    def n_tiles(self): return 12 << (2 * (self.order - self.tile_log2))
    @property
    def ppt(self): return 1 << (2 * self.tile_log2)
    @property
    def n_sh(self): return (self.sh_degree + 1) ** 2

    def c(self) -> CConfig:
        return CConfig(self.order, self.tile_log2, self.query_refine_log2, self.sh_degree, self.n_gauss, self.n_views,
                       self.r_near, self.cov_dilation_px2, self.alpha_min, self.alpha_max, self.t_eps, (C.c_float * 3)(*self.bg),
                       self.query_mode)


_lib = None


def lib():
    """Loads libuts.so; raises if it has not been built (python -m paper_2606_29794_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_29794_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.uts_strerror.restype = C.c_char_p
        L.uts_version.restype = C.c_char_p
        for n in ("uts_render_marks_bytes", "uts_hssim_scratch_bytes", "uts_depth_order_scratch_bytes", "uts_tile_query_scratch_bytes", "uts_sort_scratch_bytes", "uts_host_workspace_bytes"):
            getattr(L, n).restype = C.c_size_t
        L.uts_sort_scratch_bytes.argtypes = [C.c_uint64]
        L.uts_host_workspace_bytes.argtypes = [C.POINTER(CConfig), C.c_int, C.c_uint64]
        _lib = L
    return _lib


def _ptr(t, dtype=None):
    if t is None:
        return None
    if not t.is_cuda:
        raise RuntimeError("uts: device tensor expected (no CPU fallback)")
    if not t.is_contiguous():
        raise RuntimeError("uts: contiguous tensor expected")
    if dtype is not None and t.dtype != dtype:
        raise RuntimeError(f"uts: expected {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check(st, where):
    if st != UTS_OK:
        raise UtsError(st, where)


@dataclass
class Gaussians:
    means: torch.Tensor; scales: torch.Tensor; quats: torch.Tensor; opac: torch.Tensor; sh: torch.Tensor

    def c(self): return CGaussians(*[_ptr(t, torch.float32) for t in (self.means, self.scales, self.quats, self.opac, self.sh)])


@dataclass
class Views:
    W: torch.Tensor; b: torch.Tensor

    def c(self): return CViews(_ptr(self.W, torch.float32), _ptr(self.b, torch.float32))


@dataclass
class Proj:
    dir: torch.Tensor; lonlat: torch.Tensor; rho: torch.Tensor; conic_opac: torch.Tensor; rs: torch.Tensor
    rgb: torch.Tensor; flags: torch.Tensor

    @staticmethod
    def empty(cfg: Config, device="cuda"):
        V, P = cfg.n_views, cfg.n_gauss
        f = lambda *s: torch.empty(*s, dtype=torch.float32, device=device)
        return Proj(f(V, P, 3), f(V, P, 2), f(V, P), f(V, P, 4), f(V, P), f(V, P, 3), torch.empty(V, P, dtype=torch.uint8, device=device))

    def c(self):
        return CProj(*[_ptr(t, torch.float32) for t in (self.dir, self.lonlat, self.rho, self.conic_opac, self.rs, self.rgb)],
                     _ptr(self.flags, torch.uint8))


@dataclass
class Mask:
    """FoV mask arrays (device).  Mask.full() = whole sphere."""
    active_tiles: torch.Tensor | None = None      # int32 storage of uint32 tile ids
    n_active: int = -1
    slot_of_tile: torch.Tensor | None = None      # int32
    pixel_mask_bits: torch.Tensor | None = None   # int32 storage of uint32 words

    @staticmethod
    def full(): return Mask()

    def n_slots(self, cfg: Config): return cfg.n_tiles if self.active_tiles is None else self.n_active

    def c(self):
        return CMask(_ptr(self.active_tiles), self.n_active, _ptr(self.slot_of_tile), _ptr(self.pixel_mask_bits))


# ---------------------------------------------------------------------------------------------- the ABI calls
def uts_preprocess(cfg: Config, g: Gaussians, views: Views, out: Proj, stream=None):
    c = cfg.c()
    _check(lib().uts_preprocess(C.byref(c), g.c(), views.c(), out.c(), _stream(stream)), "uts_preprocess")


def uts_preprocess_geometry(cfg: Config, g: Gaussians, views: Views, out: Proj, stream=None):
    c = cfg.c()
    _check(lib().uts_preprocess_geometry(C.byref(c), g.c(), views.c(), out.c(), _stream(stream)), "uts_preprocess_geometry")


def uts_preprocess_color(cfg: Config, g: Gaussians, views: Views, out: Proj, stream=None):
    c = cfg.c()
    _check(lib().uts_preprocess_color(C.byref(c), g.c(), views.c(), out.c(), _stream(stream)), "uts_preprocess_color")


def uts_tile_query_scratch_bytes(cfg: Config) -> int:
    c = cfg.c()
    return int(lib().uts_tile_query_scratch_bytes(C.byref(c)))


def uts_depth_order_scratch_bytes(cfg: Config) -> int:
    c = cfg.c()
    return int(lib().uts_depth_order_scratch_bytes(C.byref(c)))


def uts_depth_order(cfg: Config, rho, emit_rank, scratch, stream=None):
    c = cfg.c()
    _check(lib().uts_depth_order(C.byref(c), _ptr(rho, torch.float32), _ptr(emit_rank, torch.int32), _ptr(scratch),
                                 C.c_size_t(scratch.numel() * scratch.element_size()), _stream(stream)), "uts_depth_order")


def uts_depth_order_static_max() -> int:
    lib().uts_depth_order_static_max.restype = C.c_uint64
    return int(lib().uts_depth_order_static_max())


def uts_depth_order_static(cfg: Config, rho, emit_rank, stream=None):
    """uts_depth_order with the scratch inside the library (no allocation anywhere); n_gauss * n_views <= uts_depth_order_static_max()."""
    c = cfg.c()
    st = lib().uts_depth_order_static(C.byref(c), _ptr(rho, torch.float32), _ptr(emit_rank, torch.int32), _stream(stream))
    if st == UTS_ERR_CAPACITY:
        raise UtsError(st, f"uts_depth_order_static: {cfg.n_gauss * cfg.n_views} records exceed the static scratch's limit of {uts_depth_order_static_max()}")
    _check(st, "uts_depth_order_static")


def uts_tile_query(cfg: Config, proj: Proj, mask: Mask, offsets, keys, vals, capacity: int, scratch, emit_rank=None, tuning: Tuning | None = None,
                   stream=None) -> int:
    """Returns the pair count.  keys=None: count only.  Raises UtsError(UTS_ERR_CAPACITY) with .needed set."""
    c = cfg.c()
    n = C.c_uint64(0)
    st = lib().uts_tile_query(C.byref(c), proj.c(), mask.c(), _ptr(emit_rank, torch.int32), _ptr(offsets, torch.int64), _ptr(keys, torch.int64), _ptr(vals, torch.int32),
                              C.c_uint64(capacity), C.byref(n), _ptr(scratch), C.c_size_t(scratch.numel() * scratch.element_size()),
                              _tuning(tuning), _stream(stream))
    if st == UTS_ERR_CAPACITY:
        e = UtsError(st, "uts_tile_query"); e.needed = int(n.value); raise e
    _check(st, "uts_tile_query")
    return int(n.value)


def uts_launch_count() -> int:
    """Kernel launches enqueued by libuts.so since it was loaded."""
    lib().uts_launch_count.restype = C.c_uint64
    return int(lib().uts_launch_count())


def uts_tile_lists_scratch_bytes(cfg: Config) -> int:
    c = cfg.c()
    lib().uts_tile_lists_scratch_bytes.restype = C.c_size_t
    return int(lib().uts_tile_lists_scratch_bytes(C.byref(c)))


def uts_tile_lists(cfg: Config, proj: Proj, mask: Mask, emit_rank, keys, vals, keys_tmp, vals_tmp, capacity: int, ranges, scratch, sort_scratch,
                   tuning: Tuning | None = None, stream=None) -> int:
    """Sorted pairs + tile ranges in one call (see include/uts.h).  Returns the pair count; raises UtsError (status
    UTS_ERR_CAPACITY, .needed = required capacity) when the buffers are too small."""
    c = cfg.c()
    n = C.c_uint64(0)
    st = lib().uts_tile_lists(C.byref(c), proj.c(), mask.c(), _ptr(emit_rank), _ptr(keys), _ptr(vals), _ptr(keys_tmp), _ptr(vals_tmp),
                              C.c_uint64(capacity), _ptr(ranges), C.byref(n), _ptr(scratch), C.c_size_t(scratch.numel() * scratch.element_size()),
                              _ptr(sort_scratch), C.c_size_t(sort_scratch.numel() * sort_scratch.element_size()), _tuning(tuning), _stream(stream))
    if st == UTS_ERR_CAPACITY:
        e = UtsError(st, "uts_tile_lists"); e.needed = int(n.value)
        raise e
    _check(st, "uts_tile_lists")
    return int(n.value)


def uts_sort_scratch_bytes(n_pairs: int) -> int:
    return int(lib().uts_sort_scratch_bytes(C.c_uint64(n_pairs)))


def uts_sort(cfg: Config, n_pairs: int, keys, vals, keys_tmp, vals_tmp, scratch, depth_presorted=False, stream=None):
    c = cfg.c()
    _check(lib().uts_sort(C.byref(c), C.c_uint64(n_pairs), _ptr(keys, torch.int64), _ptr(vals, torch.int32), _ptr(keys_tmp, torch.int64),
                          _ptr(vals_tmp, torch.int32), C.c_int(1 if depth_presorted else 0), _ptr(scratch),
                          C.c_size_t(scratch.numel() * scratch.element_size()), _stream(stream)), "uts_sort")


def uts_tile_ranges(cfg: Config, n_pairs: int, keys, ranges, stream=None):
    c = cfg.c()
    _check(lib().uts_tile_ranges(C.byref(c), C.c_uint64(n_pairs), _ptr(keys, torch.int64), _ptr(ranges, torch.int64), _stream(stream)),
           "uts_tile_ranges")


def uts_render_fwd(cfg: Config, proj: Proj, mask: Mask, ranges, vals, color, alpha, trans, n_last, stream=None):
    c = cfg.c()
    _check(lib().uts_render_fwd(C.byref(c), proj.c(), mask.c(), _ptr(ranges, torch.int64), _ptr(vals, torch.int32),
                                _ptr(color, torch.float32), _ptr(alpha, torch.float32), _ptr(trans, torch.float32),
                                _ptr(n_last, torch.int32), _stream(stream)), "uts_render_fwd")


def uts_render_fwd_counted(cfg: Config, proj: Proj, mask: Mask, ranges, vals, color, alpha, trans, n_last, work, stream=None):
    """uts_render_fwd + work counters: work = 4 int64 on the device (zeroed by the caller) -> += (evaluated by Alg.1, contributing,
    passing the patch cull, evaluated in full) pairs."""
    assert work.numel() >= 4
    c = cfg.c()
    _check(lib().uts_render_fwd_counted(C.byref(c), proj.c(), mask.c(), _ptr(ranges, torch.int64), _ptr(vals, torch.int32),
                                        _ptr(color, torch.float32), _ptr(alpha, torch.float32), _ptr(trans, torch.float32),
                                        _ptr(n_last, torch.int32), _ptr(work, torch.int64), _stream(stream)), "uts_render_fwd_counted")


def uts_render_bwd(cfg: Config, proj: Proj, mask: Mask, ranges, vals, trans, n_last, dL_dcolor, dL_dalpha, dL_drgb, dL_dconic,
                   dL_dmu2, dL_dopac, stream=None):
    c = cfg.c()
    _check(lib().uts_render_bwd(C.byref(c), proj.c(), mask.c(), _ptr(ranges, torch.int64), _ptr(vals, torch.int32),
                                _ptr(trans, torch.float32), _ptr(n_last, torch.int32), _ptr(dL_dcolor, torch.float32),
                                _ptr(dL_dalpha, torch.float32), _ptr(dL_drgb, torch.float32), _ptr(dL_dconic, torch.float32),
                                _ptr(dL_dmu2, torch.float32), _ptr(dL_dopac, torch.float32), _stream(stream)), "uts_render_bwd")


def uts_render_marks_bytes(cfg: Config, pair_capacity: int) -> int:
    c = cfg.c()
    return int(lib().uts_render_marks_bytes(C.byref(c), C.c_uint64(pair_capacity)))


def uts_render_fwd_marked(cfg: Config, proj: Proj, mask: Mask, ranges, vals, pair_capacity: int, color, alpha, trans, n_last, marks, stream=None):
    c = cfg.c()
    _check(lib().uts_render_fwd_marked(C.byref(c), proj.c(), mask.c(), _ptr(ranges), _ptr(vals), C.c_uint64(pair_capacity), _ptr(color, torch.float32),
                                       _ptr(alpha, torch.float32), _ptr(trans, torch.float32), _ptr(n_last), _ptr(marks),
                                       C.c_size_t(marks.numel() * marks.element_size()), _stream(stream)), "uts_render_fwd_marked")


def uts_render_bwd_marked(cfg: Config, proj: Proj, mask: Mask, ranges, vals, pair_capacity: int, trans, n_last, marks, dL_dcolor, dL_dalpha,
                          dL_drgb, dL_dconic, dL_dmu2, dL_dopac, stream=None):
    c = cfg.c()
    _check(lib().uts_render_bwd_marked(C.byref(c), proj.c(), mask.c(), _ptr(ranges), _ptr(vals), C.c_uint64(pair_capacity), _ptr(trans, torch.float32),
                                       _ptr(n_last), _ptr(marks), _ptr(dL_dcolor, torch.float32), _ptr(dL_dalpha, torch.float32),
                                       _ptr(dL_drgb, torch.float32), _ptr(dL_dconic, torch.float32), _ptr(dL_dmu2, torch.float32),
                                       _ptr(dL_dopac, torch.float32), _stream(stream)), "uts_render_bwd_marked")


def uts_preprocess_bwd(cfg: Config, g: Gaussians, views: Views, flags, dL_drgb, dL_dconic, dL_dmu2, dL_dmeans, dL_dscales,
                       dL_dquats, dL_dsh, stream=None):
    c = cfg.c()
    _check(lib().uts_preprocess_bwd(C.byref(c), g.c(), views.c(), _ptr(flags, torch.uint8), _ptr(dL_drgb, torch.float32),
                                    _ptr(dL_dconic, torch.float32), _ptr(dL_dmu2, torch.float32), _ptr(dL_dmeans, torch.float32),
                                    _ptr(dL_dscales, torch.float32), _ptr(dL_dquats, torch.float32), _ptr(dL_dsh, torch.float32),
                                    _stream(stream)), "uts_preprocess_bwd")


def uts_build_mask(cfg: Config, kind: str, params, device="cuda", stream=None) -> Mask:
    """kind 'cap': params = axis[3], half_angle; 'frustum': right[3], up[3], fwd[3], tan_x, tan_y."""
    c = cfg.c()
    bits = torch.empty(cfg.n_pix // 32, dtype=torch.int32, device=device)
    slot = torch.empty(cfg.n_tiles, dtype=torch.int32, device=device)
    act = torch.empty(cfg.n_tiles + 1, dtype=torch.int32, device=device)     # entry N_tile receives n_active
    prm = (C.c_double * len(params))(*[float(x) for x in params])
    n = C.c_int(0)
    _check(lib().uts_build_mask(C.byref(c), C.c_int(0 if kind == "cap" else 1), prm, _ptr(bits), _ptr(slot), _ptr(act), C.byref(n),
                                _stream(stream)), "uts_build_mask")
    return Mask(act[: n.value].contiguous(), int(n.value), slot, bits)


def uts_inv_depth_channel(cfg: Config, rho, flags, chan, stream=None):
    c = cfg.c()
    _check(lib().uts_inv_depth_channel(C.byref(c), _ptr(rho, torch.float32), _ptr(flags, torch.uint8), _ptr(chan, torch.float32), _stream(stream)),
           "uts_inv_depth_channel")


def uts_inv_depth_bwd(cfg: Config, means, views: Views, flags, dL_dchan, dL_dmeans, accumulate=True, stream=None):
    """dL_dchan: [V,P,3] (uts_render_bwd's dL_drgb on a depth-channel record) or [V,P] (uts_render_bwd_depth's dL_dinvr)."""
    c = cfg.c()
    stride = 3 if dL_dchan.dim() == 3 else 1
    _check(lib().uts_inv_depth_bwd(C.byref(c), _ptr(means, torch.float32), views.c(), _ptr(flags, torch.uint8), _ptr(dL_dchan, torch.float32),
                                   C.c_int(stride), C.c_int(1 if accumulate else 0), _ptr(dL_dmeans, torch.float32), _stream(stream)), "uts_inv_depth_bwd")


def uts_render_fwd_depth(cfg: Config, proj: Proj, mask: Mask, ranges, vals, pair_capacity: int, color, alpha, trans, n_last, depth, marks=None, stream=None):
    """Colour + inverse radial depth in one blend pass (marks=None: the plain pair)."""
    c = cfg.c()
    mb = 0 if marks is None else marks.numel() * marks.element_size()
    _check(lib().uts_render_fwd_depth(C.byref(c), proj.c(), mask.c(), _ptr(ranges), _ptr(vals), C.c_uint64(pair_capacity), _ptr(color, torch.float32),
                                      _ptr(alpha, torch.float32), _ptr(trans, torch.float32), _ptr(n_last), _ptr(depth, torch.float32), _ptr(marks),
                                      C.c_size_t(mb), _stream(stream)), "uts_render_fwd_depth")


def uts_render_bwd_depth(cfg: Config, proj: Proj, mask: Mask, ranges, vals, pair_capacity: int, trans, n_last, marks, dL_dcolor, dL_dalpha, dL_ddepth,
                         dL_drgb, dL_dconic, dL_dmu2, dL_dopac, dL_dinvr, stream=None):
    c = cfg.c()
    _check(lib().uts_render_bwd_depth(C.byref(c), proj.c(), mask.c(), _ptr(ranges), _ptr(vals), C.c_uint64(pair_capacity), _ptr(trans, torch.float32),
                                      _ptr(n_last), _ptr(marks), _ptr(dL_dcolor, torch.float32), _ptr(dL_dalpha, torch.float32),
                                      _ptr(dL_ddepth, torch.float32), _ptr(dL_drgb, torch.float32), _ptr(dL_dconic, torch.float32),
                                      _ptr(dL_dmu2, torch.float32), _ptr(dL_dopac, torch.float32), _ptr(dL_dinvr, torch.float32), _stream(stream)),
           "uts_render_bwd_depth")


def uts_rs_max_update(cfg: Config, rs, flags, rs_max, stream=None):
    c = cfg.c()
    _check(lib().uts_rs_max_update(C.byref(c), _ptr(rs, torch.float32), _ptr(flags, torch.uint8), _ptr(rs_max, torch.float32), _stream(stream)),
           "uts_rs_max_update")


CAMERA_MODELS = {"pinhole": 0, "fisheye": 1, "equirect": 2}


@dataclass
class Camera:
    """PAPER.md:477-515.  'pinhole': p0, p1 = FoV_x, FoV_y (radians); 'fisheye': p0, p1 = w_x, w_y (Eq.12); 'equirect'."""
    model: str
    width: int
    height: int
    p0: float = 0.0
    p1: float = 0.0

    def c(self): return CCamera(CAMERA_MODELS[self.model], self.width, self.height, float(self.p0), float(self.p1))


def uts_resample_fwd(cfg: Config, cam: Camera, mask: Mask, image, out, valid=None, stream=None):
    """image [S*256, C] -> out [H, W, C] (Eq.7); valid [H, W] uint8 or None."""
    c = cfg.c()
    ch = int(image.shape[-1])
    assert image.shape[0] == mask.n_slots(cfg) * 256 and tuple(out.shape) == (cam.height, cam.width, ch)
    _check(lib().uts_resample_fwd(C.byref(c), cam.c(), mask.c(), _ptr(image, torch.float32), C.c_int(ch), _ptr(out, torch.float32),
                                  _ptr(valid, torch.uint8), _stream(stream)), "uts_resample_fwd")


def uts_resample_bwd(cfg: Config, cam: Camera, mask: Mask, dL_dout, dL_dimage, stream=None):
    c = cfg.c()
    ch = int(dL_dout.shape[-1])
    assert dL_dimage.shape[0] == mask.n_slots(cfg) * 256 and int(dL_dimage.shape[-1]) == ch
    _check(lib().uts_resample_bwd(C.byref(c), cam.c(), mask.c(), _ptr(dL_dout, torch.float32), C.c_int(ch), _ptr(dL_dimage, torch.float32),
                                  _stream(stream)), "uts_resample_bwd")


def uts_build_camera_mask(cfg: Config, cam: Camera, device="cuda", stream=None) -> Mask:
    """M_C of Eq.9 from the camera intrinsics."""
    c = cfg.c()
    bits = torch.empty(cfg.n_pix // 32, dtype=torch.int32, device=device)
    slot = torch.empty(cfg.n_tiles, dtype=torch.int32, device=device)
    act = torch.empty(cfg.n_tiles + 1, dtype=torch.int32, device=device)     # entry N_tile receives n_active
    n = C.c_int(0)
    _check(lib().uts_build_camera_mask(C.byref(c), cam.c(), _ptr(bits), _ptr(slot), _ptr(act), C.byref(n), _stream(stream)),
           "uts_build_camera_mask")
    return Mask(act[: n.value].contiguous(), int(n.value), slot, bits)


def uts_depth_prefix_flags(cfg: Config, flags, emit_rank, keep: int, flags_out, stream=None):
    c = cfg.c()
    _check(lib().uts_depth_prefix_flags(C.byref(c), _ptr(flags, torch.uint8), _ptr(emit_rank), C.c_uint32(keep), _ptr(flags_out, torch.uint8),
                                        _stream(stream)), "uts_depth_prefix_flags")


def uts_count_unsaturated(cfg: Config, mask: Mask, trans, scratch, stream=None) -> int:
    c = cfg.c()
    n = C.c_uint64(0)
    _check(lib().uts_count_unsaturated(C.byref(c), mask.c(), _ptr(trans, torch.float32), C.byref(n), _ptr(scratch), _stream(stream)),
           "uts_count_unsaturated")
    return int(n.value)


def uts_hssim_scratch_bytes(cfg: Config) -> int:
    c = cfg.c()
    return int(lib().uts_hssim_scratch_bytes(C.byref(c)))


def uts_hssim_loss(cfg: Config, mask: Mask, X, G, loss3, scratch, h_map=None, dL_dX=None, lam=0.2, sigma=1.5, stream=None):
    """L = (1 - lam) L1^H + lam (1 - HSSIM) and dL/dX (Eq.10).  X, G [S*256, 3]; loss3 [3] float64 (device)."""
    c = cfg.c()
    n = mask.n_slots(cfg) * 256
    assert tuple(X.shape) == (n, 3) and tuple(G.shape) == (n, 3) and loss3.numel() == 3
    assert h_map is None or h_map.numel() == n
    assert dL_dX is None or tuple(dL_dX.shape) == (n, 3)
    _check(lib().uts_hssim_loss(C.byref(c), mask.c(), _ptr(X, torch.float32), _ptr(G, torch.float32), C.c_float(lam), C.c_float(sigma),
                                _ptr(h_map, torch.float32), _ptr(dL_dX, torch.float32), _ptr(loss3, torch.float64), _ptr(scratch),
                                C.c_size_t(scratch.numel() * scratch.element_size()), _stream(stream)), "uts_hssim_loss")


def uts_pixel_centers(order: int, first: int, n: int, device="cuda", stream=None):
    out = torch.empty(n, 3, dtype=torch.float64, device=device)
    _check(lib().uts_pixel_centers(C.c_int(order), C.c_uint64(first), C.c_uint64(n), _ptr(out), _stream(stream)), "uts_pixel_centers")
    return out


def uts_rho_max_table():
    t = (C.c_double * 14)()
    _check(lib().uts_rho_max_table(t), "uts_rho_max_table")
    return list(t)


def uts_host_workspace_bytes(cfg: Config, n_active: int, pair_capacity: int) -> int:
    c = cfg.c()
    return int(lib().uts_host_workspace_bytes(C.byref(c), C.c_int(n_active), C.c_uint64(pair_capacity)))


def uts_host_forward_backward(cfg: Config, h, mask: Mask, h_dL_dcolor, h_out, pair_capacity: int, workspace, stream=None) -> int:
    """h: dict of pinned/pageable HOST float32 tensors means, scales, quats, opac, sh, W, b.  h_out: dict of host tensors
    color, alpha and (if h_dL_dcolor is given) dL_dmeans, dL_dscales, dL_dquats, dL_dopac, dL_dsh.  Returns the pair count."""
    c = cfg.c()

    def hp(t):
        if t is None:
            return None
        assert (not t.is_cuda) and t.is_contiguous() and t.dtype == torch.float32
        return C.c_void_p(t.data_ptr())

    n = C.c_uint64(0)
    st = lib().uts_host_forward_backward(
        C.byref(c), hp(h["means"]), hp(h["scales"]), hp(h["quats"]), hp(h["opac"]), hp(h["sh"]), hp(h["W"]), hp(h["b"]), mask.c(),
        hp(h_dL_dcolor), hp(h_out["color"]), hp(h_out.get("alpha")), hp(h_out.get("dL_dmeans")), hp(h_out.get("dL_dscales")),
        hp(h_out.get("dL_dquats")), hp(h_out.get("dL_dopac")), hp(h_out.get("dL_dsh")), C.c_uint64(pair_capacity), C.byref(n),
        _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    if st == UTS_ERR_CAPACITY:
        e = UtsError(st, "uts_host_forward_backward"); e.needed = int(n.value); raise e
    _check(st, "uts_host_forward_backward")
    return int(n.value)
