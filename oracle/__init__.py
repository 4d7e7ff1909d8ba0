"""ORACLE — TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around the plain single-threaded double-precision C++ oracle in this directory
(orc_healpix.cpp, orc_raster.cpp, orc_capi.cpp), written from PAPER.md (Alg.1-2, Eq.1-6) and the readings
listed in DESIGN.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from ``paper_2606_29794_b200`` and the
CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = ["orc_healpix.cpp", "orc_raster.cpp", "orc_resample.cpp", "orc_depth.cpp", "orc_hssim.cpp", "orc_capi.cpp"]
_HDRS = ["orc_healpix.hpp", "orc_raster.hpp", "orc_resample.hpp", "orc_hssim.hpp"]
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile liboracle.so with g++ (no -ffast-math, no FMA contraction)."""
    srcs = [os.path.join(_HERE, s) for s in _SRCS]
    deps = srcs + [os.path.join(_HERE, h) for h in _HDRS]
    if (not force) and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB] + srcs
    subprocess.check_call(cmd)
    return _LIB


class _Cfg(C.Structure):
    _fields_ = [("order", C.c_int), ("tile_log2", C.c_int), ("query_refine_log2", C.c_int), ("sh_degree", C.c_int),
                ("n_gauss", C.c_int), ("n_views", C.c_int), ("r_near", C.c_float), ("cov_dilation_px2", C.c_float),
                ("alpha_min", C.c_float), ("alpha_max", C.c_float), ("t_eps", C.c_float), ("bg", C.c_float * 3),
                ("query_mode", C.c_int)]


@dataclass
class Config:
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
    query_mode: int = 0          # 0 NESTED descent (Alg.2), 1 RING scan (Alg.3)

    @property
    def n_pix(self): return 12 << (2 * self.order)
    @property
    def tile_order(self): return self.order - self.tile_log2
    @property
    def n_tiles(self): return 12 << (2 * self.tile_order)
    @property
    def ppt(self): return 1 << (2 * self.tile_log2)
    @property
    def n_sh(self): return (self.sh_degree + 1) ** 2

    def c(self) -> _Cfg:
        return _Cfg(self.order, self.tile_log2, self.query_refine_log2, self.sh_degree, self.n_gauss, self.n_views,
                    self.r_near, self.cov_dilation_px2, self.alpha_min, self.alpha_max, self.t_eps, (C.c_float * 3)(*self.bg),
                    self.query_mode)


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_npix.restype = C.c_int64
        _lib.orc_xyf2nest.restype = C.c_int64
        _lib.orc_xyf2nest.argtypes = [C.c_int, C.c_int64, C.c_int64, C.c_int]
        _lib.orc_ring_npix_in_ring.restype = C.c_int64
        _lib.orc_ring_npix_in_ring.argtypes = [C.c_int, C.c_int64]
        _lib.orc_rho_max_bruteforce.restype = C.c_double
        _lib.orc_rho_max_closed.restype = C.c_double
        _lib.orc_tile_query.restype = C.c_int64
        _lib.orc_e2e_f64.restype = C.c_double
    return _lib


def _p(a):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p)


def _f32(a): return np.ascontiguousarray(a, dtype=np.float32)
def _f64(a): return np.ascontiguousarray(a, dtype=np.float64)
def _u32(a): return None if a is None else np.ascontiguousarray(a, dtype=np.uint32)
def _i32(a): return None if a is None else np.ascontiguousarray(a, dtype=np.int32)
def _u64(a): return np.ascontiguousarray(a, dtype=np.uint64)


# ------------------------------------------------------------------ HEALPix
def nest2xyf(order, p):
    out = np.zeros(3, np.int64); lib().orc_nest2xyf(C.c_int(order), C.c_int64(int(p)), _p(out)); return tuple(int(v) for v in out)


def xyf2nest(order, x, y, f): return int(lib().orc_xyf2nest(order, int(x), int(y), int(f)))


def centers(order, which=2, first=0, n=None):
    """which: 1 = D1 plane form, 2 = D2 ring form (NESTED index), 3 = textbook RING-order centres (RING index).
    Returns (z, lam, vec_cam[n,3])."""
    if n is None:
        n = (12 << (2 * order)) - first
    z = np.zeros(n); lam = np.zeros(n); v = np.zeros((n, 3))
    lib().orc_centers(C.c_int(order), C.c_int(which), C.c_int64(first), C.c_int64(n), _p(z), _p(lam), _p(v))
    return z, lam, v


def corner(order, p, k):
    v = np.zeros(3); lib().orc_corner(C.c_int(order), C.c_int64(int(p)), C.c_int(k), _p(v)); return v


def nest2ring(order, first=0, n=None):
    if n is None: n = (12 << (2 * order)) - first
    out = np.zeros(n, np.int64); lib().orc_nest2ring(C.c_int(order), C.c_int64(first), C.c_int64(n), _p(out)); return out


def ring2nest(order, first=0, n=None):
    if n is None: n = (12 << (2 * order)) - first
    out = np.zeros(n, np.int64); lib().orc_ring2nest(C.c_int(order), C.c_int64(first), C.c_int64(n), _p(out)); return out


def ang2pix(order, z, lam):
    z = _f64(z); lam = _f64(lam); out = np.zeros(z.shape[0], np.int64)
    lib().orc_ang2pix(C.c_int(order), C.c_int64(z.shape[0]), _p(z), _p(lam), _p(out)); return out


def vec2pix(order, v):
    v = _f64(v); out = np.zeros(v.shape[0], np.int64)
    lib().orc_vec2pix(C.c_int(order), C.c_int64(v.shape[0]), _p(v), _p(out)); return out


def ring_npix_in_ring(order, i): return int(lib().orc_ring_npix_in_ring(order, int(i)))
def rho_max_bruteforce(order): return float(lib().orc_rho_max_bruteforce(C.c_int(order)))
def rho_max_closed(order): return float(lib().orc_rho_max_closed(C.c_int(order)))


def mask_bits(order, kind, params):
    """kind 'cap': params = axis[3], half_angle ; kind 'frustum': right[3], up[3], fwd[3], tan_x, tan_y."""
    n = 12 << (2 * order)
    bits = np.zeros((n + 31) // 32, np.uint32)
    prm = _f64(params)
    lib().orc_mask(C.c_int(order), C.c_int(0 if kind == "cap" else 1), _p(prm), _p(bits))
    return bits


def mask_tiles(cfg: Config, bits):
    """active tile list (ascending) and slot_of_tile from a pixel bitmap: tile active <=> any pixel active (A19)."""
    ppt = cfg.ppt
    assert ppt % 32 == 0
    w = bits.reshape(cfg.n_tiles, ppt // 32)
    act = np.flatnonzero((w != 0).any(axis=1)).astype(np.uint32)
    slot = np.full(cfg.n_tiles, -1, np.int32)
    slot[act] = np.arange(act.shape[0], dtype=np.int32)
    return act, slot


# ------------------------------------------------------------------ image synthesis (orc_resample.hpp)
CAMERA_MODELS = {"pinhole": 0, "fisheye": 1, "equirect": 2}


@dataclass
class Camera:
    """model 'pinhole' (p0, p1 = FoV_x, FoV_y in radians), 'fisheye' (p0, p1 = w_x, w_y of Eq.12), 'equirect'."""
    model: str
    width: int
    height: int
    p0: float = 0.0
    p1: float = 0.0

    def args(self):
        return (C.c_int(CAMERA_MODELS[self.model]), C.c_int(self.width), C.c_int(self.height), C.c_double(self.p0), C.c_double(self.p1))


def cam_pixel_dir(cam: Camera, u, v):
    d = np.zeros(3)
    ok = lib().orc_cam_pixel_dir(*cam.args(), C.c_double(u), C.c_double(v), _p(d))
    return d, bool(ok)


def cam_project(cam: Camera, d):
    uv = np.zeros(2)
    dd = _f64(d)
    ok = lib().orc_cam_project(*cam.args(), _p(dd), _p(uv))
    return uv, bool(ok)


def interp_weights(order, theta, lam):
    pix = np.zeros(8, np.int64); w = np.zeros(8)
    n = lib().orc_interp_weights(C.c_int(order), C.c_double(theta), C.c_double(lam), _p(pix), _p(w))
    return pix[:n], w[:n]


def resample_fwd(order, cam: Camera, image, slot_of_tile=None, pixel_mask_bits=None):
    """image [n_slot*256, C] fp32 (slot layout) -> out [H, W, C] float64, valid [H, W] uint8."""
    img = _f32(image); ch = img.shape[-1]
    out = np.zeros((cam.height, cam.width, ch)); valid = np.zeros((cam.height, cam.width), np.uint8)
    sl, mb = _i32(slot_of_tile), _u32(pixel_mask_bits)
    lib().orc_resample_fwd(C.c_int(order), *cam.args(), _p(sl), _p(mb), _p(img), C.c_int(ch), _p(out), _p(valid))
    return out, valid


def resample_bwd(order, cam: Camera, dL_dout, n_slot, slot_of_tile=None, pixel_mask_bits=None):
    g = _f64(dL_dout); ch = g.shape[-1]
    out = np.zeros((n_slot * 256, ch))
    sl, mb = _i32(slot_of_tile), _u32(pixel_mask_bits)
    lib().orc_resample_bwd(C.c_int(order), *cam.args(), _p(sl), _p(mb), C.c_int64(n_slot), _p(g), C.c_int(ch), _p(out))
    return out


def camera_mask_bits(order, cam: Camera):
    n = 12 << (2 * order)
    bits = np.zeros((n + 31) // 32, np.uint32)
    lib().orc_camera_mask(C.c_int(order), *cam.args(), _p(bits))
    return bits


# ------------------------------------------------------------------ inverse radial depth, r_s,max (orc_depth.cpp)
def inv_depth_channel(rho, flags=None):
    """rho [V,P] fp32 -> per-Gaussian channel [V,P,3] = (1/rho, 0, 0), to be blended in place of the colour (reading A29)."""
    r = _f32(rho); V, P = r.shape
    fl = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
    out = np.zeros((V, P, 3), np.float32)
    lib().orc_inv_depth_channel(C.c_int(V), C.c_int(P), _p(r), _p(fl), _p(out))
    return out


def inv_depth_bwd(means, W, b, dL_dinv, flags=None):
    """dL/dmeans [P,3] of sum_v,i dL_dinv[v,i] / ||W_v mu_i + b_v||."""
    m, Wf, bf, g = _f32(means), _f32(W), _f32(b), _f64(dL_dinv)
    V, P = g.shape
    fl = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
    out = np.zeros((P, 3))
    lib().orc_inv_depth_bwd(C.c_int(V), C.c_int(P), _p(m), _p(Wf), _p(bf), _p(fl), _p(g), _p(out))
    return out


def rs_max_update(rs, flags, rs_max):
    """r_s,max <- max(r_s,max, r_s) for visible Gaussians; returns the updated copy."""
    r = _f32(rs); V, P = r.shape
    fl = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
    out = _f32(rs_max).copy()
    lib().orc_rs_max_update(C.c_int(V), C.c_int(P), _p(r), _p(fl), _p(out))
    return out


# ------------------------------------------------------------------ resolution hierarchy (Table 6)
def select_order(width, height, omega_in):
    """Table 6: continuous target N*_side = sqrt(4 pi W H / (12 Omega_in)); returns (N*_side, k = round(log2 N*), k_L = floor, k_H = ceil)."""
    n_star = math.sqrt(4.0 * math.pi * width * height / (12.0 * omega_in))
    l2 = math.log2(n_star)
    return n_star, int(round(l2)), int(math.floor(l2)), int(math.ceil(l2))


# ------------------------------------------------------------------ L1 + HEALPix-SSIM loss (orc_hssim.cpp, NEXT-3)
def hssim_neighbor(order, p, dx, dy):
    """(pixel at offset (dx,dy) in p's face frame or -1, quarter turns of the axes)  — reading A30."""
    lib().orc_hssim_neighbor.restype = C.c_int64
    rot = C.c_int(0)
    q = lib().orc_hssim_neighbor(C.c_int(order), C.c_int64(int(p)), C.c_int(dx), C.c_int(dy), C.byref(rot))
    return int(q), int(rot.value)


def hssim_weight(face, dx, dy, sigma=1.5):
    lib().orc_hssim_weight.restype = C.c_double
    return float(lib().orc_hssim_weight(C.c_int(face), C.c_int(dx), C.c_int(dy), C.c_double(sigma)))


def hssim_loss(order, X, G, slot_of_tile=None, bits=None, lam=0.2, sigma=1.5, grad=True, q_list=None):
    """X, G [n_slot*256, 3] fp32 (slot layout).  Returns dict(loss, l1, hssim, h_map [n_slot*256], grad [n_slot*256, 3] or None).
    q_list: evaluate only these centre pixels (NESTED ids) — h_map, sums and grad then hold their terms only."""
    Xf, Gf = _f32(X), _f32(G)
    n_store = Xf.shape[0]
    st = None if slot_of_tile is None else np.ascontiguousarray(slot_of_tile, dtype=np.int32)
    bt = None if bits is None else np.ascontiguousarray(bits, dtype=np.uint32)
    h = np.zeros(n_store); g = np.zeros((n_store, 3)) if grad else None
    out = np.zeros(3)
    ql = None if q_list is None else np.ascontiguousarray(q_list, dtype=np.int64)
    lib().orc_hssim_loss(C.c_int(order), _p(st), _p(bt), C.c_int64(n_store // 256), _p(Xf), _p(Gf), C.c_double(lam), C.c_double(sigma),
                         _p(h), _p(g), _p(out), _p(ql), C.c_int64(0 if ql is None else ql.shape[0]))
    return dict(loss=float(out[0]), l1=float(out[1]), hssim=float(out[2]), h_map=h, grad=g)


# ------------------------------------------------------------------ stages (fp32 ABI arrays)
@dataclass
class ProjArrays:
    dir: np.ndarray; lonlat: np.ndarray; rho: np.ndarray; conic_opac: np.ndarray; rs: np.ndarray; rgb: np.ndarray
    flags: np.ndarray


def preprocess(cfg: Config, means, scales, quats, opac, sh, W, b) -> ProjArrays:
    V, P = cfg.n_views, cfg.n_gauss
    out = ProjArrays(np.zeros((V, P, 3), np.float32), np.zeros((V, P, 2), np.float32), np.zeros((V, P), np.float32),
                     np.zeros((V, P, 4), np.float32), np.zeros((V, P), np.float32), np.zeros((V, P, 3), np.float32),
                     np.zeros((V, P), np.uint8))
    c = cfg.c()
    args = [_f32(means), _f32(scales), _f32(quats), _f32(opac), _f32(sh), _f32(W), _f32(b)]
    lib().orc_preprocess(C.byref(c), *[_p(a) for a in args], _p(out.dir), _p(out.lonlat), _p(out.rho), _p(out.conic_opac),
                         _p(out.rs), _p(out.rgb), _p(out.flags))
    return out


def sigma_arc_both(cfg: Config, mu, s, q, W, b):
    lit = np.zeros(3); tan = np.zeros(3); J = np.zeros(6); t = np.zeros(3)
    c = cfg.c()
    lib().orc_sigma_arc_both(C.byref(c), _p(_f64(mu)), _p(_f64(s)), _p(_f64(q)), _p(_f64(W)), _p(_f64(b)), _p(lit), _p(tan), _p(J), _p(t))
    return lit, tan, J.reshape(2, 3), t


def sh_basis(degree, d):
    Y = np.zeros(16); lib().orc_sh_basis(C.c_int(degree), _p(_f64(d)), _p(Y)); return Y


def sh_basis_grad(degree, d):
    dY = np.zeros(48); lib().orc_sh_basis_grad(C.c_int(degree), _p(_f64(d)), _p(dY)); return dY.reshape(16, 3)


def tile_query(cfg: Config, proj: ProjArrays, slot_of_tile=None, brute=False, gauss_subset=None):
    """Returns offsets[V*P+1], keys, vals, info(min_margin, node_tests).  Order: (view, Gaussian id, tile) ascending."""
    V, P = cfg.n_views, cfg.n_gauss
    offsets = np.zeros(V * P + 1, np.uint64)
    mm = C.c_double(0); nt = C.c_int64(0)
    c = cfg.c()
    sub = _i32(gauss_subset)
    n = lib().orc_tile_query(C.byref(c), _p(_f32(proj.dir)), _p(_f32(proj.rho)), _p(_f32(proj.rs)), _p(proj.flags),
                             _p(_i32(slot_of_tile)), C.c_int(1 if brute else 0), _p(sub), C.c_int(0 if sub is None else sub.shape[0]),
                             _p(offsets), C.byref(mm), C.byref(nt))
    keys = np.zeros(n, np.uint64); vals = np.zeros(n, np.uint32)
    lib().orc_tile_query_fetch(_p(keys), _p(vals))
    return offsets, keys, vals, dict(min_margin=mm.value, node_tests=nt.value)


def sort_pairs(keys, vals):
    keys = _u64(keys).copy(); vals = _u32(vals).copy()
    lib().orc_sort(C.c_uint64(keys.shape[0]), _p(keys), _p(vals))
    return keys, vals


def tile_ranges(cfg: Config, keys):
    keys = _u64(keys)
    ranges = np.zeros((cfg.n_views * cfg.n_tiles, 2), np.uint64)
    c = cfg.c()
    lib().orc_tile_ranges(C.byref(c), C.c_uint64(keys.shape[0]), _p(keys), _p(ranges))
    return ranges


def render_fwd(cfg: Config, proj: ProjArrays, ranges, vals, active_tiles=None, pixel_mask_bits=None, slots_todo=None):
    """Returns color[V,S*ppt,3], alpha, n_last, margin (per pixel decision margin), counters dict."""
    V = cfg.n_views
    S = cfg.n_tiles if active_tiles is None else int(active_tiles.shape[0])
    n = V * S * cfg.ppt
    color = np.zeros((V, S * cfg.ppt, 3), np.float32); alpha = np.zeros((V, S * cfg.ppt), np.float32)
    n_last = np.zeros((V, S * cfg.ppt), np.uint32); margin = np.full((V, S * cfg.ppt), np.inf)
    ctr = np.zeros(3, np.int64)
    c = cfg.c()
    todo = _i32(slots_todo)
    lib().orc_render_fwd(C.byref(c), _p(_f32(proj.dir)), _p(_f32(proj.conic_opac)), _p(_f32(proj.rgb)),
                         _p(_u32(active_tiles)), C.c_int(S), _p(_u32(pixel_mask_bits)), _p(_u64(ranges)), _p(_u32(vals)),
                         _p(todo), C.c_int(0 if todo is None else todo.shape[0]),
                         _p(color), _p(alpha), _p(n_last), _p(margin), _p(ctr))
    return color, alpha, n_last, margin, dict(evaluated=int(ctr[0]), contributing=int(ctr[1]), early_exit_pixels=int(ctr[2]))


def render_bwd(cfg: Config, proj: ProjArrays, ranges, vals, n_last, dL_dcolor, dL_dalpha=None, active_tiles=None,
               pixel_mask_bits=None):
    """Returns dL_drgb[V,P,3], dL_dconic[V,P,3], dL_dmu2[V,P,2] (gradient w.r.t. mu'=(omega,phi)), dL_dopac[P] — float64."""
    V, P = cfg.n_views, cfg.n_gauss
    S = cfg.n_tiles if active_tiles is None else int(active_tiles.shape[0])
    d_rgb = np.zeros((V, P, 3)); d_conic = np.zeros((V, P, 3)); d_mu2 = np.zeros((V, P, 2)); d_opac = np.zeros(P)
    c = cfg.c()
    lib().orc_render_bwd(C.byref(c), _p(_f32(proj.dir)), _p(_f32(proj.conic_opac)), _p(_f32(proj.rgb)),
                         _p(_u32(active_tiles)), C.c_int(S), _p(_u32(pixel_mask_bits)), _p(_u64(ranges)), _p(_u32(vals)),
                         _p(_u32(n_last)), _p(_f32(dL_dcolor)), _p(None if dL_dalpha is None else _f32(dL_dalpha)),
                         _p(d_rgb), _p(d_conic), _p(d_mu2), _p(d_opac))
    return d_rgb, d_conic, d_mu2, d_opac


def preprocess_bwd(cfg: Config, means, scales, quats, sh, W, b, dL_drgb, dL_dconic, dL_dmu2):
    P, M = cfg.n_gauss, cfg.n_sh
    d_means = np.zeros((P, 3)); d_scales = np.zeros((P, 3)); d_quats = np.zeros((P, 4)); d_sh = np.zeros((P, M, 3))
    c = cfg.c()
    lib().orc_preprocess_bwd(C.byref(c), _p(_f32(means)), _p(_f32(scales)), _p(_f32(quats)), _p(_f32(sh)), _p(_f32(W)), _p(_f32(b)),
                             _p(_f64(dL_drgb)), _p(_f64(dL_dconic)), _p(_f64(dL_dmu2)),
                             _p(d_means), _p(d_scales), _p(d_quats), _p(d_sh))
    return d_means, d_scales, d_quats, d_sh


def e2e_f64(cfg: Config, means, scales, quats, opac, sh, W, b, ranges, vals, G_color, G_alpha=None, active_tiles=None,
            pixel_mask_bits=None, want_grad=False, want_dbg=False):
    """fp64 preprocess -> blend with FIXED lists.  Returns loss, or (loss, grads dict[, dbg8]) when want_grad."""
    P, M = cfg.n_gauss, cfg.n_sh
    S = cfg.n_tiles if active_tiles is None else int(active_tiles.shape[0])
    c = cfg.c()
    g = dict(means=np.zeros((P, 3)), scales=np.zeros((P, 3)), quats=np.zeros((P, 4)), opac=np.zeros(P), sh=np.zeros((P, M, 3)))
    dbg = np.zeros(8)
    loss = lib().orc_e2e_f64(C.byref(c), _p(_f64(means)), _p(_f64(scales)), _p(_f64(quats)), _p(_f64(opac)), _p(_f64(sh)),
                             _p(_f64(W)), _p(_f64(b)), _p(_u32(active_tiles)), C.c_int(S), _p(_u32(pixel_mask_bits)),
                             _p(_u64(ranges)), _p(_u32(vals)), _p(_f64(G_color)), _p(None if G_alpha is None else _f64(G_alpha)),
                             C.c_int(1 if want_grad else 0), _p(g["means"]), _p(g["scales"]), _p(g["quats"]), _p(g["opac"]), _p(g["sh"]),
                             _p(dbg) if want_dbg else None)
    if not want_grad:
        return loss
    return (loss, g, dbg) if want_dbg else (loss, g)


def forward_chain(cfg: Config, scene, slot_of_tile=None, active_tiles=None, pixel_mask_bits=None, brute=False):
    """The whole forward, stage by stage (fp32 at the stage boundaries, as the ABI stores).  Returns a dict."""
    proj = preprocess(cfg, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    offsets, keys, vals, qinfo = tile_query(cfg, proj, slot_of_tile, brute=brute)
    skeys, svals = sort_pairs(keys, vals)
    ranges = tile_ranges(cfg, skeys)
    color, alpha, n_last, margin, ctr = render_fwd(cfg, proj, ranges, svals, active_tiles, pixel_mask_bits)
    return dict(proj=proj, offsets=offsets, keys=keys, vals=vals, skeys=skeys, svals=svals, ranges=ranges, color=color,
                alpha=alpha, n_last=n_last, margin=margin, counters=ctr, qinfo=qinfo)
