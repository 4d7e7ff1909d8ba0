"""Seeded synthetic scene generators for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no HEALPix, no projection, no blending): it only draws the
random inputs — Gaussian parameters, view matrices, an analytic mask *descriptor* and upstream gradients — that
both the CUDA path and the test oracle consume.  The recipe is stated in DESIGN.md "Input recipe"; the scenes
stand in for the paper's datasets (Table 4), which are not available.

"N(m,s)": s is the standard deviation.  Every attribute has its own PCG64 stream seeded by (seed, config, stream).
"""
from __future__ import annotations

import math

import numpy as np

SH_C0 = 0.28209479177387814  # only used to turn a base colour in [0,1] into a DC coefficient (input recipe)

CONFIGS = {
    1: dict(name="tiny", order=6, n_gauss=1_000, sh_degree=0, n_views=1, mask=None),
    2: dict(name="panorama", order=8, n_gauss=100_000, sh_degree=3, n_views=1, mask=None),
    3: dict(name="fisheye190", order=9, n_gauss=500_000, sh_degree=3, n_views=1, mask="cap"),
    4: dict(name="large_sphere", order=10, n_gauss=2_000_000, sh_degree=3, n_views=1, mask=None),
    5: dict(name="narrow_persp_x4", order=11, n_gauss=1_000_000, sh_degree=3, n_views=4, mask="frustum"),
}

CAP_HALF_ANGLE = math.radians(95.0)
FRUSTUM_TAN = (math.tan(math.radians(30.0)), math.tan(math.radians(22.5)))


def _rng(seed, cfg_id, stream):
    return np.random.default_rng([int(seed), int(cfg_id), int(stream)])


def _uniform_dirs(rng, n):
    v = rng.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _cap_dirs(rng, n, half_angle, inside=True):
    """uniform directions inside (or outside) the cap of given half-angle about +z."""
    c = math.cos(half_angle)
    z = rng.uniform(c, 1.0, n) if inside else rng.uniform(-1.0, c, n)
    ph = rng.uniform(0.0, 2 * math.pi, n)
    s = np.sqrt(np.maximum(0.0, 1 - z * z))
    return np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1)


def _in_frustum(d, tx, ty):
    return (d[:, 2] > 0) & (np.abs(d[:, 0]) <= tx * d[:, 2]) & (np.abs(d[:, 1]) <= ty * d[:, 2])


def _frustum_dirs(rng, n, tx, ty, inside=True):
    out = np.zeros((0, 3))
    while out.shape[0] < n:
        m = max(1024, 2 * (n - out.shape[0]))
        if inside:
            x = rng.uniform(-tx, tx, m); y = rng.uniform(-ty, ty, m)
            keep = rng.uniform(0, 1, m) < (1 + x * x + y * y) ** -1.5     # solid-angle density on the plane z=1
            d = np.stack([x, y, np.ones(m)], axis=1)[keep]
            d /= np.linalg.norm(d, axis=1, keepdims=True)
        else:
            d = _uniform_dirs(rng, m)
            d = d[~_in_frustum(d, tx, ty)]
        out = np.concatenate([out, d], axis=0)
    return out[:n]


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def _random_rotation(rng):
    """A rotation matrix drawn uniformly (QR of a Gaussian matrix, signs fixed, determinant +1): an input draw, no method arithmetic."""
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))[None, :]
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def make_scene(cfg_id: int, seed: int = 0, n_gauss: int | None = None, order: int | None = None,
               sh_degree: int | None = None, n_views: int | None = None, general_view: bool = False) -> dict:
    """Returns float32 arrays means[P,3] scales[P,3] quats[P,4] opac[P] sh[P,M,3] W[V,9] b[V,3] plus
    order / sh_degree / n_views / mask descriptor.  n_gauss / order / sh_degree / n_views shrink a config for tests
    (same distributions).  general_view: every view gets its own random rotation W (tilted about all three axes) and a
    translation b ~ N(0, 0.4) (camera off the origin) instead of the configs' W = I / rotation about y, b = 0."""
    base = CONFIGS[cfg_id]
    P = int(n_gauss if n_gauss is not None else base["n_gauss"])
    k = int(order if order is not None else base["order"])
    D = int(sh_degree if sh_degree is not None else base["sh_degree"])
    V = int(n_views if n_views is not None else base["n_views"])
    M = (D + 1) ** 2
    r_dir, r_rad, r_scl, r_quat, r_op, r_col, r_pick = (_rng(seed, cfg_id, s) for s in range(7))

    if cfg_id == 1:
        dirs = _uniform_dirs(r_dir, P); rad = r_rad.uniform(2.0, 10.0, P)
        logs = r_scl.normal(-3.0, 0.5, (P, 3)); opac = _sigmoid(r_op.normal(0.0, 1.0, P))
    elif cfg_id == 2:
        dirs = _uniform_dirs(r_dir, P); rad = r_rad.uniform(1.0, 20.0, P)
        logs = r_scl.normal(-4.0, 0.7, (P, 3)); opac = _sigmoid(r_op.normal(0.0, 1.5, P))
    elif cfg_id == 3:
        inside = r_pick.uniform(0, 1, P) < 0.7
        dirs = np.where(inside[:, None], _cap_dirs(r_dir, P, CAP_HALF_ANGLE, True), _cap_dirs(r_dir, P, CAP_HALF_ANGLE, False))
        rad = r_rad.uniform(0.5, 15.0, P)
        logs = r_scl.normal(-4.5, 0.8, (P, 3)); opac = _sigmoid(r_op.normal(0.0, 1.5, P))
    elif cfg_id == 4:
        dirs = _uniform_dirs(r_dir, P); rad = np.exp(r_rad.uniform(math.log(0.5), math.log(50.0), P))
        logs = r_scl.normal(-5.0, 1.0, (P, 3))
        big = r_pick.uniform(0, 1, P) < 0.05
        logs_big = _rng(seed, cfg_id, 7).normal(-2.0, 0.5, (P, 3))
        logs = np.where(big[:, None], logs_big, logs)
        opac = _sigmoid(r_op.normal(0.0, 2.0, P))
    elif cfg_id == 5:
        inside = r_pick.uniform(0, 1, P) < 0.8
        tx, ty = FRUSTUM_TAN
        dirs = np.where(inside[:, None], _frustum_dirs(r_dir, P, tx, ty, True), _frustum_dirs(r_dir, P, tx, ty, False))
        rad = r_rad.uniform(1.0, 30.0, P)
        logs = r_scl.normal(-5.5, 0.8, (P, 3)); opac = _sigmoid(r_op.normal(0.0, 1.5, P))
    else:
        raise ValueError(cfg_id)

    q = r_quat.standard_normal((P, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    sh = np.zeros((P, M, 3))
    sh[:, 0, :] = (r_col.uniform(0.0, 1.0, (P, 3)) - 0.5) / SH_C0          # base colour U[0,1] -> DC coefficient
    if M > 1:
        sh[:, 1:, :] = r_col.normal(0.0, 0.2, (P, M - 1, 3))

    W = np.zeros((V, 9)); b = np.zeros((V, 3))
    for v in range(V):
        th = math.radians(6.0 * v) if cfg_id == 5 else 0.0                  # rotation about camera y
        c, s = math.cos(th), math.sin(th)
        W[v] = [c, 0, s, 0, 1, 0, -s, 0, c]
    if general_view:
        r_view = _rng(seed, cfg_id, 8)
        for v in range(V):
            W[v] = _random_rotation(r_view).reshape(-1)
            b[v] = r_view.normal(0.0, 0.4, 3)

    mask = None
    if base["mask"] == "cap":
        mask = dict(kind="cap", params=[0.0, 0.0, 1.0, CAP_HALF_ANGLE])
    elif base["mask"] == "frustum":
        mask = dict(kind="frustum", params=[1, 0, 0, 0, 1, 0, 0, 0, 1, FRUSTUM_TAN[0], FRUSTUM_TAN[1]])

    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return dict(cfg_id=cfg_id, name=base["name"], order=k, sh_degree=D, n_views=V, n_gauss=P, mask=mask,
                means=f32(dirs * rad[:, None]), scales=f32(np.exp(logs)), quats=f32(q), opac=f32(opac), sh=f32(sh),
                W=f32(W), b=f32(b))


def upstream_grad(n_views: int, n_pixels: int, seed: int = 0, with_alpha: bool = False):
    """dL/dcolor ~ N(0,1) iid per pixel and channel (BASELINE.json configs: 'random upstream gradient')."""
    r = np.random.default_rng([int(seed), 999])
    g = r.standard_normal((n_views, n_pixels, 3), dtype=np.float32)
    if with_alpha:
        return g, r.standard_normal((n_views, n_pixels), dtype=np.float32)
    return g
