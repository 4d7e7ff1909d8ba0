"""Host logic of the small-disc path of the CUDA tile query: csrc/uts_window_query.cuh (angle -> cell map, face gluing, window of
candidate tiles settled by the defining predicate) is __host__ __device__; tests/hostlogic/window_query_host.cu drives it on the
CPU and the results must equal the oracle's: pixel of a direction, neighbour across face edges, and the tile sets of Alg.2
(reading A6) and Alg.3, bit for bit — on the shrunk configs, every refinement, masks, and discs centred on / next to the poles, the
8 vertices shared by three faces, face edges, with radii up to the largest the path accepts.  No GPU needed."""
import ctypes as C
import math
import os
import shutil
import subprocess
import tempfile

import numpy as np
import pytest

import oracle as orc
from helpers import ocfg, oracle_mask, small_scene

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.fixture(scope="module")
def hostlib():
    if not os.path.exists(NVCC) and shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    out = os.path.join(tempfile.mkdtemp(prefix="uts_hostlogic_"), "winq_host.so")
    subprocess.check_call([NVCC if os.path.exists(NVCC) else "nvcc", "-O2", "-std=c++17", "-shared", "-Xcompiler", "-fPIC", "-w", "--extended-lambda",
                           "-I", os.path.join(ROOT, "include"), "-I", os.path.join(ROOT, "paper_2606_29794_b200", "csrc"),
                           os.path.join(ROOT, "tests", "hostlogic", "window_query_host.cu"), "-o", out])
    L = C.CDLL(out)
    L.window_query_host.restype = C.c_int
    L.extended_cell_host.restype = C.c_int64
    return L


def _pix(L, order, v):
    v = np.ascontiguousarray(v, np.float64)
    out = np.zeros(v.shape[0], np.int64)
    L.vec_to_pixel_host(C.c_int(order), C.c_int64(v.shape[0]), v.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
    return out


def test_direction_to_pixel_round_trip_and_oracle(hostlib):
    for order in range(0, 8):
        _, _, v = orc.centers(order, 2)
        assert np.array_equal(_pix(hostlib, order, v), np.arange(12 << (2 * order)))
    rng = np.random.default_rng(3)
    v = rng.standard_normal((200_000, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
    v[:2000, [0, 2]] *= 1e-3; v[:2000] /= np.linalg.norm(v[:2000], axis=1, keepdims=True)       # near the poles
    for order in (0, 1, 3, 8, 13):
        assert np.array_equal(_pix(hostlib, order, v), orc.vec2pix(order, v)), order
    # hierarchy: the pixel at order o is the parent of the pixel at order o + 3
    assert np.array_equal(_pix(hostlib, 9, v) >> 6, _pix(hostlib, 6, v))


def test_fp32_centres_are_within_the_chord_margin(hostlib):
    rng = np.random.default_rng(4)
    for order in (2, 6, 10, 12):
        N = 1 << order
        worst = 0.0
        for _ in range(4000):
            f, x, y = int(rng.integers(12)), int(rng.integers(N)), int(rng.integers(N))
            if rng.random() < 0.2:
                x, y = (N - 1 - int(rng.integers(3)), N - 1 - int(rng.integers(3)))                  # next to the pole / lower vertex
            c32 = (C.c_float * 3)(); c64 = (C.c_double * 3)()
            hostlib.cell_centers_host(order, f, x, y, c32, c64)
            worst = max(worst, max(abs(c32[i] - c64[i]) for i in range(3)))
            p = orc.xyf2nest(order, x, y, f)
            _, _, want = orc.centers(order, 2, first=p, n=1)
            assert max(abs(c64[i] - want[0, i]) for i in range(3)) < 5e-15
        assert worst < 1.2e-6, (order, worst)


@pytest.mark.parametrize("order", [2, 3, 5])
def test_extended_cells_equal_the_oracle_neighbour_map(hostlib, order):
    """Cell (x + dx, y + dy) of the extended frame of p's face, |dx|, |dy| <= 3, against the oracle's neighbour function (derived
    from shared-corner geometry, pinned in test_oracle_hssim.py): same pixel, or both 'does not exist'."""
    N = 1 << order
    rng = np.random.default_rng(order)
    pix = np.arange(12 * N * N) if order <= 3 else np.unique(np.concatenate([rng.integers(0, 12 * N * N, 600),
                                                                               [orc.xyf2nest(order, x, y, f) for f in range(12) for x in (0, 1, N - 2, N - 1) for y in (0, 1, N - 2, N - 1)]]))
    for p in pix:
        x, y, f = orc.nest2xyf(order, int(p))
        for dy in range(-3, 4):
            for dx in range(-3, 4):
                if not (-N <= x + dx < 2 * N and -N <= y + dy < 2 * N):
                    continue
                got = hostlib.extended_cell_host(order, f, x + dx, y + dy)
                want, _ = orc.hssim_neighbor(order, int(p), dx, dy)
                assert got == want, (order, int(p), (x, y, f), (dx, dy), got, want)


def _host_sets(L, oc, pr, mode, slot=None):
    kt, kq = oc.tile_order, oc.tile_order + oc.query_refine_log2
    rho_q = 0.0 if mode == 1 else orc.rho_max_closed(kq)
    rho_t = orc.rho_max_closed(kt)
    buf = np.zeros(64, np.uint32)
    sp = None if slot is None else np.ascontiguousarray(slot, np.int32).ctypes.data_as(C.c_void_p)
    out = []
    for i in range(oc.n_gauss):
        if pr.flags[0, i] & 1:
            out.append(None); continue
        d = np.ascontiguousarray(pr.dir[0, i], np.float32)
        R = min(math.pi, float(pr.rs[0, i]) + rho_q)
        n = L.window_query_host(kt, kq, d.ctypes.data_as(C.c_void_p), C.c_double(R), C.c_double(rho_t), sp, buf.ctypes.data_as(C.c_void_p), 64)
        out.append(None if n < 0 else buf[:n].copy())
    return out


def _check(L, sc, refine, mode, tweak=None, min_taken=0.3, masked=False):
    oc = ocfg(sc, query_refine_log2=refine, query_mode=mode)
    pr = orc.preprocess(oc, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    if tweak is not None:
        tweak(pr)
    slot = oracle_mask(oc, sc)[2] if masked else None
    off, keys, vals, info = orc.tile_query(oc, pr, slot)
    assert info["min_margin"] > 1e-12
    tiles = (keys >> np.uint64(32)).astype(np.uint32)
    got = _host_sets(L, oc, pr, mode, slot)
    taken = 0
    for i in range(oc.n_gauss):
        if got[i] is None:
            continue
        taken += 1
        want = tiles[int(off[i]):int(off[i + 1])]
        assert np.array_equal(got[i], want), (i, pr.dir[0, i], pr.rs[0, i], got[i], want)
    assert taken >= min_taken * oc.n_gauss, (taken, oc.n_gauss)


@pytest.mark.parametrize("mode", [0, 1], ids=["nested-set", "ring-set"])
@pytest.mark.parametrize("cfg_id,P,order,refine", [(1, 1000, 7, 2), (2, 1500, 8, 2), (4, 1500, 8, 2), (4, 600, 7, 1), (1, 600, 7, 0),
                                                   (4, 500, 7, 3), (2, 500, 8, 4), (5, 1500, 10, 2), (2, 1000, 12, 2)])
def test_window_query_equals_oracle(hostlib, cfg_id, P, order, refine, mode):
    _check(hostlib, small_scene(cfg_id, P, order, n_views=1), refine, mode)


@pytest.mark.parametrize("cfg_id,order", [(3, 8), (5, 9)])
def test_window_query_respects_the_mask(hostlib, cfg_id, order):
    _check(hostlib, small_scene(cfg_id, 1500, order, n_views=1), 2, 0, masked=True)


@pytest.mark.parametrize("mode", [0, 1], ids=["nested-set", "ring-set"])
@pytest.mark.parametrize("order,refine", [(7, 2), (8, 2), (7, 0), (8, 4), (11, 2)])
def test_window_query_at_poles_three_face_vertices_and_edges(hostlib, order, refine, mode):
    """Disc centres ON and next to the poles, the 8 vertices shared by three faces (z = +-2/3, longitude c pi/2), the 4-face
    vertices (z = 0, longitude pi/4 + c pi/2), along face edges, and random; radii spread over the three window sizes, a third of
    them within 0.1 % of the largest radius a window size accepts."""
    n = 420
    sc = small_scene(4, n, order)
    rng = np.random.default_rng(100 * order + refine)
    kt = order - 4
    Nt = 1 << kt

    def tweak(pr):
        d = rng.standard_normal((n, 3))
        special = []
        for sgn in (1, -1):
            special.append([0, 0, sgn])                                                     # poles (HEALPix frame x, y, z)
            for c in range(4):
                lam = c * math.pi / 2
                special.append([math.sqrt(5) / 3 * math.cos(lam), math.sqrt(5) / 3 * math.sin(lam), sgn * 2 / 3])   # 3-face vertices
        for c in range(4):
            lam = math.pi / 4 + c * math.pi / 2
            special.append([math.cos(lam), math.sin(lam), 0.0])                             # 4-face vertices on the equator
        special = np.array(special)
        k = special.shape[0]
        for rep in range(6):                                                                # exactly on, and jittered by a fraction of a tile
            jit = (0.0 if rep == 0 else 0.7 / Nt) * rng.standard_normal((k, 3))
            d[rep * k:(rep + 1) * k] = special + jit
        # along face edges: the meridians lambda = c pi/2 above z = 2/3 and the belt lines z = +-(2/3)(1 - 2 |lambda - lambda_c| ... ) sampled
        e0 = 6 * k
        zz = rng.uniform(0.67, 0.999, 40); lam = rng.integers(0, 4, 40) * math.pi / 2
        d[e0:e0 + 40] = np.stack([np.sqrt(1 - zz * zz) * np.cos(lam), np.sqrt(1 - zz * zz) * np.sin(lam), zz * rng.choice([-1, 1], 40)], 1)
        tt = rng.uniform(0, 1, 40); cc = rng.integers(0, 4, 40)
        zb = (2 / 3) * (1 - 2 * tt) ; lb = (cc + 0.5 * tt) * math.pi / 2                     # edge from a 3-face vertex down to the equator vertex
        d[e0 + 40:e0 + 80] = np.stack([np.sqrt(1 - zb * zb) * np.cos(lb), np.sqrt(1 - zb * zb) * np.sin(lb), zb], 1)
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        cam = np.stack([d[:, 1], d[:, 2], d[:, 0]], 1)                                      # HEALPix (x,y,z) -> camera (y_hp, z_hp, x_hp)
        pr.dir[0] = cam.astype(np.float32)
        pr.lonlat[0, :, 0] = np.arctan2(cam[:, 0], cam[:, 2]).astype(np.float32)
        pr.lonlat[0, :, 1] = np.arctan2(cam[:, 1], np.hypot(cam[:, 0], cam[:, 2])).astype(np.float32)
        rho_q = 0.0 if mode == 1 else orc.rho_max_closed(kt + refine)
        w = rng.integers(1, 4, n)
        Rmax = 0.98 * 0.6 * w / Nt
        R = np.where(rng.random(n) < 0.33, Rmax * (1 - 1e-3 * rng.random(n)), Rmax * rng.uniform(0.2, 1.0, n))
        pr.rs[0] = np.maximum(R - rho_q, 1e-5).astype(np.float32)
        pr.flags[0] = 0
    _check(hostlib, sc, refine, mode, tweak, min_taken=0.6)
