"""Host logic of the CUDA tile query: csrc/uts_ring_query.cuh (ring intervals + integer tile-row masks) is __host__ __device__;
tests/hostlogic/ring_query_host.cu drives it on the CPU for one disc at a time and the resulting tile sets must equal the
oracle's (Alg.2 reading A6 and Alg.3), bit for bit, on the shrunk configs, on discs over / on the poles, on every refinement and
on whole-sphere discs.  No GPU needed: nvcc compiles the driver as host code."""
import ctypes as C
import math
import os
import shutil
import subprocess
import tempfile

import numpy as np
import pytest

import oracle as orc
from helpers import ocfg, small_scene

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.fixture(scope="module")
def hostlib():
    if not os.path.exists(NVCC) and shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    out = os.path.join(tempfile.mkdtemp(prefix="uts_hostlogic_"), "ringq_host.so")
    subprocess.check_call([NVCC if os.path.exists(NVCC) else "nvcc", "-O2", "-std=c++17", "-shared", "-Xcompiler", "-fPIC", "-w",
                           "-I", os.path.join(ROOT, "include"), "-I", os.path.join(ROOT, "paper_2606_29794_b200", "csrc"),
                           os.path.join(ROOT, "tests", "hostlogic", "ring_query_host.cu"), "-o", out])
    L = C.CDLL(out)
    L.ring_query_host.restype = C.c_int
    return L


def _host_sets(L, oc, pr, mode):
    kt, kq = oc.tile_order, oc.tile_order + oc.query_refine_log2
    rho_q = 0.0 if mode == 1 else orc.rho_max_closed(kq)
    buf = np.zeros(oc.n_tiles, np.uint32)
    nr = C.c_int(0)
    out = []
    for i in range(oc.n_gauss):
        if pr.flags[0, i] & 1:
            out.append(np.zeros(0, np.uint32)); continue
        d = np.ascontiguousarray(pr.dir[0, i], np.float32)
        R = min(math.pi, float(pr.rs[0, i]) + rho_q)
        n = L.ring_query_host(kt, kq, d.ctypes.data_as(C.c_void_p), C.c_float(pr.lonlat[0, i, 0]), C.c_float(pr.lonlat[0, i, 1]), C.c_double(R),
                              buf.ctypes.data_as(C.c_void_p), buf.shape[0], C.byref(nr))
        out.append(buf[:n].copy())
    return out


def _check(L, sc, refine, mode, tweak=None):
    oc = ocfg(sc, query_refine_log2=refine, query_mode=mode)
    pr = orc.preprocess(oc, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    if tweak is not None:
        tweak(pr)
    off, keys, vals, info = orc.tile_query(oc, pr)
    assert info["min_margin"] > 1e-12
    tiles = (keys >> np.uint64(32)).astype(np.uint32)
    got = _host_sets(L, oc, pr, mode)
    for i in range(oc.n_gauss):
        want = tiles[int(off[i]):int(off[i + 1])]
        assert np.array_equal(got[i], want), (i, pr.dir[0, i], pr.rs[0, i], got[i][:8], want[:8], got[i].shape, want.shape)


@pytest.mark.parametrize("mode", [0, 1], ids=["nested-set", "ring-set"])
@pytest.mark.parametrize("cfg_id,P,order,refine", [(1, 1000, 6, 2), (2, 600, 8, 2), (4, 600, 7, 2), (4, 300, 6, 1), (1, 300, 5, 0),
                                                   (4, 300, 6, 3), (4, 200, 6, 4), (4, 150, 4, 2), (3, 400, 9, 2), (5, 400, 10, 2)])
def test_ring_interval_query_equals_oracle(hostlib, cfg_id, P, order, refine, mode):
    _check(hostlib, small_scene(cfg_id, P, order, n_views=1), refine, mode)


@pytest.mark.parametrize("mode", [0, 1], ids=["nested-set", "ring-set"])
@pytest.mark.parametrize("order,refine", [(6, 2), (7, 2), (5, 0), (6, 4)])
def test_ring_interval_query_poles_large_and_whole_sphere(hostlib, order, refine, mode):
    sc = small_scene(4, 64, order)
    rng = np.random.default_rng(5)

    def tweak(pr):
        d = rng.standard_normal((64, 3))
        d[:8] = [[0.02, 1, 0.01], [0, 1, 0], [0.3, -1, 0.2], [0, -1, 0], [1, 0.05, 0], [0.1, 0.2, -1], [1e-4, 1, 0], [0, -1, 1e-5]]
        d[8:24, 1] = np.where(np.arange(16) % 2 == 0, 1, -1) * (1.0 + 4.0 * rng.random(16))        # near the poles
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        pr.dir[0] = d.astype(np.float32)
        pr.lonlat[0, :, 0] = np.arctan2(d[:, 0], d[:, 2]).astype(np.float32)            # Eq.1 PAPER.md:72 for the hand-made directions
        pr.lonlat[0, :, 1] = np.arctan2(d[:, 1], np.hypot(d[:, 0], d[:, 2])).astype(np.float32)
        rs = np.exp(rng.uniform(math.log(0.003), math.log(3.2), 64))
        rs[:8] = [0.3, 0.21, 0.9, 0.08, math.pi, 2.5, 0.4, 1.6]
        pr.rs[0] = np.minimum(rs, math.pi).astype(np.float32)
        pr.flags[0] = 0
    _check(hostlib, sc, refine, mode, tweak)
