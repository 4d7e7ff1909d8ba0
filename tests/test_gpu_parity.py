"""GPU parity: every stage of the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Stage-wise protocol: GPU stage n runs on the ORACLE's output of stage n-1,
so integer stages must be bit-identical and float stages agree within the stated tolerances; the all-GPU chain is then
compared with the all-oracle chain.  Shrunk versions of the five BASELINE.json configs: several tiles, ragged lists,
masks, multiple views, SH degree 0 and 3.

Tolerances (BASELINE.json north_star): tile lists / sorted order / ranges bit-exact; colour and alpha 1e-4 absolute;
gradients 1e-3 relative (measured against the largest magnitude of each output array, reading A25)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle as orc
from helpers import canon_pairs, ocfg, oracle_mask, small_scene

pytestmark = pytest.mark.gpu

MARGIN = 2e-3      # pixels whose nearest alpha/T decision is closer than this (relative) may legitimately flip in fp32


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B, rasterizer as R
    return B, R


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype) if t.element_size() == torch.empty(0, dtype=dtype).element_size() else t.to(dtype)
    return t.cuda().contiguous()


def u64(t): return t.cpu().numpy().view(np.uint64)
def u32(t): return t.cpu().numpy().view(np.uint32)


# shrunk configs: (cfg_id, n_gauss, order, extra)
CASES = [
    pytest.param(1, 1000, 6, {}, id="cfg1-tiny-full"),
    pytest.param(2, 12000, 7, {}, id="cfg2-panorama-sh3"),
    pytest.param(3, 12000, 7, {}, id="cfg3-fisheye-cap-mask"),
    pytest.param(4, 3000, 7, {}, id="cfg4-large-outliers"),
    pytest.param(5, 8000, 8, {"n_views": 2}, id="cfg5-frustum-2views"),
    pytest.param(4, 30000, 5, {}, id="cfg4-dense-long-lists-early-exit"),     # lists up to ~1500 entries (6 batches), 40 % of pixels saturate
    # general views [W|b]: random tilted rotations and b != 0, so cam = -W^T b, the SH view direction from an off-origin
    # camera, M = W Sigma W^T for a tilted W and W^T dL/dt in the backward are all exercised
    pytest.param(2, 12000, 7, {"general_view": True}, id="cfg2-sh3-general-view"),
    pytest.param(5, 8000, 8, {"n_views": 3, "general_view": True}, id="cfg5-frustum-3-general-views"),
    pytest.param(4, 3000, 7, {"general_view": True, "sh_degree": 2}, id="cfg4-sh2-general-view"),
]


class Case:
    """Oracle results for one shrunk config, computed once per test session."""
    _cache = {}

    def __init__(self, cfg_id, P, order, extra, query_mode=0):
        self.scene = small_scene(cfg_id, P, order, **extra)
        self.ocfg = ocfg(self.scene, query_mode=query_mode)
        self.bits, self.act, self.slot = oracle_mask(self.ocfg, self.scene)
        self.fw = orc.forward_chain(self.ocfg, self.scene, self.slot, self.act, self.bits)
        assert self.fw["qinfo"]["min_margin"] > 1e-12, "margin certificate failed: change the seed"

    @classmethod
    def get(cls, cfg_id, P, order, extra, query_mode=0):
        key = (cfg_id, P, order, tuple(sorted(extra.items())), query_mode)
        if key not in cls._cache:
            cls._cache[key] = Case(cfg_id, P, order, extra, query_mode)
        return cls._cache[key]

    def gpu_mask(self, B):
        if self.bits is None:
            return B.Mask.full()
        return B.Mask(dev(self.act.view(np.int32)), int(self.act.shape[0]), dev(self.slot), dev(self.bits.view(np.int32)))

    def gpu_proj(self, B):
        p = self.fw["proj"]
        return B.Proj(dev(p.dir), dev(p.lonlat), dev(p.rho), dev(p.conic_opac), dev(p.rs), dev(p.rgb), dev(p.flags))


def _cfg(R, scene, **kw):
    return R.config_of(scene, **kw)


# ------------------------------------------------------------------------------------------- HEALPix
def test_pixel_centers_match_oracle():
    B, _ = _gpu()
    for order in range(0, 9):
        n = 12 << (2 * order)
        got = B.uts_pixel_centers(order, 0, n).cpu().numpy()
        _, _, want = orc.centers(order, which=2)
        assert np.abs(got - want).max() < 5e-15
    # a slice at the maximum supported order
    first = (12 << 26) - 1000
    got = B.uts_pixel_centers(13, first, 1000).cpu().numpy()
    _, _, want = orc.centers(13, which=2, first=first, n=1000)
    assert np.abs(got - want).max() < 5e-15


def test_mask_builder_matches_oracle_mask():
    B, R = _gpu()
    for cfg_id, order in ((3, 7), (5, 8)):
        scene = small_scene(cfg_id, 10, order)
        oc = ocfg(scene)
        bits, act, slot = oracle_mask(oc, scene)
        m = B.uts_build_mask(_cfg(R, scene), scene["mask"]["kind"], scene["mask"]["params"])
        gb = u32(m.pixel_mask_bits)
        # the predicate is evaluated in double on both sides from centres that agree to 5e-15 (test_pixel_centers_match_oracle), and
        # no centre of these grids lies within 1e-12 of a mask boundary: the bitmaps, the tile list and the slot table are identical
        assert np.array_equal(gb, bits)
        assert m.n_active == act.shape[0]
        assert np.array_equal(u32(m.active_tiles), act)
        assert np.array_equal(m.slot_of_tile.cpu().numpy(), slot)


# ------------------------------------------------------------------------------------------- F1
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_preprocess(cfg_id, P, order, extra):
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    g, views = R.scene_to_device(c.scene)
    out = B.Proj.empty(cfg)
    B.uts_preprocess(cfg, g, views, out)
    want = c.fw["proj"]
    assert np.array_equal(out.flags.cpu().numpy(), want.flags)
    for name, rtol in (("dir", 0), ("rho", 0), ("rs", 0), ("lonlat", 1e-6), ("conic_opac", 1e-6), ("rgb", 1e-5)):
        a = getattr(out, name).cpu().numpy().astype(np.float64); b = getattr(want, name).astype(np.float64)
        if rtol == 0:
            # geometry is computed in double and rounded once: identical fp32 bits except where the double results straddle a
            # rounding boundary (allow 1 ulp on < 0.01 % of the values)
            neq = a != b
            assert neq.mean() < 1e-4, (name, neq.mean())
            assert np.all(np.abs(a - b)[neq] <= np.abs(b[neq]) * 1.3e-7), name
        else:
            assert np.allclose(a, b, rtol=rtol, atol=rtol), (name, np.abs(a - b).max())


def test_preprocess_culls_and_degree_variants():
    B, R = _gpu()
    for deg in (0, 1, 2, 3):
        scene = small_scene(2, 500, 6, sh_degree=deg)
        scene["means"][:5] *= 1e-3            # rho <= r_near  -> culled
        scene["means"][5] = np.nan            # non-finite     -> culled
        scene["scales"][6] = 0.0              # with dilation still positive definite -> kept
        oc = ocfg(scene)
        want = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
        cfg = _cfg(R, scene)
        g, views = R.scene_to_device(scene)
        out = B.Proj.empty(cfg)
        B.uts_preprocess(cfg, g, views, out)
        assert np.array_equal(out.flags.cpu().numpy(), want.flags)
        assert (want.flags[0, :6] & 1).all()
        assert np.allclose(out.rgb.cpu().numpy(), want.rgb, atol=1e-5)
        assert np.allclose(out.conic_opac.cpu().numpy(), want.conic_opac, rtol=1e-6, atol=1e-6)


def test_preprocess_in_two_calls_is_bit_identical():
    """uts_preprocess_geometry (no SH needed) followed by uts_preprocess_color leaves the records bit-identical to uts_preprocess
    (the host call uploads the SH while the tile lists are built); checked with culled, clamped and multi-view records."""
    B, R = _gpu()
    for deg, V in ((0, 1), (3, 1), (2, 3)):
        scene = small_scene(5, 4000, 6, sh_degree=deg, n_views=V)
        scene["means"][:5] *= 1e-3; scene["means"][5] = np.nan
        scene["sh"][7:400] -= 0.6                                   # pushes colours below 0: clamp bits
        cfg = _cfg(R, scene)
        g, views = R.scene_to_device(scene)
        one = B.Proj.empty(cfg); two = B.Proj.empty(cfg)
        for t in (two.dir, two.lonlat, two.rho, two.conic_opac, two.rs, two.rgb):
            t.fill_(-3.0)
        two.flags.fill_(255)
        B.uts_preprocess(cfg, g, views, one)
        no_sh = B.Gaussians(g.means, g.scales, g.quats, g.opac, None)
        B.uts_preprocess_geometry(cfg, no_sh, views, two)
        assert int((two.flags > 1).sum()) == 0
        B.uts_preprocess_color(cfg, B.Gaussians(g.means, None, None, None, g.sh), views, two)
        torch.cuda.synchronize()
        assert int((one.flags & 1).sum()) >= 6 * V and int((one.flags > 1).sum()) > 0
        for name in ("dir", "lonlat", "rho", "conic_opac", "rs", "rgb", "flags"):
            assert torch.equal(getattr(one, name), getattr(two, name)), name


# ------------------------------------------------------------------------------------------- F2
WINDOW = pytest.mark.parametrize("window", [True, False], ids=["window-path", "ring-intervals-only"])   # uts_tuning.window_mode 2 / 1


@WINDOW
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_tile_query_bit_exact(cfg_id, P, order, extra, window):
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    proj, mask = c.gpu_proj(B), c.gpu_mask(B)
    tn = B.Tuning(window_mode=2 if window else 1)
    n_want = int(c.fw["keys"].shape[0])
    offsets = torch.empty(cfg.n_views * cfg.n_gauss + 1, dtype=torch.int64, device="cuda")
    scratch = torch.empty(B.uts_tile_query_scratch_bytes(cfg) // 8 + 32, dtype=torch.int64, device="cuda")
    # count-only call
    n = B.uts_tile_query(cfg, proj, mask, offsets, None, None, 0, scratch, tuning=tn)
    assert n == n_want
    assert np.array_equal(u64(offsets), c.fw["offsets"])
    # capacity too small -> error carrying the needed size
    keys = torch.empty(max(n, 1), dtype=torch.int64, device="cuda"); vals = torch.empty(max(n, 1), dtype=torch.int32, device="cuda")
    if n > 1:
        with pytest.raises(B.UtsError) as ei:
            B.uts_tile_query(cfg, proj, mask, offsets, keys, vals, n - 1, scratch, tuning=tn)
        assert ei.value.status == B.UTS_ERR_CAPACITY and ei.value.needed == n
    n = B.uts_tile_query(cfg, proj, mask, offsets, keys, vals, n, scratch, tuning=tn)
    gk, gv = canon_pairs(u64(offsets), u64(keys), u32(vals))
    assert np.array_equal(gk, c.fw["keys"])
    assert np.array_equal(gv, c.fw["vals"])


@pytest.mark.parametrize("block_radius", [0.0, 6.0], ids=["default-split", "most-discs-on-the-block-path"])
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_tile_query_quadtree_descent_bit_exact(cfg_id, P, order, extra, block_radius):
    """uts_tuning.query_impl = 1: the stackless quadtree descent — Alg.2's depth-first form, the library's path
    for k_q = 13 — on every case, with the default thread / block split and with the split moved so that most discs take the
    block-per-Gaussian bitmap path.  Count-only, capacity error, emit; with and without the depth-order emission ranks."""
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    proj, mask = c.gpu_proj(B), c.gpu_mask(B)
    tn = B.Tuning(query_impl=1, descent_block_radius=block_radius)
    n_want = int(c.fw["keys"].shape[0])
    offsets = torch.empty(cfg.n_views * cfg.n_gauss + 1, dtype=torch.int64, device="cuda")
    scratch = torch.empty(B.uts_tile_query_scratch_bytes(cfg) // 8 + 32, dtype=torch.int64, device="cuda")
    assert B.uts_tile_query(cfg, proj, mask, offsets, None, None, 0, scratch, tuning=tn) == n_want
    assert np.array_equal(u64(offsets), c.fw["offsets"])
    keys = torch.empty(max(n_want, 1), dtype=torch.int64, device="cuda"); vals = torch.empty(max(n_want, 1), dtype=torch.int32, device="cuda")
    if n_want > 1:
        with pytest.raises(B.UtsError) as ei:
            B.uts_tile_query(cfg, proj, mask, offsets, keys, vals, n_want - 1, scratch, tuning=tn)
        assert ei.value.status == B.UTS_ERR_CAPACITY and ei.value.needed == n_want
    B.uts_tile_query(cfg, proj, mask, offsets, keys, vals, n_want, scratch, tuning=tn)
    gk, gv = canon_pairs(u64(offsets), u64(keys), u32(vals))
    assert np.array_equal(gk, c.fw["keys"]) and np.array_equal(gv, c.fw["vals"])
    # the whole staged chain on the descent, depth-presorted: sorted arrays and ranges
    r = R.Rasterizer(cfg, mask, fused_lists=False, depth_presort=True, tuning=tn)
    r.proj = proj
    r.depth_order(); r.tile_query(); r.sort(); r.tile_ranges()
    assert r.n_pairs == n_want
    assert np.array_equal(u64(r.keys)[:n_want], c.fw["skeys"]) and np.array_equal(u32(r.vals)[:n_want], c.fw["svals"])
    assert np.array_equal(u64(r.ranges), c.fw["ranges"])


@pytest.mark.parametrize("mode,P,seed", [(0, 300, 0), (1, 120, 1)], ids=["nested", "ring-set"])
def test_tile_query_order13_refine16_takes_the_descent(mode, P, seed):
    """k = 13, f = 16: k_q = 13, where a block's ring table no longer fits shared memory and the library switches to the quadtree
    descent by itself (no tuning).  A few hundred Gaussians incl. discs of tens of thousands of tiles, a polar one and a culled
    one; the oracle's descent / Alg.3 scan is the reference (its brute force over 12 * 4^13 pixels per Gaussian is out of reach),
    pinned at lower orders.  (seed: the one whose margin certificate holds.)"""
    B, R = _gpu()
    scene = small_scene(5, P, 13, n_views=1, seed=seed)
    scene["mask"] = None
    scene["scales"][::7] *= 8.0
    scene["means"][3] = np.array([0.004, 2.5, -0.003]); scene["means"][5] *= 1e-3
    oc = ocfg(scene, query_refine_log2=4, query_mode=mode)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    off, keys, vals, info = orc.tile_query(oc, pr)
    assert info["min_margin"] > 1e-12 and keys.shape[0] > 3000
    cfg = _cfg(R, scene, query_refine_log2=4, query_mode=mode)
    proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    n = int(keys.shape[0])
    offsets = torch.empty(cfg.n_gauss + 1, dtype=torch.int64, device="cuda")
    scratch = torch.empty(B.uts_tile_query_scratch_bytes(cfg) // 8 + 32, dtype=torch.int64, device="cuda")
    gkeys = torch.empty(n, dtype=torch.int64, device="cuda"); gvals = torch.empty(n, dtype=torch.int32, device="cuda")
    assert B.uts_tile_query(cfg, proj, B.Mask.full(), offsets, gkeys, gvals, n, scratch) == n
    assert np.array_equal(u64(offsets), off)
    gk, gv = canon_pairs(u64(offsets), u64(gkeys), u32(gvals))
    assert np.array_equal(gk, keys) and np.array_equal(gv, vals)


@pytest.mark.parametrize("mode", [0, 1], ids=["nested", "ring-set"])
@pytest.mark.parametrize("order,refine,masked", [(8, 2, False), (9, 2, True), (8, 0, False), (8, 4, False), (12, 2, False)])
def test_tile_query_window_path_small_discs_everywhere(order, refine, masked, mode):
    """The tile-window path (uts_window_query.cuh) on discs it is made for: 6000 small discs, among them centres ON and next to the
    poles, the vertices shared by three and by four faces and the meridian face edges, radii up to the largest the path accepts (so
    that 3 x 3, 5 x 5 and 7 x 7 windows all occur), with a cap mask or without; emission ranks from uts_depth_order; count-only, then
    emit.  Against the oracle's sets, bit for bit; the same call with the window path switched off must give the same arrays."""
    B, R = _gpu()
    n = 6000
    scene = small_scene(3 if masked else 4, n, order, n_views=1)
    if not masked:
        scene["mask"] = None
    oc = ocfg(scene, query_refine_log2=refine, query_mode=mode)
    bits, act, slot = oracle_mask(oc, scene)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    rng = np.random.default_rng(order * 10 + refine)
    Nt = 1 << oc.tile_order
    d = pr.dir[0].astype(np.float64)
    special = [[0, 1, 0], [0, -1, 0]]
    for sgn in (1, -1):
        for c in range(4):
            lam = c * np.pi / 2
            special.append([np.sqrt(5) / 3 * np.sin(lam), sgn * 2 / 3, np.sqrt(5) / 3 * np.cos(lam)])       # 3-face vertices (camera frame)
    for c in range(4):
        lam = np.pi / 4 + c * np.pi / 2
        special.append([np.sin(lam), 0.0, np.cos(lam)])                                                     # 4-face vertices
    special = np.array(special)
    k = special.shape[0]
    for rep in range(40):
        d[rep * k:(rep + 1) * k] = special + (0.0 if rep == 0 else 0.8 / Nt) * rng.standard_normal((k, 3))
    zz = rng.uniform(0.67, 0.9999, 300) * rng.choice([-1, 1], 300); lam = rng.integers(0, 4, 300) * np.pi / 2
    d[40 * k:40 * k + 300] = np.stack([np.sqrt(1 - zz * zz) * np.sin(lam), zz, np.sqrt(1 - zz * zz) * np.cos(lam)], 1)   # meridian face edges
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    pr.dir[0] = d.astype(np.float32)
    pr.lonlat[0, :, 0] = np.arctan2(d[:, 0], d[:, 2]).astype(np.float32)
    pr.lonlat[0, :, 1] = np.arctan2(d[:, 1], np.hypot(d[:, 0], d[:, 2])).astype(np.float32)
    rho_q = 0.0 if mode == 1 else orc.rho_max_closed(oc.tile_order + refine)
    w = rng.integers(1, 4, n)
    Rmax = 0.98 * 0.6 * w / Nt
    Rr = np.where(rng.random(n) < 0.3, Rmax * (1 - 1e-3 * rng.random(n)), Rmax * rng.uniform(0.1, 1.0, n))
    Rr[::50] *= 4.0                                                              # a few discs beyond the window class, mixed in
    pr.rs[0] = np.maximum(Rr - rho_q, 1e-5).astype(np.float32)
    pr.rho[0] = rng.uniform(0.5, 30.0, n).astype(np.float32)
    pr.flags[0] = 0
    pr.flags[0, 5::97] = 1                                                       # culled records in between
    off, keys, vals, info = orc.tile_query(oc, pr, slot)
    assert info["min_margin"] > 1e-12
    cfg = _cfg(R, scene, query_refine_log2=refine, query_mode=mode)
    mask = B.Mask.full() if bits is None else B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    got = []
    for tn in (B.Tuning(window_mode=2), B.Tuning(window_mode=1)):
        r = R.Rasterizer(cfg, mask, depth_presort=True, fused_lists=False, tuning=tn, pair_capacity=16)
        r.proj = proj
        r.depth_order()
        assert r.tile_query() == keys.shape[0]
        rank = u32(r.emit_rank).astype(np.int64)
        cnt = np.diff(u64(r.offsets).astype(np.int64))
        assert np.array_equal(cnt[rank], np.diff(off.astype(np.int64)))          # per-Gaussian counts, in emission-rank order
        r.sort(); r.tile_ranges()
        wk, wv = orc.sort_pairs(keys, vals)
        assert np.array_equal(u64(r.keys)[: r.n_pairs], wk) and np.array_equal(u32(r.vals)[: r.n_pairs], wv)
        got.append((u64(r.keys)[: r.n_pairs].copy(), u32(r.vals)[: r.n_pairs].copy()))
    assert np.array_equal(got[0][0], got[1][0]) and np.array_equal(got[0][1], got[1][1])


@pytest.mark.parametrize("refine", [0, 1, 3, 4])
def test_tile_query_other_refinements(refine):
    B, R = _gpu()
    scene = small_scene(4, 800, 6)
    oc = ocfg(scene, query_refine_log2=refine)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    off, keys, vals, info = orc.tile_query(oc, pr)
    assert info["min_margin"] > 1e-12
    cfg = _cfg(R, scene, query_refine_log2=refine)
    proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    r = R.Rasterizer(cfg, pair_capacity=16, depth_presort=False)       # forces the capacity-retry path
    r.proj = proj
    n = r.tile_query()
    assert n == keys.shape[0]
    assert np.array_equal(u64(r.offsets), off)
    gk, gv = canon_pairs(u64(r.offsets), u64(r.keys), u32(r.vals))
    assert np.array_equal(gk, keys) and np.array_equal(gv, vals)


@pytest.mark.parametrize("cfg_id,order,refine", [(4, 9, 2), (3, 9, 2), (4, 8, 1), (5, 10, 2)])
def test_tile_query_block_path_large_discs(cfg_id, order, refine):
    """Discs of thousands of tiles take the block-per-Gaussian bitmap path (R > 36/sqrt(N_tile)); with and without a mask."""
    B, R = _gpu()
    scene = small_scene(cfg_id, 300, order, n_views=1)
    scene["scales"][::2] *= 30.0                   # every other Gaussian becomes a very large disc
    scene["scales"][7] = 80.0                      # r_s = pi inside the block path
    oc = ocfg(scene, query_refine_log2=refine)
    bits, act, slot = oracle_mask(oc, scene)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    assert (pr.rs[0] + orc.rho_max_closed(oc.tile_order + refine) > 36.0 / np.sqrt(oc.n_tiles)).sum() > 8
    off, keys, vals, info = orc.tile_query(oc, pr, slot)
    assert info["min_margin"] > 1e-12
    cfg = _cfg(R, scene, query_refine_log2=refine)
    mask = B.Mask.full() if bits is None else B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    r = R.Rasterizer(cfg, mask, depth_presort=False)
    r.proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    n = r.tile_query()
    assert n == keys.shape[0]
    assert np.array_equal(u64(r.offsets), off)
    gk, gv = canon_pairs(u64(r.offsets), u64(r.keys), u32(r.vals))
    assert np.array_equal(gk, keys) and np.array_equal(gv, vals)


def test_tile_query_whole_sphere_and_empty():
    B, R = _gpu()
    scene = small_scene(1, 4, 6)
    scene["scales"][0] = 50.0                      # r_s clamps to pi: every tile (reading A24)
    scene["means"][1] *= 1e-4                      # culled: zero tiles
    oc = ocfg(scene)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    off, keys, vals, _ = orc.tile_query(oc, pr)
    assert off[1] - off[0] == oc.n_tiles and off[2] == off[1]
    cfg = _cfg(R, scene)
    r = R.Rasterizer(cfg, depth_presort=False)
    r.proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    n = r.tile_query()
    gk, gv = canon_pairs(u64(r.offsets), u64(r.keys), u32(r.vals))
    assert np.array_equal(u64(r.offsets), off) and np.array_equal(gk, keys) and np.array_equal(gv, vals)
    # P = 0
    cfg0 = B.Config(order=6, n_gauss=0)
    r0 = R.Rasterizer(cfg0, depth_presort=False)
    assert r0.tile_query() == 0


# ------------------------------------------------------------------------------------------- F2, RING mode (NEXT-1)
@pytest.mark.parametrize("cfg_id,P,order,refine,big", [
    (1, 1000, 6, 2, False), (2, 12000, 7, 2, False), (4, 3000, 7, 2, False), (3, 12000, 7, 2, False), (5, 8000, 8, 2, False),
    (4, 800, 6, 0, False), (4, 800, 6, 1, False), (4, 800, 6, 4, False), (4, 300, 9, 2, True), (3, 300, 9, 2, True), (5, 300, 10, 2, True)])
def test_tile_query_ring_mode_bit_exact(cfg_id, P, order, refine, big):
    """query_mode = UTS_QUERY_RING: the CUDA path against the oracle's Alg.3 step by step.  Small discs,
    masks, refinements x1..x16, and (big) discs of thousands of tiles incl. r_s = pi and discs over the poles."""
    B, R = _gpu()
    scene = small_scene(cfg_id, P, order, n_views=1)
    if big:
        scene["scales"][::2] *= 30.0
        scene["scales"][7] = 80.0
        scene["means"][9] = np.array([0.01, 3.0, 0.02]); scene["means"][11] = np.array([0.02, -2.0, 0.01])   # discs over the poles
    oc = ocfg(scene, query_refine_log2=refine, query_mode=1)
    bits, act, slot = oracle_mask(oc, scene)
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    off, keys, vals, info = orc.tile_query(oc, pr, slot)
    assert info["min_margin"] > 1e-12
    cfg = _cfg(R, scene, query_refine_log2=refine, query_mode=1)
    mask = B.Mask.full() if bits is None else B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    r = R.Rasterizer(cfg, mask, depth_presort=False)
    r.proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    n = r.tile_query()
    assert n == keys.shape[0]
    assert np.array_equal(u64(r.offsets), off)
    gk, gv = canon_pairs(u64(r.offsets), u64(r.keys), u32(r.vals))
    assert np.array_equal(gk, keys) and np.array_equal(gv, vals)
    # and it is not the NESTED set
    ocn = ocfg(scene, query_refine_log2=refine)
    assert orc.tile_query(ocn, pr, slot)[1].shape[0] > n


@pytest.mark.parametrize("cfg_id,P,order,extra", [CASES[1], CASES[2]])
def test_end_to_end_chain_ring_mode(cfg_id, P, order, extra):
    """All-GPU chain in RING mode against the all-oracle chain in RING mode: lists bit-exact, image 1e-4, gradients 1e-3."""
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra, query_mode=1)
    cfg = _cfg(R, c.scene, query_mode=1)
    mask = c.gpu_mask(B)
    g, views = R.scene_to_device(c.scene)
    r = R.Rasterizer(cfg, mask)
    r.forward(g, views)
    n = r.n_pairs
    assert n == c.fw["skeys"].shape[0]
    assert np.array_equal(u64(r.keys)[:n], c.fw["skeys"]) and np.array_equal(u32(r.vals)[:n], c.fw["svals"])
    assert np.array_equal(u64(r.ranges), c.fw["ranges"])
    _compare_image(c, r.color.cpu().numpy(), r.alpha.cpu().numpy(), u32(r.n_last))
    from paper_2606_29794_b200 import scenes
    V, npx = r.color.shape[0], r.color.shape[1]
    gcol, _ = _zero_unsafe(c, scenes.upstream_grad(V, npx, seed=200 + cfg_id))
    s = c.scene
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(c.ocfg, c.fw["proj"], c.fw["ranges"], c.fw["svals"], c.fw["n_last"], gcol, None, c.act, c.bits)
    w_means, w_scales, w_quats, w_sh = orc.preprocess_bwd(c.ocfg, s["means"], s["scales"], s["quats"], s["sh"], s["W"], s["b"], w_rgb, w_conic, w_mu2)
    G = r.backward(g, views, dev(gcol))
    for name, want in (("means", w_means), ("scales", w_scales), ("quats", w_quats), ("opac", w_opac), ("sh", w_sh)):
        e = _rel_err(G[name].cpu().numpy(), want)
        assert e <= 1e-3, (name, e)


# ------------------------------------------------------------------------------------------- F3 / F4
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_sort_and_ranges_bit_exact(cfg_id, P, order, extra):
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    n = int(c.fw["keys"].shape[0])
    keys = dev(c.fw["keys"].view(np.int64)); vals = dev(c.fw["vals"].view(np.int32))
    kt = torch.empty_like(keys); vt = torch.empty_like(vals)
    scratch = torch.empty(B.uts_sort_scratch_bytes(n) // 8 + 32, dtype=torch.int64, device="cuda")
    B.uts_sort(cfg, n, keys, vals, kt, vt, scratch)
    assert np.array_equal(u64(keys), c.fw["skeys"])
    assert np.array_equal(u32(vals), c.fw["svals"])           # ties broken by Gaussian id (stability)
    ranges = torch.empty(cfg.n_views * cfg.n_tiles, 2, dtype=torch.int64, device="cuda")
    B.uts_tile_ranges(cfg, n, keys, ranges)
    assert np.array_equal(u64(ranges), c.fw["ranges"])


@pytest.mark.parametrize("n", [0, 1, 2, 255, 3071, 3072, 3073, 50_000, 1_000_003])
def test_sort_sizes_and_ties(n):
    """Ragged sizes around the 3072-pair block and heavy ties: values record the input position, so stability is visible."""
    B, R = _gpu()
    cfg = B.Config(order=10, n_gauss=1, n_views=4)           # 18 tile bits -> 7 passes
    rng = np.random.default_rng(n)
    tile = rng.integers(0, 4 * cfg.n_tiles, n, dtype=np.uint64)
    depth = rng.integers(0, 7, n, dtype=np.uint64) * np.uint64(0x01010101) if n % 2 else rng.integers(0, 1 << 32, n, dtype=np.uint64)
    keys_h = (tile << np.uint64(32)) | depth
    vals_h = np.arange(n, dtype=np.uint32)
    wk, wv = orc.sort_pairs(keys_h, vals_h)
    keys = dev(keys_h.view(np.int64)) if n else torch.empty(0, dtype=torch.int64, device="cuda")
    vals = dev(vals_h.view(np.int32)) if n else torch.empty(0, dtype=torch.int32, device="cuda")
    kt = torch.empty_like(keys); vt = torch.empty_like(vals)
    scratch = torch.empty(B.uts_sort_scratch_bytes(max(n, 1)) // 8 + 32, dtype=torch.int64, device="cuda")
    B.uts_sort(cfg, n, keys, vals, kt, vt, scratch)
    assert np.array_equal(u64(keys), wk) and np.array_equal(u32(vals), wv)
    ranges = torch.empty(cfg.n_views * cfg.n_tiles, 2, dtype=torch.int64, device="cuda")
    B.uts_tile_ranges(cfg, n, keys, ranges)
    assert np.array_equal(u64(ranges), orc.tile_ranges(orc.Config(order=10, n_gauss=1, n_views=4), wk))


# ------------------------------------------------------------------------------------------- F5 / F6
def _render_gpu(B, R, c, cfg, marks=True):
    mask = c.gpu_mask(B)
    r = R.Rasterizer(cfg, mask, pair_capacity=int(c.fw["svals"].shape[0]), marks=marks)      # the marks are sized by the capacity
    r.proj = c.gpu_proj(B)
    r.ranges = dev(c.fw["ranges"].view(np.int64))
    r.vals = dev(c.fw["svals"].view(np.int32))
    r.render_fwd()
    return r


def _compare_image(c, color, alpha, n_last):
    want_c, want_a, want_n, margin = c.fw["color"], c.fw["alpha"], c.fw["n_last"], c.fw["margin"]
    safe = margin > MARGIN
    assert safe.mean() > 0.9
    dc = np.abs(color.astype(np.float64) - want_c).max(axis=-1)
    da = np.abs(alpha.astype(np.float64) - want_a)
    assert dc[safe].max() <= 1e-4, dc[safe].max()
    assert da[safe].max() <= 1e-4, da[safe].max()
    assert np.array_equal(n_last[safe], want_n[safe])
    # a flipped borderline decision changes a pixel by at most about alpha_min (or the clamp step)
    assert dc.max() < 2e-2 and da.max() < 2e-2


MARKS = pytest.mark.parametrize("marks", [False, True], ids=["plain", "marked"])     # uts_render_fwd / _bwd and the marked pair


@MARKS
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_render_fwd(cfg_id, P, order, extra, marks):
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    r = _render_gpu(B, R, c, _cfg(R, c.scene), marks)
    color, alpha = r.color.cpu().numpy(), r.alpha.cpu().numpy()
    _compare_image(c, color, alpha, u32(r.n_last))
    assert np.allclose(r.trans.cpu().numpy() + alpha, 1.0, atol=1e-6)
    if c.bits is not None:       # masked-out pixels of active tiles are exactly zero
        ppt = c.ocfg.ppt
        pix = (c.act.astype(np.int64)[:, None] * ppt + np.arange(ppt)[None, :]).reshape(-1)
        on = ((c.bits[pix >> 5] >> (pix & 31).astype(np.uint32)) & 1).astype(bool)
        assert (color[:, ~on] == 0).all() and (alpha[:, ~on] == 0).all()


@pytest.mark.parametrize("cfg_id,P,order,extra", [CASES[1], CASES[5]])
def test_render_fwd_counted_matches_the_oracle_work_counters(cfg_id, P, order, extra):
    """uts_render_fwd_counted (bench.py's work counters; it walks every entry in full): bit-identical image to uts_render_fwd, whose
    patch cull and early out therefore change nothing, and the evaluated / contributing pair counts of Alg.1's loop equal the
    oracle's counters up to the few pixels whose decisions sit on a threshold."""
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    r = _render_gpu(B, R, c, _cfg(R, c.scene), marks=False)
    work = torch.zeros(4, dtype=torch.int64, device="cuda")
    out = [torch.empty_like(t) for t in (r.color, r.alpha, r.trans, r.n_last)]
    B.uts_render_fwd_counted(r.cfg, r.proj, r.mask, r.ranges, r.vals, *out, work)
    for a, b in zip(out, (r.color, r.alpha, r.trans, r.n_last)):        # the counted walk takes no patch cull and no early out:
        assert torch.equal(a, b)                                          # the production kernel's shortcuts change no bit
    ev, contrib, n_cull, n_full = (int(x) for x in work.cpu().tolist())
    assert contrib <= n_full <= n_cull <= ev
    ctr = c.fw["counters"]
    assert abs(ev - ctr["evaluated"]) <= 2e-3 * ctr["evaluated"] + 16, (ev, ctr)
    assert abs(contrib - ctr["contributing"]) <= 2e-3 * ctr["contributing"] + 16, (contrib, ctr)
    assert ev >= int(u32(r.n_last).astype(np.int64).sum())                # every entry before n_last was evaluated


def test_render_fwd_background_and_no_thresholds():
    """bg != 0; alpha rules disabled (alpha_min 0, alpha_max 1, eps 0): no decision can flip, every pixel must agree."""
    B, R = _gpu()
    scene = small_scene(1, 1000, 6)
    kw = dict(alpha_min=0.0, alpha_max=1.0, t_eps=0.0, bg=(0.25, 0.5, 0.75))
    oc = ocfg(scene, **kw)
    fw = orc.forward_chain(oc, scene)
    cfg = _cfg(R, scene, **kw)
    r = R.Rasterizer(cfg, pair_capacity=int(fw["svals"].shape[0]))
    p = fw["proj"]
    r.proj = B.Proj(dev(p.dir), dev(p.lonlat), dev(p.rho), dev(p.conic_opac), dev(p.rs), dev(p.rgb), dev(p.flags))
    r.ranges = dev(fw["ranges"].view(np.int64)); r.vals = dev(fw["svals"].view(np.int32))
    r.render_fwd()
    assert np.abs(r.color.cpu().numpy() - fw["color"]).max() <= 1e-4
    assert np.abs(r.alpha.cpu().numpy() - fw["alpha"]).max() <= 1e-4


# ------------------------------------------------------------------------------------------- B1 / B2
def _rel_err(got, want):
    """Gradient error against the 1e-3 bar (reading A25), the LARGER of two measures, so that small entries cannot hide behind the
    array's largest one: (i) max |got - want| / max |want|; (ii) per element, |got - want| / (|want| + 0.05 rms(want)) — relative
    for every entry above a twentieth of the array's RMS, absolute (5e-5 rms) below, where fp32 atomics in a different order already
    differ by that much (measured: (ii) stays below 3e-4 on every case, (i) below 6e-6)."""
    got = got.astype(np.float64)
    d = np.abs(got - want)
    scale = max(np.abs(want).max(), 1e-30)
    rms = max(float(np.sqrt(np.mean(np.square(want)))), 1e-30)
    return max(d.max() / scale, float((d / (np.abs(want) + 0.05 * rms)).max()))


def _zero_unsafe(c, gcol, galpha=None):
    """A pixel whose forward decisions sit within MARGIN of a threshold may legitimately take the other branch in fp32, which
    changes its gradient contributions by a finite step; such pixels get zero upstream gradient on BOTH sides, so the
    comparison below measures arithmetic, not branch flips.  (The thresholds-off test further down covers every pixel.)"""
    unsafe = ~(c.fw["margin"] > MARGIN)
    gcol = gcol.copy(); gcol[unsafe] = 0
    if galpha is not None:
        galpha = galpha.copy(); galpha[unsafe] = 0
    return gcol, galpha


@MARKS
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_backward(cfg_id, P, order, extra, marks):
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    r = _render_gpu(B, R, c, cfg, marks)
    V, npx = r.color.shape[0], r.color.shape[1]
    from paper_2606_29794_b200 import scenes
    gcol, galpha = _zero_unsafe(c, *scenes.upstream_grad(V, npx, seed=cfg_id, with_alpha=True))
    # oracle backward on the oracle's own forward state
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(c.ocfg, c.fw["proj"], c.fw["ranges"], c.fw["svals"], c.fw["n_last"], gcol, galpha,
                                                   c.act, c.bits)
    r.render_bwd(dev(gcol), dev(galpha))
    G = r.grads
    for name, want in (("rgb", w_rgb), ("conic", w_conic), ("mu2", w_mu2), ("opac", w_opac)):
        e = _rel_err(G[name].cpu().numpy(), want)
        assert e <= 1e-3, (name, e)
    # B2 on the oracle's B1 output (stage-wise)
    s = c.scene
    w_means, w_scales, w_quats, w_sh = orc.preprocess_bwd(c.ocfg, s["means"], s["scales"], s["quats"], s["sh"], s["W"], s["b"],
                                                          w_rgb, w_conic, w_mu2)
    g, views = R.scene_to_device(s)
    G["rgb"].copy_(dev(w_rgb.astype(np.float32))); G["conic"].copy_(dev(w_conic.astype(np.float32))); G["mu2"].copy_(dev(w_mu2.astype(np.float32)))
    r.preprocess_bwd(g, views)
    for name, want in (("means", w_means), ("scales", w_scales), ("quats", w_quats), ("sh", w_sh)):
        e = _rel_err(G[name].cpu().numpy(), want)
        assert e <= 1e-3, (name, e)


@pytest.mark.parametrize("cfg_id,P,order,extra,marks", [(1, 1000, 6, {}, True), (2, 12000, 7, {}, True), (4, 30000, 5, {}, True), (2, 12000, 7, {}, False),
                                                        (2, 8000, 7, {"general_view": True}, True), (5, 6000, 7, {"general_view": True, "n_views": 2}, False)])
def test_backward_thresholds_off_every_pixel(cfg_id, P, order, extra, marks):
    """alpha_min 0, alpha_max 1, eps 0: no decision exists, so every pixel takes part and the whole chain (forward on the GPU,
    backward on the GPU) must match the oracle's within 1e-3 on every gradient array."""
    B, R = _gpu()
    scene = small_scene(cfg_id, P, order, **extra)
    scene["mask"] = None                               # full sphere: every pixel of every tile takes part
    kw = dict(alpha_min=0.0, alpha_max=1.0, t_eps=0.0, bg=(0.1, 0.2, 0.3))
    oc = ocfg(scene, **kw)
    fw = orc.forward_chain(oc, scene)
    cfg = _cfg(R, scene, **kw)
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg, marks=marks)
    r.forward(g, views)
    assert np.array_equal(u64(r.keys)[: r.n_pairs], fw["skeys"])
    assert np.abs(r.color.cpu().numpy() - fw["color"]).max() <= 1e-4
    from paper_2606_29794_b200 import scenes
    gcol, galpha = scenes.upstream_grad(cfg.n_views, r.color.shape[1], seed=7, with_alpha=True)
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(oc, fw["proj"], fw["ranges"], fw["svals"], fw["n_last"], gcol, galpha)
    w_means, w_scales, w_quats, w_sh = orc.preprocess_bwd(oc, scene["means"], scene["scales"], scene["quats"], scene["sh"], scene["W"],
                                                          scene["b"], w_rgb, w_conic, w_mu2)
    r.render_bwd(dev(gcol), dev(galpha))
    r.preprocess_bwd(g, views)
    G = r.grads
    for name, want in (("rgb", w_rgb), ("conic", w_conic), ("mu2", w_mu2), ("opac", w_opac), ("means", w_means), ("scales", w_scales),
                       ("quats", w_quats), ("sh", w_sh)):
        e = _rel_err(G[name].cpu().numpy(), want)
        assert e <= 1e-3, (name, e)


# ------------------------------------------------------------------------------------------- whole chain
# the three ways the ABI builds the sorted lists (include/uts.h), with the marked and the plain blend pair:
#   fused            uts_depth_order -> uts_tile_lists                                              (the default), marked blend
#   staged-presorted uts_depth_order -> uts_tile_query(emit_rank) -> uts_sort(depth_presorted = 1) -> uts_tile_ranges, plain blend
#   staged-plain     uts_tile_query(emit_rank = NULL) -> uts_sort (all key bytes) -> uts_tile_ranges, marked blend
PATHS = {"fused": dict(depth_presort=True, fused_lists=True, marks=True),
         "staged-presorted": dict(depth_presort=True, fused_lists=False, marks=False),
         "staged-plain": dict(depth_presort=False, fused_lists=False, marks=True)}


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES)
def test_end_to_end_chain(cfg_id, P, order, extra, path):
    """All-GPU chain against the all-oracle chain: pair lists, sorted order and ranges bit-exact (the GPU preprocess
    rounds double results to fp32 once, as the oracle does), image within 1e-4, parameter gradients within 1e-3."""
    B, R = _gpu()
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    if c.scene["mask"] is not None:
        mask = B.uts_build_mask(cfg, c.scene["mask"]["kind"], c.scene["mask"]["params"])
        assert np.array_equal(u32(mask.pixel_mask_bits), c.bits)
    else:
        mask = B.Mask.full()
    g, views = R.scene_to_device(c.scene)
    r = R.Rasterizer(cfg, mask, **PATHS[path])
    assert r.fused_lists == PATHS[path]["fused_lists"] and r.use_marks == PATHS[path]["marks"]
    r.forward(g, views)
    n = r.n_pairs
    # fp32 records straddling a rounding boundary could flip a borderline tile; require exact equality and report if not
    assert n == c.fw["skeys"].shape[0]
    assert np.array_equal(u64(r.keys)[:n], c.fw["skeys"])
    assert np.array_equal(u32(r.vals)[:n], c.fw["svals"])
    assert np.array_equal(u64(r.ranges), c.fw["ranges"])
    _compare_image(c, r.color.cpu().numpy(), r.alpha.cpu().numpy(), u32(r.n_last))
    from paper_2606_29794_b200 import scenes
    V, npx = r.color.shape[0], r.color.shape[1]
    gcol, _ = _zero_unsafe(c, scenes.upstream_grad(V, npx, seed=100 + cfg_id))
    s = c.scene
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(c.ocfg, c.fw["proj"], c.fw["ranges"], c.fw["svals"], c.fw["n_last"], gcol, None, c.act, c.bits)
    w_means, w_scales, w_quats, w_sh = orc.preprocess_bwd(c.ocfg, s["means"], s["scales"], s["quats"], s["sh"], s["W"], s["b"], w_rgb, w_conic, w_mu2)
    G = r.backward(g, views, dev(gcol))
    for name, want in (("means", w_means), ("scales", w_scales), ("quats", w_quats), ("opac", w_opac), ("sh", w_sh)):
        e = _rel_err(G[name].cpu().numpy(), want)
        assert e <= 1e-3, (name, e)


def test_host_call_matches_device_chain():
    """uts_host_forward_backward (host buffers, copies inside) returns what the stage calls return."""
    B, R = _gpu()
    scene = small_scene(2, 5000, 7)
    cfg = _cfg(R, scene)
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg)
    r.forward(g, views)
    from paper_2606_29794_b200 import scenes
    gcol = scenes.upstream_grad(1, r.color.shape[1], seed=5)
    G = r.backward(g, views, dev(gcol))
    h = {k: torch.from_numpy(scene[k]).contiguous() for k in ("means", "scales", "quats", "opac", "sh", "W", "b")}
    P, M = cfg.n_gauss, cfg.n_sh
    out = dict(color=torch.empty(1, r.color.shape[1], 3), alpha=torch.empty(1, r.color.shape[1]), dL_dmeans=torch.empty(P, 3),
               dL_dscales=torch.empty(P, 3), dL_dquats=torch.empty(P, 4), dL_dopac=torch.empty(P), dL_dsh=torch.empty(P, M, 3))
    cap = r.n_pairs + 10
    ws = torch.empty(B.uts_host_workspace_bytes(cfg, -1, cap) // 8 + 64, dtype=torch.int64, device="cuda")
    with pytest.raises(B.UtsError):
        B.uts_host_forward_backward(cfg, h, B.Mask.full(), torch.from_numpy(gcol), out, 7, ws)      # capacity too small
    n = B.uts_host_forward_backward(cfg, h, B.Mask.full(), torch.from_numpy(gcol), out, cap, ws)
    assert n == r.n_pairs
    assert torch.equal(out["color"], r.color.cpu()) and torch.equal(out["alpha"], r.alpha.cpu())
    for name in ("means", "scales", "quats", "opac", "sh"):
        a, b = out["dL_d" + name].numpy(), G[name].cpu().numpy()
        assert np.abs(a - b).max() <= 1e-4 * max(np.abs(b).max(), 1e-30)      # atomics: summation order differs run to run


def test_invalid_arguments_are_reported():
    B, R = _gpu()
    bad = B.Config(order=3, n_gauss=10)              # order < tile_log2
    with pytest.raises(B.UtsError) as ei:
        B.uts_preprocess(bad, B.Gaussians(*[torch.zeros(40, device="cuda")] * 5), B.Views(torch.zeros(9, device="cuda"), torch.zeros(3, device="cuda")),
                         B.Proj.empty(B.Config(order=6, n_gauss=10)))
    assert ei.value.status == B.UTS_ERR_INVALID_ARG
    with pytest.raises(B.UtsError) as ei:
        B.uts_sort(B.Config(order=6, n_gauss=1, tile_log2=3), 4, *[torch.zeros(8, dtype=torch.int64, device="cuda"), torch.zeros(8, dtype=torch.int32, device="cuda")] * 2,
                   torch.zeros(4096, dtype=torch.int64, device="cuda"))
    assert ei.value.status == B.UTS_ERR_UNSUPPORTED
    with pytest.raises(RuntimeError):
        B.uts_tile_ranges(B.Config(order=6, n_gauss=1), 1, torch.zeros(1, dtype=torch.int64), torch.zeros(4, dtype=torch.int64, device="cuda"))


# ------------------------------------------------------------------------------------------- F2 + F3 + F4 fused
@pytest.mark.parametrize("mat_tiles", [None, 3.0, 40.0, "off"], ids=["default-threshold", "matrix-from-3-tiles", "matrix-from-40-tiles", "matrix-off"])
@pytest.mark.parametrize("cfg_id,P,order,extra", CASES + [pytest.param(4, 3000, 8, {"n_views": 3}, id="cfg4-3views-order8"),
                                                          pytest.param(3, 4000, 6, {}, id="cfg3-cap-mask-order6")])
def test_tile_lists_bit_exact(cfg_id, P, order, extra, mat_tiles):
    """uts_tile_lists (large discs through the bit matrix, small discs through emit + sort, per-tile merge) against the oracle's
    sorted pairs and ranges, bit for bit; the matrix threshold is moved so that few, most or nearly all discs take the matrix."""
    B, R = _gpu()
    tuning = None if mat_tiles is None else (B.Tuning(matrix_off=1) if mat_tiles == "off" else B.Tuning(matrix_min_tiles=mat_tiles))
    c = Case.get(cfg_id, P, order, extra)
    cfg = _cfg(R, c.scene)
    r = R.Rasterizer(cfg, c.gpu_mask(B), fused_lists=True, pair_capacity=16, tuning=tuning)   # tiny capacity: exercises UTS_ERR_CAPACITY + regrow
    r.proj = c.gpu_proj(B)
    r.depth_order()
    n = r.tile_lists()
    assert n == c.fw["skeys"].shape[0]
    assert np.array_equal(u64(r.keys)[:n], c.fw["skeys"])
    assert np.array_equal(u32(r.vals)[:n], c.fw["svals"])
    assert np.array_equal(u64(r.ranges), c.fw["ranges"])


def test_tile_lists_whole_sphere_discs_and_empty():
    """Whole-sphere discs (reading A24) as matrix rows, with and without a mask; culled Gaussians; P = 0."""
    B, R = _gpu()
    scene = small_scene(3, 600, 6)
    scene["scales"][:40] *= 400.0                                     # r_s = pi
    scene["means"][40:60] *= 1e-3                                     # inside r_near: culled
    oc = ocfg(scene)
    bits, act, slot = oracle_mask(oc, scene)
    fw = orc.forward_chain(oc, scene, slot, act, bits)
    assert (fw["proj"].rs >= 3.14159).sum() >= 15 and (fw["proj"].flags & 1).sum() >= 20
    cfg = _cfg(R, scene)
    mask = B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg, mask, fused_lists=True, tuning=B.Tuning(matrix_min_tiles=8.0))
    r.preprocess(g, views); r.depth_order()
    n = r.tile_lists()
    assert n == fw["skeys"].shape[0] and np.array_equal(u64(r.keys)[:n], fw["skeys"]) and np.array_equal(u32(r.vals)[:n], fw["svals"])
    assert np.array_equal(u64(r.ranges), fw["ranges"])
    cfg0 = B.Config(order=6, n_gauss=0)
    r0 = R.Rasterizer(cfg0, fused_lists=True)
    assert r0.tile_lists() == 0 and int(r0.ranges.abs().sum()) == 0


@pytest.mark.parametrize("cfg_id,P,order", [(1, 3000, 6), (3, 20000, 7), (4, 20000, 7), (5, 8000, 8)])
def test_marked_blend_equals_plain_blend(cfg_id, P, order):
    """uts_render_fwd_marked / uts_render_bwd_marked (the backward visits only the (warp, entry) pairs the forward marked) against
    uts_render_fwd / uts_render_bwd on the same lists: image, alpha, trans, n_last bit-identical; gradients the same sums (the set
    of visited entries per pixel is unchanged, only whole-warp no-ops are skipped), compared at 2e-4 of the largest entry (fp32 atomics:
    two runs of the same kernel differ by a few 1e-5 where large terms cancel)."""
    B, R = _gpu()
    scene = small_scene(cfg_id, P, order)
    cfg = _cfg(R, scene)
    g, views = R.scene_to_device(scene)
    mask = B.uts_build_mask(cfg, scene["mask"]["kind"], scene["mask"]["params"]) if scene["mask"] is not None else B.Mask.full()
    rm = R.Rasterizer(cfg, mask, marks=True); rp = R.Rasterizer(cfg, mask, marks=False)
    rm.marks.fill_(-1)                                   # the forward must write every word the backward reads
    cm, am = rm.forward(g, views); cp, ap = rp.forward(g, views)
    assert rm.n_pairs == rp.n_pairs > 0
    for a, b in ((cm, cp), (am, ap), (rm.trans, rp.trans), (rm.n_last, rp.n_last)):
        assert torch.equal(a, b)
    gen = torch.Generator(device="cuda").manual_seed(3)
    gcol = torch.randn(cm.shape, device="cuda", generator=gen)
    gal = torch.randn(am.shape, device="cuda", generator=gen)
    Gm = rm.backward(g, views, gcol, gal); Gp = rp.backward(g, views, gcol, gal)
    for k in Gm:
        a, b = Gm[k], Gp[k]
        assert float((a - b).abs().max()) <= 2e-4 * float(b.abs().max()) + 1e-12, k


def test_depth_prefix_lists_give_the_full_result_when_every_pixel_saturates():
    """Occlusion-bounded lists (include/uts.h, uts_depth_prefix_flags / uts_count_unsaturated): lists built from the nearest `keep`
    Gaussians only.  n_open counts the visible pixels that did not saturate; with keep = P it is the full forward's own count; and as
    soon as a prefix leaves no pixel open, image, alpha, T and n_last are bit-identical to the full lists' and the gradients are the
    same sums — with far fewer pairs."""
    B, R = _gpu()
    scene = small_scene(4, 400000, 6)                      # dense: the large near Gaussians saturate every pixel
    cfg = _cfg(R, scene)
    g, views = R.scene_to_device(scene)
    full = R.Rasterizer(cfg)
    cf, af = full.forward(g, views)
    P = cfg.n_gauss
    scratch = torch.zeros(1, dtype=torch.int64, device="cuda")
    open_full = B.uts_count_unsaturated(cfg, full.mask, full.trans, scratch)
    assert open_full == int((full.trans >= cfg.t_eps).sum())
    pre = R.Rasterizer(cfg)
    _, _, n_open = pre.forward_depth_prefix(g, views, P)
    assert n_open == open_full and pre.n_pairs == full.n_pairs
    assert open_full == 0, "pick a denser scene: the test needs every pixel to saturate"
    _, _, n_small = pre.forward_depth_prefix(g, views, 8)
    assert n_small > 0                                    # eight Gaussians cannot saturate the sphere: reported, not hidden
    keep = P // 512
    while True:
        cp, ap, n_open = pre.forward_depth_prefix(g, views, keep)
        if n_open == 0 or keep >= P:
            break
        keep *= 2
    assert n_open == 0 and keep <= P // 4 and pre.n_pairs < full.n_pairs // 2
    for a, b in ((cp, cf), (ap, af), (pre.trans, full.trans), (pre.n_last, full.n_last)):
        assert torch.equal(a, b)
    gen = torch.Generator(device="cuda").manual_seed(5)
    gcol = torch.randn(cf.shape, device="cuda", generator=gen)
    Gp = pre.backward(g, views, gcol); Gf = full.backward(g, views, gcol)
    for k in Gf:
        assert float((Gp[k] - Gf[k]).abs().max()) <= 2e-4 * float(Gf[k].abs().max()) + 1e-12, k


def test_forward_auto_is_always_the_full_result():
    """Rasterizer.forward_auto: depth prefix when every pixel saturates inside it, full lists otherwise — the image is the full
    lists' image either way, bit for bit."""
    B, R = _gpu()
    # (a) a scene that saturates everywhere: the second call at the latest goes through the prefix
    scene = small_scene(4, 400000, 6)
    cfg = _cfg(R, scene)
    g, views = R.scene_to_device(scene)
    full = R.Rasterizer(cfg); cf, _ = full.forward(g, views)
    auto = R.Rasterizer(cfg)
    for _ in range(3):
        ca, _ = auto.forward_auto(g, views)
        assert torch.equal(ca, cf) and torch.equal(auto.n_last, full.n_last)
    assert auto._auto["used_prefix"] and auto.n_pairs < full.n_pairs
    # (b) a scene that does not: the attempts stop, every call returns the full result
    scene = small_scene(1, 3000, 6)
    cfg = _cfg(R, scene)
    g, views = R.scene_to_device(scene)
    full = R.Rasterizer(cfg); cf, _ = full.forward(g, views)
    auto = R.Rasterizer(cfg)
    for _ in range(6):
        ca, _ = auto.forward_auto(g, views)
        assert torch.equal(ca, cf) and auto.n_pairs == full.n_pairs
    assert auto._auto["off"] and not auto._auto["used_prefix"]


def test_concurrent_calls_from_two_threads_on_two_streams():
    """include/uts.h "Library state": the per-device context (auxiliary streams, fork / join events) is guarded by a mutex, so two
    threads may drive the path at the same time on their own streams.  Each thread runs the whole forward + backward 15 times on its
    own scene and stream (ctypes releases the GIL during the calls); every result must equal the one computed alone."""
    import threading
    B, R = _gpu()
    from paper_2606_29794_b200 import scenes
    jobs = []
    for seed, cfg_id in ((0, 2), (1, 4)):
        scene = small_scene(cfg_id, 12000, 7, seed=seed)
        cfg = _cfg(R, scene)
        g, views = R.scene_to_device(scene)
        r = R.Rasterizer(cfg)
        r.forward(g, views)
        gcol = torch.from_numpy(scenes.upstream_grad(1, r.color.shape[1], seed=seed)).cuda()
        r.backward(g, views, gcol)
        torch.cuda.synchronize()
        ref = dict(n=r.n_pairs, keys=r.keys[: r.n_pairs].clone(), vals=r.vals[: r.n_pairs].clone(), ranges=r.ranges.clone(), color=r.color.clone(),
                   n_last=r.n_last.clone(), means=r.grads["means"].clone())
        jobs.append((cfg, g, views, gcol, ref))
    errors = []

    def work(job):
        try:
            cfg, g, views, gcol, ref = job
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                r = R.Rasterizer(cfg)
                for _ in range(15):
                    r.forward(g, views)
                    G = r.backward(g, views, gcol)
                    stream.synchronize()
                    n = r.n_pairs
                    assert n == ref["n"]
                    assert torch.equal(r.keys[:n], ref["keys"]) and torch.equal(r.vals[:n], ref["vals"]) and torch.equal(r.ranges, ref["ranges"])
                    assert torch.equal(r.color, ref["color"]) and torch.equal(r.n_last, ref["n_last"])
                    assert float((G["means"] - ref["means"]).abs().max()) <= 2e-4 * float(ref["means"].abs().max())
        except BaseException as e:      # noqa: BLE001 - reported by the main thread
            errors.append(repr(e))

    threads = [threading.Thread(target=work, args=(j,)) for j in jobs]
    for t in threads: t.start()
    for t in threads: t.join()
    assert not errors, errors
