"""Pins for the oracle's rasteriser stages (Alg.1, Eq.1-6) against closed forms, brute force and
invariants.  The paper prints no worked numeric example, so image-level parity with the authors' code is unpinned;
every stage below is pinned by something other than itself."""
import math

import numpy as np
import pytest

import oracle as orc
from helpers import ocfg, small_scene

I3 = np.eye(3).reshape(1, 9)
Z3 = np.zeros((1, 3))


def _rot_y(th):
    c, s = math.cos(th), math.sin(th)
    return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]])


def _rand_rot(rng):
    q = rng.standard_normal(4); q /= np.linalg.norm(q)
    return q


# ------------------------------------------------------------------ O1 preprocess
def test_projection_eq1_and_jacobian_fd():
    # Eq.1 retyped in numpy; J compared with central differences of Eq.1
    rng = np.random.default_rng(0)
    cfg = orc.Config(order=6, n_gauss=1, cov_dilation_px2=0.0)
    pi_ = lambda t: np.array([math.atan2(t[0], t[2]), math.atan2(t[1], math.hypot(t[0], t[2]))])
    for _ in range(20):
        mu = rng.standard_normal(3) * 3
        W = _rot_y(rng.uniform(0, 6)) @ np.array([[1, 0, 0], [0, 0, -1], [0, 1, 0]])
        b = rng.standard_normal(3)
        _, _, J, t = orc.sigma_arc_both(cfg, mu, [0.1, 0.2, 0.3], _rand_rot(rng), W.reshape(-1), b)
        assert np.allclose(t, W @ mu + b, atol=1e-14)
        Jfd = np.zeros((2, 3))
        for k in range(3):
            e = np.zeros(3); e[k] = 1e-6
            Jfd[:, k] = (pi_(t + e) - pi_(t - e)) / 2e-6
        assert np.abs(J - Jfd).max() < 1e-8
    # the fp32 stage: lon/lat/rho/dir
    mu = np.array([[1.0, 2.0, 3.0]], np.float32)
    cfg = orc.Config(order=6, n_gauss=1)
    pr = orc.preprocess(cfg, mu, [[.1, .1, .1]], [[1, 0, 0, 0]], [0.5], np.zeros((1, 1, 3)), I3, Z3)
    assert pr.lonlat[0, 0, 0] == pytest.approx(math.atan2(1, 3), rel=1e-6)
    assert pr.lonlat[0, 0, 1] == pytest.approx(math.atan2(2, math.hypot(1, 3)), rel=1e-6)
    assert pr.rho[0, 0] == pytest.approx(math.sqrt(14), rel=1e-6)
    assert np.allclose(pr.dir[0, 0], mu[0] / math.sqrt(14), atol=1e-7)


def test_sigma_arc_literal_eq2_equals_tangent_basis():
    # Alg.1 l.6 literal S_phi J W Sigma W^T J^T S_phi^T  ==  [e;n] M [e;n]^T / rho^2  (S_phi J = [e;n]/rho)
    rng = np.random.default_rng(1)
    cfg = orc.Config(order=6, n_gauss=1, cov_dilation_px2=0.0)
    for _ in range(50):
        mu = rng.standard_normal(3) * 2
        if rng.uniform() < 0.3:
            mu[[0, 2]] *= 1e-3          # near a pole
        lit, tan, _, _ = orc.sigma_arc_both(cfg, mu, np.exp(rng.normal(-2, 1, 3)), _rand_rot(rng), _rot_y(rng.uniform(0, 6)).reshape(-1), rng.standard_normal(3) * 0.1)
        assert np.allclose(lit, tan, rtol=1e-9, atol=1e-18)


def test_isotropic_gaussian_closed_form():
    # s=(sig,sig,sig) => Sigma_arc = (sig/rho)^2 I + h I for any rotation and direction; r_s = 3 sqrt((sig/rho)^2+h)
    rng = np.random.default_rng(2)
    for k, dil in ((6, 0.3), (8, 0.0)):
        cfg = orc.Config(order=k, n_gauss=1, cov_dilation_px2=dil)
        h = float(np.float32(dil)) * 4 * math.pi / cfg.n_pix      # the config field is fp32
        for _ in range(20):
            mu = rng.standard_normal(3) * 4; sig = math.exp(rng.normal(-3, 1))
            lit, _, _, t = orc.sigma_arc_both(cfg, mu, [sig] * 3, _rand_rot(rng), _rot_y(rng.uniform(0, 6)).reshape(-1), [0, 0, 0])
            rho = np.linalg.norm(t)
            assert lit[0] == pytest.approx((sig / rho) ** 2 + h, rel=1e-10)
            assert lit[2] == pytest.approx((sig / rho) ** 2 + h, rel=1e-10)
            assert abs(lit[1]) < 1e-12 * lit[0]
            pr = orc.preprocess(cfg, [mu], [[sig] * 3], [_rand_rot(rng)], [0.7], np.zeros((1, 1, 3)), I3, Z3)
            rho = np.linalg.norm(np.float32(mu).astype(np.float64))
            sig32 = float(np.float32(sig))
            var = (sig32 / rho) ** 2 + h
            assert pr.rs[0, 0] == pytest.approx(min(math.pi, 3 * math.sqrt(var)), rel=1e-6)
            assert pr.conic_opac[0, 0, 0] == pytest.approx(1 / var, rel=1e-5)
            assert pr.conic_opac[0, 0, 2] == pytest.approx(1 / var, rel=1e-5)
            assert abs(pr.conic_opac[0, 0, 1]) < 1e-6 / var
            assert pr.conic_opac[0, 0, 3] == pytest.approx(0.7, rel=1e-6)


def test_sigma_arc_invariant_under_rotation_about_polar_axis():
    rng = np.random.default_rng(3)
    cfg = orc.Config(order=6, n_gauss=1)
    mu = rng.standard_normal(3); s = np.exp(rng.normal(-2, 0.5, 3)); q = _rand_rot(rng)
    a, _, _, _ = orc.sigma_arc_both(cfg, mu, s, q, np.eye(3).reshape(-1), [0, 0, 0])
    b, _, _, _ = orc.sigma_arc_both(cfg, mu, s, q, _rot_y(1.234).reshape(-1), [0, 0, 0])
    assert np.allclose(a, b, rtol=1e-12)


def test_cull_rules():
    cfg = orc.Config(order=6, n_gauss=3)
    means = np.array([[0, 0, 0.1], [0, 0, 1.0], [np.nan, 0, 1]], np.float32)      # rho <= r_near ; ok ; non-finite
    pr = orc.preprocess(cfg, means, np.full((3, 3), .1), np.tile([1, 0, 0, 0], (3, 1)), [.5] * 3, np.zeros((3, 1, 3)), I3, Z3)
    assert list(pr.flags[0] & 1) == [1, 0, 1]
    assert pr.rs[0, 0] == 0 and pr.rs[0, 2] == 0


def test_sh_degree0_colour_and_clamp_flag():
    cfg = orc.Config(order=6, n_gauss=2, sh_degree=0)
    sh = np.array([[[1.0, -3.0, 0.0]], [[0.5, 0.5, 0.5]]], np.float32)
    pr = orc.preprocess(cfg, [[0, 0, 2], [0, 1, 2]], np.full((2, 3), .1), np.tile([1, 0, 0, 0], (2, 1)), [.5, .5], sh, I3, Z3)
    assert pr.rgb[0, 0, 0] == pytest.approx(0.5 + 0.28209479177387814, rel=1e-6)
    assert pr.rgb[0, 0, 1] == 0.0 and pr.flags[0, 0] == 0b0100          # G channel clamped -> bit 2
    assert pr.rgb[0, 0, 2] == pytest.approx(0.5)
    assert pr.flags[0, 1] == 0


def test_sh_basis_orthonormal_by_healpix_quadrature():
    # sum_p Y_a Y_b Omega_pix = delta_ab: pins every constant and sign pattern of the 16 basis functions up to an overall
    # sign per function, and is an end-to-end use of the equal-area grid.  Signs: degree-1 convention (-y, z, -x) below.
    k = 6
    _, _, v = orc.centers(k, 2)
    Y = np.stack([orc.sh_basis(3, d) for d in v])
    G = Y.T @ Y * (4 * math.pi / v.shape[0])
    assert np.abs(G - np.eye(16)).max() < 2e-4
    d = np.array([0.3, -0.5, 0.8]); d /= np.linalg.norm(d)
    Y = orc.sh_basis(3, d)
    c1 = math.sqrt(3 / (4 * math.pi))
    assert np.allclose(Y[1:4], [-c1 * d[1], c1 * d[2], -c1 * d[0]])
    # gradient of the basis polynomials vs central differences
    dY = orc.sh_basis_grad(3, d)
    for kk in range(3):
        e = np.zeros(3); e[kk] = 1e-6
        assert np.allclose(dY[:, kk], (orc.sh_basis(3, d + e) - orc.sh_basis(3, d - e)) / 2e-6, atol=1e-8)


# ------------------------------------------------------------------ O2 tile query
@pytest.mark.parametrize("cfg_id,P,order,refine", [(1, 1000, 6, 2), (2, 400, 8, 2), (4, 300, 7, 2), (4, 200, 6, 1), (1, 200, 5, 0)])
def test_tile_query_descent_equals_bruteforce(cfg_id, P, order, refine):
    sc = small_scene(cfg_id, P, order)
    cfg = ocfg(sc, query_refine_log2=refine)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    o1, k1, v1, i1 = orc.tile_query(cfg, pr, brute=True)
    o2, k2, v2, i2 = orc.tile_query(cfg, pr, brute=False)
    assert i1["min_margin"] > 1e-12          # margin certificate: no decision is borderline
    assert np.array_equal(o1, o2) and np.array_equal(k1, k2) and np.array_equal(v1, v2)
    assert i2["node_tests"] < i1["node_tests"]
    # order (Gaussian id, tile) ascending, each tile once per Gaussian; key layout (tile<<32)|bits(rho32)
    tiles = (k1 >> np.uint64(32)).astype(np.int64)
    for i in range(cfg.n_gauss):
        seg = tiles[int(o1[i]):int(o1[i + 1])]
        assert np.all(np.diff(seg) > 0)
        assert np.all(v1[int(o1[i]):int(o1[i + 1])] == i)
    assert np.array_equal((k1 & np.uint64(0xFFFFFFFF)).astype(np.uint32), pr.rho[0].view(np.uint32)[v1])


def test_tile_query_is_superset_of_fine_centres_within_rs_and_handles_huge():
    # conservative: every tile owning an order-k pixel centre within r_s is in the set (no contribution within 3 sigma is lost)
    sc = small_scene(4, 150, 6)
    cfg = ocfg(sc)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    pr.rs[0, :3] = np.float32(math.pi)                # r_s >= pi => all tiles (A24)
    off, keys, vals, _ = orc.tile_query(cfg, pr)
    _, _, vpix = orc.centers(cfg.order, 2)
    tiles = (keys >> np.uint64(32)).astype(np.int64)
    for i in range(cfg.n_gauss):
        mine = set(tiles[int(off[i]):int(off[i + 1])].tolist())
        u = pr.dir[0, i].astype(np.float64); u /= np.linalg.norm(u)
        inside = np.flatnonzero(vpix @ u >= math.cos(min(math.pi, float(pr.rs[0, i]))))
        assert set((inside >> (2 * cfg.tile_log2)).tolist()) <= mine
        if i < 3:
            assert len(mine) == cfg.n_tiles


def test_tile_query_respects_mask_and_views():
    sc = small_scene(5, 300, 7, n_views=2)
    cfg = ocfg(sc)
    bits = orc.mask_bits(cfg.order, sc["mask"]["kind"], sc["mask"]["params"])
    act, slot = orc.mask_tiles(cfg, bits)
    assert 0 < act.shape[0] < cfg.n_tiles
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    off, keys, vals, _ = orc.tile_query(cfg, pr, slot_of_tile=slot)
    offf, keysf, valsf, _ = orc.tile_query(cfg, pr)
    tid = (keys >> np.uint64(32)).astype(np.int64)
    assert np.all(slot[tid % cfg.n_tiles] >= 0)
    tf = (keysf >> np.uint64(32)).astype(np.int64)
    keep = slot[tf % cfg.n_tiles] >= 0
    assert np.array_equal(keysf[keep], keys) and np.array_equal(valsf[keep], vals)
    # view index lives in the tile field: second half of the Gaussians x views order belongs to view 1
    assert np.all(tid[int(off[cfg.n_gauss]):] >= cfg.n_tiles) and np.all(tid[:int(off[cfg.n_gauss])] < cfg.n_tiles)


# ------------------------------------------------------------------ O2', RING scan (Alg.3; NEXT-1)
@pytest.mark.parametrize("cfg_id,P,order,refine", [(1, 1000, 6, 2), (2, 400, 8, 2), (4, 300, 7, 2), (4, 200, 6, 1), (1, 200, 5, 0), (4, 150, 6, 3)])
def test_ring_scan_equals_bruteforce_centres_within_rs(cfg_id, P, order, refine):
    """Alg.3 step by step == the plain definition it computes: tiles owning an order-k_q pixel whose CENTRE is within r_s
    (no PixRad margin), by a literal loop over every Gaussian x every order-k_q pixel."""
    sc = small_scene(cfg_id, P, order)
    cfg = ocfg(sc, query_refine_log2=refine, query_mode=1)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    o1, k1, v1, i1 = orc.tile_query(cfg, pr, brute=True)
    o2, k2, v2, i2 = orc.tile_query(cfg, pr, brute=False)
    assert i1["min_margin"] > 1e-12
    assert np.array_equal(o1, o2) and np.array_equal(k1, k2) and np.array_equal(v1, v2)
    # the brute-force set re-derived here in numpy from the oracle's pixel centres (independent of orc.tile_query)
    _, _, vq = orc.centers(cfg.tile_order + refine, 2)
    tiles = (k2 >> np.uint64(32)).astype(np.int64)
    for i in range(0, cfg.n_gauss, 7):
        u = pr.dir[0, i].astype(np.float64); u /= np.linalg.norm(u)
        inside = np.flatnonzero(vq @ u >= math.cos(min(math.pi, float(pr.rs[0, i]))))
        assert sorted(set((inside >> (2 * refine)).tolist())) == tiles[int(o2[i]):int(o2[i + 1])].tolist()
    # non-conservative: a subset of the NESTED set ("at the expense of quality"), strictly smaller on these scenes
    cfgn = ocfg(sc, query_refine_log2=refine)
    on, kn, vn, _ = orc.tile_query(cfgn, pr)
    assert set(zip(k2.tolist(), v2.tolist())) <= set(zip(kn.tolist(), vn.tolist())) and k2.shape[0] < kn.shape[0]


def test_ring_scan_poles_full_rings_and_whole_sphere():
    """Branches of Alg.3: disc over a pole (l.2 clamp, l.16 full rings), centre exactly at a pole (l.9), r_s = pi."""
    sc = small_scene(1, 6, 6)
    cfg = ocfg(sc, query_mode=1)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    d = np.array([[0.02, 1, 0.01], [0.0, 1.0, 0.0], [0.3, -1, 0.2], [0, -1, 0], [1, 0.05, 0], [0.1, 0.2, -1]], np.float64)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    pr.dir[0] = d.astype(np.float32)
    pr.rs[0] = np.array([0.3, 0.21, 0.9, 0.08, math.pi, 2.5], np.float32)
    o1, k1, v1, i1 = orc.tile_query(cfg, pr, brute=True)
    o2, k2, v2, i2 = orc.tile_query(cfg, pr, brute=False)
    assert i1["min_margin"] > 1e-12
    assert np.array_equal(o1, o2) and np.array_equal(k1, k2) and np.array_equal(v1, v2)
    assert int(o2[5] - o2[4]) == cfg.n_tiles                 # r_s = pi: every tile
    assert int(o2[2] - o2[1]) > 0 and int(o2[4] - o2[3]) > 0  # discs centred exactly on the poles are found


def test_ring_scan_respects_mask():
    sc = small_scene(5, 300, 7, n_views=2)
    cfg = ocfg(sc, query_mode=1)
    bits = orc.mask_bits(cfg.order, sc["mask"]["kind"], sc["mask"]["params"])
    act, slot = orc.mask_tiles(cfg, bits)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    off, keys, vals, _ = orc.tile_query(cfg, pr, slot_of_tile=slot)
    offf, keysf, valsf, _ = orc.tile_query(cfg, pr)
    tf = (keysf >> np.uint64(32)).astype(np.int64)
    keep = slot[tf % cfg.n_tiles] >= 0
    assert np.array_equal(keysf[keep], keys) and np.array_equal(valsf[keep], vals)


# ------------------------------------------------------------------ O3 / O4
def test_sort_and_ranges_properties():
    sc = small_scene(2, 3000, 7)
    cfg = ocfg(sc)
    pr = orc.preprocess(cfg, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
    # force depth ties to exercise the id tie-break
    pr.rho[0, ::2] = pr.rho[0, 0]
    _, keys, vals, _ = orc.tile_query(cfg, pr)
    sk, sv = orc.sort_pairs(keys, vals)
    assert np.all(np.diff(sk.astype(np.int64) >> 1) >= 0) and np.all(sk[1:] >= sk[:-1])
    order = np.lexsort((vals, keys))                     # (key, then Gaussian id): the unique total order of A9
    assert np.array_equal(sk, keys[order]) and np.array_equal(sv, vals[order])
    rg = orc.tile_ranges(cfg, sk)
    assert int((rg[:, 1] - rg[:, 0]).sum()) == keys.shape[0]
    tid = (sk >> np.uint64(32)).astype(np.int64)
    for t in np.random.default_rng(0).integers(0, cfg.n_tiles, 50):
        s, e = int(rg[t, 0]), int(rg[t, 1])
        assert np.all(tid[s:e] == t)
        assert (s == e == 0) == (not np.any(tid == t)) or (s < e)


# ------------------------------------------------------------------ O5 blend forward
def _haversine(lon1, lat1, lon2, lat2):
    # textbook haversine [35]
    h = np.sin((lat2 - lat1) / 2) ** 2 + np.cos(lat1) * np.cos(lat2) * np.sin((lon2 - lon1) / 2) ** 2
    return 2 * np.arcsin(np.sqrt(np.clip(h, 0, 1)))


def _pix_lonlat(order):
    z, lam, _ = orc.centers(order, 2)
    return lam, np.arcsin(z)


def _one_scene(means, scales, quats, opac, sh):
    P = len(means)
    return dict(means=np.float32(means), scales=np.float32(scales), quats=np.float32(quats), opac=np.float32(opac),
                sh=np.float32(sh).reshape(P, -1, 3), W=np.float32(I3), b=np.float32(Z3), order=None, n_gauss=P, n_views=1, sh_degree=0)


@pytest.mark.parametrize("mu", [[0.3, 0.2, 2.0], [1.0, -2.5, 0.4], [-0.02, 3.0, 0.01], [-2.0, 0.1, -1.0]])
def test_single_isotropic_gaussian_analytic(mu):
    # alpha(p) = o exp(-d_gc^2 / (2 sigma_ang^2)) with alpha rules disabled; d_gc from an independent haversine
    k = 6; sig = 0.25; o = 0.8
    cfg = orc.Config(order=k, n_gauss=1, alpha_min=0.0, alpha_max=1.0, t_eps=0.0)
    q = np.array([0.9, 0.1, -0.3, 0.2]); q /= np.linalg.norm(q)      # unit quaternion (A14: used as given)
    sc = _one_scene([mu], [[sig] * 3], [q], [o], [[1.0, 0.5, -0.2]])
    out = orc.forward_chain(cfg, sc)
    mu32 = np.float32(mu).astype(np.float64)
    rho = np.linalg.norm(mu32)
    lon_g, lat_g = math.atan2(mu32[0], mu32[2]), math.atan2(mu32[1], math.hypot(mu32[0], mu32[2]))
    lon_p, lat_p = _pix_lonlat(k)
    var = (float(np.float32(sig)) / rho) ** 2 + float(np.float32(0.3)) * 4 * math.pi / cfg.n_pix
    alpha = float(np.float32(o)) * np.exp(-_haversine(lon_g, lat_g, lon_p, lat_p) ** 2 / (2 * var))
    rgb = 0.5 + 0.28209479177387814 * np.float32([1.0, 0.5, -0.2]).astype(np.float64)
    # pixels of the Gaussian's tiles get the analytic value, all other pixels get 0
    tiles = (out["keys"] >> np.uint64(32)).astype(np.int64)
    in_list = np.isin(np.arange(cfg.n_pix) >> 8, tiles)
    assert in_list.any() and (alpha[~in_list].max(initial=0) < math.exp(-4.5) * o)     # nothing within 3 sigma is lost
    want = np.where(in_list[:, None], alpha[:, None] * rgb[None, :], 0.0)
    assert np.abs(out["color"][0] - want).max() < 5e-6
    assert np.abs(out["alpha"][0] - np.where(in_list, alpha, 0)).max() < 5e-6


def test_two_gaussians_closed_form_and_depth_order():
    # Eq.6: c1 a1 + c2 a2 (1 - a1), nearer Gaussian first whatever the input order
    k = 5
    cfg = orc.Config(order=k, n_gauss=2, alpha_min=0.0, alpha_max=1.0, t_eps=0.0, cov_dilation_px2=0.0)
    near = ([0.1, 0.2, 1.5], 0.3, 0.6, [1.0, 0.0, 0.0]); far = ([0.3, 0.1, 4.0], 1.0, 0.9, [0.0, 1.0, 0.5])
    lon_p, lat_p = _pix_lonlat(k)
    res = []
    for order in ((near, far), (far, near)):
        sc = _one_scene([g[0] for g in order], [[g[1]] * 3 for g in order], [[1, 0, 0, 0]] * 2, [g[2] for g in order], [[g[3]] for g in order])
        out = orc.forward_chain(cfg, sc)
        res.append(out["color"][0])
        al = []
        for g in (near, far):
            m = np.float32(g[0]).astype(np.float64); rho = np.linalg.norm(m)
            d = _haversine(math.atan2(m[0], m[2]), math.atan2(m[1], math.hypot(m[0], m[2])), lon_p, lat_p)
            al.append(float(np.float32(g[2])) * np.exp(-d ** 2 / (2 * (float(np.float32(g[1])) / rho) ** 2)))
        c1 = 0.5 + 0.28209479177387814 * np.float64(np.float32(near[3])); c2 = 0.5 + 0.28209479177387814 * np.float64(np.float32(far[3]))
        want = al[0][:, None] * c1 + (al[1] * (1 - al[0]))[:, None] * c2
        tiles = (out["skeys"] >> np.uint64(32)).astype(np.int64)
        both = np.zeros(cfg.n_tiles, int); np.add.at(both, tiles, 1)
        sel = np.repeat(both == 2, 256)
        assert sel.sum() > 0
        assert np.abs(out["color"][0][sel] - want[sel]).max() < 5e-6
        assert np.abs(out["alpha"][0][sel] - (1 - (1 - al[0]) * (1 - al[1]))[sel]).max() < 5e-6
    assert np.array_equal(res[0], res[1])


def test_alpha_rules_and_termination_order():
    # Alg.1 l.23-27 (A7): accumulate, update T, then test T < eps; alpha_max clamp; alpha_min skip; bg; alpha = 1 - T
    k = 4
    cfg = orc.Config(order=k, n_gauss=3, cov_dilation_px2=0.0, bg=(0.25, 0.5, 1.0))
    # three huge co-centred opaque Gaussians: alpha clamps at 0.99 each: T = 1e-2, 1e-4, (1e-6 never reached: 1e-4 < eps? no: T=1e-4 is not < 1e-4)
    sc = _one_scene([[0, 0, 1.0], [0, 0, 2.0], [0, 0, 3.0]], [[50.0] * 3] * 3, [[1, 0, 0, 0]] * 3, [0.999] * 3, [[[1.0, 1.0, 1.0]]] * 3)
    out = orc.forward_chain(cfg, sc)
    c = 0.5 + 0.28209479177387814
    # fp64 arithmetic: T after two = 0.01*0.01 (float32 alpha_max 0.99 -> 0.9900000095): T2 slightly < 1e-4 -> break after 2
    amax = float(np.float32(0.99)); T1 = 1 - amax; T2 = T1 * (1 - amax)
    n_expected = 2 if T2 < float(np.float32(1e-4)) else 3
    assert np.all(out["n_last"][0] == n_expected)
    T = T2 if n_expected == 2 else T2 * (1 - amax)
    want = c * (1 - T) + T * np.array([0.25, 0.5, 1.0])
    assert np.abs(out["color"][0] - want).max() < 1e-6
    assert np.abs(out["alpha"][0] - (1 - T)).max() < 1e-6
    # alpha_min: a faint Gaussian contributes nothing and leaves n_last = 0
    sc = _one_scene([[0, 0, 1.0]], [[50.0] * 3], [[1, 0, 0, 0]], [0.003], [[[1.0, 1.0, 1.0]]])
    cfg1 = orc.Config(order=k, n_gauss=1, cov_dilation_px2=0.0)
    out = orc.forward_chain(cfg1, sc)
    assert np.all(out["n_last"] == 0) and np.all(out["color"] == 0) and np.all(out["alpha"] == 0)
    assert out["counters"]["evaluated"] == cfg1.n_pix and out["counters"]["contributing"] == 0


def test_permutation_invariance_and_fourfold_symmetry():
    sc = small_scene(1, 300, 5)
    cfg = ocfg(sc)
    base = orc.forward_chain(cfg, sc)
    perm = np.random.default_rng(0).permutation(sc["n_gauss"])
    sp = dict(sc); 
    for key in ("means", "scales", "quats", "opac", "sh"):
        sp[key] = sc[key][perm]
    out = orc.forward_chain(cfg, sp)
    assert np.abs(out["color"] - base["color"]).max() < 1e-6 and np.array_equal(out["n_last"], base["n_last"])
    # rotating the scene about the polar (camera y) axis by pi/2 shifts faces by one column (HEALPix 4-fold symmetry)
    sr = dict(sc); sr["W"] = np.float32(_rot_y(math.pi / 2).reshape(1, 9))
    out = orc.forward_chain(cfg, sr)
    nf = cfg.n_pix // 12
    img = base["color"][0].reshape(12, nf, 3); rot = out["color"][0].reshape(12, nf, 3)
    for f in range(12):
        r, c = divmod(f, 4)
        assert np.abs(rot[4 * r + (c + 1) % 4] - img[f]).max() < 2e-5


def test_mask_semantics():
    # A19: inactive tiles get no pairs; inactive pixels of active tiles output 0 / n_last 0; active pixels equal the unmasked render
    sc = small_scene(3, 400, 6)
    cfg = ocfg(sc)
    bits = orc.mask_bits(cfg.order, sc["mask"]["kind"], sc["mask"]["params"])
    act, slot = orc.mask_tiles(cfg, bits)
    full = orc.forward_chain(cfg, sc)
    msk = orc.forward_chain(cfg, sc, slot_of_tile=slot, active_tiles=act, pixel_mask_bits=bits)
    on = np.unpackbits(bits.view(np.uint8), bitorder="little").astype(bool)
    pix = (act.astype(np.int64)[:, None] * 256 + np.arange(256)[None, :]).reshape(-1)
    assert msk["color"].shape[1] == act.shape[0] * 256
    sel = on[pix]
    assert np.array_equal(msk["color"][0][sel], full["color"][0][pix][sel])
    assert np.all(msk["color"][0][~sel] == 0) and np.all(msk["n_last"][0][~sel] == 0) and np.all(msk["alpha"][0][~sel] == 0)


# ------------------------------------------------------------------ rotation / anisotropy / SH sign pins
def _rodrigues(axis, th):
    """Rotation by angle th about `axis` (right-handed, active): R = I + sin(th) K + (1 - cos(th)) K^2 — textbook, built here
    without the oracle's QuatToMat."""
    a = np.asarray(axis, np.float64); a = a / np.linalg.norm(a)
    K = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + math.sin(th) * K + (1 - math.cos(th)) * (K @ K)


@pytest.mark.parametrize("dil", [0.0, 0.3])
def test_single_anisotropic_rotated_gaussian_from_first_principles(dil):
    """Pins QuatToMat (R, not R^T; Alg.1 l.4 PAPER.md:537), the (east,north) orientation of SphericalOffset and the sign of
    the conic's off-diagonal (Eq.2) — none of which an isotropic Gaussian can see.  ONE strongly anisotropic
    Gaussian (scales 0.02 / 0.1 / 0.3) with a non-trivial rotation, a tilted view W and b != 0, alpha rules disabled.
    Expected value, numpy only: Sigma3D = R diag(s^2) R^T with R from Rodrigues' formula on the axis-angle the quaternion
    encodes; Sigma2 = E (W Sigma3D W^T) E^T / rho^2 (+ h I) in an ARBITRARY orthonormal tangent basis E at the Gaussian's
    direction (not the oracle's east/north: the quadratic form does not depend on the basis); delta = the pixel direction's
    log-map offset in that basis; alpha = o exp(-delta^T Sigma2^-1 delta / 2).  (1) log-map offset: equality to rounding;
    (2) gnomonic (pinhole-on-the-tangent-plane) offset, the flat-space limit of EWA splatting: agreement to O((sigma/rho)^2)."""
    k = 9
    cfg = orc.Config(order=k, n_gauss=1, alpha_min=0.0, alpha_max=1.0, t_eps=0.0, cov_dilation_px2=dil)
    axis = np.array([0.3, -0.5, 0.8]); axis /= np.linalg.norm(axis); th = 1.1
    q32 = np.float32(np.concatenate([[math.cos(th / 2)], math.sin(th / 2) * axis]))
    s32 = np.float32([0.02, 0.1, 0.3]); mu32 = np.float32([2.6, 2.1, -4.4]); o32 = np.float32(0.85)
    W32 = np.float32(_rodrigues([1.0, 0.4, -0.2], 0.7)); b32 = np.float32([0.3, -0.2, 0.5])
    sh0 = np.float32([1.0, 0.5, -0.2])
    sc = dict(means=mu32[None], scales=s32[None], quats=q32[None], opac=np.float32([o32]), sh=sh0.reshape(1, 1, 3),
              W=W32.reshape(1, 9), b=b32[None], order=k, n_gauss=1, n_views=1, sh_degree=0)
    out = orc.forward_chain(cfg, sc)

    s, mu, o, W, b = (a.astype(np.float64) for a in (s32, mu32, o32, W32, b32))
    R = _rodrigues(axis, th)
    Sigma = R @ np.diag(s * s) @ R.T
    t = W @ mu + b; rho = np.linalg.norm(t); u = t / rho
    e1 = np.cross(u, [0.2, 0.9, -0.4]); e1 /= np.linalg.norm(e1); e2 = np.cross(u, e1)
    E = np.stack([e1, e2])
    h = float(np.float32(dil)) * 4 * math.pi / cfg.n_pix
    S2 = E @ (W @ Sigma @ W.T) @ E.T / rho ** 2 + h * np.eye(2)
    ev = np.linalg.eigvalsh(S2)
    assert ev[1] / ev[0] > 8 and abs(S2[0, 1]) > 0.1 * ev[1]               # really anisotropic, really oblique in this basis
    Q = np.linalg.inv(S2)
    _, _, w = orc.centers(k, 2)
    c = w @ u; tau = w - c[:, None] * u[None, :]; sn = np.linalg.norm(tau, axis=1)
    g = np.arctan2(sn, c)
    d_log = (tau @ E.T) * (g / np.maximum(sn, 1e-300))[:, None]
    a_log = o * np.exp(-0.5 * np.einsum("pi,ij,pj->p", d_log, Q, d_log))
    rgb = 0.5 + 0.28209479177387814 * sh0.astype(np.float64)
    tiles = (out["keys"] >> np.uint64(32)).astype(np.int64)
    in_list = np.isin(np.arange(cfg.n_pix) >> 8, tiles)
    assert 3 <= np.unique(tiles).shape[0] and a_log[~in_list].max(initial=0) < math.exp(-4.5) * o
    assert (a_log[in_list] > 0.5).sum() > 100                               # the Gaussian is resolved by many pixels
    assert np.abs(out["alpha"][0] - np.where(in_list, a_log, 0)).max() < 5e-6
    assert np.abs(out["color"][0] - np.where(in_list[:, None], a_log[:, None] * rgb[None, :], 0)).max() < 5e-6
    # r_s = 3 sqrt(lambda_max) from the same independent matrix
    assert out["proj"].rs[0, 0] == pytest.approx(3 * math.sqrt(ev[1]), rel=1e-6)
    # (2) flat-space limit: pinhole projection onto the tangent plane at u
    front = c > 0.5
    d_gn = (w @ E.T) / np.where(front, c, 1.0)[:, None]
    a_gn = np.where(front, o * np.exp(-0.5 * np.einsum("pi,ij,pj->p", d_gn, Q, d_gn)), 0.0)
    sig_max = math.sqrt(ev[1])
    err = np.abs(out["alpha"][0] - a_gn)[in_list].max()
    assert err < 2.0 * sig_max ** 2 and sig_max ** 2 < 2e-3, (err, sig_max)
    # what a transposed R (or swapped tangent axes) would give is far outside both tolerances
    S2_T = E @ (W @ (R.T @ np.diag(s * s) @ R) @ W.T) @ E.T / rho ** 2 + h * np.eye(2)
    a_T = o * np.exp(-0.5 * np.einsum("pi,ij,pj->p", d_log, np.linalg.inv(S2_T), d_log))
    assert np.abs(a_T - a_log)[in_list].max() > 0.3


def test_sh_basis_signs_against_scipy_complex_harmonics():
    """Degree 0-3 constants AND signs of the real SH basis (reading A13) against a library routine: the convention is the real
    form of the complex harmonics with the Condon-Shortley phase kept, index l^2 + l + m:
        m > 0: sqrt(2) Re Y_l^m,   m = 0: Y_l^0,   m < 0: sqrt(2) Im Y_l^|m|
    (degree 1 then reads (-y, z, -x) sqrt(3/4pi), the convention stated in SURVEY 8c O1.5).  scipy evaluates Y_l^m through
    Legendre recurrences, not through the polynomial table the oracle restates."""
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(11)
    for _ in range(25):
        d = rng.standard_normal(3); d /= np.linalg.norm(d)
        theta, phi = math.acos(d[2]), math.atan2(d[1], d[0])
        want = []
        for l in range(4):
            for m in range(-l, l + 1):
                y = complex(sph_harm_y(l, abs(m), theta, phi))
                want.append(y.real if m == 0 else math.sqrt(2) * (y.real if m > 0 else y.imag))
        assert np.allclose(orc.sh_basis(3, d), want, rtol=0, atol=1e-12)
