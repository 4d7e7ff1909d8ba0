"""Finite-difference pins for the oracle's backward (Eq.3-4): the analytic gradients of the fp64
pipeline preprocess -> blend (lists held fixed) must equal central differences of the oracle's own fp64 forward,
for every parameter group.  Also pins the literal Eq.3 term against the definition Eq.2."""
import math

import numpy as np
import pytest

import oracle as orc
from helpers import ocfg, small_scene


def _setup(cfg_id, P, order, sh_degree, rules, seed=0, n_views=1, scale_boost=1.0):
    sc = small_scene(cfg_id, P, order, seed=seed, sh_degree=sh_degree, n_views=n_views)
    sc["scales"] = sc["scales"] * np.float32(scale_boost)
    kw = {} if rules else dict(alpha_min=0.0, alpha_max=1.0, t_eps=0.0)
    cfg = ocfg(sc, **kw)
    if n_views > 1:
        th = 0.4
        sc["W"][1] = np.float32([math.cos(th), 0, math.sin(th), 0, 1, 0, -math.sin(th), 0, math.cos(th)])
        sc["b"][1] = np.float32([0.05, -0.1, 0.2])
    fw = orc.forward_chain(cfg, sc)
    S = cfg.n_tiles * cfg.ppt
    rng = np.random.default_rng(5)
    G = rng.standard_normal((cfg.n_views, S, 3)); Ga = rng.standard_normal((cfg.n_views, S))
    params = {k: sc[k].astype(np.float64) for k in ("means", "scales", "quats", "opac", "sh", "W", "b")}
    return cfg, sc, fw, params, G, Ga


def _loss(cfg, p, fw, G, Ga, **kw):
    return orc.e2e_f64(cfg, p["means"], p["scales"], p["quats"], p["opac"], p["sh"], p["W"], p["b"], fw["ranges"], fw["svals"], G, Ga, **kw)


@pytest.mark.parametrize("cfg_id,P,order,D,rules,V", [(1, 40, 4, 0, False, 1), (1, 40, 4, 3, True, 1), (2, 60, 5, 3, False, 2), (4, 30, 5, 2, True, 1)])
def test_gradients_match_central_differences(cfg_id, P, order, D, rules, V):
    cfg, sc, fw, p, G, Ga = _setup(cfg_id, P, order, D, rules, n_views=V, scale_boost=3.0)
    loss, g = _loss(cfg, p, fw, G, Ga, want_grad=True)
    assert np.isfinite(loss)
    rng = np.random.default_rng(11)
    worst = 0.0
    for name in ("means", "scales", "quats", "opac", "sh"):
        arr = p[name]; ga = g[name]
        scale = np.abs(ga).max()
        assert scale > 0, name
        flat_idx = rng.choice(arr.size, size=min(arr.size, 25), replace=False)
        for fi in flat_idx:
            idx = np.unravel_index(fi, arr.shape)
            h = 1e-6 * max(1.0, abs(arr[idx])) if name != "scales" else 1e-6 * arr[idx]
            old = arr[idx]
            arr[idx] = old + h; lp = _loss(cfg, p, fw, G, Ga)
            arr[idx] = old - h; lm = _loss(cfg, p, fw, G, Ga)
            arr[idx] = old
            fd = (lp - lm) / (2 * h)
            err = abs(fd - ga[idx]) / max(scale * 1e-3, abs(fd))
            worst = max(worst, err)
            assert err < 2e-5, (name, idx, fd, ga[idx])
    assert worst < 2e-5


def test_directional_derivative_end_to_end():
    # <g, delta> == (L(x+e delta) - L(x-e delta)) / 2e over all parameters at once (config-1 distributions)
    cfg, sc, fw, p, G, Ga = _setup(1, 120, 5, 1, True, seed=3, scale_boost=2.0)
    loss, g = _loss(cfg, p, fw, G, Ga, want_grad=True)
    rng = np.random.default_rng(2)
    for _ in range(3):
        delta = {k: rng.standard_normal(p[k].shape) * (0.01 if k != "scales" else 0.01 * p[k]) for k in ("means", "scales", "quats", "opac", "sh")}
        e = 1e-5
        pp = {k: (p[k] + e * delta[k] if k in delta else p[k]) for k in p}
        pm = {k: (p[k] - e * delta[k] if k in delta else p[k]) for k in p}
        fd = (_loss(cfg, pp, fw, G, Ga) - _loss(cfg, pm, fw, G, Ga)) / (2 * e)
        an = sum(float((g[k] * delta[k]).sum()) for k in delta)
        assert fd == pytest.approx(an, rel=2e-5, abs=1e-9)


def test_eq3_literal_term_is_the_phi_derivative_of_eq2():
    # Eq.3: L_phi|S_phi = -sin(phi) (2 cos(phi) s_ww L_a + s_wp L_b) must be d/dphi of
    # <L_arc, S_phi Sigma_rad S_phi^T> at fixed Sigma_rad (Eq.2) with the off-diagonal stored once (A15).
    cfg, sc, fw, p, G, Ga = _setup(1, 10, 4, 0, False, scale_boost=4.0)
    loss, g, dbg = _loss(cfg, p, fw, G, Ga, want_grad=True, want_dbg=True)
    eq3, La, Lb, Lc, sww, swp, spp, phi = dbg
    assert abs(eq3) > 0
    def L(ph):
        S = np.diag([math.cos(ph), 1.0]); Sr = np.array([[sww, swp], [swp, spp]])
        A = S @ Sr @ S.T
        return La * A[0, 0] + Lb * A[0, 1] + Lc * A[1, 1]
    fd = (L(phi + 1e-6) - L(phi - 1e-6)) / 2e-6
    assert eq3 == pytest.approx(fd, rel=1e-7)


def test_stagewise_fp32_backward_consistent_with_fp64_chain():
    # the fp32-ABI stage functions (render_bwd -> preprocess_bwd) reproduce the fp64 chain up to fp32 rounding of the records
    cfg, sc, fw, p, G, Ga = _setup(2, 80, 5, 3, True, scale_boost=2.0)
    loss, g = _loss(cfg, p, fw, G, Ga, want_grad=True)
    d_rgb, d_conic, d_mu2, d_opac = orc.render_bwd(cfg, fw["proj"], fw["ranges"], fw["svals"], fw["n_last"], G.astype(np.float32), Ga.astype(np.float32))
    dm, ds, dq, dsh = orc.preprocess_bwd(cfg, sc["means"], sc["scales"], sc["quats"], sc["sh"], sc["W"], sc["b"], d_rgb, d_conic, d_mu2)
    for a, b in ((dm, g["means"]), (ds, g["scales"]), (dq, g["quats"]), (dsh, g["sh"]), (d_opac, g["opac"])):
        assert np.abs(a - b).max() <= 2e-4 * np.abs(b).max()
