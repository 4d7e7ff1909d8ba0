"""Pins of the oracle's inverse-radial-depth channel and r_s,max buffer (oracle/orc_depth.cpp; SURVEY §8f NEXT-4;
PAPER.md:96, 147; reading A29)."""
import dataclasses

import numpy as np

import oracle as orc
from helpers import ocfg, small_scene


def test_equal_radius_scene_depth_is_alpha_over_r():
    """All Gaussians at the same radius r0: D(p) = r0^-1 sum_i alpha_i T_i = (1 - T_final) / r0 = alpha(p) / r0 for every pixel."""
    sc = small_scene(1, 400, 5)
    r0 = 3.0
    m = sc["means"].astype(np.float64)
    sc["means"] = (m / np.linalg.norm(m, axis=1, keepdims=True) * r0).astype(np.float32)
    cfg = ocfg(sc)
    fw = orc.forward_chain(cfg, sc)
    pr = fw["proj"]
    chan = orc.inv_depth_channel(pr.rho, pr.flags)
    assert np.array_equal(chan[..., 1:], np.zeros_like(chan[..., 1:]))
    pd = dataclasses.replace(pr, rgb=chan)
    D, alpha, n_last, _, _ = orc.render_fwd(cfg, pd, fw["ranges"], fw["svals"])
    assert np.array_equal(n_last, fw["n_last"])                        # same lists, same decisions: the channel does not touch alpha
    inv = 1.0 / pr.rho.astype(np.float64)                                 # the records' own fp32 radii (all within 1 ulp of r0)
    assert np.abs(inv - 1 / r0).max() < 1e-6
    assert (alpha > 0.05).sum() > 100
    assert np.abs(D[..., 0] - alpha / r0).max() < 2e-6
    assert np.all(D[..., 1:] == 0)


def test_inv_depth_gradient_matches_finite_differences():
    """d/dmu of sum_{v,i} g[v,i] / ||W_v mu_i + b_v|| against central differences (independent of the -t/r^3 formula)."""
    rng = np.random.default_rng(2)
    P, V = 7, 3
    means = rng.normal(size=(P, 3)).astype(np.float32) * 2
    W = np.stack([np.linalg.qr(rng.normal(size=(3, 3)))[0] for _ in range(V)]).astype(np.float32).reshape(V, 9)
    b = rng.normal(size=(V, 3)).astype(np.float32)
    g = rng.normal(size=(V, P))

    def loss(mu):
        t = np.einsum("vrc,pc->vpr", W.reshape(V, 3, 3).astype(np.float64), mu) + b.astype(np.float64)[:, None, :]
        return float((g / np.linalg.norm(t, axis=-1)).sum())

    got = orc.inv_depth_bwd(means, W, b, g)
    mu0 = means.astype(np.float64)
    for i in range(P):
        for c in range(3):
            e = np.zeros_like(mu0); e[i, c] = 1e-6
            fd = (loss(mu0 + e) - loss(mu0 - e)) / 2e-6
            assert abs(fd - got[i, c]) < 1e-7 * max(1.0, abs(fd)), (i, c, fd, got[i, c])
    # culled Gaussians take no gradient
    flags = np.zeros((V, P), np.uint8); flags[:, 2] = 1
    got2 = orc.inv_depth_bwd(means, W, b, g, flags)
    assert np.all(got2[2] == 0) and np.allclose(np.delete(got2, 2, 0), np.delete(got, 2, 0))


def test_rs_max_buffer():
    rs = np.float32([[0.1, 0.5, 0.3, 0.9], [0.2, 0.4, 0.8, 0.05]])
    flags = np.uint8([[0, 0, 1, 0], [0, 1, 0, 0]])
    buf = np.float32([0.15, 0.0, 0.0, 1.0])
    out = orc.rs_max_update(rs, flags, buf)
    assert np.array_equal(out, np.float32([0.2, 0.5, 0.8, 1.0]))          # culled entries (0.3 in view 0, 0.4 in view 1) are ignored
    assert np.array_equal(orc.rs_max_update(rs, flags, out), out)         # idempotent
    assert np.all(out >= buf)                                             # monotone
