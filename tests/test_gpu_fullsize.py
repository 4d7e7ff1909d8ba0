"""Full-size parity for the BASELINE.json configs (config 2 whole frame; config 3 = cap mask, config 4 = the bench workload and
config 5 = frustum mask + 4 views on sampled tiles), in the launch configuration bench.py times.  The oracle cannot run a whole frame in seconds, so: (1) properties that hold at any size are checked on the
whole output on the device; (2) a random sample of tiles is rendered by the oracle from its OWN complete lists and compared
element by element (list contents bit-exact, colour/alpha 1e-4, n_last); (3) the backward is run with an upstream gradient
that is zero outside the sampled tiles, which the oracle can then reproduce exactly from the sample (1e-3)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle as orc
from helpers import ocfg, oracle_mask, oracle_on_tiles
from paper_2606_29794_b200 import scenes

pytestmark = pytest.mark.gpu
MARGIN = 2e-3


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B, rasterizer as R
    return B, R


def _rel(got, want):
    return np.abs(got.astype(np.float64) - want).max() / max(np.abs(want).max(), 1e-30)


def test_config2_whole_frame_against_the_oracle():
    """BASELINE.json config 2 (Nside 256, 100k Gaussians, SH3) is small enough for the oracle to run WHOLE (about 25 s on one core):
    every pair, every pixel and every gradient entry of the full-size frame is compared."""
    B, R = _gpu()
    scene = scenes.make_scene(2, seed=0)
    cfg = R.config_of(scene)
    oc = ocfg(scene)
    fw = orc.forward_chain(oc, scene)
    assert fw["qinfo"]["min_margin"] > 1e-12
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg)
    r.forward(g, views)
    n = r.n_pairs
    assert n == fw["skeys"].shape[0]
    assert np.array_equal(r.keys[:n].cpu().numpy().view(np.uint64), fw["skeys"])
    assert np.array_equal(r.vals[:n].cpu().numpy().view(np.uint32), fw["svals"])
    assert np.array_equal(r.ranges.cpu().numpy().view(np.uint64), fw["ranges"])
    safe = fw["margin"] > MARGIN
    assert safe.mean() > 0.98
    col, al = r.color.cpu().numpy(), r.alpha.cpu().numpy()
    assert np.abs(col - fw["color"]).max(axis=-1)[safe].max() <= 1e-4 and np.abs(al - fw["alpha"])[safe].max() <= 1e-4
    assert np.array_equal(r.n_last.cpu().numpy().view(np.uint32)[safe], fw["n_last"][safe])
    assert np.abs(col - fw["color"]).max() < 2e-2
    gcol = scenes.upstream_grad(1, col.shape[1], seed=12)
    gcol[~safe] = 0                                                             # decisions within MARGIN of a threshold: excluded on both sides
    G = r.backward(g, views, torch.from_numpy(gcol).cuda())
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(oc, fw["proj"], fw["ranges"], fw["svals"], fw["n_last"], gcol)
    w = orc.preprocess_bwd(oc, scene["means"], scene["scales"], scene["quats"], scene["sh"], scene["W"], scene["b"], w_rgb, w_conic, w_mu2)
    for name, want in zip(("means", "scales", "quats", "sh"), w):
        assert _rel(G[name].cpu().numpy(), want) <= 1e-3, name
    assert _rel(G["opac"].cpu().numpy(), w_opac) <= 1e-3


@pytest.mark.parametrize("cfg_id,n_sample", [(3, 32), (4, 16), (5, 16)], ids=["config3-fisheye-cap", "config4-large-sphere", "config5-frustum-4views"])
def test_full_size_properties_and_sampled_tiles(cfg_id, n_sample):
    B, R = _gpu()
    scene = scenes.make_scene(cfg_id, seed=0)
    cfg = R.config_of(scene)
    oc = ocfg(scene)
    mask = B.Mask.full() if scene["mask"] is None else B.uts_build_mask(cfg, scene["mask"]["kind"], scene["mask"]["params"])
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg, mask)
    r.forward(g, views)
    n = r.n_pairs
    V, NT, ppt = cfg.n_views, cfg.n_tiles, cfg.ppt
    keys, vals = r.keys[:n], r.vals[:n]
    # ---- (1) properties on the whole output
    hi = keys >> 32
    assert bool((keys[1:] >= keys[:-1]).all())                                   # sorted (keys < 2^63: signed compare is fine)
    tie = keys[1:] == keys[:-1]
    assert bool((vals[1:][tie] > vals[:-1][tie]).all())                          # ties broken by Gaussian id
    rg = r.ranges
    lens = rg[:, 1] - rg[:, 0]
    assert int(lens.sum()) == n                                                  # ranges partition the pair array
    nz = lens > 0
    ids = torch.arange(V * NT, device="cuda")[nz]
    assert bool((hi[rg[nz, 0]] == ids).all()) and bool((hi[rg[nz, 1] - 1] == ids).all())
    assert int((hi[1:] != hi[:-1]).sum()) + 1 == int(nz.sum())                   # one run per non-empty tile
    if mask.slot_of_tile is not None:                                            # inactive tiles receive no pairs
        inactive = (mask.slot_of_tile < 0).repeat(V)
        assert int(lens[inactive].sum()) == 0
    assert bool(torch.isfinite(r.color).all()) and float(r.alpha.min()) >= 0.0 and float(r.alpha.max()) <= 1.0 + 1e-6
    # the plain 6/7-pass sort of the (view, Gaussian, tile)-ordered emission gives the same arrays as the depth-presorted path
    r2 = R.Rasterizer(cfg, mask, pair_capacity=n, depth_presort=False)
    r2.preprocess(g, views); r2.tile_query(); r2.sort()
    assert r2.n_pairs == n and torch.equal(r2.keys[:n], keys) and torch.equal(r2.vals[:n], vals)
    del r2
    # ---- (2) sampled tiles against the oracle's own complete lists
    bits, act, slot = oracle_mask(oc, scene)
    if act is not None:
        assert np.array_equal(mask.active_tiles.cpu().numpy().view(np.uint32), act)   # same mask on both sides
    rng = np.random.default_rng(123)
    pool = np.arange(NT) if act is None else act.astype(np.int64)
    pick = np.sort(rng.choice(pool, n_sample, replace=False))
    o = oracle_on_tiles(oc, scene, pick, bits)
    assert o["qinfo"]["min_margin"] > 1e-12
    rg_h = rg.cpu().numpy()
    slot_of = (lambda t: t) if act is None else (lambda t: int(slot[t]))
    safe_all = []
    for v in range(V):
        for si, t in enumerate(pick):
            a, b = (int(x) for x in o["ranges"][v * NT + t])
            ga, gb = (int(x) for x in rg_h[v * NT + t])
            assert gb - ga == b - a
            assert np.array_equal(vals[ga:gb].cpu().numpy().view(np.uint32), o["svals"][a:b])          # list content and order
            assert np.array_equal(keys[ga:gb].cpu().numpy().view(np.uint64), o["skeys"][a:b])
            s0 = slot_of(int(t)) * ppt
            col = r.color[v, s0:s0 + ppt].cpu().numpy(); al = r.alpha[v, s0:s0 + ppt].cpu().numpy()
            nl = r.n_last[v, s0:s0 + ppt].cpu().numpy().view(np.uint32)
            wc, wa, wn = o["color"][v, si * ppt:(si + 1) * ppt], o["alpha"][v, si * ppt:(si + 1) * ppt], o["n_last"][v, si * ppt:(si + 1) * ppt]
            safe = o["margin"][v, si * ppt:(si + 1) * ppt] > MARGIN
            safe_all.append(safe)
            assert np.abs(col - wc).max(axis=-1)[safe].max(initial=0) <= 1e-4
            assert np.abs(al - wa)[safe].max(initial=0) <= 1e-4
            assert np.array_equal(nl[safe], wn[safe])
            assert np.abs(col - wc).max() < 2e-2
    assert np.concatenate(safe_all).mean() > 0.9
    # ---- (3) backward with the upstream gradient confined to the sampled tiles
    S = r.S
    gcol = np.zeros((V, S * ppt, 3), np.float32)
    gs = scenes.upstream_grad(V, n_sample * ppt, seed=9)
    for v in range(V):
        for si, t in enumerate(pick):
            blk = gs[v, si * ppt:(si + 1) * ppt].copy()
            blk[~(o["margin"][v, si * ppt:(si + 1) * ppt] > MARGIN)] = 0          # decisions within MARGIN of a threshold: excluded on both sides
            gs[v, si * ppt:(si + 1) * ppt] = blk
            s0 = slot_of(int(t)) * ppt
            gcol[v, s0:s0 + ppt] = blk
    G = r.backward(g, views, torch.from_numpy(gcol).cuda())
    w_rgb, w_conic, w_mu2, w_opac = orc.render_bwd(oc, o["proj"], o["ranges"], o["svals"], o["n_last"], gs, None, o["sact"], bits)
    w = orc.preprocess_bwd(oc, scene["means"], scene["scales"], scene["quats"], scene["sh"], scene["W"], scene["b"], w_rgb, w_conic, w_mu2)
    for name, want in zip(("means", "scales", "quats", "sh"), w):
        assert _rel(G[name].cpu().numpy(), want) <= 1e-3, name
    assert _rel(G["opac"].cpu().numpy(), w_opac) <= 1e-3
