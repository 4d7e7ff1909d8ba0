"""GPU parity of the inverse radial depth channel and the r_s,max buffer (include/uts.h
uts_inv_depth_channel / uts_inv_depth_bwd / uts_rs_max_update) against the oracle (oracle/orc_depth.cpp), through the C ABI.
The depth image is the ordinary blend (uts_render_fwd / uts_render_bwd) on a record whose rgb is the channel (reading A29).
Tolerances: channel 1 ulp of fp32; depth image 1e-4 absolute x max(1/rho); gradients 1e-3 of each array's largest entry."""
import dataclasses

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle as orc
from helpers import ocfg, small_scene

pytestmark = pytest.mark.gpu
MARGIN = 2e-3


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B, rasterizer as R
    return B, R


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda().contiguous()


@pytest.mark.parametrize("cfg_id,P,order,extra", [(2, 8000, 6, {}), (5, 6000, 8, {"n_views": 2})], ids=["panorama", "frustum-2views"])
def test_depth_image_and_gradients(cfg_id, P, order, extra):
    B, R = _gpu()
    scene = small_scene(cfg_id, P, order, **extra)
    oc = ocfg(scene)
    from helpers import oracle_mask
    bits, act, slot = oracle_mask(oc, scene)
    fw = orc.forward_chain(oc, scene, slot, act, bits)
    pr = fw["proj"]
    V = oc.n_views
    # ---- channel
    cfg = R.config_of(scene)
    chan = torch.empty(V, P, 3, dtype=torch.float32, device="cuda")
    B.uts_inv_depth_channel(cfg, dev(pr.rho), dev(pr.flags), chan)
    want_chan = orc.inv_depth_channel(pr.rho, pr.flags)
    got_chan = chan.cpu().numpy()
    assert np.abs(got_chan - want_chan).max() <= 1.2e-7 * np.abs(want_chan).max()
    # ---- depth image: the blend on the oracle's lists with rgb := channel
    pd = dataclasses.replace(pr, rgb=want_chan)
    D, _, n_last, margin, _ = orc.render_fwd(oc, pd, fw["ranges"], fw["svals"], act, bits)
    mask = B.Mask.full() if bits is None else B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    r = R.Rasterizer(cfg, mask, pair_capacity=int(fw["svals"].shape[0]))
    r.proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(want_chan), dev(pr.flags))
    r.ranges = dev(fw["ranges"].view(np.int64)); r.vals = dev(fw["svals"].view(np.int32))
    r.render_fwd()
    safe = margin > MARGIN
    scale = float(want_chan.max())
    err = np.abs(r.color.cpu().numpy()[..., 0] - D[..., 0])[safe].max()
    assert err <= 1e-4 * max(1.0, scale), err
    assert (D[..., 0] > 0).sum() > 1000
    # ---- backward: dL/dD -> dL/d(1/rho) (+ alpha-path terms) -> means
    rng = np.random.default_rng(cfg_id)
    gD = np.zeros(D.shape, np.float32); gD[..., 0] = rng.normal(size=D.shape[:-1]).astype(np.float32)
    gD[~safe] = 0
    w_chan, w_conic, w_mu2, w_opac = orc.render_bwd(oc, pd, fw["ranges"], fw["svals"], n_last, gD, None, act, bits)
    r.render_bwd(dev(gD), None)
    G = r.grads
    for name, want in (("rgb", w_chan), ("conic", w_conic), ("mu2", w_mu2), ("opac", w_opac)):
        e = np.abs(G[name].cpu().numpy() - want).max() / max(np.abs(want).max(), 1e-30)
        assert e <= 1e-3, (name, e)
    want_means = orc.inv_depth_bwd(scene["means"], scene["W"], scene["b"], w_chan[..., 0], pr.flags)
    g, views = R.scene_to_device(scene)
    base = torch.full((P, 3), 0.5, dtype=torch.float32, device="cuda")
    B.uts_inv_depth_bwd(cfg, g.means, views, dev(pr.flags), dev(w_chan.astype(np.float32)), base, accumulate=True)
    e = np.abs(base.cpu().numpy() - 0.5 - want_means).max() / max(np.abs(want_means).max(), 1e-30)
    assert e <= 1e-3, e
    B.uts_inv_depth_bwd(cfg, g.means, views, dev(pr.flags), dev(w_chan.astype(np.float32)), base, accumulate=False)
    e = np.abs(base.cpu().numpy() - want_means).max() / max(np.abs(want_means).max(), 1e-30)
    assert e <= 1e-3, e


@pytest.mark.parametrize("marks", [True, False], ids=["marked", "plain"])
@pytest.mark.parametrize("cfg_id,P,order,extra", [(2, 8000, 6, {}), (5, 6000, 8, {"n_views": 2, "general_view": True})], ids=["panorama", "frustum-2-general-views"])
def test_depth_as_fourth_blend_channel(cfg_id, P, order, extra, marks):
    """uts_render_fwd_depth / uts_render_bwd_depth: colour and inverse radial depth in ONE blend pass.  The colour outputs
    are bit-identical to uts_render_fwd's; the depth image equals the oracle's blend of the channel 1/rho; the gradients equal the SUM
    of the oracle's colour-loss and depth-loss backward passes, and dL_dinvr feeds uts_inv_depth_bwd (stride 1)."""
    B, R = _gpu()
    scene = small_scene(cfg_id, P, order, **extra)
    oc = ocfg(scene)
    from helpers import oracle_mask
    from paper_2606_29794_b200 import scenes
    bits, act, slot = oracle_mask(oc, scene)
    fw = orc.forward_chain(oc, scene, slot, act, bits)
    pr = fw["proj"]
    V = oc.n_views
    want_chan = orc.inv_depth_channel(pr.rho, pr.flags)
    pd = dataclasses.replace(pr, rgb=want_chan)
    D, _, n_last, margin_d, _ = orc.render_fwd(oc, pd, fw["ranges"], fw["svals"], act, bits)
    cfg = R.config_of(scene)
    mask = B.Mask.full() if bits is None else B.Mask(dev(act.view(np.int32)), int(act.shape[0]), dev(slot), dev(bits.view(np.int32)))
    r = R.Rasterizer(cfg, mask, pair_capacity=int(fw["svals"].shape[0]), marks=marks)
    r.proj = B.Proj(dev(pr.dir), dev(pr.lonlat), dev(pr.rho), dev(pr.conic_opac), dev(pr.rs), dev(pr.rgb), dev(pr.flags))
    r.ranges = dev(fw["ranges"].view(np.int64)); r.vals = dev(fw["svals"].view(np.int32))
    r.render_fwd()
    ref = [t.clone() for t in (r.color, r.alpha, r.trans, r.n_last)]
    for t in (r.color, r.alpha, r.trans, r.n_last):
        t.fill_(7)
    depth = torch.full_like(r.alpha, -1.0)
    B.uts_render_fwd_depth(cfg, r.proj, mask, r.ranges, r.vals, r.capacity, r.color, r.alpha, r.trans, r.n_last, depth, r.marks)
    for a, b in zip(ref, (r.color, r.alpha, r.trans, r.n_last)):
        assert torch.equal(a, b)
    safe = (fw["margin"] > MARGIN) & (margin_d > MARGIN)
    scale = float(want_chan.max())
    assert np.abs(depth.cpu().numpy() - D[..., 0])[safe].max() <= 1e-4 * max(1.0, scale)
    assert float(depth.min()) >= 0.0 and (D[..., 0] > 0).sum() > 1000
    # ---- backward: both losses at once
    npx = r.color.shape[1]
    gcol = scenes.upstream_grad(V, npx, seed=3); gcol[~safe] = 0
    rng = np.random.default_rng(cfg_id + 10)
    gD = np.zeros(D.shape, np.float32); gD[..., 0] = rng.normal(size=D.shape[:-1]).astype(np.float32); gD[~safe] = 0
    w_rgb, c1, m1, o1 = orc.render_bwd(oc, pr, fw["ranges"], fw["svals"], fw["n_last"], gcol, None, act, bits)
    w_chan, c2, m2, o2 = orc.render_bwd(oc, pd, fw["ranges"], fw["svals"], n_last, gD, None, act, bits)
    G = r._alloc_grads()
    invr = torch.full((V, P), 9.0, dtype=torch.float32, device="cuda")
    B.uts_render_bwd_depth(cfg, r.proj, mask, r.ranges, r.vals, r.capacity, r.trans, r.n_last, r.marks, dev(gcol), None, dev(np.ascontiguousarray(gD[..., 0])),
                           G["rgb"], G["conic"], G["mu2"], G["opac"], invr)
    for name, want in (("rgb", w_rgb), ("conic", c1 + c2), ("mu2", m1 + m2), ("opac", o1 + o2)):
        e = np.abs(G[name].cpu().numpy() - want).max() / max(np.abs(want).max(), 1e-30)
        assert e <= 1e-3, (name, e)
    e = np.abs(invr.cpu().numpy() - w_chan[..., 0]).max() / max(np.abs(w_chan[..., 0]).max(), 1e-30)
    assert e <= 1e-3, e
    want_means = orc.inv_depth_bwd(scene["means"], scene["W"], scene["b"], w_chan[..., 0], pr.flags)
    g, views = R.scene_to_device(scene)
    out = torch.zeros(P, 3, dtype=torch.float32, device="cuda")
    B.uts_inv_depth_bwd(cfg, g.means, views, dev(pr.flags), dev(np.ascontiguousarray(w_chan[..., 0].astype(np.float32))), out, accumulate=False)
    e = np.abs(out.cpu().numpy() - want_means).max() / max(np.abs(want_means).max(), 1e-30)
    assert e <= 1e-3, e


def test_rs_max_update_matches_oracle():
    B, R = _gpu()
    rng = np.random.default_rng(0)
    V, P = 3, 5000
    rs = rng.uniform(0, 3.2, size=(V, P)).astype(np.float32)
    flags = (rng.uniform(size=(V, P)) < 0.2).astype(np.uint8) | (rng.integers(0, 8, size=(V, P)).astype(np.uint8) << 1)
    buf = rng.uniform(0, 2.0, size=P).astype(np.float32)
    cfg = B.Config(order=6, n_gauss=P, n_views=V)
    t = dev(buf.copy())
    B.uts_rs_max_update(cfg, dev(rs), dev(flags), t)
    assert np.array_equal(t.cpu().numpy(), orc.rs_max_update(rs, flags, buf))
