"""GPU parity of the image-synthesis step (include/uts.h uts_resample_fwd / uts_resample_bwd /
uts_build_camera_mask) against the oracle (oracle/orc_resample.cpp), through the C ABI.

Tolerances: the visibility mask is integer work -> bit-exact (cameras whose domain boundary does not pass exactly through pixel
centres); interpolated values 1e-5 absolute on N(0,1) images (fp32 weights and accumulation, geometry in double on both sides);
the adjoint 1e-5 of the largest entry (fp32 atomics, summation order not fixed)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle as orc

pytestmark = pytest.mark.gpu


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B
    return B


CAMS = [("pinhole", 160, 120, np.radians(70.0), np.radians(50.0)),
        ("pinhole", 97, 61, np.radians(121.0), np.radians(33.0)),
        ("fisheye", 128, 128, 190.0 / 180.0, 190.0 / 180.0),
        ("fisheye", 150, 90, 200.0 / 180.0, 140.0 / 180.0),
        ("equirect", 256, 128, 0.0, 0.0)]


def both(B, spec):
    return orc.Camera(*spec), B.Camera(*spec)


@pytest.mark.parametrize("spec", CAMS, ids=lambda s: f"{s[0]}-{s[1]}x{s[2]}")
@pytest.mark.parametrize("order", [4, 7])
def test_camera_mask_bit_exact(spec, order):
    B = _gpu()
    ocam, gcam = both(B, spec)
    cfg = B.Config(order=order, n_gauss=1)
    m = B.uts_build_camera_mask(cfg, gcam)
    want = orc.camera_mask_bits(order, ocam)
    got = m.pixel_mask_bits.cpu().numpy().view(np.uint32)
    assert np.array_equal(got, want)
    oc = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    act, slot = orc.mask_tiles(oc, want)
    assert m.n_active == act.shape[0]
    assert np.array_equal(m.active_tiles.cpu().numpy().view(np.uint32), act)
    assert np.array_equal(m.slot_of_tile.cpu().numpy(), slot)


@pytest.mark.parametrize("spec", CAMS, ids=lambda s: f"{s[0]}-{s[1]}x{s[2]}")
@pytest.mark.parametrize("order,masked", [(4, False), (6, True), (8, False)])
def test_resample_fwd_bwd_match_oracle(spec, order, masked):
    B = _gpu()
    ocam, gcam = both(B, spec)
    cfg = B.Config(order=order, n_gauss=1)
    oc = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    rng = np.random.default_rng(order * 7 + len(spec[0]))
    if masked:
        mask = B.uts_build_camera_mask(cfg, gcam)
        bits = orc.camera_mask_bits(order, ocam)
        act, slot = orc.mask_tiles(oc, bits)
        n_slot = act.shape[0]
    else:
        mask, bits, slot, n_slot = B.Mask.full(), None, None, oc.n_tiles
    ch = 3
    img = rng.normal(size=(n_slot * 256, ch)).astype(np.float32)
    want, wvalid = orc.resample_fwd(order, ocam, img, slot, bits)
    out = torch.empty(ocam.height, ocam.width, ch, dtype=torch.float32, device="cuda")
    valid = torch.empty(ocam.height, ocam.width, dtype=torch.uint8, device="cuda")
    B.uts_resample_fwd(cfg, gcam, mask, torch.from_numpy(img).cuda(), out, valid)
    assert np.array_equal(valid.cpu().numpy(), wvalid)
    err = np.abs(out.cpu().numpy() - want).max()
    assert err <= 1e-5, err
    assert wvalid.sum() > 0.3 * wvalid.size
    # adjoint
    g = rng.normal(size=(ocam.height, ocam.width, ch)).astype(np.float32)
    wantb = orc.resample_bwd(order, ocam, g, n_slot, slot, bits)
    gi = torch.full((n_slot * 256, ch), 7.0, dtype=torch.float32, device="cuda")            # the call zeroes it
    B.uts_resample_bwd(cfg, gcam, mask, torch.from_numpy(g).cuda(), gi)
    errb = np.abs(gi.cpu().numpy() - wantb).max() / max(np.abs(wantb).max(), 1e-30)
    assert errb <= 1e-5, errb


def test_resample_single_channel_and_poles():
    """Equirectangular output covers both poles (the 4-pixel pole rule) and the 0 / 2 pi seam; 1 channel (e.g. alpha)."""
    B = _gpu()
    spec = ("equirect", 48, 2048, 0.0, 0.0)                    # tall image: 33 rows lie between each pole and the first ring
    ocam, gcam = both(B, spec)
    order = 4
    cfg = B.Config(order=order, n_gauss=1)
    img = np.random.default_rng(5).normal(size=(12 * 256, 1)).astype(np.float32)
    want, _ = orc.resample_fwd(order, ocam, img)
    out = torch.empty(2048, 48, 1, dtype=torch.float32, device="cuda")
    B.uts_resample_fwd(cfg, gcam, B.Mask.full(), torch.from_numpy(img).cuda(), out, None)
    assert np.abs(out.cpu().numpy() - want).max() <= 1e-5


def test_resample_full_size_sampled():
    """BASELINE.json config 4's grid (Nside 1024) to a 2048 x 1024 equirectangular image: 400 sampled output pixels against the
    oracle's per-pixel pieces (P_C, Interp_H support), and the constant-field property on every pixel."""
    B = _gpu()
    order = 10
    cfg = B.Config(order=order, n_gauss=1)
    npix = 12 << (2 * order)
    gen = torch.Generator(device="cuda"); gen.manual_seed(3)
    img = torch.randn(npix, 3, device="cuda", generator=gen)
    gcam = B.Camera("equirect", 2048, 1024)
    out = torch.empty(1024, 2048, 3, dtype=torch.float32, device="cuda")
    B.uts_resample_fwd(cfg, gcam, B.Mask.full(), img, out, None)
    host = img.cpu().numpy()
    got = out.cpu().numpy()
    ocam = orc.Camera("equirect", 2048, 1024)
    rng = np.random.default_rng(0)
    worst = 0.0
    for _ in range(400):
        i, j = int(rng.integers(0, 2048)), int(rng.integers(0, 1024))
        d, ok = orc.cam_pixel_dir(ocam, i + 0.5, j + 0.5)
        th = np.arctan2(np.hypot(d[0], d[2]), d[1]); lam = np.arctan2(d[0], d[2]) % (2 * np.pi)
        pix, w = orc.interp_weights(order, th, lam)
        worst = max(worst, np.abs((w[:, None] * host[pix]).sum(0) - got[j, i]).max())
    assert worst <= 1e-5, worst
    one = torch.ones(npix, 1, device="cuda")
    o1 = torch.empty(1024, 2048, 1, dtype=torch.float32, device="cuda")
    B.uts_resample_fwd(cfg, gcam, B.Mask.full(), one, o1, None)
    assert float((o1 - 1).abs().max()) <= 1e-6


def test_render_then_resample_chain():
    """Hot path -> image: a shrunk fisheye scene rendered on the camera's own mask (uts_build_camera_mask), resampled to the
    fisheye image; compared with the oracle's chain on the same mask."""
    B = _gpu()
    from paper_2606_29794_b200 import rasterizer as R
    from helpers import ocfg, small_scene
    scene = small_scene(3, 6000, 7)
    spec = ("fisheye", 200, 200, 190.0 / 180.0, 190.0 / 180.0)
    ocam, gcam = both(B, spec)
    oc = ocfg(scene)
    bits = orc.camera_mask_bits(oc.order, ocam)
    act, slot = orc.mask_tiles(oc, bits)
    fw = orc.forward_chain(oc, scene, slot, act, bits)
    want, wvalid = orc.resample_fwd(oc.order, ocam, fw["color"][0].astype(np.float32), slot, bits)
    cfg = R.config_of(scene)
    mask = B.uts_build_camera_mask(cfg, gcam)
    g, views = R.scene_to_device(scene)
    r = R.Rasterizer(cfg, mask=mask)
    r.forward(g, views)
    out = torch.empty(200, 200, 3, dtype=torch.float32, device="cuda")
    B.uts_resample_fwd(cfg, gcam, mask, r.color[0].contiguous(), out, None)
    # the HEALPix image itself agrees to 1e-4 except at pixels within the alpha/T decision margin; interpolation is a convex
    # combination, so the resampled image inherits the bound wherever its four samples are outside the margin zone
    safe_h = fw["margin"][0] > 2e-3
    w_img = np.where(safe_h, 0.0, 1.0).astype(np.float32).reshape(-1, 1)
    touched, _ = orc.resample_fwd(oc.order, ocam, w_img, slot, bits)
    ok = (touched[..., 0] == 0) & (wvalid == 1)
    assert ok.sum() > 0.5 * wvalid.sum()
    err = np.abs(out.cpu().numpy() - want)[ok].max()
    assert err <= 1e-4, err
