"""Pins of the oracle's image-synthesis part (oracle/orc_resample.cpp): camera models P_C / Pi_C^-1
(Eq.11-15), the visibility mask (Eq.9), Interp_H (Eq.7, reading A26) and its adjoint.

None of these tests retypes the oracle's formulas: they use closed-form special cases, round trips, brute force over the
pixel set, exactness on functions the scheme must reproduce, solid-angle counts and the adjoint identity."""
import numpy as np
import pytest

import oracle as orc

CAMS = [orc.Camera("pinhole", 96, 64, np.radians(70.0), np.radians(50.0)),
        orc.Camera("fisheye", 96, 64, 1.0, 1.0),
        orc.Camera("fisheye", 96, 80, 190.0 / 180.0, 150.0 / 180.0),
        orc.Camera("equirect", 128, 64)]


def test_pinhole_closed_forms():
    cam = orc.Camera("pinhole", 640, 480, np.radians(90.0), np.radians(60.0))
    d, ok = orc.cam_pixel_dir(cam, 320.0, 240.0)
    assert ok and np.allclose(d, [0, 0, 1], atol=1e-15)                       # principal point looks down the optical axis
    d, ok = orc.cam_pixel_dir(cam, 640.0 - 1e-9, 240.0)                       # right edge: half FoV_x = 45 deg off axis
    assert ok and abs(np.degrees(np.arctan2(d[0], d[2])) - 45.0) < 1e-6 and abs(d[1]) < 1e-15
    d, ok = orc.cam_pixel_dir(cam, 320.0, 0.0)                                # top edge: half FoV_y = 30 deg
    assert ok and abs(np.degrees(np.arctan2(-d[1], d[2])) - 30.0) < 1e-9
    assert not orc.cam_pixel_dir(cam, 640.5, 10.0)[1] and not orc.cam_pixel_dir(cam, -0.5, 10.0)[1]
    assert not orc.cam_project(cam, np.array([0.0, 0.0, -1.0]))[1]             # behind the camera


def test_fisheye_closed_forms():
    # isotropic 180 deg fisheye (w = 1): the incident angle grows linearly with the radius, 90 deg at the rim (Eq.14 with a = W/2)
    cam = orc.Camera("fisheye", 400, 400, 1.0, 1.0)
    for frac in (0.0, 0.25, 0.5, 1.0):
        d, ok = orc.cam_pixel_dir(cam, 200.0 + 200.0 * frac, 200.0)
        assert ok
        assert abs(np.degrees(np.arccos(np.clip(d[2], -1, 1))) - 90.0 * frac) < 1e-9
        assert abs(d[1]) < 1e-12 and d[0] >= -1e-15
    assert not orc.cam_pixel_dir(cam, 200.0 + 200.0 * 0.72, 200.0 + 200.0 * 0.72)[1]     # outside the inscribed ellipse
    # anisotropic: w_eff interpolates between w_x (horizontal) and w_y (vertical), Eq.12
    cam = orc.Camera("fisheye", 400, 200, 190.0 / 180.0, 120.0 / 180.0)
    d, _ = orc.cam_pixel_dir(cam, 400.0, 100.0)
    assert abs(np.degrees(np.arccos(d[2])) - 95.0) < 1e-9                     # horizontal rim: half of 190 deg
    d, _ = orc.cam_pixel_dir(cam, 200.0, 200.0)
    assert abs(np.degrees(np.arccos(d[2])) - 60.0) < 1e-9                     # vertical rim: half of 120 deg


def test_equirect_closed_forms():
    cam = orc.Camera("equirect", 360, 180)
    d, ok = orc.cam_pixel_dir(cam, 180.0, 90.0)
    assert ok and np.allclose(d, [0, 0, 1], atol=1e-15)                       # centre: omega = 0, phi = 0
    d, _ = orc.cam_pixel_dir(cam, 270.0, 90.0)
    assert np.allclose(d, [1, 0, 0], atol=1e-15)                              # omega = +90 deg -> camera +x (Eq.1 convention)
    d, _ = orc.cam_pixel_dir(cam, 180.0, 0.0)
    assert np.allclose(d, [0, 1, 0], atol=1e-15)                              # top row: phi = +90 deg


@pytest.mark.parametrize("cam", CAMS, ids=lambda c: f"{c.model}-{c.p0:.2f}")
def test_project_inverts_pixel_dir(cam):
    rng = np.random.default_rng(1)
    n_in = 0
    for _ in range(400):
        u, v = rng.uniform(0, cam.width), rng.uniform(0, cam.height)
        d, ok = orc.cam_pixel_dir(cam, u, v)
        assert abs(np.linalg.norm(d) - 1) < 1e-12
        if not ok:
            continue
        n_in += 1
        uv, ok2 = orc.cam_project(cam, d)
        assert ok2 and np.allclose(uv, [u, v], atol=1e-8)
    assert n_in > 200


def test_camera_mask_solid_angles():
    """Pixel counts of M_C against the solid angles PAPER.md:62 gives: 4 asin(sin tx sin ty) (perspective), 2 pi (1 - cos t)
    (isotropic fisheye), 4 pi (equirect)."""
    order = 6
    npix = 12 << (2 * order)
    tx, ty = np.radians(35.0), np.radians(25.0)
    bits = orc.camera_mask_bits(order, orc.Camera("pinhole", 640, 480, 2 * tx, 2 * ty))
    cnt = int(np.unpackbits(bits.view(np.uint8)).sum())
    want = npix * 4 * np.arcsin(np.sin(tx) * np.sin(ty)) / (4 * np.pi)
    assert abs(cnt - want) < 6 * np.sqrt(npix) * 0.25
    bits = orc.camera_mask_bits(order, orc.Camera("fisheye", 512, 512, 1.0, 1.0))
    cnt = int(np.unpackbits(bits.view(np.uint8)).sum())
    assert abs(cnt - npix / 2) < 4 * np.sqrt(npix)                              # hemisphere
    bits = orc.camera_mask_bits(order, orc.Camera("fisheye", 512, 512, 190.0 / 180, 190.0 / 180))
    cnt = int(np.unpackbits(bits.view(np.uint8)).sum())
    assert abs(cnt - npix * (1 - np.cos(np.radians(95.0))) / 2) < 4 * np.sqrt(npix)
    bits = orc.camera_mask_bits(order, orc.Camera("equirect", 64, 32))
    assert int(np.unpackbits(bits.view(np.uint8)).sum()) == npix


@pytest.mark.parametrize("order", [0, 1, 3, 5])
def test_interp_weights_invariants_and_bruteforce(order):
    """Weights are a partition of unity; away from the poles the support is the two longitude-nearest centres on each of the two
    bracketing rings, found here by brute force over ALL pixel centres (independent of the oracle's ring arithmetic)."""
    z, lam, _ = orc.centers(order, which=1)
    theta_c = np.arccos(np.clip(z, -1, 1))
    ring_thetas = np.unique(np.round(theta_c, 12))
    rng = np.random.default_rng(order)
    for _ in range(300):
        th = np.arccos(rng.uniform(-1, 1)); la = rng.uniform(0, 2 * np.pi)
        pix, w = orc.interp_weights(order, th, la)
        assert abs(w.sum() - 1) < 1e-12 and (w >= -1e-15).all()
        if th < ring_thetas[0] or th > ring_thetas[-1]:
            assert len(pix) == 6                                            # ring pair + the 4 pixels that stand for the pole
            continue
        above = ring_thetas[ring_thetas <= th].max(); below = ring_thetas[ring_thetas > th].min() if (ring_thetas > th).any() else None
        want = set()
        for rt in (above, below):
            if rt is None:
                continue
            on = np.flatnonzero(np.abs(theta_c - rt) < 1e-9)
            dl = np.abs((lam[on] - la + np.pi) % (2 * np.pi) - np.pi)
            want.update(on[np.argsort(dl)[:2]].tolist())
        got = set(pix[w > 1e-9].tolist())
        assert got <= want, (th, la, got, want)
    # at a pixel centre the interpolant returns that pixel
    for p in rng.choice(z.shape[0], min(50, z.shape[0]), replace=False):
        pix, w = orc.interp_weights(order, theta_c[p], lam[p])
        assert abs(w[pix == p].sum() - 1) < 1e-9


def test_interp_reproduces_ring_linear_functions():
    """Bilinear in (colatitude, longitude): a field that is a function of the ring colatitude only is reproduced wherever it is linear
    in colatitude, i.e. f = theta exactly between the first and the last ring; f = longitude away from the 0 / 2 pi seam."""
    order = 4
    z, lam, _ = orc.centers(order, which=1)
    theta_c = np.arccos(np.clip(z, -1, 1))
    rng = np.random.default_rng(7)
    for _ in range(300):
        th = rng.uniform(theta_c.min(), theta_c.max()); la = rng.uniform(0.6, 2 * np.pi - 0.6)
        pix, w = orc.interp_weights(order, th, la)
        assert abs((w * theta_c[pix]).sum() - th) < 1e-12
        assert abs((w * lam[pix]).sum() - la) < 1e-12
    # beyond the first ring the value runs linearly in theta from the ring-1 mean (pole) to the ring value
    t1 = theta_c.min()
    f = np.where(np.abs(theta_c - t1) < 1e-12, 5.0, 0.0)
    pix, w = orc.interp_weights(order, 0.25 * t1, 1.0)
    assert abs((w * f[pix]).sum() - 5.0) < 1e-12
    g = lam.copy()                                                           # ring 1 has 4 pixels at pi/4 + k pi/2: mean = pi
    pix, w = orc.interp_weights(order, 0.0, 1.0)
    assert abs((w * g[pix]).sum() - np.pi) < 1e-12


@pytest.mark.parametrize("cam", CAMS, ids=lambda c: f"{c.model}-{c.p0:.2f}")
def test_resample_constant_and_smooth_field(cam):
    order = 5
    npix = 12 << (2 * order)
    one = np.ones((npix, 1), np.float32)
    out, valid = orc.resample_fwd(order, cam, one)
    assert np.allclose(out[valid == 1], 1.0, atol=1e-12) and np.all(out[valid == 0] == 0)
    # a smooth field sampled at the pixel centres is recovered to second order in the pixel size
    dirs = orc.centers(order, which=2)[2]
    a = np.array([0.3, -0.5, 0.8])
    img = (dirs @ a).astype(np.float32).reshape(-1, 1)
    out, valid = orc.resample_fwd(order, cam, img)
    err = 0.0
    for j in range(0, cam.height, 7):
        for i in range(0, cam.width, 5):
            if valid[j, i]:
                d, _ = orc.cam_pixel_dir(cam, i + 0.5, j + 0.5)
                err = max(err, abs(out[j, i, 0] - d @ a))
    # pixel size 1.8 deg: (0.032 rad)^2 ~ 1e-3; next to the poles ring 1 has 4 pixels 90 deg apart: (1 - cos 45 deg) sin(theta_1) = 7.5e-3
    assert err < (8e-3 if cam.model == "equirect" else 3e-3), err


@pytest.mark.parametrize("cam", CAMS[:2], ids=lambda c: c.model)
def test_resample_mask_renormalisation_and_adjoint(cam):
    order = 4
    cfg = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    bits = orc.camera_mask_bits(order, cam)
    act, slot = orc.mask_tiles(cfg, bits)
    n_slot = act.shape[0]
    rng = np.random.default_rng(3)
    one = np.ones((n_slot * 256, 2), np.float32)
    out, valid = orc.resample_fwd(order, cam, one, slot, bits)
    inside = out[..., 0] > 0
    assert np.allclose(out[inside], 1.0, atol=1e-12)                          # dropped weights are renormalised (A27)
    assert inside.sum() >= 0.97 * valid.sum()
    # adjoint identity <R x, y> = <x, R^T y>
    x = rng.normal(size=(n_slot * 256, 2)).astype(np.float32)
    y = rng.normal(size=(cam.height, cam.width, 2))
    Rx, _ = orc.resample_fwd(order, cam, x, slot, bits)
    Rty = orc.resample_bwd(order, cam, y, n_slot, slot, bits)
    assert abs((Rx * y).sum() - (x.astype(np.float64) * Rty).sum()) < 1e-9 * max(1.0, abs((Rx * y).sum()))
    # pixels the mask switches off receive no gradient
    off = np.ones(n_slot * 256, bool)
    pm = np.unpackbits(bits.view(np.uint8), bitorder="little").astype(bool)
    for t, s in enumerate(slot):
        if s >= 0:
            off[s * 256:(s + 1) * 256] = ~pm[t * 256:(t + 1) * 256]
    assert np.all(Rty[off] == 0)
