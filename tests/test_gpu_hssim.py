"""GPU parity of the L1 + HEALPix-SSIM loss (include/uts.h uts_hssim_loss) against the oracle
(oracle/orc_hssim.cpp), through the C ABI.  PAPER.md:135-143, Eq.10; readings A30-A35.

Tolerances: the kernel works in fp32 with the window sums taken about the centre pixel's value, the oracle in
fp64.  h_q: 5e-5 absolute (h in [-1, 1]); L, L1^H, HSSIM: 2e-6 absolute (fp64 accumulation of fp32 per-pixel terms);
dL/dX: 2e-4 of the largest entry (fp32 SSIM derivatives; atomics, summation order not fixed)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle as orc

pytestmark = pytest.mark.gpu

TOL_H, TOL_L, TOL_G = 5e-5, 2e-6, 2e-4


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B
    return B


def _images(order, n_store, seed, kind):
    """Seeded synthetic (rendered, ground truth) pair in [0,1]: a smooth field of the storage index plus noise, like a render
    against its photograph ('natural'); independent uniform noise ('noise'); identical images ('same'); flat images ('flat')."""
    rng = np.random.default_rng(seed)
    i = np.arange(n_store, dtype=np.float64)[:, None]
    if kind == "natural":
        base = 0.5 + 0.35 * np.sin(i * np.array([[0.011, 0.007, 0.003]]) + np.array([[0.0, 1.0, 2.0]]))
        X = base + 0.05 * rng.normal(size=(n_store, 3))
        G = base + 0.08 * rng.normal(size=(n_store, 3)) + 0.02
    elif kind == "noise":
        X, G = rng.uniform(size=(n_store, 3)), rng.uniform(size=(n_store, 3))
    elif kind == "same":
        X = rng.uniform(size=(n_store, 3)); G = X
    else:
        X = np.full((n_store, 3), 0.25); G = np.full((n_store, 3), 0.75)
    return np.clip(X, 0, 1).astype(np.float32), np.clip(G, 0, 1).astype(np.float32)


def _run(B, cfg, mask, X, G, lam=0.2, sigma=1.5, grad=True, hmap=True):
    n = X.shape[0]
    dX = torch.from_numpy(X).cuda(); dG = torch.from_numpy(G).cuda()
    loss3 = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")
    scratch = torch.empty(B.uts_hssim_scratch_bytes(cfg), dtype=torch.uint8, device="cuda")
    h = torch.full((n,), -7.0, dtype=torch.float32, device="cuda") if hmap else None
    g = torch.full((n, 3), -7.0, dtype=torch.float32, device="cuda") if grad else None
    B.uts_hssim_loss(cfg, mask, dX, dG, loss3, scratch, h_map=h, dL_dX=g, lam=lam, sigma=sigma)
    torch.cuda.synchronize()
    return loss3.cpu().numpy(), None if h is None else h.cpu().numpy(), None if g is None else g.cpu().numpy()


def _compare(got, want, grad=True):
    l3, h, g = got
    assert abs(l3[0] - want["loss"]) <= TOL_L and abs(l3[1] - want["l1"]) <= TOL_L and abs(l3[2] - want["hssim"]) <= TOL_L, (l3, want["loss"], want["l1"], want["hssim"])
    assert np.abs(h - want["h_map"]).max(initial=0.0) <= TOL_H
    if grad:
        scale = np.abs(want["grad"]).max(initial=0.0)
        assert np.abs(g - want["grad"]).max(initial=0.0) <= TOL_G * scale + 1e-12


@pytest.mark.parametrize("kind", ["natural", "noise"])
@pytest.mark.parametrize("order", [4, 5, 6])
def test_full_sphere_matches_oracle(order, kind):
    """Every face edge, both pole crossings and all 8 three-face vertices are inside the image; order 4 has faces of one tile
    (every tile touches four edges), order 6 has interior tiles and a ragged mix of edge tiles."""
    B = _gpu()
    cfg = B.Config(order=order, n_gauss=1)
    n = (12 << (2 * order))
    X, G = _images(order, n, order * 11 + len(kind), kind)
    want = orc.hssim_loss(order, X, G)
    _compare(_run(B, cfg, B.Mask.full(), X, G), want)


CAMS = [("fisheye", 128, 128, 190.0 / 180.0, 190.0 / 180.0), ("pinhole", 160, 120, np.radians(70.0), np.radians(50.0)),
        ("fisheye", 150, 90, 200.0 / 180.0, 140.0 / 180.0)]


@pytest.mark.parametrize("spec", CAMS, ids=lambda s: f"{s[0]}-{s[1]}x{s[2]}")
@pytest.mark.parametrize("order", [5, 7])
def test_camera_mask_matches_oracle(spec, order):
    """FoV masks: windows cut by M_C = 0 (weights renormalised, A32), inactive tiles in the apron, slot layout != tile layout."""
    B = _gpu()
    cfg = B.Config(order=order, n_gauss=1)
    oc = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    mask = B.uts_build_camera_mask(cfg, B.Camera(*spec))
    bits = orc.camera_mask_bits(order, orc.Camera(*spec))
    act, slot = orc.mask_tiles(oc, bits)
    assert mask.n_active == act.shape[0]
    X, G = _images(order, act.shape[0] * 256, order + spec[1], "natural")
    want = orc.hssim_loss(order, X, G, slot_of_tile=slot, bits=bits)
    _compare(_run(B, cfg, mask, X, G), want)


@pytest.mark.parametrize("axis,half", [((0.0, 1.0, 0.0), 0.9), ((0.0, -1.0, 0.0), 0.5), ((0.6, 0.64, 0.48), 1.3), ((1.0, 0.0, 0.0), 0.05)])
def test_cap_masks_match_oracle(axis, half):
    """Caps about the poles (the quarter-turn gluing of the polar faces inside the window), about a general axis covering 3-face
    vertices, and a cap smaller than a window (few valid pixels, heavy renormalisation)."""
    B = _gpu()
    order = 6
    cfg = B.Config(order=order, n_gauss=1)
    oc = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    mask = B.uts_build_mask(cfg, "cap", list(axis) + [half])
    bits = orc.mask_bits(order, "cap", list(axis) + [half])
    act, slot = orc.mask_tiles(oc, bits)
    assert mask.n_active == act.shape[0] > 0
    X, G = _images(order, act.shape[0] * 256, int(half * 100), "noise")
    want = orc.hssim_loss(order, X, G, slot_of_tile=slot, bits=bits, lam=0.35, sigma=2.0)
    _compare(_run(B, cfg, mask, X, G, lam=0.35, sigma=2.0), want)


def test_identical_and_flat_images():
    """X = G: h = 1 everywhere, L = 0, gradient ~ 0 (SSIM has a maximum there; L1's subgradient at 0 is taken as 0).  Flat
    X = a, G = b: h = (2ab + C1) / (a^2 + b^2 + C1) exactly, for any window."""
    B = _gpu()
    order = 5
    cfg = B.Config(order=order, n_gauss=1)
    n = 12 << (2 * order)
    X, G = _images(order, n, 3, "same")
    l3, h, g = _run(B, cfg, B.Mask.full(), X, G)
    assert abs(l3[0]) <= TOL_L and abs(l3[1]) <= 1e-12 and abs(l3[2] - 1.0) <= TOL_L
    assert np.abs(h - 1.0).max() <= TOL_H
    assert np.abs(g).max() <= 1e-6 / n * 50
    X, G = _images(order, n, 3, "flat")
    l3, h, g = _run(B, cfg, B.Mask.full(), X, G)
    want = (2 * 0.25 * 0.75 + 1e-4) / (0.25 ** 2 + 0.75 ** 2 + 1e-4)
    assert np.abs(h - want).max() <= 1e-6
    assert abs(l3[1] - 0.5) <= 1e-7 and abs(l3[2] - want) <= 1e-6
    _compare((l3, h, g), orc.hssim_loss(order, X, G))


def test_forward_only_and_no_map():
    B = _gpu()
    order = 5
    cfg = B.Config(order=order, n_gauss=1)
    n = 12 << (2 * order)
    X, G = _images(order, n, 9, "natural")
    want = orc.hssim_loss(order, X, G, grad=False)
    l3, h, g = _run(B, cfg, B.Mask.full(), X, G, grad=False, hmap=False)
    assert h is None and g is None
    assert abs(l3[0] - want["loss"]) <= TOL_L and abs(l3[2] - want["hssim"]) <= TOL_L


def test_empty_mask():
    """No visible pixel: L = L1 = HSSIM = 0 (the oracle's convention), nothing launched over the image."""
    B = _gpu()
    order = 5
    cfg = B.Config(order=order, n_gauss=1)
    z = torch.zeros(1, dtype=torch.int32, device="cuda")          # n_active = 0 of a non-null list
    mask = B.Mask(z, 0, torch.full((cfg.n_tiles,), -1, dtype=torch.int32, device="cuda"), torch.zeros(cfg.n_pix // 32, dtype=torch.int32, device="cuda"))
    X = np.zeros((0, 3), np.float32)
    l3, h, g = _run(B, cfg, mask, X, X)
    assert np.array_equal(l3, np.zeros(3))


def test_chain_render_loss_backward():
    """The loss's gradient is what uts_render_bwd consumes: render a small scene, take dL/dI from uts_hssim_loss against a seeded
    target, and compare with the oracle's loss gradient on the GPU's own image (same input on both sides)."""
    B = _gpu()
    from paper_2606_29794_b200 import scenes
    from paper_2606_29794_b200.rasterizer import Rasterizer, config_of, scene_to_device
    sc = scenes.make_scene(1, seed=2, n_gauss=3000, order=6)
    cfg = config_of(sc)
    g_dev, views = scene_to_device(sc)
    r = Rasterizer(cfg, B.Mask.full())
    color, _ = r.forward(g_dev, views)
    img = color[0].contiguous()
    n = img.shape[0]
    rng = np.random.default_rng(4)
    G = np.clip(img.cpu().numpy() + 0.05 * rng.normal(size=(n, 3)), 0, 1).astype(np.float32)
    loss3 = torch.empty(3, dtype=torch.float64, device="cuda")
    g = torch.empty(n, 3, dtype=torch.float32, device="cuda")
    scratch = torch.empty(B.uts_hssim_scratch_bytes(cfg), dtype=torch.uint8, device="cuda")
    B.uts_hssim_loss(cfg, r.mask, img, torch.from_numpy(G).cuda(), loss3, scratch, dL_dX=g)
    torch.cuda.synchronize()
    want = orc.hssim_loss(6, img.cpu().numpy(), G)
    assert abs(loss3[0].item() - want["loss"]) <= TOL_L
    assert np.abs(g.cpu().numpy() - want["grad"]).max() <= TOL_G * np.abs(want["grad"]).max()
    grads = r.backward(g_dev, views, g.view(1, n, 3))
    torch.cuda.synchronize()
    assert all(bool(torch.isfinite(v).all()) for v in grads.values()) and float(grads["means"].abs().max()) > 0


def _sample_pixels(order, rng, n_random):
    """Pixels where the window meets every kind of face boundary — the four corners of every face (both poles, the eight 3-face
    vertices, the 4-face vertices), edge midpoints — plus random ones."""
    N = 1 << order
    def nest(f, x, y):
        p = 0
        for b in range(order):
            p |= ((x >> b) & 1) << (2 * b) | ((y >> b) & 1) << (2 * b + 1)
        return (f << (2 * order)) | p
    pts = []
    for f in range(12):
        for (x, y) in [(0, 0), (N - 1, 0), (0, N - 1), (N - 1, N - 1), (N // 2, 0), (0, N // 2), (N - 1, N // 2), (N // 2, N - 1), (3, N - 2), (N - 4, 2)]:
            pts.append(nest(f, x, y))
    pts += list(rng.integers(0, 12 << (2 * order), size=n_random))
    return np.unique(np.array(pts, np.int64))


@pytest.mark.parametrize("masked", [False, True], ids=["config4-full-sphere", "fisheye-mask"])
def test_full_size_sampled_against_oracle(masked):
    """BASELINE.json's image size (order 10, Nside 1024: 12.6 M pixels), the launch bench.py times under extras.hssim_loss.  The
    oracle evaluates a sample: the centres P (face corners, edges, random) and every pixel of their windows, Q; h is compared on all
    of Q, the gradient on P (every centre whose window holds a pixel of P is in Q, by the window's symmetry, pinned in
    tests/test_oracle_hssim.py).  Whole-image properties: HSSIM = mean of the kernel's own h_map, L1^H = the plain mean of |X - G|."""
    B = _gpu()
    order = 10
    cfg = B.Config(order=order, n_gauss=1)
    oc = orc.Config(order=order, n_gauss=1, n_views=1, sh_degree=0)
    rng = np.random.default_rng(21 + masked)
    if masked:
        spec = ("fisheye", 2048, 2048, 200.0 / 180.0, 200.0 / 180.0)
        mask = B.uts_build_camera_mask(cfg, B.Camera(*spec))
        bits = orc.camera_mask_bits(order, orc.Camera(*spec))
        act, slot = orc.mask_tiles(oc, bits)
        n = act.shape[0] * 256
    else:
        mask, bits, slot, n = B.Mask.full(), None, None, 12 << (2 * order)
    X, G = _images(order, n, 5, "natural")
    P = _sample_pixels(order, rng, 150)
    Q = set()
    for p in P:
        for dy in range(-5, 6):
            for dx in range(-5, 6):
                q, _ = orc.hssim_neighbor(order, int(p), dx, dy)
                if q >= 0:
                    Q.add(q)
    Q = np.array(sorted(Q), np.int64)
    want = orc.hssim_loss(order, X, G, slot_of_tile=slot, bits=bits, q_list=Q)
    l3, h, g = _run(B, cfg, mask, X, G)

    def store(p):
        if bits is not None and not (bits[p >> 5] >> (p & 31)) & 1:
            return -1
        s = p >> 8 if slot is None else slot[p >> 8]
        return -1 if s < 0 else s * 256 + (p & 255)
    iQ = np.array([store(int(q)) for q in Q]); iQ = iQ[iQ >= 0]
    iP = np.array([store(int(p)) for p in P]); iP = iP[iP >= 0]
    assert iQ.size > 5000 and iP.size > (60 if masked else 250)
    assert np.abs(h[iQ] - want["h_map"][iQ]).max() <= TOL_H
    scale = np.abs(want["grad"][iP]).max()
    assert np.abs(g[iP] - want["grad"][iP]).max() <= TOL_G * scale
    n_valid = n if bits is None else int(sum(bin(int(w)).count("1") for w in bits))
    assert abs(l3[2] - h.astype(np.float64).sum() / n_valid) <= TOL_L
    if bits is None:
        assert abs(l3[1] - np.abs(X.astype(np.float64) - G).mean()) <= TOL_L
    assert abs(l3[0] - (0.8 * l3[1] + 0.2 * (1 - l3[2]))) <= 1e-8              # lambda is an fp32 argument of the ABI


def test_max_order_flat_images():
    """Order 13 (Nside 8192, 8.05e8 pixels: the largest grid uts_config accepts; 3 * n_store exceeds 2^31, so every storage index
    has to be 64-bit).  Flat X = a, G = b: h = (2ab + C1) / (a^2 + b^2 + C1) at every pixel for any window, L1^H = |a - b|, and
    dL/dX = (1 - lambda) sign(a - b) / (3 N) + the SSIM term, whose window weights sum to 1: the same value at every pixel."""
    B = _gpu()
    if torch.cuda.mem_get_info()[0] < 40e9:
        pytest.skip("needs 40 GB of free device memory")
    order = 13
    cfg = B.Config(order=order, n_gauss=1)
    n = 12 << (2 * order)
    a, b, lam = 0.25, 0.75, 0.2
    X = torch.full((n, 3), a, dtype=torch.float32, device="cuda"); G = torch.full((n, 3), b, dtype=torch.float32, device="cuda")
    h = torch.empty(n, dtype=torch.float32, device="cuda"); g = torch.empty(n, 3, dtype=torch.float32, device="cuda")
    loss3 = torch.empty(3, dtype=torch.float64, device="cuda")
    scratch = torch.empty(B.uts_hssim_scratch_bytes(cfg), dtype=torch.uint8, device="cuda")
    B.uts_hssim_loss(cfg, B.Mask.full(), X, G, loss3, scratch, h_map=h, dL_dX=g, lam=lam)
    torch.cuda.synchronize()
    want = (2 * a * b + 1e-4) / (a * a + b * b + 1e-4)
    assert float((h - want).abs().max()) <= 1e-6
    l3 = loss3.cpu().numpy()
    assert abs(l3[1] - abs(a - b)) <= 1e-7 and abs(l3[2] - want) <= 1e-6
    # d ssim / dx for flat windows: only the mean path is left, (2 b b1 - 2 a a1) / b1^2 with a1 = 2ab + C1, b1 = a^2 + b^2 + C1
    a1, b1 = 2 * a * b + 1e-4, a * a + b * b + 1e-4
    dssim = (2 * b * b1 - 2 * a * a1) / (b1 * b1)
    gw = ((1 - lam) * (-1.0) - lam * dssim) / (3.0 * n)
    # "the same value" holds where every window that contains the pixel uses one kernel and is complete: face interiors (across a
    # face edge the zone's kernel changes, at 3-face vertices taps are missing, and the normalised weights a pixel receives no longer
    # sum to 1).  Checked on pixels at least 8 from the face edges, tile corners and tile edges included; everywhere else bounded.
    rng = np.random.default_rng(13)
    N = 1 << order
    xs = np.concatenate([rng.integers(8, N - 8, 1500), 16 * rng.integers(1, N // 16 - 1, 500), 16 * rng.integers(1, N // 16 - 1, 500) - 1])
    ys = np.concatenate([rng.integers(8, N - 8, 1500), 16 * rng.integers(1, N // 16 - 1, 500) - 1, rng.integers(8, N - 8, 500)])
    fs = rng.integers(0, 12, xs.shape[0])
    p = np.zeros(xs.shape[0], np.int64)
    for bit in range(order):
        p |= ((xs >> bit) & 1) << (2 * bit) | ((ys >> bit) & 1) << (2 * bit + 1)
    p |= fs.astype(np.int64) << (2 * order)
    gs = g[torch.from_numpy(p).cuda()]
    assert float((gs / gw - 1.0).abs().max()) <= 2e-4
    assert float((g / gw - 1.0).abs().max()) <= 0.15
    del X, G, h, g
    torch.cuda.empty_cache()
