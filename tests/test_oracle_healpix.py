"""Pins for the oracle's HEALPix geometry (§3.1, Table 6).

The paper prints no formula for Nest2Lonlat; the oracle is pinned by what the paper and HEALPix fix:
12*Nside^2 pixels of equal area, the NESTED quadtree hierarchy, RING<->NESTED being two orders of the same pixels,
two independent derivations of the centres (plane form D1, ring form D2) plus the textbook RING-order centre,
Nside=1 closed-form centres, and the ring structure.
"""
import math

import numpy as np
import pytest

import oracle as orc


def test_npix_and_xyf_roundtrip():
    # PAPER.md:60 N_pix = 12 Nside^2 ; PAPER.md:64 (x,y,f) parameterisation
    for k in range(0, 7):
        n = 12 * (1 << k) ** 2
        assert orc.lib().orc_npix(k) == n
        for p in np.random.default_rng(k).integers(0, n, 200):
            x, y, f = orc.nest2xyf(k, p)
            assert 0 <= x < (1 << k) and 0 <= y < (1 << k) and 0 <= f < 12
            assert orc.xyf2nest(k, x, y, f) == p
    # bit interleave: x in the even bits, y in the odd bits
    assert orc.nest2xyf(3, 0b000001) == (1, 0, 0)
    assert orc.nest2xyf(3, 0b000010) == (0, 1, 0)
    assert orc.nest2xyf(3, 0b100100 + 5 * 64) == (0b010, 0b100, 5)


def test_nside1_closed_form_centres():
    # Nside=1: z = +2/3 (f=0-3), 0 (f=4-7), -2/3 (f=8-11); lam = pi/4 + c*pi/2 polar rows, c*pi/2 equatorial row
    for which in (1, 2):
        z, lam, _ = orc.centers(0, which)
        for f in range(12):
            r, c = divmod(f, 4)
            assert z[f] == pytest.approx([2 / 3, 0.0, -2 / 3][r], abs=1e-15)
            want = (math.pi / 4 + c * math.pi / 2) if r != 1 else c * math.pi / 2
            assert lam[f] == pytest.approx(want, abs=1e-15)


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4, 5, 6])
def test_D1_equals_D2_equals_ring_textbook(k):
    z1, l1, v1 = orc.centers(k, 1)
    z2, l2, v2 = orc.centers(k, 2)
    assert np.abs(v1 - v2).max() < 1e-14
    assert np.abs(z1 - z2).max() < 1e-14
    # textbook RING-order centre of the RING index of each NESTED pixel
    ring = orc.nest2ring(k)
    _, _, v3all = orc.centers(k, 3)
    assert np.abs(v3all[ring] - v2).max() < 1e-14
    # unit vectors, all distinct
    assert np.abs(np.linalg.norm(v2, axis=1) - 1).max() < 1e-15
    assert np.unique(np.round(v2, 12), axis=0).shape[0] == v2.shape[0]


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4, 5, 6, 7, 8])
def test_ring_nest_bijection(k):
    n = 12 << (2 * k)
    r = orc.nest2ring(k)
    assert np.array_equal(np.sort(r), np.arange(n))
    if k <= 6:
        back = orc.ring2nest(k)          # through ang2pix of the textbook centre
        assert np.array_equal(back[r], np.arange(n))


def test_ring_structure():
    # ring i (1..4Nside-1) has 4*min(i,Nside,4Nside-i) pixels, all at one z; RING index increases with ring then longitude
    k = 4; ns = 1 << k
    z, lam, _ = orc.centers(k, 3)
    pos = 0
    for i in range(1, 4 * ns):
        m = orc.ring_npix_in_ring(k, i)
        assert m == 4 * min(i, ns, 4 * ns - i)
        zz = z[pos:pos + m]; ll = lam[pos:pos + m]
        assert np.ptp(zz) < 1e-15
        assert np.all(np.diff(ll) > 0)
        # closed-form z of ring i
        if i < ns: want = 1 - i * i / (3 * ns * ns)
        elif i > 3 * ns: want = -1 + (4 * ns - i) ** 2 / (3 * ns * ns)
        else: want = (2 * ns - i) * 2 / (3 * ns)
        assert zz[0] == pytest.approx(want, abs=1e-15)
        pos += m
    assert pos == 12 * ns * ns


@pytest.mark.parametrize("k", [1, 3, 5, 7])
def test_pix_ang_pix_roundtrip_and_hierarchy(k):
    z, lam, v = orc.centers(k, 2)
    n = z.shape[0]
    assert np.array_equal(orc.ang2pix(k, z, lam), np.arange(n))
    assert np.array_equal(orc.vec2pix(k, v), np.arange(n))
    # parent contains its children's centres (PAPER.md:64 quadtree): ang2pix at order k-1 of a child centre = p>>2
    assert np.array_equal(orc.ang2pix(k - 1, z, lam), np.arange(n) >> 2)
    # tile of a pixel = p >> 2*log2(B)  (Alg.1 l.18 AncestorTile), checked geometrically two levels up
    if k >= 2:
        assert np.array_equal(orc.ang2pix(k - 2, z, lam), np.arange(n) >> 4)


def test_equal_area_exact_counts():
    # every order-k pixel contains exactly 4^5 order-(k+5) centres (equal area + hierarchy), via ang2pix (geometric, not bit shifts)
    k = 1
    z, lam, _ = orc.centers(k + 5, 1)
    counts = np.bincount(orc.ang2pix(k, z, lam), minlength=12 << (2 * k))
    assert np.all(counts == 1024)


def test_equal_area_monte_carlo():
    # 2M uniform directions: per-pixel counts consistent with binomial (Omega_pix = 4pi/N_pix)
    k = 3; n = 12 << (2 * k); m = 2_000_000
    rng = np.random.default_rng(1)
    v = rng.standard_normal((m, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
    counts = np.bincount(orc.vec2pix(k, v), minlength=n)
    mean = m / n; sd = math.sqrt(mean * (1 - 1 / n))
    zscore = (counts - mean) / sd
    assert np.abs(zscore).max() < 5.0
    assert abs(zscore.std() - 1.0) < 0.1


def test_rho_max_closed_equals_bruteforce():
    # PixRad(o) of Alg.2
    for o in range(0, 8):
        assert orc.rho_max_closed(o) == pytest.approx(orc.rho_max_bruteforce(o), rel=1e-13)
    assert orc.rho_max_closed(0) == pytest.approx(math.acos(2 / 3), rel=1e-14)
    # asymptotically ~ 1.044 sqrt(Omega_pix)
    o = 12
    assert orc.rho_max_closed(o) / math.sqrt(4 * math.pi / (12 << (2 * o))) == pytest.approx(1.044, abs=2e-3)


def test_rho_max_bounds_all_descendant_centres():
    # the bound Alg.2's pruning relies on: every descendant centre lies within rho_max(o) of the node centre
    for o in (0, 1, 2, 3):
        _, _, vn = orc.centers(o, 2)
        for d in (1, 2, 3, 4):
            _, _, vc = orc.centers(o + d, 2)
            parent = np.arange(vc.shape[0]) >> (2 * d)
            cosang = np.clip(np.einsum("ij,ij->i", vc, vn[parent]), -1, 1)
            assert np.arccos(cosang).max() <= orc.rho_max_closed(o) + 1e-12


def test_mask_solid_angles():
    # cap 2pi(1-cos theta); frustum 4 asin(sin tx sin ty)
    k = 6; n = 12 << (2 * k)
    bits = orc.mask_bits(k, "cap", [0, 0, 1, math.radians(95)])
    frac = np.unpackbits(bits.view(np.uint8)).sum() / n
    assert frac == pytest.approx((1 - math.cos(math.radians(95))) / 2, abs=2e-3)
    tx, ty = math.tan(math.radians(30)), math.tan(math.radians(22.5))
    bits = orc.mask_bits(k, "frustum", [1, 0, 0, 0, 1, 0, 0, 0, 1, tx, ty])
    frac = np.unpackbits(bits.view(np.uint8)).sum() / n
    assert frac == pytest.approx(4 * math.asin(math.sin(math.radians(30)) * math.sin(math.radians(22.5))) / (4 * math.pi), abs=2e-3)
