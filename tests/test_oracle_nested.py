"""Pins of the oracle's NESTED -> RING index map (oracle/nested.py): it is a bijection, the identity at
Nside 1 (one pixel per base face, faces numbered along the rings), every NESTED pixel centre computed from the
HEALPix projection plane coincides with a RING pixel centre (checked inside nest2ring to 1e-9), the four
children of a pixel surround their parent's centre, z -> -z maps face f of the north cap to face f + 8, and -- the pin
of the east/west orientation inside a face (which interleaved bit is ix) -- the published Nside-2 table
(tests/golden/healpix_nest2ring_nside2.txt) plus the same orientation at every resolution."""
import os

import numpy as np
import pytest

import oracle as O
from oracle import nested


@pytest.mark.parametrize("nside", [1, 2, 4, 16, 64])
def test_bijection(nside):
    r = nested.nest2ring(nside)
    assert np.array_equal(np.sort(r), np.arange(12 * nside * nside))


def test_nside1_is_identity():
    assert np.array_equal(nested.nest2ring(1), np.arange(12))


@pytest.mark.parametrize("nside", [2, 8, 32])
def test_children_surround_parent(nside):
    """NESTED hierarchy: pixels 4p .. 4p+3 at Nside are the children of pixel p at Nside/2; the mean of the
    children's unit vectors points at the parent's centre (to a small fraction of the pixel size)."""
    def vec(ns, ring_idx):
        a = O.pix2ang(ns, ring_idx)
        return np.stack([a["s"] * np.cos(a["phi"]), a["s"] * np.sin(a["phi"]), a["z"]], 1)
    rc, rp = nested.nest2ring(nside), nested.nest2ring(nside // 2)
    vc, vp = vec(nside, rc), vec(nside // 2, rp)
    mean = vc.reshape(-1, 4, 3).mean(1)
    mean /= np.linalg.norm(mean, axis=1)[:, None]
    ang = np.arccos(np.clip(np.sum(mean * vp, 1), -1, 1))
    pix = np.sqrt(4 * np.pi / (12 * (nside // 2) ** 2))
    assert ang.max() < 0.2 * pix
    # and every child is closer to its own parent than to 3 pixel sizes
    d = np.arccos(np.clip(np.sum(vc * np.repeat(vp, 4, 0), 1), -1, 1))
    assert d.max() < 0.8 * pix


def test_north_south_faces_mirror():
    nside = 8
    r = nested.nest2ring(nside)
    a = O.pix2ang(nside, r)
    n2 = nside * nside
    for f in range(4):
        zn = np.sort(a["z"][f * n2:(f + 1) * n2])
        zs = np.sort(-a["z"][(f + 8) * n2:(f + 9) * n2])
        np.testing.assert_allclose(zn, zs, atol=1e-14)
        assert a["z"][f * n2:(f + 1) * n2].min() > -1e-9 - 2.0 / 3.0 * 0 - 0.01   # north faces reach down to the equator only
    assert np.all(np.abs(a["z"][4 * n2:8 * n2]) <= 2.0 / 3.0 + 1e-12)              # equatorial faces stay in the belt


def test_published_nside2_table():
    """The Nside-2 NESTED -> RING table of Gorski et al. 2005 (Fig. 4), written out by hand in tests/golden/: swapping the
    two interleaved bits (east <-> west inside every face) or mis-placing a face fails here."""
    path = os.path.join(os.path.dirname(__file__), "golden", "healpix_nest2ring_nside2.txt")
    want = np.array([int(l) for l in open(path) if l.strip() and not l.startswith("#")], np.int64)
    assert want.size == 48 and np.array_equal(np.sort(want), np.arange(48))
    assert np.array_equal(nested.nest2ring(2), want)


@pytest.mark.parametrize("nside", [2, 4, 16, 128])
def test_child_1_is_east_of_child_2(nside):
    """NESTED bit order at every level: of the four children 4p .. 4p+3 of a pixel, child 0 is the southernmost, child 3
    the northernmost, and child 1 lies EAST (larger phi) of child 2 (Gorski et al. 2005, Fig. 4: the even bits of the
    in-face index count along the north-east axis).  Checked away from the poles' phi wrap by comparing on the circle."""
    r = nested.nest2ring(nside)
    a = O.pix2ang(nside, r)
    z, phi = a["z"].reshape(-1, 4), a["phi"].reshape(-1, 4)
    assert np.all(z[:, 0] < z[:, 1]) and np.all(z[:, 0] < z[:, 2]) and np.all(z[:, 3] > z[:, 1]) and np.all(z[:, 3] > z[:, 2])
    d = np.mod(phi[:, 1] - phi[:, 2] + np.pi, 2 * np.pi) - np.pi          # signed azimuth difference east - west
    assert np.all(d > 0)
