"""Pins of the oracle's NESTED -> RING index map (oracle/nested.py): it is a bijection, the identity at
Nside 1 (one pixel per base face, faces numbered along the rings), every NESTED pixel centre computed from the
HEALPix projection plane coincides with a RING pixel centre (checked inside nest2ring to 1e-9), the four
children of a pixel surround their parent's centre, and z -> -z maps face f of the north cap to face f + 8."""
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
