"""Pins for the oracle's HEALPix RING geometry and its kernel-table evaluation (CPU only).

The paper only cites HEALPix; the layout pinned here is the published one
(tests/golden/healpix_ring_nside1_nside2.txt) plus invariants of the scheme.
"""
import os

import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append(line.split())
    return rows


def test_explicit_layout_nside1_nside2():
    rows = _load("healpix_ring_nside1_nside2.txt")
    den = {1: (3.0, 4.0), 2: (12.0, 8.0)}
    for nside in (1, 2):
        sel = [(int(r[1]), int(r[2]), int(r[3])) for r in rows if int(r[0]) == nside]
        assert len(sel) == 12 * nside * nside
        pa = O.pix2ang(nside, [s[0] for s in sel])
        z = np.array([s[1] for s in sel]) / den[nside][0]
        phi = np.array([s[2] for s in sel]) * np.pi / den[nside][1]
        np.testing.assert_allclose(pa["z"], z, rtol=0, atol=2e-16)
        np.testing.assert_allclose(pa["phi"], phi, rtol=0, atol=1e-15)
        np.testing.assert_allclose(pa["s"], np.sqrt(1 - z * z), rtol=0, atol=2e-16)


@pytest.mark.parametrize("nside", [1, 2, 3, 4, 7, 16, 64, 256])
def test_ring_table_invariants(nside):
    t = O.ring_table(nside)
    nr = 4 * nside - 1
    npix = 12 * nside * nside
    assert O.npix(nside) == npix
    assert t["npr"].sum() == npix
    # starts are the running sum of ring lengths
    np.testing.assert_array_equal(t["start"], np.concatenate(([0], np.cumsum(t["npr"])[:-1])))
    # cap rings have 4i pixels, belt rings 4N
    i = np.arange(1, nr + 1)
    ip = np.minimum(np.minimum(i, nside), 4 * nside - i)
    np.testing.assert_array_equal(t["npr"], 4 * ip)
    # z strictly decreasing, north/south mirror, equator at z = 0
    assert np.all(np.diff(t["z"]) < 0)
    np.testing.assert_allclose(t["z"], -t["z"][::-1], rtol=0, atol=1e-16)
    assert t["z"][2 * nside - 1] == 0.0
    np.testing.assert_array_equal(t["npr"], t["npr"][::-1])
    np.testing.assert_allclose(t["phi0"], t["phi0"][::-1], rtol=0, atol=0)
    # equal-area property: ring i's pixels have area 4pi/npix, so the z-extent of the cap down to
    # the boundary below ring i is (pixels so far) * 2/npix; the ring centre lies inside it
    zb_above = 1.0 - 2.0 * t["start"] / npix
    zb_below = 1.0 - 2.0 * (t["start"] + t["npr"]) / npix
    assert np.all(t["z"] < zb_above + 1e-15) and np.all(t["z"] > zb_below - 1e-15)
    # s^2 + z^2 = 1
    np.testing.assert_allclose(t["s"] ** 2 + t["z"] ** 2, 1.0, rtol=0, atol=4e-16)
    # phi: first pixel at dphi/2 unless shifted (belt rings with (i-N) odd) where it is 0
    np.testing.assert_allclose(t["dphi"] * t["npr"], 2 * np.pi, rtol=1e-15)
    sh = (i >= nside) & (i <= 3 * nside) & ((i - nside) % 2 == 1)
    np.testing.assert_array_equal(t["shifted"], sh.astype(np.int32))
    np.testing.assert_allclose(t["phi0"], np.where(sh, 0.0, 0.5 * t["dphi"]), rtol=0, atol=0)


@pytest.mark.parametrize("nside", [1, 2, 5, 8, 32])
def test_pix2ang_roundtrip_and_sums(nside):
    npix = 12 * nside * nside
    pa = O.pix2ang(nside, np.arange(npix))
    t = O.ring_table(nside)
    # pixel index = ring start + k, and k < ring length
    np.testing.assert_array_equal(t["start"][pa["ring"] - 1] + pa["k"], np.arange(npix))
    assert np.all(pa["k"] < t["npr"][pa["ring"] - 1]) and np.all(pa["k"] >= 0)
    # sum of unit vectors vanishes (4-fold + mirror symmetry), mean z^2 ~ 1/3 (equal-area quadrature)
    x, y, z = pa["s"] * np.cos(pa["phi"]), pa["s"] * np.sin(pa["phi"]), pa["z"]
    assert abs(x.sum()) < 1e-10 and abs(y.sum()) < 1e-10 and abs(z.sum()) < 1e-10
    assert abs((z * z).mean() - 1.0 / 3.0) < 0.2 / nside ** 2 + 1e-15
    # phi inside [0, 2pi)
    assert pa["phi"].min() >= 0 and pa["phi"].max() < 2 * np.pi


def test_pix2ang_rejects_out_of_range():
    with pytest.raises(ValueError):
        O.pix2ang(4, [12 * 16])
    with pytest.raises(ValueError):
        O.pix2ang(4, [-1])


def test_kernel_eval_is_linear_interpolation_on_uniform_cos_nodes():
    theta_max = 0.3
    c = np.cos(theta_max)
    n = 9
    T = np.array([3.0, -1.0, 4.0, 1.0, -5.0, 9.0, 2.0, 6.0, 5.0])
    x = c + np.arange(n) * (1 - c) / (n - 1)
    # nodes reproduce the table; index 0 is x = cos(theta_max), index n-1 is x = 1
    for i in range(n):
        assert abs(O.kernel_eval(T, theta_max, x[i]) - T[i]) < 1e-12
    # midpoints are averages; quarter points are 3:1 blends
    for i in range(n - 1):
        assert abs(O.kernel_eval(T, theta_max, 0.5 * (x[i] + x[i + 1])) - 0.5 * (T[i] + T[i + 1])) < 1e-12
        assert abs(O.kernel_eval(T, theta_max, 0.75 * x[i] + 0.25 * x[i + 1])
                   - (0.75 * T[i] + 0.25 * T[i + 1])) < 1e-12
    # x above 1 (round-off of a self pair) clamps to the last node
    assert O.kernel_eval(T, theta_max, 1.0 + 3e-16) == T[-1]
    assert O.kernel_eval(T, theta_max, 1.0) == T[-1]


def test_canonical_dot_matches_vector_dot():
    """z z' + s s' cos(dphi) is the unit-vector dot product (spherical law of cosines)."""
    nside = 8
    npix = 12 * nside * nside
    pa = O.pix2ang(nside, np.arange(npix))
    v = np.stack([pa["s"] * np.cos(pa["phi"]), pa["s"] * np.sin(pa["phi"]), pa["z"]], 1)
    rng = np.random.default_rng(0)
    p, q = rng.integers(0, npix, 2000), rng.integers(0, npix, 2000)
    canon = pa["z"][p] * pa["z"][q] + (pa["s"][p] * pa["s"][q]) * np.cos(pa["phi"][p] - pa["phi"][q])
    np.testing.assert_allclose(canon, np.einsum("ij,ij->i", v[p], v[q]), rtol=0, atol=5e-16)
