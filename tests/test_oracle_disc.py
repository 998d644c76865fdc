"""Pins for the oracle's ring-range disc query and its run-end counter (CPU only).

BASELINE.json north_star: "At Nside 16, the disc-query neighbour sets equal the brute-force sets
exactly"; SURVEY.md 8c.6 rows "disc query = brute force", "pair totals", "identity limit".
"""
import os

import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DEG = np.pi / 180.0
ARCMIN = np.pi / 10800.0


def _totals():
    rows = {}
    with open(os.path.join(GOLD, "pair_totals.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a = line.split()
                rows[(int(a[0]), int(a[1]))] = (int(a[2]), int(a[3]), int(a[4]))
    return rows


@pytest.mark.parametrize("nside", [4, 8, 16])
@pytest.mark.parametrize("theta_deg", [3.4, 13.6, 30.0, 75.0, 179.0])
def test_disc_query_equals_brute_force_sets(nside, theta_deg):
    """Neighbour SETS (not just counts) agree for every output pixel, incl. pole-containing discs
    and near-full-sphere discs (wrap through phi = 0)."""
    npix = 12 * nside * nside
    th = theta_deg * DEG
    for p in range(npix):
        a = np.sort(O.neighbours(nside, th, p, O.MODE_DISC))
        b = np.sort(O.neighbours(nside, th, p, O.MODE_BRUTE))
        assert a.size == np.unique(a).size, "disc query returned a pixel twice"
        np.testing.assert_array_equal(a, b)


def test_brute_force_is_the_definition():
    """Brute-force neighbour set re-derived here in numpy from unit vectors of the published
    Nside-2 layout (golden file), independent of the oracle's geometry code."""
    rows = []
    with open(os.path.join(GOLD, "healpix_ring_nside1_nside2.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a = line.split()
                if int(a[0]) == 2:
                    rows.append((int(a[2]) / 12.0, int(a[3]) * np.pi / 8.0))
    z = np.array([r[0] for r in rows]); phi = np.array([r[1] for r in rows])
    s = np.sqrt(1 - z * z)
    v = np.stack([s * np.cos(phi), s * np.sin(phi), z], 1)
    for theta_deg in (20.0, 35.0, 61.0, 100.0):
        c = np.cos(theta_deg * DEG)
        d = v @ v.T
        # stay away from knife edges so the vector form and the canonical form agree
        assert np.min(np.abs(d - c)) > 1e-9
        for p in range(48):
            want = np.nonzero(d[p] >= c)[0]
            got = np.sort(O.neighbours(2, theta_deg * DEG, p, O.MODE_BRUTE))
            np.testing.assert_array_equal(got, want)


def test_pair_totals_nside16_and_nside64():
    tot = _totals()
    # Nside 16, theta_max = 13.6 deg: brute force AND disc query AND run-end counter
    T16 = tot[(16, 816)][0]
    m = np.zeros(12 * 16 * 16, np.float32)
    _, c_b, s_b = O.convolve(16, None, 13.6 * DEG, [], mode=O.MODE_BRUTE)
    _, c_d, s_d = O.convolve(16, None, 13.6 * DEG, [], mode=O.MODE_DISC)
    c_r, s_r = O.count(16, 13.6 * DEG)
    assert int(c_b.sum()) == T16
    np.testing.assert_array_equal(c_b, c_d); np.testing.assert_array_equal(s_b, s_d)
    np.testing.assert_array_equal(c_b, c_r); np.testing.assert_array_equal(s_b, s_r)
    # config 1 (Nside 64, 3.4 deg): exact total and per-pixel min/max
    T64, lo, hi = tot[(64, 204)]
    _, c_d, s_d = O.convolve(64, None, 3.4 * DEG, [], mode=O.MODE_DISC)
    assert int(c_d.sum()) == T64 and c_d.min() == lo and c_d.max() == hi
    c_r, s_r = O.count(64, 3.4 * DEG)
    np.testing.assert_array_equal(c_d, c_r); np.testing.assert_array_equal(s_d, s_r)
    # north / equator / south split quoted in SURVEY.md 8a
    t = O.ring_table(64)
    eq0, eq1 = t["start"][2 * 64 - 1], t["start"][2 * 64 - 1] + t["npr"][2 * 64 - 1]
    assert (int(c_d[:eq0].sum()), int(c_d[eq0:eq1].sum()), int(c_d[eq1:].sum())) == \
        (1046852, 10496, 1046852)


@pytest.mark.slow
def test_pair_total_config2_full_sphere():
    T, lo, hi = _totals()[(256, 90)]
    c, _ = O.count(256, 1.5 * DEG)
    assert int(c.sum()) == T and c.min() == lo and c.max() == hi


def test_pair_totals_large_nside_on_symmetric_subset():
    """Configs 3-5: whole-sphere totals cost minutes; instead check the per-pixel min/max bounds of
    the golden file on sampled pixels, and the exact north == south mirror symmetry of counts."""
    tot = _totals()
    rng = np.random.default_rng(5)
    for nside, am in ((1024, 30), (2048, 20), (2048, 60)):
        _, lo, hi = tot[(nside, am)]
        npix = 12 * nside * nside
        sel = np.unique(np.concatenate([rng.integers(0, npix, 300), [0, 3, npix - 1, npix // 2]]))
        c, s = O.count(nside, am * ARCMIN, sel=sel)
        assert c.min() >= lo and c.max() <= hi
        # mirror pixel: same ring position in the southern ring 4N - i
        pa = O.pix2ang(nside, sel)
        t = O.ring_table(nside)
        mir = t["start"][4 * nside - pa["ring"] - 1] + pa["k"]
        cm, _ = O.count(nside, am * ARCMIN, sel=mir)
        np.testing.assert_array_equal(c, cm)


def test_run_end_counter_equals_exhaustive_on_samples():
    """sco_count (walks in from the run ends) == sco_convolve's exhaustive candidate test."""
    rng = np.random.default_rng(11)
    for nside, th in ((128, 2.0 * DEG), (1024, 30 * ARCMIN), (2048, 60 * ARCMIN), (37, 9.0 * DEG)):
        npix = 12 * nside * nside
        sel = np.unique(np.concatenate([rng.integers(0, npix, 200), np.arange(0, 24),
                                        np.arange(npix - 24, npix)]))
        _, c1, s1 = O.convolve(nside, None, th, [], sel=sel)
        c2, s2 = O.count(nside, th, sel=sel)
        np.testing.assert_array_equal(c1, c2); np.testing.assert_array_equal(s1, s2)


def test_identity_limit():
    """theta_max below the nearest-neighbour distance: count == 1, out = Omega * T[n-1] * m exactly."""
    nside = 16
    npix = 12 * nside * nside
    th = 0.2 / nside           # pixel spacing ~ 1/nside
    T = np.linspace(0.3, 2.5, 17)
    m = np.random.default_rng(3).standard_normal(npix).astype(np.float32)
    out, c, s = O.convolve(nside, T, th, [m])
    assert np.all(c == 1)
    np.testing.assert_array_equal(s, np.arange(npix, dtype=np.uint64))
    # self-pair dot = z^2 + s^2 is 1 - O(1e-16); the table coordinate amplifies that by
    # (n-1)/(1-c) ~ 2e5, so "exactly" means to ~1e-11 relative
    np.testing.assert_allclose(out[0], 4 * np.pi / npix * T[-1] * m.astype(np.float64), rtol=1e-10)


def test_neighbour_relation_is_symmetric():
    """q in N(p) <=> p in N(q), bitwise (dot_pq == dot_qp because (s_p s_q) is grouped)."""
    nside, th = 8, 17.0 * DEG
    npix = 12 * nside * nside
    A = np.zeros((npix, npix), bool)
    for p in range(npix):
        A[p, O.neighbours(nside, th, p)] = True
    assert np.array_equal(A, A.T) and np.all(np.diag(A))
