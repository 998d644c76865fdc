"""Pins of the oracle's two-zone kernel table ("half the available interpolation nodes within
the first 1/16 of the available support"; reading R11), against what the mathematics fixes:
node values, the uniform table when both zones have the same spacing, exactness for kernels that are
linear in x = cos(theta) (brute-force sum over the oracle's own neighbour list), a kink at the zone
boundary, and monotone node placement with half the nodes inside zone_frac * theta_max."""
import numpy as np
import pytest

import oracle as O
from oracle import sco
from workloads import gen


def test_node_placement():
    theta, n, f = 240 * gen.ARCMIN, 4096, 1.0 / 16.0
    x, th = gen.zoned_table_nodes(theta, n, f)
    assert x.size == n and np.all(np.diff(x) > 0)
    assert x[0] == pytest.approx(np.cos(theta), abs=1e-15) and x[-1] == 1.0
    inner = th <= f * theta * (1 + 1e-9)
    assert inner.sum() == n // 2                       # half the nodes within the first 1/16 of the support
    assert th[n // 2] == pytest.approx(f * theta, rel=1e-9)
    # uniform in x inside each zone
    assert np.allclose(np.diff(x[: n // 2 + 1]), np.diff(x[: n // 2 + 1])[0], rtol=1e-9)
    assert np.allclose(np.diff(x[n // 2:]), np.diff(x[n // 2:])[0], rtol=1e-9)


def test_nodes_are_reproduced_and_midpoints_are_means():
    theta, n, f = 3.0 * gen.DEG, 32, 0.125
    x, _ = gen.zoned_table_nodes(theta, n, f)
    T = np.sin(40.0 * x) + x ** 3
    for i in range(n):
        assert sco.kernel_eval_zoned(T, theta, f, x[i]) == pytest.approx(T[i], abs=1e-13)
    for i in range(n - 1):
        xm = 0.5 * (x[i] + x[i + 1])
        assert sco.kernel_eval_zoned(T, theta, f, xm) == pytest.approx(0.5 * (T[i] + T[i + 1]), abs=1e-12)
    # argument above 1 (self pair rounding) clamps to the last node
    assert sco.kernel_eval_zoned(T, theta, f, 1.0 + 1e-15) == pytest.approx(T[-1], abs=1e-13)


def test_equal_spacing_zones_equal_the_uniform_table():
    """If (x1 - c) / h == (1 - x1) / (h - 1) the node set IS the uniform one: both evaluations and both
    convolutions must agree to round-off (pins the index arithmetic of both zones against the pinned
    uniform path)."""
    nside, theta, n = 16, 11.0 * gen.DEG, 64
    h, c = n // 2, np.cos(theta)
    x1 = (h + c * (h - 1)) / (n - 1)
    f = np.arccos(x1) / theta
    xu, _ = gen.table_nodes(theta, n)
    xz, _ = gen.zoned_table_nodes(theta, n, f)
    np.testing.assert_allclose(xz, xu, rtol=0, atol=1e-14)
    T = np.cos(25.0 * xu) * np.exp(3 * (xu - 1))
    for xx in np.linspace(c, 1.0, 777):
        assert sco.kernel_eval_zoned(T, theta, f, xx) == pytest.approx(sco.kernel_eval(T, theta, xx), abs=1e-12)
    m = gen.noise_map(12 * nside * nside, 5)
    a, ca, sa = O.convolve(nside, T, theta, [m])
    b, cb, sb = O.convolve(nside, T, theta, [m], zone_frac=f)
    np.testing.assert_array_equal(ca, cb)
    np.testing.assert_allclose(b, a, rtol=0, atol=1e-13 * np.max(np.abs(a)))


@pytest.mark.parametrize("f", [1.0 / 16.0, 0.3, 0.77])
def test_kernel_linear_in_x_is_exact(f):
    """K(x) = a + b x is reproduced exactly by linear interpolation on ANY node set, so the convolution must
    equal Omega * sum_q (a + b dot_pq) m_q over the neighbour list, with dot_pq from the unit vectors."""
    nside, theta, n = 8, 20.0 * gen.DEG, 16
    npix = 12 * nside * nside
    x, _ = gen.zoned_table_nodes(theta, n, f)
    a_, b_ = 0.7, -1.9
    T = a_ + b_ * x
    m = gen.noise_map(npix, 6).astype(np.float64)
    out, cnt, _ = O.convolve(nside, T, theta, [m.astype(np.float32)], zone_frac=f)
    ang = O.pix2ang(nside, np.arange(npix))
    v = np.stack([ang["s"] * np.cos(ang["phi"]), ang["s"] * np.sin(ang["phi"]), ang["z"]], 1)
    omega = 4 * np.pi / npix
    for p in (0, 5, 100, 383, 400, npix - 1):
        q = O.neighbours(nside, theta, p)
        assert q.size == cnt[p]
        dots = np.minimum(v[q] @ v[p], 1.0)
        want = omega * np.sum((a_ + b_ * dots) * m[q].astype(np.float32))
        assert out[0][p] == pytest.approx(want, rel=1e-12, abs=1e-15)


def test_kink_at_zone_boundary_is_exact():
    """A kernel that is piecewise linear in x with its only kink at x1 is exact on the two-zone table."""
    theta, n, f = 10.0 * gen.DEG, 12, 0.25
    x, _ = gen.zoned_table_nodes(theta, n, f)
    x1 = np.cos(f * theta)
    K = lambda xx: 2.0 * abs(xx - x1) + 0.1 * xx
    T = np.array([K(xx) for xx in x])
    for xx in np.linspace(np.cos(theta), 1.0, 501):
        assert sco.kernel_eval_zoned(T, theta, f, xx) == pytest.approx(K(xx), abs=1e-13)


def test_bad_arguments():
    m = [gen.noise_map(12, 1)]
    with pytest.raises(Exception):
        O.convolve(1, np.ones(5), 1.0, m, zone_frac=0.5)      # odd n
    with pytest.raises(Exception):
        O.convolve(1, np.ones(2), 1.0, m, zone_frac=0.5)      # n < 4
    with pytest.raises(Exception):
        O.convolve(1, np.ones(8), 1.0, m, zone_frac=1.0)      # zone_frac must be < 1
