"""The paper-style table generator (workloads/splitfit.py; Eq. 1-6): properties the least-squares
split must have, on a small problem (l_max 384)."""
import numpy as np

from workloads import gen, splitfit


def _problem():
    lmax, fwhm = 384, 60 * gen.ARCMIN
    return lmax, splitfit.gaussian_beam_ell(fwhm, lmax)


def test_legendre_recurrence_against_closed_forms():
    x = np.linspace(-1, 1, 9)
    P = splitfit.legendre_matrix(4, x)
    np.testing.assert_allclose(P[2], 0.5 * (3 * x ** 2 - 1), atol=1e-14)
    np.testing.assert_allclose(P[3], 0.5 * (5 * x ** 3 - 3 * x), atol=1e-14)
    np.testing.assert_allclose(P[4], (35 * x ** 4 - 30 * x ** 2 + 3) / 8, atol=1e-14)


def test_split_reproduces_the_kernel_and_needs_enough_support():
    lmax, K = _problem()
    errs = []
    for theta_cut in (1.0 * gen.DEG, 2.0 * gen.DEG, 4.0 * gen.DEG):
        r = splitfit.split_fit(K, ell_cut=128, theta_cut=theta_cut, n_nodes=256)
        # below l_cut the l-space part absorbs the residual exactly (identity block of Eq. 5)
        assert np.max(np.abs((K - r["K_tilde_ell"])[:128])) < 1e-8 * K[0]
        assert r["K_hat_theta"].size == 256 and r["K_hat_ell"].size == 128
        errs.append(r["sigma2_frac"])
    # a real-space support of about one beam width is too narrow; two and four are enough (Eq. 6, alpha = 1;
    # not monotone beyond that: the 1e-6 singular-value cut damps differently for every support)
    assert errs[0] > 1e-6 > max(errs[1], errs[2])


def test_real_space_part_is_compact_and_feeds_the_table_format():
    """The fitted real-space kernel lives on the library's node set x_j = c + j (1-c)/(n-1): it can be passed to
    sc_plan_create / the oracle unchanged, and its Legendre transform carries the high-l part of K_l."""
    lmax, K = _problem()
    theta_cut = 3.0 * gen.DEG
    r = splitfit.split_fit(K, ell_cut=128, theta_cut=theta_cut, n_nodes=256)
    x_lib, _ = gen.table_nodes(theta_cut, 256)
    np.testing.assert_allclose(r["x"], x_lib, atol=1e-15)
    w = np.full(256, (1 - np.cos(theta_cut)) / 255)
    w[[0, -1]] *= 0.5
    b = 2 * np.pi * splitfit.legendre_matrix(lmax, r["x"]) @ (w * r["K_hat_theta"])
    hi = np.arange(lmax + 1) >= 128
    assert np.sum((2 * np.arange(lmax + 1) + 1)[hi] * (K - b)[hi] ** 2) <= 1e-6 * np.sum((2 * np.arange(lmax + 1) + 1) * K ** 2)
