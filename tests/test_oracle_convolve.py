"""Pins for the oracle's convolution against closed forms and invariants (CPU only).

BASELINE.json north_star: constant map -> Omega * Sum K ~ 2 pi Int K dx; Y_10 / Y_20 maps -> b_l * map
with b_l = 2 pi Int K(x) P_l(x) dx; linearity; operator symmetry <a, C b> = <C a, b>.
Tolerances are the measured discretisation errors of SURVEY.md 8c.6 (the paper states none).
"""
import os

import numpy as np
import pytest
from scipy.integrate import quad
from scipy.special import eval_legendre

import oracle as O
from workloads import gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _b_ell_golden():
    out = {}
    with open(os.path.join(GOLD, "b_ell.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a = line.split()
                out[(int(a[0]), int(a[1]))] = float(a[2])
    return out


def _b_ell_quad(cfg, ell):
    """2 pi Int_c^1 K(x) P_l(x) dx of the ANALYTIC truncated Gaussian, in theta to keep it smooth."""
    sigma = cfg.fwhm / 2.3548
    f = lambda th: np.exp(-0.5 * (th / sigma) ** 2) * eval_legendre(ell, np.cos(th)) * np.sin(th)
    v, _ = quad(f, 0.0, cfg.theta_max, epsabs=0, epsrel=1e-13, limit=400)
    return 2 * np.pi * v


def test_golden_b_ell_matches_quadrature():
    g = _b_ell_golden()
    for (c, ell), val in g.items():
        cfg = gen.config(c)
        assert abs(_b_ell_quad(cfg, ell) / val - 1) < 2e-9, (c, ell)


def _belt(nside, margin):
    t = O.ring_table(nside)
    lo, hi = nside + margin, 3 * nside - margin        # ring numbers
    return slice(int(t["start"][lo - 1]), int(t["start"][hi - 1] + t["npr"][hi - 1]))


def _relrms(a, b):
    return np.sqrt(np.mean((a - b) ** 2) / np.mean(b ** 2))


def test_constant_map_config1():
    cfg = gen.config(1)
    b0 = _b_ell_golden()[(1, 0)]
    T = gen.table_for(cfg)
    one = np.ones(cfg.npix, np.float32)
    out, cnt, _ = O.convolve(cfg.nside, T, cfg.theta_max, [one])
    out = out[0]
    belt = _belt(cfg.nside, 4)
    # mean +2.7e-5, belt max 1.5e-4 / rms 7e-5, all-sky rms 6.2e-4, poles -4.3 %
    assert abs(out.mean() / b0 - 1) < 1e-4
    assert np.max(np.abs(out[belt] / b0 - 1)) < 3e-4
    assert _relrms(out, np.full_like(out, b0)) < 2e-3
    assert -0.06 < out[0] / b0 - 1 < -0.03
    # and equals Omega * Sum_q Kt by definition: re-sum with the neighbour list of a few pixels
    for p in (0, 777, cfg.npix // 2, cfg.npix - 1):
        q = O.neighbours(cfg.nside, cfg.theta_max, p)
        assert q.size == cnt[p]


@pytest.mark.parametrize("ell,tol_belt,tol_all", [(1, 1.5e-4, 2.5e-3), (2, 1.5e-4, 3e-3),
                                                    (30, 1.5e-4, 1e-2), (60, 2.5e-4, None)])
def test_zonal_eigenfunctions_config1(ell, tol_belt, tol_all):
    """m = P_l(z) (prop. to Y_l0) -> b_l m.  l = 60 has b_l/b_0 = 0.67: a wrong kernel scale, a
    reversed table or a wrong normalisation fails here even though l <= 2 barely sees the kernel."""
    cfg = gen.config(1)
    bl = _b_ell_golden()[(1, ell)]
    T = gen.table_for(cfg)
    m = gen.legendre_map(cfg.nside, ell).astype(np.float32)
    out, _, _ = O.convolve(cfg.nside, T, cfg.theta_max, [m])
    ref = bl * m.astype(np.float64)
    belt = _belt(cfg.nside, 4)
    # normalise by the all-sky rms of the reference (zonal maps have nodes in the belt)
    scale = np.sqrt(np.mean(ref ** 2))
    assert np.sqrt(np.mean((out[0][belt] - ref[belt]) ** 2)) / scale < tol_belt
    if tol_all is not None:
        assert _relrms(out[0], ref) < tol_all
    # discriminating power: the neighbouring multiplier b_{l+-} must NOT fit at high l
    if ell >= 30:
        wrong = _b_ell_golden()[(1, 100 if ell == 60 else 60)]
        assert np.sqrt(np.mean((out[0][belt] - wrong / bl * ref[belt]) ** 2)) / scale > 50 * tol_belt


@pytest.mark.slow
def test_zonal_eigenfunctions_config2_belt_sample():
    """Config 2 (Nside 256, truncation at 7 sigma): belt rel-rms 1.5e-7 (l <= 4), 4.8e-7 (l = 120)
    per SURVEY.md 8c.6; checked on every 16th belt ring to keep the CPU suite short."""
    cfg = gen.config(2)
    g = _b_ell_golden()
    # The config's own 4096-node table carries a lerp bias of (h/sigma^2)^2/12 ~ +3e-6 (K is convex
    # in x); the pin is against the ANALYTIC b_l, so use a 2^17-node table here (bias ~3e-9) and
    # check the 4096-node bias separately below.
    T = gen.gaussian_table(cfg.fwhm, cfg.theta_max, 1 << 17)
    t = O.ring_table(cfg.nside)
    rings = np.arange(cfg.nside + 8, 3 * cfg.nside - 8, 16)
    sel = np.concatenate([np.arange(t["start"][r - 1], t["start"][r - 1] + t["npr"][r - 1], 7)
                          for r in rings])
    for ell, tol in ((0, 1e-6), (2, 2e-6), (4, 2e-6), (120, 5e-6)):
        m = gen.legendre_map(cfg.nside, ell).astype(np.float32)
        out, _, _ = O.convolve(cfg.nside, T, cfg.theta_max, [m], sel=sel)
        ref = g[(2, ell)] * m.astype(np.float64)
        scale = np.sqrt(np.mean(ref ** 2))
        assert np.sqrt(np.mean((out[0] - ref[sel]) ** 2)) / scale < tol, ell
    # 4096-node table: constant map is biased high by ~ (h/sigma^2)^2/12, h = (1-c)/(n-1)
    one = np.ones(cfg.npix, np.float32)
    out, _, _ = O.convolve(cfg.nside, gen.table_for(cfg), cfg.theta_max, [one], sel=sel)
    sigma2 = (cfg.fwhm / 2.3548) ** 2
    h = (1 - np.cos(cfg.theta_max)) / (cfg.n_table - 1)
    bias = (h / sigma2) ** 2 / 12
    assert abs(np.mean(out[0]) / g[(2, 0)] - 1 - bias) < 0.15 * bias


def test_linearity():
    nside, th = 32, 0.12
    npix = 12 * nside * nside
    rng = np.random.default_rng(1)
    T = rng.standard_normal(257)
    a = rng.standard_normal(npix).astype(np.float32)
    b = rng.standard_normal(npix).astype(np.float32)
    # alpha a + beta b must be exactly representable in fp32 for the identity to hold to fp64
    # round-off: use power-of-two weights on maps quantised to 12 bits
    a = np.round(a * 256) / 256
    b = np.round(b * 256) / 256
    comb = (0.5 * a - 2.0 * b).astype(np.float32)
    assert np.array_equal(comb.astype(np.float64), 0.5 * a.astype(np.float64) - 2.0 * b)
    out, _, _ = O.convolve(nside, T, th, [a, b, comb])
    np.testing.assert_allclose(out[2], 0.5 * out[0] - 2.0 * out[1], rtol=0,
                               atol=1e-14 * np.abs(out).max())


def test_operator_symmetry():
    """<a, C b> = <C a, b> to fp64 round-off (K radial => symmetric weights, Omega uniform)."""
    for nside, th in ((16, 0.3), (64, 3.4 * np.pi / 180)):
        npix = 12 * nside * nside
        rng = np.random.default_rng(nside)
        T = rng.standard_normal(513)
        a = rng.standard_normal(npix).astype(np.float32)
        b = rng.standard_normal(npix).astype(np.float32)
        out, _, _ = O.convolve(nside, T, th, [a, b])
        lhs = np.dot(a.astype(np.float64), out[1])
        rhs = np.dot(out[0], b.astype(np.float64))
        norm = np.linalg.norm(a) * np.linalg.norm(out[1])
        assert abs(lhs - rhs) < 1e-13 * norm


def test_convolve_equals_explicit_sum_on_tiny_map():
    """out(p) re-summed here from the brute-force neighbour list, numpy lerp of the table in x."""
    nside, th = 4, 0.5
    npix = 12 * nside * nside
    rng = np.random.default_rng(9)
    n = 33
    T = rng.standard_normal(n)
    m = rng.standard_normal(npix).astype(np.float32)
    out, cnt, sig = O.convolve(nside, T, th, [m], mode=O.MODE_BRUTE)
    pa = O.pix2ang(nside, np.arange(npix))
    c = np.cos(th)
    xn = c + np.arange(n) * (1 - c) / (n - 1)
    for p in range(npix):
        q = O.neighbours(nside, th, p, O.MODE_BRUTE)
        d = pa["z"][p] * pa["z"][q] + (pa["s"][p] * pa["s"][q]) * np.cos(pa["phi"][p] - pa["phi"][q])
        K = np.interp(np.minimum(d, 1.0), xn, T)
        want = 4 * np.pi / npix * np.sum(K * m[q].astype(np.float64))
        assert abs(out[0][p] - want) < 1e-13 * np.abs(out).max()
        assert cnt[p] == q.size and sig[p] == q.sum()


def test_selected_outputs_match_full_run():
    cfg = gen.config(1)
    T = gen.table_for(cfg)
    m = gen.noise_map(cfg.npix, 0)
    sel = gen.sample_pixels(cfg.nside, 200, seed=1)
    full, cf, sf = O.convolve(cfg.nside, T, cfg.theta_max, [m])
    part, cp, sp = O.convolve(cfg.nside, T, cfg.theta_max, [m], sel=sel)
    np.testing.assert_array_equal(full[0][sel], part[0])
    np.testing.assert_array_equal(cf[sel], cp)
    np.testing.assert_array_equal(sf[sel], sp)


def test_split_table_shape_config4():
    """SURVEY.md 8c.4 shape check of the config-4 stand-in kernel: K_r(0) = 0.65067, minimum
    -0.1297 near 5.30', zero crossings near 3.46', 9.33', 16.35'; exactly 0 at theta_max."""
    cfg = gen.config(4)
    T = gen.table_for(cfg)
    _, theta = gen.table_nodes(cfg.theta_max, cfg.n_table)
    am = theta / gen.ARCMIN
    assert abs(T[-1] - 0.65067) < 2e-5
    assert T[0] == 0.0
    i = np.argmin(T)
    assert abs(T[i] + 0.1297) < 2e-4 and abs(am[i] - 5.30) < 0.05
    zc = am[np.nonzero(np.diff(np.sign(T[1:])))[0] + 1]
    assert len(zc) == 3
    np.testing.assert_allclose(np.sort(zc), [3.46, 9.33, 16.35], atol=0.03)
