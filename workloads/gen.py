"""Seeded synthetic inputs for the real-space spherical convolution (maps and kernel tables).

This module serves BOTH the oracle-side tests and the CUDA-side tests / bench.  It holds none of
the method's arithmetic (no neighbour search, no interpolation, no summation): it only produces
input arrays.  numpy/scipy only.

The inputs stand in for the paper's workload -- HEALPix Nside 2048 white-noise ("uniform-noise")
maps convolved with arc-minute beams, PAPER.md:76, :86, :124 -- whose actual kernels derive from
the WMAP-7 spectrum and are not available here.  The five configurations
are BASELINE.json's `configs`, verbatim.
"""
from dataclasses import dataclass, field
from typing import Tuple

import numpy as np

ARCMIN = np.pi / 10800.0
DEG = np.pi / 180.0


@dataclass(frozen=True)
class Config:
    name: str
    nside: int
    theta_max: float                 # radians
    n_table: int
    kernel: str                      # "gauss" | "split"
    fwhm: float                      # radians
    seeds: Tuple[int, ...]           # one N(0,1) map per seed
    ylm_map: bool = False            # append the l<=4 band-limited map (config 2)
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def npix(self):
        return 12 * self.nside * self.nside

    @property
    def batch(self):
        return len(self.seeds) + (1 if self.ylm_map else 0)


CONFIGS = (
    Config("cfg1_nside64_gauss2deg", 64, 3.4 * DEG, 4096, "gauss", 2.0 * DEG, (0,)),
    Config("cfg2_nside256_gauss30am", 256, 1.5 * DEG, 4096, "gauss", 30 * ARCMIN, (1,), ylm_map=True),
    Config("cfg3_nside1024_gauss10am", 1024, 30 * ARCMIN, 8192, "gauss", 10 * ARCMIN, (2,)),
    Config("cfg4_nside2048_split5am", 2048, 20 * ARCMIN, 16384, "split", 5 * ARCMIN, (3,),
           extra=dict(l_split=1500, taper_from=15 * ARCMIN)),
    Config("cfg5_nside2048_gauss20am_b3", 2048, 60 * ARCMIN, 16384, "gauss", 20 * ARCMIN, (4, 5, 6)),
    # NOT a BASELINE.json config: the paper's own worked example (7' beam, l_cut 1500, theta_cut 240',
    # PAPER.md:94-96, Fig. 3-4) as a split-like stand-in table -- context for Eq. 7's 8.0 s on a GTX 480
    Config("cfg6_paper_nside2048_split7am_240am", 2048, 240 * ARCMIN, 16384, "split", 7 * ARCMIN, (7,),
           extra=dict(l_split=1500, taper_from=200 * ARCMIN)),
)


def config(i: int) -> Config:
    """BASELINE.json configs[i-1] (1-based as in SURVEY.md); 6 = the paper-scale extra (see CONFIGS)."""
    return CONFIGS[i - 1]


# ---------------------------------------------------------------------------------------------
# maps
# ---------------------------------------------------------------------------------------------
def noise_map(npix: int, seed: int) -> np.ndarray:
    """fp32 i.i.d. N(0,1) map ("uniform-noise input map").  Philox counter RNG so the
    same seed gives the same map on every machine."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    return rng.standard_normal(npix, dtype=np.float32)


def ring_zphi(nside: int):
    """(z, phi) of every RING pixel centre, fp64 -- used only to *evaluate input functions* on the
    pixel grid (Y_lm maps, zonal maps); standard HEALPix ring formulas (Gorski et al. 2005)."""
    N = nside
    i = np.arange(1, 4 * N, dtype=np.int64)
    ip = np.where(i < N, i, np.where(i <= 3 * N, N, 4 * N - i))
    zc = 1.0 - ip.astype(np.float64) ** 2 / (3.0 * N * N)
    z = np.where(i < N, zc, np.where(i <= 3 * N, (2.0 * N - i) * 2.0 / (3.0 * N), -zc))
    shifted = (i >= N) & (i <= 3 * N) & (((i - N) & 1) == 1)
    n = 4 * ip
    ring = np.repeat(np.arange(4 * N - 1), n)
    start = np.concatenate(([0], np.cumsum(n)[:-1]))
    k = np.arange(12 * N * N, dtype=np.int64) - start[ring]
    dphi = 2.0 * np.pi / n
    phi = (k + np.where(shifted, 0.0, 0.5)[ring]) * dphi[ring]
    return z[ring], phi


def legendre_map(nside: int, ell: int) -> np.ndarray:
    """fp64 zonal map P_ell(z_p) (proportional to Y_ell,0)."""
    from scipy.special import eval_legendre
    z, _ = ring_zphi(nside)
    return eval_legendre(ell, z)


def ylm_map(nside: int, seed: int, lmax: int = 4) -> np.ndarray:
    """Band-limited map m = sum_{l<=lmax} sum_m a_lm Y^real_lm with (lmax+1)^2 coefficients ~N(0,1)
    drawn in (l, m=-l..l) order (BASELINE.json config 2).  Built in fp64."""
    from scipy.special import sph_harm_y
    rng = np.random.Generator(np.random.Philox(key=seed))
    z, phi = ring_zphi(nside)
    theta = np.arccos(z)
    out = np.zeros(z.shape, np.float64)
    for l in range(lmax + 1):
        for m in range(-l, l + 1):
            a = rng.standard_normal()
            Y = sph_harm_y(l, abs(m), theta, phi)
            if m == 0:
                y = Y.real
            elif m > 0:
                y = np.sqrt(2.0) * (-1) ** m * Y.real
            else:
                y = np.sqrt(2.0) * (-1) ** m * Y.imag
            out += a * y
    return out


def maps_for(cfg: Config):
    """List of the config's fp32 input maps."""
    maps = [noise_map(cfg.npix, s) for s in cfg.seeds]
    if cfg.ylm_map:
        maps.append(ylm_map(cfg.nside, seed=1000 + cfg.seeds[0]).astype(np.float32))
    return maps


# ---------------------------------------------------------------------------------------------
# kernel tables: n samples K(x_i), x_i = c + i (1-c)/(n-1), c = cos(theta_max)  (x_{n-1} = 1)
# ---------------------------------------------------------------------------------------------
def table_nodes(theta_max: float, n: int):
    """(x_i, theta_i) of the table nodes; theta from 1 - x to keep small angles accurate."""
    c = np.cos(theta_max)
    i = np.arange(n, dtype=np.float64)
    one_minus_x = (n - 1 - i) * ((1.0 - c) / (n - 1))
    x = c + i * ((1.0 - c) / (n - 1))
    theta = 2.0 * np.arcsin(np.sqrt(0.5 * one_minus_x))
    return x, theta


def zoned_table_nodes(theta_max: float, n: int, zone_frac: float):
    """Nodes of the two-zone table (reading R11): n even, h = n / 2,
    x1 = cos(zone_frac theta_max); x_i = c + i (x1 - c) / h for i < h, x_i = x1 + (i - h)(1 - x1)/(h - 1)
    for i >= h.  -> (x_i, theta_i = acos x_i); x_0 = cos(theta_max), x_{n-1} = 1."""
    if n < 4 or n % 2 or not (0.0 < zone_frac < 1.0):
        raise ValueError("n even >= 4 and 0 < zone_frac < 1")
    h = n // 2
    c, x1 = np.cos(theta_max), np.cos(zone_frac * theta_max)
    x = np.concatenate([c + np.arange(h) * (x1 - c) / h, x1 + np.arange(h) * (1.0 - x1) / (h - 1)])
    x[-1] = 1.0
    return x, np.arccos(np.clip(x, -1.0, 1.0))


def gaussian_table(fwhm: float, theta_max: float, n: int) -> np.ndarray:
    """K(theta) = exp(-theta^2 / 2 sigma^2), sigma = FWHM / 2.3548 (as BASELINE.json writes it;
    'Gaussian beam with a given FWHM')."""
    sigma = fwhm / 2.3548
    _, theta = table_nodes(theta_max, n)
    return np.exp(-0.5 * (theta / sigma) ** 2)


def split_table(fwhm: float, theta_max: float, n: int, l_split: int, taper_from: float) -> np.ndarray:
    """Stand-in for the paper's truncated real-space kernel (Fig. 3-4), whose LSQ/SVD
    fit needs the WMAP-7 spectrum: K_r = [Gaussian - its l<=l_split Legendre-truncated part] times a
    cosine taper from `taper_from` to 0 at theta_max (BASELINE.json config 4)."""
    sigma = fwhm / 2.3548
    x, theta = table_nodes(theta_max, n)
    kg = np.exp(-0.5 * (theta / sigma) ** 2)
    # b_l of the flat-sky Gaussian, K_low(x) = sum_l (2l+1)/(4 pi) b_l P_l(x), 3-term recurrence
    p0, p1 = np.ones_like(x), x.copy()
    klow = np.zeros_like(x)
    for l in range(l_split + 1):
        bl = 2.0 * np.pi * sigma * sigma * np.exp(-0.5 * l * (l + 1) * sigma * sigma)
        pl = p0 if l == 0 else p1
        klow += (2 * l + 1) / (4.0 * np.pi) * bl * pl
        if l >= 1:
            p0, p1 = p1, ((2 * l + 1) * x * p1 - l * p0) / (l + 1)
    taper = np.where(theta <= taper_from, 1.0,
                     0.5 * (1.0 + np.cos(np.pi * (theta - taper_from) / (theta_max - taper_from))))
    taper = np.where(theta >= theta_max, 0.0, taper)
    return (kg - klow) * taper


def table_for(cfg: Config) -> np.ndarray:
    if cfg.kernel == "gauss":
        return gaussian_table(cfg.fwhm, cfg.theta_max, cfg.n_table)
    if cfg.kernel == "split":
        return split_table(cfg.fwhm, cfg.theta_max, cfg.n_table, cfg.extra["l_split"],
                           cfg.extra["taper_from"])
    raise ValueError(cfg.kernel)


def sample_pixels(nside: int, n: int, seed: int) -> np.ndarray:
    """Deterministic sample of output pixels for full-size parity: both pole caps' first/last
    pixels, the cap/belt boundary rings, the equator, plus `n` seeded random pixels."""
    N = nside
    npix = 12 * N * N
    ncap = 2 * N * (N - 1)
    fixed = [0, 1, 2, 3, 4, 11, 12, npix - 1, npix - 4, npix - 5, npix - 12,
             ncap - 1, ncap, ncap + 1, ncap + 4 * N - 1, ncap + 4 * N,
             npix - ncap - 1, npix - ncap, npix // 2, npix // 2 - 1, npix // 2 + 4 * N]
    fixed = [p for p in fixed if 0 <= p < npix]
    rng = np.random.Generator(np.random.Philox(key=seed))
    rnd = rng.integers(0, npix, size=n, dtype=np.int64)
    return np.unique(np.concatenate([np.asarray(fixed, np.int64), rnd]))
