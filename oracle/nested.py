"""NESTED -> RING pixel index map for the oracle side (TEST INFRASTRUCTURE; shares nothing with the CUDA path).

Independent route: a NESTED pixel p = face * nside^2 + interleave(ix, iy) is located in the HEALPix
projection plane (Gorski et al. 2005, Fig. 4; the paper only cites HEALPix): the 12 base
faces are squares rotated by 45 degrees with centres
    faces 0-3: (x, y) = (pi/4 + f pi/2,  pi/4),  faces 4-7: ((f-4) pi/2, 0),  faces 8-11: (pi/4 + (f-8) pi/2, -pi/4),
and pixel (ix, iy) of a face sits at  x = x_c + (ix - iy) pi/(4 nside),  y = y_c + (ix + iy + 1 - nside) pi/(4 nside).
The plane maps to the sphere by  z = 8 y / (3 pi), phi = x  for |y| <= pi/4  and
z = sign(y)(1 - sigma^2/3), phi = x_t + (x - x_t)/sigma  with sigma = 2 - 4|y|/pi and x_t the centre of the
polar triangle, otherwise.  The RING pixel is then the one whose centre (ring table of the oracle) coincides
with (z, phi); `nest2ring` checks that it does to 1e-9, so a wrong formula cannot pass silently.
"""
import numpy as np

from . import sco


def _deinterleave(v):
    v = v.astype(np.int64)
    ix = np.zeros_like(v)
    iy = np.zeros_like(v)
    for b in range(31):
        ix |= ((v >> (2 * b)) & 1) << b
        iy |= ((v >> (2 * b + 1)) & 1) << b
    return ix, iy


def nest2ring(nside):
    """-> int64 array r with r[p_nested] = p_ring for all 12 nside^2 pixels (nside a power of two)."""
    if nside < 1 or nside & (nside - 1):
        raise ValueError("nside must be a power of two")
    npix = 12 * nside * nside
    p = np.arange(npix, dtype=np.int64)
    face = p // (nside * nside)
    ix, iy = _deinterleave(p % (nside * nside))
    xc = np.where(face < 4, np.pi / 4 + face * np.pi / 2,
                  np.where(face < 8, (face - 4) * np.pi / 2, np.pi / 4 + (face - 8) * np.pi / 2))
    yc = np.where(face < 4, np.pi / 4, np.where(face < 8, 0.0, -np.pi / 4))
    x = xc + (ix - iy) * np.pi / (4 * nside)
    y = yc + (ix + iy + 1 - nside) * np.pi / (4 * nside)
    ay = np.abs(y)
    eq = ay <= np.pi / 4 + 1e-14
    sigma = 2.0 - 4.0 * ay / np.pi
    z = np.where(eq, 8.0 * y / (3.0 * np.pi), np.sign(y) * (1.0 - sigma * sigma / 3.0))
    xt = np.pi / 4 + np.floor(x / (np.pi / 2)) * np.pi / 2
    with np.errstate(divide="ignore", invalid="ignore"):
        phi = np.where(eq, x, xt + (x - xt) / np.where(sigma > 0, sigma, 1.0))
    phi = np.mod(phi, 2 * np.pi)
    t = sco.ring_table(nside)
    zr = np.asarray(t["z"], np.float64)                   # decreasing with ring number
    ring = np.abs(zr[None, :] - z[:, None]).argmin(1) if npix <= 3072 else None
    if ring is None:                                       # large maps: search in the sorted z table
        idx = np.searchsorted(-zr, -z)
        idx = np.clip(idx, 1, zr.size - 1)
        ring = np.where(np.abs(zr[idx] - z) < np.abs(zr[idx - 1] - z), idx, idx - 1)
    assert np.max(np.abs(zr[ring] - z)) < 1e-9, "pixel centre is not on a ring"
    dphi = np.asarray(t["dphi"])[ring]
    phi0 = np.asarray(t["phi0"])[ring]
    npr = np.asarray(t["npr"])[ring].astype(np.int64)
    k = np.rint((phi - phi0) / dphi).astype(np.int64) % npr
    dd = np.abs(np.mod(phi0 + k * dphi - phi + np.pi, 2 * np.pi) - np.pi)
    assert np.max(dd) < 1e-9, "pixel centre is not a ring pixel centre"
    return np.asarray(t["start"], np.int64)[ring] + k
