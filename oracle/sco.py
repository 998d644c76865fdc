"""ctypes binding of oracle/libsco.so (argument marshalling only; see oracle/sco.h).

TEST INFRASTRUCTURE: not importable from the product package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MODE_DISC, MODE_BRUTE = 0, 1
_lib = None


def load():
    """Build (if stale) and load libsco.so."""
    global _lib
    if _lib is None:
        path = _build.build()
        lib = C.CDLL(path)
        i32, i64, dbl, vp = C.c_int, C.c_int64, C.c_double, C.c_void_p
        lib.sco_npix.argtypes = [i32, vp]
        lib.sco_ring_table.argtypes = [i32] + [vp] * 7
        lib.sco_pix2ang.argtypes = [i32, i64] + [vp] * 6
        lib.sco_kernel_eval.argtypes = [vp, i32, dbl, dbl]
        lib.sco_kernel_eval.restype = dbl
        lib.sco_kernel_eval_zoned.argtypes = [vp, i32, dbl, dbl, dbl]
        lib.sco_kernel_eval_zoned.restype = dbl
        lib.sco_convolve_zoned.argtypes = [i32, vp, i32, dbl, dbl, vp, vp, i32, i64, vp, vp, vp, i32, i32]
        lib.sco_neighbours.argtypes = [i32, dbl, i64, i32, vp, i64, vp]
        lib.sco_convolve.argtypes = [i32, vp, i32, dbl, vp, vp, i32, i64, vp, vp, vp, i32, i32]
        lib.sco_count.argtypes = [i32, dbl, i64, vp, vp, vp, i32]
        lib.sco_last_threads.restype = i32
        _lib = lib
    return _lib


def _chk(rc, what):
    if rc != 0:
        raise ValueError(f"{what} failed with oracle status {rc}")


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def npix(nside):
    out = C.c_int64(0)
    _chk(load().sco_npix(nside, C.byref(out)), "sco_npix")
    return out.value


def ring_table(nside):
    """dict of per-ring arrays (index = ring number - 1)."""
    nr = 4 * nside - 1
    t = dict(start=np.zeros(nr, np.int64), npr=np.zeros(nr, np.int32), z=np.zeros(nr),
             s=np.zeros(nr), phi0=np.zeros(nr), dphi=np.zeros(nr), shifted=np.zeros(nr, np.int32))
    _chk(load().sco_ring_table(nside, *[_ptr(t[k]) for k in
                                        ("start", "npr", "z", "s", "phi0", "dphi", "shifted")]),
         "sco_ring_table")
    return t


def pix2ang(nside, pix):
    pix = np.ascontiguousarray(pix, np.int64)
    n = pix.size
    ring, k = np.zeros(n, np.int32), np.zeros(n, np.int32)
    z, s, phi = np.zeros(n), np.zeros(n), np.zeros(n)
    _chk(load().sco_pix2ang(nside, n, _ptr(pix), _ptr(ring), _ptr(k), _ptr(z), _ptr(s), _ptr(phi)),
         "sco_pix2ang")
    return dict(ring=ring, k=k, z=z, s=s, phi=phi)


def kernel_eval(ktable, theta_max, x):
    kt = np.ascontiguousarray(ktable, np.float64)
    return load().sco_kernel_eval(_ptr(kt), kt.size, float(theta_max), float(x))


def kernel_eval_zoned(ktable, theta_max, zone_frac, x):
    kt = np.ascontiguousarray(ktable, np.float64)
    return load().sco_kernel_eval_zoned(_ptr(kt), kt.size, float(theta_max), float(zone_frac), float(x))


def neighbours(nside, theta_max, p, mode=MODE_DISC):
    lib = load()
    n = C.c_int64(0)
    _chk(lib.sco_neighbours(nside, float(theta_max), int(p), mode, None, 0, C.byref(n)),
         "sco_neighbours")
    buf = np.zeros(max(n.value, 1), np.int64)
    _chk(lib.sco_neighbours(nside, float(theta_max), int(p), mode, _ptr(buf), buf.size, C.byref(n)),
         "sco_neighbours")
    return buf[:n.value].copy()


def convolve(nside, ktable, theta_max, maps, sel=None, mode=MODE_DISC, nthreads=0,
             want_counts=True, zone_frac=None):
    """maps: sequence of B fp32 arrays (N_pix).  Returns (out[B, n_out] fp64, counts, sigs).
    zone_frac: None = uniform table in cos(theta); else the two-zone table of sco_kernel_eval_zoned."""
    lib = load()
    maps = [np.ascontiguousarray(m, np.float32) for m in maps]
    B = len(maps)
    N = npix(nside)
    for m in maps:
        if m.shape != (N,):
            raise ValueError("map has wrong shape")
    sel_a = None if sel is None else np.ascontiguousarray(sel, np.int64)
    nout = N if sel_a is None else sel_a.size
    out = np.zeros((max(B, 1), nout), np.float64)
    kt = None if ktable is None else np.ascontiguousarray(ktable, np.float64)
    in_ptrs = (C.c_void_p * max(B, 1))(*[m.ctypes.data for m in maps])
    out_ptrs = (C.c_void_p * max(B, 1))(*[out[b].ctypes.data for b in range(max(B, 1))])
    counts = np.zeros(nout, np.int32) if want_counts else None
    sigs = np.zeros(nout, np.uint64) if want_counts else None
    if zone_frac is None:
        _chk(lib.sco_convolve(nside, _ptr(kt), 0 if kt is None else kt.size, float(theta_max),
                              in_ptrs, out_ptrs, B, nout if sel_a is not None else 0, _ptr(sel_a),
                              _ptr(counts), _ptr(sigs), mode, nthreads), "sco_convolve")
    else:
        _chk(lib.sco_convolve_zoned(nside, _ptr(kt), 0 if kt is None else kt.size, float(theta_max),
                                    float(zone_frac), in_ptrs, out_ptrs, B,
                                    nout if sel_a is not None else 0, _ptr(sel_a),
                                    _ptr(counts), _ptr(sigs), mode, nthreads), "sco_convolve_zoned")
    return out[:B], counts, sigs


def count(nside, theta_max, sel=None, nthreads=0):
    lib = load()
    N = npix(nside)
    sel_a = None if sel is None else np.ascontiguousarray(sel, np.int64)
    nout = N if sel_a is None else sel_a.size
    counts, sigs = np.zeros(nout, np.int32), np.zeros(nout, np.uint64)
    _chk(lib.sco_count(nside, float(theta_max), nout if sel_a is not None else 0, _ptr(sel_a),
                       _ptr(counts), _ptr(sigs), nthreads), "sco_count")
    return counts, sigs


def last_threads():
    return load().sco_last_threads()


class Oracle:
    """Convenience holder of (nside, ktable, theta_max)."""

    def __init__(self, nside, ktable, theta_max):
        self.nside, self.theta_max = int(nside), float(theta_max)
        self.ktable = np.ascontiguousarray(ktable, np.float64)

    def convolve(self, maps, **kw):
        return convolve(self.nside, self.ktable, self.theta_max, maps, **kw)
