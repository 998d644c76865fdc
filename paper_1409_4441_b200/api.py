"""ctypes binding of libsc.so: same names as include/sc.h, marshalling only."""
import ctypes as C
import os

import numpy as np

from . import build as _build

SC_ORDER_RING, SC_ORDER_NESTED = 0, 1
SC_PATH_AUTO, SC_PATH_GENERIC = 0, 1

# every symbol include/sc.h declares
SC_K_POLAR, SC_K_SYM, SC_K_BELT, SC_K_COUNT = 0, 1, 2, 3
KERNEL_NAMES = ("generic_warp_kernel", "sym_kernel", "belt_kernel")

EXPORTS = ("sc_plan_create", "sc_plan_create_zoned", "sc_convolve", "sc_convolve_host", "sc_convolve_profile", "sc_plan_partition",
           "sc_band_partition", "sc_convolve_band", "sc_cap_rows", "sc_convolve_cap",
           "sc_plan_destroy", "sc_plan_set_path",
           "sc_plan_info", "sc_debug_neighbour_counts", "sc_neighbour_counts_static", "sc_debug_stats", "sc_debug_fma_peak", "sc_last_launch_count", "sc_plan_double_coordinate",
           "sc_status_string", "sc_last_cuda_error", "sc_version")

_lib = None


class ScError(RuntimeError):
    def __init__(self, status, what):
        l = lib()
        msg = l.sc_status_string(status).decode()
        cuda = l.sc_last_cuda_error().decode()
        super().__init__(f"{what}: {msg}" + (f" [{cuda}]" if cuda and status == 4 else ""))
        self.status = status


def lib():
    """Load libsc.so (building it with nvcc if the sources are newer).  Raises if unavailable."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if os.environ.get("SC_NO_BUILD") != "1":
            path = _build.build()
        l = C.CDLL(path)
        vp, i32, dbl = C.c_void_p, C.c_int, C.c_double
        l.sc_plan_create.argtypes = [C.POINTER(vp), i32, i32, vp, i32, dbl, i32]
        l.sc_plan_create_zoned.argtypes = [C.POINTER(vp), i32, i32, vp, i32, dbl, dbl, i32]
        l.sc_convolve.argtypes = [vp, vp, vp, i32, vp]
        l.sc_convolve_host.argtypes = [vp, vp, vp, i32]
        l.sc_convolve_profile.argtypes = [vp, vp, vp, i32, vp, vp]
        l.sc_plan_partition.argtypes = [vp, vp, vp]
        l.sc_band_partition.argtypes = [vp, i32, i32, vp, vp, vp, vp]
        l.sc_convolve_band.argtypes = [vp, i32, i32, vp, vp, i32, vp]
        l.sc_cap_rows.argtypes = [vp, i32, vp, vp]
        l.sc_convolve_cap.argtypes = [vp, i32, vp, vp, i32, vp]
        l.sc_plan_destroy.argtypes = [vp]
        l.sc_plan_set_path.argtypes = [vp, i32]
        l.sc_plan_info.argtypes = [vp, vp, vp, vp, vp]
        l.sc_debug_neighbour_counts.argtypes = [vp, vp, vp, vp]
        l.sc_neighbour_counts_static.argtypes = [vp, vp, vp, vp]
        l.sc_debug_stats.argtypes = [vp, vp, vp, vp]
        l.sc_last_launch_count.argtypes = [vp]
        l.sc_plan_double_coordinate.argtypes = [vp]
        l.sc_debug_fma_peak.argtypes = [i32, vp, vp]
        for f in ("sc_status_string", "sc_last_cuda_error", "sc_version"):
            getattr(l, f).restype = C.c_char_p
        l.sc_status_string.argtypes = [i32]
        _lib = l
    return _lib


def _chk(st, what):
    if st != 0:
        raise ScError(st, what)


def sc_version():
    return lib().sc_version().decode()


def sc_plan_create(nside, ordering, ktable, theta_max, max_batch=1):
    """-> opaque plan handle (int).  ktable: host fp64 array, K at x_i = c + i(1-c)/(n-1)."""
    kt = np.ascontiguousarray(ktable, np.float64)
    h = C.c_void_p(None)
    _chk(lib().sc_plan_create(C.byref(h), int(nside), int(ordering), kt.ctypes.data_as(C.c_void_p),
                              int(kt.size), float(theta_max), int(max_batch)), "sc_plan_create")
    return h.value


def sc_plan_create_zoned(nside, ordering, ktable, theta_max, zone_frac, max_batch=1):
    """Two-zone table (include/sc.h): ktable at the zoned nodes, zone_frac in (0, 1)."""
    kt = np.ascontiguousarray(ktable, np.float64)
    h = C.c_void_p(None)
    _chk(lib().sc_plan_create_zoned(C.byref(h), int(nside), int(ordering), kt.ctypes.data_as(C.c_void_p),
                                    int(kt.size), float(theta_max), float(zone_frac), int(max_batch)),
         "sc_plan_create_zoned")
    return h.value


def _ptr_array(ptrs):
    return (C.c_void_p * len(ptrs))(*[int(p) for p in ptrs])


def sc_convolve(plan, in_ptrs, out_ptrs, stream=0):
    """in_ptrs / out_ptrs: sequences of B device addresses (ints); stream: cudaStream_t as int."""
    if len(in_ptrs) != len(out_ptrs):
        raise ValueError("in/out batch mismatch")
    _chk(lib().sc_convolve(plan, _ptr_array(in_ptrs), _ptr_array(out_ptrs), len(in_ptrs),
                           C.c_void_p(int(stream) or None)), "sc_convolve")


def sc_convolve_host(plan, in_ptrs, out_ptrs):
    """Same with HOST addresses (end-to-end call, copies inside, synchronous)."""
    if len(in_ptrs) != len(out_ptrs):
        raise ValueError("in/out batch mismatch")
    _chk(lib().sc_convolve_host(plan, _ptr_array(in_ptrs), _ptr_array(out_ptrs), len(in_ptrs)),
         "sc_convolve_host")


def sc_convolve_profile(plan, in_ptrs, out_ptrs, stream=0):
    """Measurement only: one step with events around every kernel -> per-kernel ms (tuple of SC_K_COUNT)."""
    if len(in_ptrs) != len(out_ptrs):
        raise ValueError("in/out batch mismatch")
    ms = (C.c_float * SC_K_COUNT)()
    _chk(lib().sc_convolve_profile(plan, _ptr_array(in_ptrs), _ptr_array(out_ptrs), len(in_ptrs),
                                   C.c_void_p(int(stream) or None), ms), "sc_convolve_profile")
    return tuple(float(x) for x in ms)


def sc_plan_partition(plan):
    pr, fb = C.c_int(0), C.c_int(0)
    _chk(lib().sc_plan_partition(plan, C.byref(pr), C.byref(fb)), "sc_plan_partition")
    return dict(polar_rings=pr.value, first_belt_ring=fb.value)


def sc_band_partition(plan, world, rank):
    """-> dict(ring_lo, ring_hi, out_rows=(o0, o1, o2, o3), in_rows=(i0, i1, i2, i3)) of latitude band `rank`."""
    lo, hi = C.c_int(0), C.c_int(0)
    orow, irow = (C.c_int64 * 4)(), (C.c_int64 * 4)()
    _chk(lib().sc_band_partition(plan, int(world), int(rank), C.byref(lo), C.byref(hi), orow, irow), "sc_band_partition")
    return dict(ring_lo=lo.value, ring_hi=hi.value, out_rows=tuple(orow), in_rows=tuple(irow))


def sc_convolve_band(plan, ring_lo, ring_hi, in_ptrs, out_ptrs, stream=0):
    """sc_convolve restricted to base rings ring_lo .. ring_hi and their southern mirrors."""
    if len(in_ptrs) != len(out_ptrs):
        raise ValueError("in/out batch mismatch")
    _chk(lib().sc_convolve_band(plan, int(ring_lo), int(ring_hi), _ptr_array(in_ptrs), _ptr_array(out_ptrs),
                                len(in_ptrs), C.c_void_p(int(stream) or None)), "sc_convolve_band")


def sc_cap_rows(plan, ring_hi):
    """-> dict(out_rows=(0, o1), in_rows=(0, i1)): pixel ranges written / read by sc_convolve_cap(ring_hi)."""
    orow, irow = (C.c_int64 * 2)(), (C.c_int64 * 2)()
    _chk(lib().sc_cap_rows(plan, int(ring_hi), orow, irow), "sc_cap_rows")
    return dict(out_rows=tuple(orow), in_rows=tuple(irow))


def sc_convolve_cap(plan, ring_hi, in_ptrs, out_ptrs, stream=0):
    """North polar cap only: output rings 1 .. ring_hi, no southern mirror images (include/sc.h)."""
    if len(in_ptrs) != len(out_ptrs):
        raise ValueError("in/out batch mismatch")
    _chk(lib().sc_convolve_cap(plan, int(ring_hi), _ptr_array(in_ptrs), _ptr_array(out_ptrs), len(in_ptrs),
                               C.c_void_p(int(stream) or None)), "sc_convolve_cap")


def sc_plan_destroy(plan):
    _chk(lib().sc_plan_destroy(plan), "sc_plan_destroy")


def sc_plan_set_path(plan, path):
    _chk(lib().sc_plan_set_path(plan, int(path)), "sc_plan_set_path")


def sc_plan_info(plan):
    npix, tot, nke = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    c = C.c_double(0)
    _chk(lib().sc_plan_info(plan, C.byref(npix), C.byref(tot), C.byref(c), C.byref(nke)), "sc_plan_info")
    return dict(npix=npix.value, total_pairs=tot.value, cos_theta_max=c.value, n_knife_edge=nke.value)


def sc_debug_stats(plan):
    n, e, g = C.c_int64(0), C.c_double(0), C.c_double(0)
    _chk(lib().sc_debug_stats(plan, C.byref(n), C.byref(e), C.byref(g)), "sc_debug_stats")
    return dict(n_uncertain=n.value, max_t_err=e.value, guard_band=g.value)


def sc_debug_neighbour_counts(plan, count_ptr, sig_ptr=0, stream=0):
    _chk(lib().sc_debug_neighbour_counts(plan, C.c_void_p(int(count_ptr)), C.c_void_p(int(sig_ptr) or None),
                                         C.c_void_p(int(stream) or None)), "sc_debug_neighbour_counts")


SC_STATIC_MAX_NPIX = 196608     # include/sc.h: entries of the static device scratch (nside <= 128)


def sc_neighbour_counts_static(plan, count_ptr, sig_ptr=0, stream=0):
    """sc_debug_neighbour_counts without any allocation (static device scratch; 12 nside^2 <= SC_STATIC_MAX_NPIX)."""
    _chk(lib().sc_neighbour_counts_static(plan, C.c_void_p(int(count_ptr)), C.c_void_p(int(sig_ptr) or None),
                                          C.c_void_p(int(stream) or None)),
         f"sc_neighbour_counts_static (static scratch holds {SC_STATIC_MAX_NPIX} pixels: nside <= 128)")


def sc_debug_fma_peak(packed=True):
    """Measurement only: sustained FP32 FMA/s of the current device (FFMA2 loop if packed else scalar FFMA;
    packed = 2: FFMA2 with the operand pattern of the kernels' accumulation)."""
    v, ms = C.c_double(0), C.c_double(0)
    _chk(lib().sc_debug_fma_peak(int(packed), C.byref(v), C.byref(ms)), "sc_debug_fma_peak")
    return dict(fma_per_s=v.value, elapsed_ms=ms.value)


def sc_last_launch_count(plan):
    return lib().sc_last_launch_count(plan)


def sc_plan_double_coordinate(plan):
    return lib().sc_plan_double_coordinate(plan)


class Plan:
    """Convenience owner of a plan for torch users: maps are torch CUDA fp32 tensors."""

    def __init__(self, nside, ktable, theta_max, max_batch=1, ordering=SC_ORDER_RING, zone_frac=None):
        self.nside = int(nside)
        self.npix = 12 * self.nside * self.nside
        if zone_frac is None:
            self.handle = sc_plan_create(nside, ordering, ktable, theta_max, max_batch)
        else:
            self.handle = sc_plan_create_zoned(nside, ordering, ktable, theta_max, zone_frac, max_batch)

    def close(self):
        if getattr(self, "handle", None):
            sc_plan_destroy(self.handle)
            self.handle = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def info(self):
        d = sc_plan_info(self.handle)
        d.update(sc_debug_stats(self.handle))
        d["double_coordinate"] = sc_plan_double_coordinate(self.handle)
        return d

    def set_path(self, path):
        sc_plan_set_path(self.handle, path)

    def convolve(self, maps, out=None):
        """maps: list of CUDA fp32 tensors (N_pix) -> list of output tensors; async on the current
        torch stream."""
        import torch
        for m in maps:
            if not (m.is_cuda and m.dtype == torch.float32 and m.is_contiguous() and m.numel() == self.npix):
                raise ValueError("maps must be contiguous CUDA fp32 tensors of N_pix elements")
        if out is None:
            out = [torch.empty_like(m) for m in maps]
        sc_convolve(self.handle, [m.data_ptr() for m in maps], [o.data_ptr() for o in out],
                    torch.cuda.current_stream().cuda_stream)
        return out

    def convolve_profile(self, maps, out):
        """Measurement only: one step, returns {kernel name: device ms} (synchronises the stream)."""
        import torch
        ms = sc_convolve_profile(self.handle, [m.data_ptr() for m in maps], [o.data_ptr() for o in out],
                                 torch.cuda.current_stream().cuda_stream)
        return dict(zip(KERNEL_NAMES, ms))

    def partition(self):
        return sc_plan_partition(self.handle)

    def band(self, world, rank):
        return sc_band_partition(self.handle, world, rank)

    def convolve_band(self, ring_lo, ring_hi, maps, out):
        """Band version of convolve(): reads/writes only the band's rows of the full-size tensors."""
        import torch
        sc_convolve_band(self.handle, ring_lo, ring_hi, [m.data_ptr() for m in maps], [o.data_ptr() for o in out],
                         torch.cuda.current_stream().cuda_stream)
        return out

    def cap_rows(self, ring_hi):
        return sc_cap_rows(self.handle, ring_hi)

    def convolve_cap(self, ring_hi, maps, out):
        """North polar cap only: maps / out are CUDA fp32 tensors holding at least the rows of cap_rows(ring_hi)."""
        import torch
        sc_convolve_cap(self.handle, ring_hi, [m.data_ptr() for m in maps], [o.data_ptr() for o in out],
                        torch.cuda.current_stream().cuda_stream)
        return out

    def convolve_host(self, maps, out=None):
        """maps: list of host fp32 numpy arrays or CPU tensors (N_pix) -> list of numpy arrays."""
        arrs = [np.ascontiguousarray(m, np.float32) if not hasattr(m, "data_ptr") else m for m in maps]
        if out is None:
            out = [np.empty(self.npix, np.float32) for _ in arrs]
        ptr = lambda a: a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        sc_convolve_host(self.handle, [ptr(a) for a in arrs], [ptr(o) for o in out])
        return out

    def neighbour_counts(self, want_sig=True):
        import torch
        cnt = torch.empty(self.npix, dtype=torch.int32, device="cuda")
        sig = torch.empty(self.npix, dtype=torch.int64, device="cuda") if want_sig else None
        sc_debug_neighbour_counts(self.handle, cnt.data_ptr(), sig.data_ptr() if want_sig else 0,
                                  torch.cuda.current_stream().cuda_stream)
        return cnt, sig
