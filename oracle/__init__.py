"""fp64 CPU oracle for the real-space spherical convolution (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_1409_4441_b200 and shares no code with it.
"""
from .sco import (Oracle, load, npix, ring_table, pix2ang, kernel_eval, kernel_eval_zoned, neighbours,  # noqa: F401
                  convolve, count, last_threads, MODE_DISC, MODE_BRUTE)
