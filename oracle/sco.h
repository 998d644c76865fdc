/*
 * sco.h -- C ABI of the ORACLE ("sco" = spherical-convolution oracle).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.  It shares no code,
 * header, table or constant with the CUDA path under paper_1409_4441_b200/ and neither side
 * includes or imports the other.
 *
 * What it computes (BASELINE.json north_star; the operation the paper calls "convolving a ...
 * map with a radial kernel" applied in real space with a kernel truncated at theta_cut,
 * PAPER.md:11, :33 Eq. 1 context, :66 section 2):
 *
 *     out[b][p] = Omega_pix * SUM_{q : dot(p,q) >= cos(theta_max)} Kt(dot(p,q)) * (double) m_b[q]
 *
 * with Omega_pix = 4 pi / N_pix, on a HEALPix RING-ordered map (the paper only cites HEALPix,
 * PAPER.md:76, :216; the standard ring scheme is restated in sco.cpp, reading R2).
 * Everything is plain fp64, one pair at a time, no blocking/fusion/reordering.
 *
 * Pins: tests/test_oracle_*.py (-m "not gpu"): explicit Nside 1 / 2 layouts, brute force vs disc
 * query, exact pair totals, identity limit, constant map -> b_0, zonal eigenfunctions -> b_l,
 * linearity, operator symmetry; two-zone table: equals the uniform table when the zones have equal
 * spacing, exact for kernels linear in x, node values reproduced.  Nothing here is "parity unpinned" except where DESIGN.md says so.
 */
#ifndef SCO_H
#define SCO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { SCO_OK = 0, SCO_ERR_ARG = 1, SCO_ERR_ALLOC = 2 };
enum { SCO_MODE_DISC = 0, SCO_MODE_BRUTE = 1 };

/* N_pix = 12 nside^2.  nside >= 1 (any integer, RING needs no power of two). */
int sco_npix(int nside, int64_t *npix);

/* Ring tables, rings i = 1 .. 4*nside-1 stored at index i-1 (all arrays length 4*nside-1).
 * start: index of the ring's first pixel; npr: pixels in the ring; z = cos(colatitude);
 * s = sin(colatitude); phi of pixel k (0-based in ring) = phi0 + k * dphi; shifted = 1 on belt
 * rings whose first pixel sits at phi = 0. Any output pointer may be NULL. */
int sco_ring_table(int nside, int64_t *start, int32_t *npr, double *z, double *s,
                   double *phi0, double *dphi, int32_t *shifted);

/* RING pixel index -> ring number (1-based), index in ring, z, s, phi.  Outputs may be NULL. */
int sco_pix2ang(int nside, int64_t n, const int64_t *pix, int32_t *ring, int32_t *k_in_ring,
                double *z, double *s, double *phi);

/* Linear-interpolated kernel table Kt(x) of SURVEY.md 8c.3 / DESIGN.md reading R5:
 * nodes x_i = c + i (1-c)/(n-1), c = cos(theta_max). */
double sco_kernel_eval(const double *ktable, int n_table, double theta_max, double x);

/* Two-zone table (reading R11): n_table even >= 4, h = n_table / 2,
 * x1 = cos(zone_frac * theta_max), 0 < zone_frac < 1.  Nodes i < h: x_i = c + i (x1 - c) / h (outer zone);
 * nodes i >= h: x_i = x1 + (i - h)(1 - x1) / (h - 1) (inner zone: half the nodes next to theta = 0).
 * Linear interpolation in x between adjacent nodes. */
double sco_kernel_eval_zoned(const double *ktable, int n_table, double theta_max, double zone_frac, double x);

/* Neighbour list of one output pixel, ascending ring then ascending in-ring order of visit.
 * buf may be NULL (count only). Returns the count in *n_out (even if > cap). */
int sco_neighbours(int nside, double theta_max, int64_t p, int mode,
                   int64_t *buf, int64_t cap, int64_t *n_out);

/* The convolution.  in[b]: N_pix fp32 values.  If sel == NULL every pixel is an output and
 * out[b] has N_pix doubles; otherwise out[b][j] (and counts[j], sigs[j]) refer to pixel sel[j],
 * j < n_sel.  counts = number of neighbours, sigs = sum of neighbour pixel indices (uint64).
 * counts / sigs / out may be NULL (B may be 0 for a count-only pass that still tests every pair).
 * mode: SCO_MODE_DISC (ring-range disc query, every candidate tested) or SCO_MODE_BRUTE
 * (every pixel of the sphere tested; tiny nside only).  nthreads <= 0: all cores. */
int sco_convolve(int nside, const double *ktable, int n_table, double theta_max,
                 const float *const *in, double *const *out, int B,
                 int64_t n_sel, const int64_t *sel,
                 int32_t *counts, uint64_t *sigs, int mode, int nthreads);

/* The same convolution with the two-zone table of sco_kernel_eval_zoned. */
int sco_convolve_zoned(int nside, const double *ktable, int n_table, double theta_max, double zone_frac,
                       const float *const *in, double *const *out, int B,
                       int64_t n_sel, const int64_t *sel,
                       int32_t *counts, uint64_t *sigs, int mode, int nthreads);

/* Count-only pass that locates the two ends of every (pixel, ring) run with the same fp64 test
 * instead of testing every interior pixel (uses: inclusion along a ring is one contiguous arc).
 * Pinned against sco_convolve's exhaustive counts in tests.  sel as above. */
int sco_count(int nside, double theta_max, int64_t n_sel, const int64_t *sel,
              int32_t *counts, uint64_t *sigs, int nthreads);

/* threads the last parallel call used */
int sco_last_threads(void);

#ifdef __cplusplus
}
#endif
#endif
