/*
 * sco.cpp -- the ORACLE: a plain, slow, fp64 CPU statement of the real-space spherical
 * convolution on a HEALPix RING map.  TEST INFRASTRUCTURE (see sco.h).  Build:
 *     g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -fPIC -shared oracle/sco.cpp -o oracle/libsco.so
 * -ffp-contract=off matters: the inclusion test below is specified without FMA contraction
 * (reading R4).
 *
 * Definition followed (BASELINE.json north_star; "convolving a real or synthetic map
 * with a radial kernel", PAPER.md:33 real-space kernel truncated at theta_cut, PAPER.md:66 the
 * real-space portion applied on the GPU):
 *     out(p) = Omega_pix * SUM_{q : theta_pq <= theta_max} K(cos theta_pq) * m(q),
 *     Omega_pix = 4 pi / N_pix.
 * HEALPix is only cited by the paper; the RING scheme of Gorski et al. 2005 is
 * restated here from its defining formulas:
 *   rings i = 1 .. 4N-1 north to south; pixels-per-quadrant i_p = i (i < N), N (N <= i <= 3N),
 *   4N-i (i > 3N); ring length n_i = 4 i_p;
 *   z_i = 1 - i^2/(3N^2) (north cap), (2N-i) 2/(3N) (belt), -(1 - (4N-i)^2/(3N^2)) (south cap);
 *   first pixel of ring: 2i(i-1) (north cap), 2N(N-1) + (i-N) 4N (belt), N_pix - 2i'(i'+1), i' = 4N-i;
 *   phi of pixel k (0-based) = phi0_i + k dphi_i, dphi_i = 2 pi / n_i, phi0_i = dphi_i / 2 except
 *   phi0_i = 0 on belt rings with (i - N) odd.
 * Canonical fp64 evaluation order (this file is the authority on inclusion decisions):
 *   s = sqrt((1.0 - z) * (1.0 + z));  phi = phi0 + k * dphi;
 *   dot = z_p * z_q + (s_p * s_q) * cos(phi_p - phi_q);      included  <=>  dot >= cos(theta_max).
 */
#include "sco.h"
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Ring {
    int64_t start;
    int32_t n;
    int32_t shifted;
    double z, s, phi0, dphi;
};

int g_last_threads = 1;

/* ring i (1-based) of an Nside = N map */
Ring ring_geom(int N, int i) {
    Ring R;
    const int64_t npix = 12LL * N * N;
    int64_t ip;
    if (i < N) {
        ip = i;
        R.z = 1.0 - (double)((int64_t)i * i) / (3.0 * N * N);
        R.start = 2LL * i * (i - 1);
        R.shifted = 0;
    } else if (i <= 3 * N) {
        ip = N;
        R.z = (2.0 * N - i) * 2.0 / (3.0 * N);
        R.start = 2LL * N * (N - 1) + (int64_t)(i - N) * 4LL * N;
        R.shifted = ((i - N) & 1) ? 1 : 0;
    } else {
        const int64_t ii = 4LL * N - i;
        ip = ii;
        R.z = -(1.0 - (double)(ii * ii) / (3.0 * N * N));
        R.start = npix - 2LL * ii * (ii + 1);
        R.shifted = 0;
    }
    R.n = (int32_t)(4 * ip);
    R.s = std::sqrt((1.0 - R.z) * (1.0 + R.z));
    R.dphi = 2.0 * M_PI / R.n;
    R.phi0 = R.shifted ? 0.0 : 0.5 * R.dphi;
    return R;
}

std::vector<Ring> all_rings(int N) {
    std::vector<Ring> v(4 * N - 1);
    for (int i = 1; i <= 4 * N - 1; ++i) v[i - 1] = ring_geom(N, i);
    return v;
}

/* ring (1-based) that holds RING pixel p: the unique i with start_i <= p < start_i + n_i */
int ring_of_pixel(int N, int64_t p) {
    const int64_t npix = 12LL * N * N, ncap = 2LL * N * (N - 1);
    if (p < ncap) {                       /* north cap: 2i(i-1) <= p < 2i(i+1) */
        int64_t i = (int64_t)((1.0 + std::sqrt(1.0 + 2.0 * (double)p)) / 2.0);
        while (i > 1 && 2 * i * (i - 1) > p) --i;
        while (2 * i * (i + 1) <= p) ++i;
        return (int)i;
    }
    if (p < npix - ncap) return (int)(N + (p - ncap) / (4LL * N));
    const int64_t pm = npix - 1 - p;      /* mirror into the north cap numbering */
    int64_t i = (int64_t)((1.0 + std::sqrt(1.0 + 2.0 * (double)pm)) / 2.0);
    while (i > 1 && 2 * i * (i - 1) > pm) --i;
    while (2 * i * (i + 1) <= pm) ++i;
    return (int)(4LL * N - i);
}

inline double pix_phi(const Ring &R, int64_t k) { return R.phi0 + (double)k * R.dphi; }

/* the canonical inclusion quantity */
inline double pair_dot(double zp, double sp, double phip, double zq, double sq, double phiq) {
    return zp * zq + (sp * sq) * std::cos(phip - phiq);
}

/* Kt(x): SURVEY.md 8c.3 / DESIGN.md R5.  x_i = c + i (1-c)/(n-1); clamp x to <= 1. */
inline double kernel_eval(const double *T, int n, double c, double x) {
    if (x > 1.0) x = 1.0;
    const double t = (x - c) / (1.0 - c) * (double)(n - 1);
    long i = (long)std::floor(t);
    if (i < 0) i = 0;
    if (i > n - 2) i = n - 2;
    const double f = t - (double)i;
    return T[i] + f * (T[i + 1] - T[i]);
}

/* Two-zone table (reading R11 of PAPER.md:106 "half the available interpolation nodes within the
 * first 1/16 of the available support"): n nodes (n even, >= 4), h = n/2, x1 = cos(zone_frac * theta_max).
 * Nodes i = 0 .. h-1 (outer zone):  x_i = c + i (x1 - c) / h;  nodes i = h .. n-1 (inner zone, next to
 * theta = 0):  x_i = x1 + (i - h)(1 - x1) / (h - 1).  Linear interpolation in x between adjacent nodes. */
inline double kernel_eval_zoned(const double *T, int n, double c, double x1, double x) {
    if (x > 1.0) x = 1.0;
    const int h = n / 2;
    long i;
    double f;
    if (x >= x1) {
        const double s = (x - x1) / (1.0 - x1) * (double)(h - 1);
        i = (long)std::floor(s);
        if (i < 0) i = 0;
        if (i > h - 2) i = h - 2;
        f = s - (double)i;
        i += h;
    } else {
        const double s = (x - c) / (x1 - c) * (double)h;
        i = (long)std::floor(s);
        if (i < 0) i = 0;
        if (i > h - 1) i = h - 1;
        f = s - (double)i;
    }
    return T[i] + f * (T[i + 1] - T[i]);
}

inline int64_t floordiv(int64_t a, int64_t b) { int64_t q = a / b, r = a % b; return (r != 0 && ((r < 0) != (b < 0))) ? q - 1 : q; }
inline int64_t posmod(int64_t a, int64_t n) { int64_t r = a % n; return r < 0 ? r + n : r; }

/*
 * Ring-range disc query: candidate pixels of ring Rq for an output pixel at (zp, sp, phip).
 * Returns false if the ring cannot hold a neighbour.  Otherwise [k_first, k_first + k_count) is a
 * superset (in-ring indices, to be taken mod n) of the included arc, padded by PAD pixels per side;
 * the caller applies the canonical test to every candidate.  (Inclusion along a ring is one
 * contiguous arc centred on phi_p because cos(dphi) is monotone in |dphi| on [0, pi].)
 */
const int PAD = 2;
inline bool ring_candidates(const Ring &Rq, double zp, double sp, double phip, double c,
                            int64_t &k_first, int64_t &k_count) {
    const double ss = sp * Rq.s;
    const double rho = (c - zp * Rq.z) / ss;      /* need cos(dphi) >= rho */
    if (rho > 1.0 + 1e-9) return false;
    double H;
    if (rho <= -1.0) H = M_PI; else H = std::acos(rho > 1.0 ? 1.0 : rho);
    const double klo = (phip - H - Rq.phi0) / Rq.dphi, khi = (phip + H - Rq.phi0) / Rq.dphi;
    const int64_t a = (int64_t)std::floor(klo) - PAD, b = (int64_t)std::ceil(khi) + PAD;
    if (b - a + 1 >= Rq.n) { k_first = 0; k_count = Rq.n; }
    else { k_first = a; k_count = b - a + 1; }
    return true;
}

/* rings that can hold a neighbour of a point on ring ip (1-based): contiguous interval around ip */
inline void ring_interval(const std::vector<Ring> &R, int ip, double c, int &lo, int &hi) {
    const int nr = (int)R.size();
    const Ring &P = R[ip - 1];
    lo = ip; hi = ip;
    /* closest approach of two rings is at dphi = 0: cos(theta - theta') = z z' + s s'.  1e-9 slack,
       then one more ring, keeps the interval a strict superset; every candidate is tested anyway. */
    while (lo > 1 && P.z * R[lo - 2].z + P.s * R[lo - 2].s >= c - 1e-9) --lo;
    while (hi < nr && P.z * R[hi].z + P.s * R[hi].s >= c - 1e-9) ++hi;
    if (lo > 1) --lo;
    if (hi < nr) ++hi;
}

struct Acc {          /* per-output accumulators */
    int64_t count = 0;
    uint64_t sig = 0;
};

/* one output pixel, disc-query mode */
template <class F> inline void visit_disc(int N, const std::vector<Ring> &R, double c, int64_t p, F &&f) {
    const int ip = ring_of_pixel(N, p);
    const Ring &P = R[ip - 1];
    const double phip = pix_phi(P, p - P.start);
    int lo, hi; ring_interval(R, ip, c, lo, hi);
    for (int iq = lo; iq <= hi; ++iq) {
        const Ring &Q = R[iq - 1];
        int64_t k0, kc;
        if (!ring_candidates(Q, P.z, P.s, phip, c, k0, kc)) continue;
        for (int64_t j = 0; j < kc; ++j) {
            const int64_t k = posmod(k0 + j, Q.n);
            const double d = pair_dot(P.z, P.s, phip, Q.z, Q.s, pix_phi(Q, k));
            if (d >= c) f(Q.start + k, d);
        }
    }
}

/* one output pixel, brute force: every pixel of the sphere */
template <class F> inline void visit_brute(int N, const std::vector<Ring> &R, double c, int64_t p, F &&f) {
    const int ip = ring_of_pixel(N, p);
    const Ring &P = R[ip - 1];
    const double phip = pix_phi(P, p - P.start);
    for (size_t r = 0; r < R.size(); ++r) {
        const Ring &Q = R[r];
        for (int64_t k = 0; k < Q.n; ++k) {
            const double d = pair_dot(P.z, P.s, phip, Q.z, Q.s, pix_phi(Q, k));
            if (d >= c) f(Q.start + k, d);
        }
    }
}

int resolve_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    return nthreads;
}

}  // namespace

extern "C" {

int sco_last_threads(void) { return g_last_threads; }

int sco_npix(int nside, int64_t *npix) {
    if (nside < 1 || !npix) return SCO_ERR_ARG;
    *npix = 12LL * nside * nside;
    return SCO_OK;
}

int sco_ring_table(int nside, int64_t *start, int32_t *npr, double *z, double *s,
                   double *phi0, double *dphi, int32_t *shifted) {
    if (nside < 1) return SCO_ERR_ARG;
    for (int i = 1; i <= 4 * nside - 1; ++i) {
        const Ring R = ring_geom(nside, i);
        if (start) start[i - 1] = R.start;
        if (npr) npr[i - 1] = R.n;
        if (z) z[i - 1] = R.z;
        if (s) s[i - 1] = R.s;
        if (phi0) phi0[i - 1] = R.phi0;
        if (dphi) dphi[i - 1] = R.dphi;
        if (shifted) shifted[i - 1] = R.shifted;
    }
    return SCO_OK;
}

int sco_pix2ang(int nside, int64_t n, const int64_t *pix, int32_t *ring, int32_t *k_in_ring,
                double *z, double *s, double *phi) {
    if (nside < 1 || n < 0 || (!pix && n > 0)) return SCO_ERR_ARG;
    const int64_t npix = 12LL * nside * nside;
    for (int64_t j = 0; j < n; ++j) {
        if (pix[j] < 0 || pix[j] >= npix) return SCO_ERR_ARG;
        const int i = ring_of_pixel(nside, pix[j]);
        const Ring R = ring_geom(nside, i);
        const int64_t k = pix[j] - R.start;
        if (ring) ring[j] = i;
        if (k_in_ring) k_in_ring[j] = (int32_t)k;
        if (z) z[j] = R.z;
        if (s) s[j] = R.s;
        if (phi) phi[j] = pix_phi(R, k);
    }
    return SCO_OK;
}

double sco_kernel_eval(const double *ktable, int n_table, double theta_max, double x) {
    return kernel_eval(ktable, n_table, std::cos(theta_max), x);
}

double sco_kernel_eval_zoned(const double *ktable, int n_table, double theta_max, double zone_frac, double x) {
    return kernel_eval_zoned(ktable, n_table, std::cos(theta_max), std::cos(zone_frac * theta_max), x);
}

int sco_neighbours(int nside, double theta_max, int64_t p, int mode,
                   int64_t *buf, int64_t cap, int64_t *n_out) {
    if (nside < 1 || !n_out || !(theta_max > 0.0)) return SCO_ERR_ARG;
    const int64_t npix = 12LL * nside * nside;
    if (p < 0 || p >= npix) return SCO_ERR_ARG;
    const std::vector<Ring> R = all_rings(nside);
    const double c = std::cos(theta_max);
    int64_t cnt = 0;
    auto f = [&](int64_t q, double) { if (buf && cnt < cap) buf[cnt] = q; ++cnt; };
    if (mode == SCO_MODE_BRUTE) visit_brute(nside, R, c, p, f); else visit_disc(nside, R, c, p, f);
    *n_out = cnt;
    return SCO_OK;
}

static int convolve_impl(int nside, const double *ktable, int n_table, double theta_max, double zone_frac,
                         const float *const *in, double *const *out, int B,
                         int64_t n_sel, const int64_t *sel,
                         int32_t *counts, uint64_t *sigs, int mode, int nthreads) {
    if (nside < 1 || B < 0 || !(theta_max > 0.0) || theta_max > M_PI) return SCO_ERR_ARG;
    const bool zoned = zone_frac > 0.0;
    if (zoned && (zone_frac >= 1.0 || n_table < 4 || (n_table & 1))) return SCO_ERR_ARG;
    const double x1 = zoned ? std::cos(zone_frac * theta_max) : 0.0;
    if (B > 0 && (!ktable || n_table < 2 || !in || !out)) return SCO_ERR_ARG;
    if (B > 16) return SCO_ERR_ARG;
    const int64_t npix = 12LL * nside * nside;
    const int64_t nout = sel ? n_sel : npix;
    if (sel) for (int64_t j = 0; j < n_sel; ++j) if (sel[j] < 0 || sel[j] >= npix) return SCO_ERR_ARG;
    const std::vector<Ring> R = all_rings(nside);
    const double c = std::cos(theta_max);
    const double omega = 4.0 * M_PI / (double)npix;
    nthreads = resolve_threads(nthreads);
    g_last_threads = nthreads;
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads)
    for (int64_t j = 0; j < nout; ++j) {
        const int64_t p = sel ? sel[j] : j;
        double sum[16];
        for (int b = 0; b < B; ++b) sum[b] = 0.0;
        int64_t cnt = 0; uint64_t sg = 0;
        auto f = [&](int64_t q, double d) {
            ++cnt; sg += (uint64_t)q;
            if (B > 0) {
                const double K = zoned ? kernel_eval_zoned(ktable, n_table, c, x1, d) : kernel_eval(ktable, n_table, c, d);
                for (int b = 0; b < B; ++b) sum[b] += K * (double)in[b][q];
            }
        };
        if (mode == SCO_MODE_BRUTE) visit_brute(nside, R, c, p, f); else visit_disc(nside, R, c, p, f);
        for (int b = 0; b < B; ++b) out[b][j] = omega * sum[b];
        if (counts) counts[j] = (int32_t)cnt;
        if (sigs) sigs[j] = sg;
    }
    return SCO_OK;
}

int sco_convolve(int nside, const double *ktable, int n_table, double theta_max,
                 const float *const *in, double *const *out, int B,
                 int64_t n_sel, const int64_t *sel,
                 int32_t *counts, uint64_t *sigs, int mode, int nthreads) {
    return convolve_impl(nside, ktable, n_table, theta_max, 0.0, in, out, B, n_sel, sel, counts, sigs, mode, nthreads);
}

int sco_convolve_zoned(int nside, const double *ktable, int n_table, double theta_max, double zone_frac,
                       const float *const *in, double *const *out, int B,
                       int64_t n_sel, const int64_t *sel,
                       int32_t *counts, uint64_t *sigs, int mode, int nthreads) {
    if (!(zone_frac > 0.0)) return SCO_ERR_ARG;
    return convolve_impl(nside, ktable, n_table, theta_max, zone_frac, in, out, B, n_sel, sel, counts, sigs, mode, nthreads);
}

int sco_count(int nside, double theta_max, int64_t n_sel, const int64_t *sel,
              int32_t *counts, uint64_t *sigs, int nthreads) {
    if (nside < 1 || !(theta_max > 0.0) || theta_max > M_PI) return SCO_ERR_ARG;
    const int64_t npix = 12LL * nside * nside;
    const int64_t nout = sel ? n_sel : npix;
    if (sel) for (int64_t j = 0; j < n_sel; ++j) if (sel[j] < 0 || sel[j] >= npix) return SCO_ERR_ARG;
    const std::vector<Ring> R = all_rings(nside);
    const double c = std::cos(theta_max);
    nthreads = resolve_threads(nthreads);
    g_last_threads = nthreads;
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthreads)
    for (int64_t j = 0; j < nout; ++j) {
        const int64_t p = sel ? sel[j] : j;
        const int ip = ring_of_pixel(nside, p);
        const Ring &P = R[ip - 1];
        const double phip = pix_phi(P, p - P.start);
        int lo, hi; ring_interval(R, ip, c, lo, hi);
        int64_t cnt = 0; uint64_t sg = 0;
        for (int iq = lo; iq <= hi; ++iq) {
            const Ring &Q = R[iq - 1];
            int64_t k0, kc;
            if (!ring_candidates(Q, P.z, P.s, phip, c, k0, kc)) continue;
            auto inc = [&](int64_t k) {
                return pair_dot(P.z, P.s, phip, Q.z, Q.s, pix_phi(Q, posmod(k, Q.n))) >= c;
            };
            if (kc >= Q.n) {            /* whole ring is candidate: test every pixel */
                for (int64_t k = 0; k < Q.n; ++k) if (inc(k)) { ++cnt; sg += (uint64_t)(Q.start + k); }
                continue;
            }
            /* candidates [k0, k0+kc) hold the whole arc with PAD excluded pixels on each side:
               walk inwards from both ends to the first included pixel. */
            int64_t a = k0, b = k0 + kc - 1;
            while (a <= b && !inc(a)) ++a;
            while (b >= a && !inc(b)) --b;
            for (int64_t k = a; k <= b; ++k) { ++cnt; sg += (uint64_t)(Q.start + posmod(k, Q.n)); }
        }
        if (counts) counts[j] = (int32_t)cnt;
        if (sigs) sigs[j] = sg;
    }
    return SCO_OK;
}

}  // extern "C"
