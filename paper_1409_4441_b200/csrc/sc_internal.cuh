// sc_internal.cuh -- structures and device helpers shared by the kernels of libsc (product code;
// shares nothing with oracle/).  See include/sc.h for the operation and DESIGN.md for the design.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sc {

constexpr int kMaxB = 4;          // maps per launch (larger batches are chunked by the host)
constexpr int kTabPad = 64;       // zero entries appended to the device table (t clamps to tmax+1)

// Device view of a plan.  Passed to kernels by value.
struct Dev {
    int nside, nrings, npix, ncap;        // ncap = 2 N (N-1): pixels in one polar cap (rings 1..N-1)
    int ntab;                             // n: table nodes
    float tmax;                           // n-1: table coordinate of theta_max
    float eps;                            // guard half-width in table cells: |t - tmax| <= eps -> fp64 decision
    float omega;                          // 4 pi / N_pix
    double c;                             // cos(theta_max), host libm
    double scale;                         // (n-1)/(1-c): t = (1 - dot) * scale
    double ke_band;                       // |dot - c| <= ke_band -> knife-edge (host decides)
    // ring tables, index = ring number - 1, rings 1 .. 4N-1
    const double *z, *s, *phi0, *dphi;    // canonical fp64 geometry (R4)
    const int *start, *npr;               // first pixel, pixels in ring
    const int *rlo, *rhi;                 // candidate input-ring interval (1-based, inclusive)
    // device interpolation table: K(t) = tab[i].x + t * tab[i].y for t in [i, i+1), t = (1-dot)*scale
    // (two-zone plans: K = tab[i].x + (tau - i) tab[i].y and tabh[i].x + (tau - i - 1/2) tabh[i].y)
    const float2 *tab;
    // same cells for the half-cell-shifted coordinate t' = t - 1/2 (fast kernel: round(t') = floor(t)):
    // K(t) = tabh[i].x + t' * tabh[i].y
    const float2 *tabh;
    // knife-edge overrides decided on the host, sorted by key = p * npix + q
    const unsigned long long *ke_key;
    const unsigned char *ke_in;
    int n_ke;
    // two-zone table (R11): the lookup coordinate is tau = min(z_alpha t, z_beta + z_gamma t), t = (1-dot) scale
    int zoned, z_hm1;                     // z_hm1 = n/2 - 1: cells of the inner zone
    float z_alpha, z_gamma, z_t1g;        // inner zone: tau = z_alpha t; outer zone: tau = z_hm1 + z_gamma t - z_t1g
    // steep tables: the table coordinate of every pair is formed in fp64
    // and split into cell + position in the cell; the tables are then in the cell-local form of the two-zone mode
    int hp;
};

// 1 - cos d for |d| <= pi in fp64: 2 sin^2(d/2) (generic kernels, any azimuth difference)
__device__ __forceinline__ double one_minus_cos_f64(double d) {
    const double sh = sin(0.5 * d);
    return 2.0 * sh * sh;
}
// ... and for |d| <= 0.9 rad by its even series through d^16 (next term < 1e-14 relative): the fast kernels
__device__ __forceinline__ double one_minus_cos_poly_f64(double d) {
    const double y = d * d;
    double p = -1.0 / 20922789888000.0;                  // 16!
    p = fma(y, p, 1.0 / 87178291200.0);                  // 14!
    p = fma(y, p, -1.0 / 479001600.0);                   // 12!
    p = fma(y, p, 1.0 / 3628800.0);                      // 10!
    p = fma(y, p, -1.0 / 40320.0);
    p = fma(y, p, 1.0 / 720.0);
    p = fma(y, p, -1.0 / 24.0);
    p = fma(y, p, 0.5);
    return y * p;
}

// Audit outputs (plan creation / debug only)
struct Audit {
    unsigned long long *total_pairs;      // sum of counts
    unsigned long long *n_uncertain;      // pairs decided in fp64
    unsigned int *max_t_err_bits;         // max |t32 - t64| as float bits
    unsigned long long *ke_list;          // recorded knife-edge pairs: key | (gpu verdict << 63)
    unsigned int *ke_count;
    unsigned int ke_cap;
};

struct Maps {
    const float *in[kMaxB];
    float *out[kMaxB];
};

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------

// ring (1-based) and in-ring index of RING pixel p
__device__ __forceinline__ int ring_of_pixel(const Dev &P, int p, int &k) {
    const int N = P.nside;
    int ring;
    if (p < P.ncap) {
        int i = (int)(0.5 * (1.0 + sqrt(1.0 + 2.0 * (double)p)));
        while (i > 1 && 2 * i * (i - 1) > p) --i;
        while (2 * i * (i + 1) <= p) ++i;
        ring = i;
    } else if (p < P.npix - P.ncap) {
        ring = N + (p - P.ncap) / (4 * N);
    } else {
        const int pm = P.npix - 1 - p;
        int i = (int)(0.5 * (1.0 + sqrt(1.0 + 2.0 * (double)pm)));
        while (i > 1 && 2 * i * (i - 1) > pm) --i;
        while (2 * i * (i + 1) <= pm) ++i;
        ring = 4 * N - i;
    }
    k = p - P.start[ring - 1];
    return ring;
}

// The canonical fp64 inclusion quantity, R4: every operation individually rounded
// (no FMA contraction), phi = phi0 + k*dphi with k the in-ring index in [0, n).
__device__ __forceinline__ double canonical_dot(const Dev &P, int rp, int kp, int rq, int kq) {
    const double phip = __dadd_rn(P.phi0[rp - 1], __dmul_rn((double)kp, P.dphi[rp - 1]));
    const double phiq = __dadd_rn(P.phi0[rq - 1], __dmul_rn((double)kq, P.dphi[rq - 1]));
    const double cd = cos(__dsub_rn(phip, phiq));
    return __dadd_rn(__dmul_rn(P.z[rp - 1], P.z[rq - 1]),
                     __dmul_rn(__dmul_rn(P.s[rp - 1], P.s[rq - 1]), cd));
}

// Two-zone table: cell j and position f in [0, 1] inside it for table coordinate t (0 <= t <= tmax).  The
// outer-zone coordinate is formed relative to the zone start so that pairs just outside the inner zone, where
// the kernel is steep, keep full fp32 resolution (adding the cell offset first would cost 3 digits).
__device__ __forceinline__ void zoned_cell(const Dev &P, float t, int &j, float &f) {
    const float w1 = t * P.z_alpha, w2 = fmaf(t, P.z_gamma, -P.z_t1g);
    const bool outer = w2 + (float)P.z_hm1 < w1;
    const float w = fmaxf(outer ? w2 : w1, 0.f);
    const int off = outer ? P.z_hm1 : 0;
    int i = (int)w;
    if (i + off > P.ntab - 2) i = P.ntab - 2 - off;
    j = i + off;
    f = w - (float)i;
}

// The symmetric images of a pair (rotations by pi/2, z -> -z, the reflection phi -> pi/2 - phi) have the same z z' and
// s s' bit for bit and azimuth differences that agree up to the rounding of phi0 + k dphi (a few 1e-16 rad), so their
// canonical dots differ by less than 1e-14.  If one image is further than this from cos(theta_max), all images share its
// verdict and need not be evaluated one by one (the guard band is ~3e-10 wide in these units: 1 pair in 30 goes on).
constexpr double kImageMargin = 1e-11;

// Exact decision for one pair (slow path).  If `au` is given the pair is also audited.
static __device__ __noinline__ bool exact_included(const Dev &P, int rp, int kp, int rq, int kq, float t32,
                                            const Audit *au) {
    const double dot = canonical_dot(P, rp, kp, rq, kq);
    bool in = dot >= P.c;
    const bool knife = fabs(dot - P.c) <= P.ke_band;
    if (knife) {
        const unsigned long long key =
            (unsigned long long)(P.start[rp - 1] + kp) * (unsigned long long)P.npix +
            (unsigned long long)(P.start[rq - 1] + kq);
        int lo = 0, hi = P.n_ke - 1;
        while (lo <= hi) {                 // host verdicts win
            const int mid = (lo + hi) >> 1;
            const unsigned long long km = P.ke_key[mid];
            if (km == key) { in = P.ke_in[mid] != 0; break; }
            if (km < key) lo = mid + 1; else hi = mid - 1;
        }
        if (au && au->ke_list) {
            const unsigned int slot = atomicAdd(au->ke_count, 1u);
            if (slot < au->ke_cap) au->ke_list[slot] = key | ((unsigned long long)(dot >= P.c) << 63);
        }
    }
    if (au) {
        atomicAdd(au->n_uncertain, 1ull);
        const double t64 = (1.0 - dot) * P.scale;
        const float err = fabsf((float)((double)t32 - t64));
        atomicMax(au->max_t_err_bits, __float_as_uint(err));
    }
    return in;
}

}  // namespace sc
