// sc_plan.cu -- host side of libsc: the C ABI of include/sc.h, plan construction (HEALPix RING
// ring tables, device interpolation table, input-ring intervals, knife-edge audit) and kernel
// dispatch.  Product code: shares nothing with oracle/.
#include "../../include/sc.h"
#include "sc_internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace sc {
cudaError_t launch_generic_conv(const Dev &P, const Maps &io, int B, int a0, int a1, int b0, int b1, cudaStream_t st);
cudaError_t launch_generic_conv_warp(const Dev &P, const Maps &io, int B, int a0, int a1, int b0, int b1, cudaStream_t st,
                                     bool overlap = false);
cudaError_t launch_generic_count(const Dev &P, int *count_dev, unsigned long long *sig_dev, const Audit *au, cudaStream_t st);
struct FastPlan;
FastPlan *fast_plan_create(const Dev &P, const std::vector<double> &z, const std::vector<double> &s,
                           int max_batch, int *polar_rings, cudaError_t *err);
void fast_plan_destroy(FastPlan *fp);
cudaError_t fast_convolve(FastPlan *fp, const Dev &P, const Maps &io, int B, cudaStream_t st, int *launches, cudaEvent_t *ev);
int fast_first_belt_ring(const FastPlan *fp);
cudaError_t fast_launch(FastPlan *fp, const Dev &P, const Maps &io, int B, int which, cudaStream_t st, int *launches, int chunk);
int fast_chunk_count(const FastPlan *fp, int B, int kind);
cudaError_t reorder_f32(int nside, int dir, const float *src, float *dst, cudaStream_t st);
cudaError_t reorder_i32(int nside, int dir, const int *src, int *dst, cudaStream_t st);
cudaError_t reorder_u64(int nside, int dir, const unsigned long long *src, unsigned long long *dst, cudaStream_t st);
cudaError_t fast_launch_band(FastPlan *fp, const Dev &P, const Maps &io, int B, int lo, int hi, cudaStream_t st, int *launches);
void fast_chunk_rings(const FastPlan *fp, int B, int kind, int i, int *lo, int *hi);
cudaError_t fast_launch_cap(FastPlan *fp, const Dev &P, const Maps &io, int ring_hi, cudaStream_t st, int *launches);
bool fast_available(const FastPlan *fp, int B);
}  // namespace sc

namespace {
thread_local std::string g_cuda_err;

bool cuda_ok(cudaError_t e, const char *what) {
    if (e == cudaSuccess) return true;
    g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return false;
}
#define SC_CUDA(call) do { if (!cuda_ok((call), #call)) return SC_ERR_CUDA; } while (0)

// One ring of the HEALPix RING scheme (Gorski et al. 2005; the paper only cites it, PAPER.md:76,
// :216).  Canonical fp64 evaluation of DESIGN.md R4: this order of operations fixes the last bit
// of z, s, phi0, dphi and therefore of the inclusion test.
struct RingGeom { int start, n, shifted; double z, s, phi0, dphi; };

RingGeom healpix_ring(int N, int i) {
    RingGeom g;
    const int64_t npix = 12LL * N * N;
    if (i < N) {                                   // north polar cap
        g.n = 4 * i;
        g.start = (int)(2LL * i * (i - 1));
        g.z = 1.0 - (double)((int64_t)i * i) / (3.0 * N * N);
        g.shifted = 0;
    } else if (i <= 3 * N) {                       // equatorial belt
        g.n = 4 * N;
        g.start = (int)(2LL * N * (N - 1) + (int64_t)(i - N) * 4 * N);
        g.z = (2.0 * N - i) * 2.0 / (3.0 * N);
        g.shifted = (i - N) & 1;
    } else {                                       // south polar cap
        const int64_t m = 4LL * N - i;
        g.n = (int)(4 * m);
        g.start = (int)(npix - 2 * m * (m + 1));
        g.z = -(1.0 - (double)(m * m) / (3.0 * N * N));
        g.shifted = 0;
    }
    g.s = std::sqrt((1.0 - g.z) * (1.0 + g.z));
    g.dphi = 2.0 * M_PI / g.n;
    g.phi0 = g.shifted ? 0.0 : 0.5 * g.dphi;
    return g;
}

template <class T> sc_status upload(const std::vector<T> &h, T **d) {
    *d = nullptr;
    const size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(T);
    if (!cuda_ok(cudaMalloc((void **)d, bytes), "cudaMalloc")) return SC_ERR_ALLOC;
    if (!h.empty()) SC_CUDA(cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return SC_OK;
}
}  // namespace

struct sc_plan {
    sc::Dev dev{};
    int device = 0;
    int max_batch = 1;
    int path = SC_PATH_AUTO;
    int64_t total_pairs = 0, n_knife = 0, n_uncertain = 0;
    double max_t_err = 0.0;
    std::vector<RingGeom> rings;
    std::vector<void *> owned;                 // device allocations
    // end-to-end staging
    float *stage_in = nullptr, *stage_out = nullptr;
    int stage_maps = 0;
    cudaStream_t own_stream = nullptr, comp_stream = nullptr, d2h_stream = nullptr;
    std::vector<cudaEvent_t> events;           // pool for the pipelined host entry
    std::vector<int> rlo_h, rhi_h;             // host copies of the candidate input-ring interval of every ring
    mutable int last_launches = 0;
    sc::FastPlan *fast = nullptr;
    int polar_rings = 0;                       // rings 1..polar_rings and their southern mirrors use the generic kernel
    // NESTED plans: the kernels run on plan-owned RING buffers (nest_maps maps in, nest_maps maps out)
    int nested = 0;
    float *nest_in = nullptr, *nest_out = nullptr;
    int nest_maps = 0;                         // min(max_batch, maps per launch): larger batches run in chunks of this size
};

namespace {

template <class T> sc_status upload_owned(sc_plan *pl, const std::vector<T> &h, const T **d) {
    T *p = nullptr;
    sc_status st = upload(h, &p);
    if (st != SC_OK) return st;
    pl->owned.push_back(p);
    *d = p;
    return SC_OK;
}

void pix_to_ring(const sc_plan *pl, int64_t p, int &ring, int &k) {
    // largest ring with start <= p
    int lo = 0, hi = (int)pl->rings.size() - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (pl->rings[mid].start <= p) lo = mid; else hi = mid - 1;
    }
    ring = lo + 1;
    k = (int)(p - pl->rings[lo].start);
}

// Host verdict for a knife-edge pair: the canonical test with the host libm (R4).
bool host_included(const sc_plan *pl, int64_t p, int64_t q) {
    int rp, kp, rq, kq;
    pix_to_ring(pl, p, rp, kp);
    pix_to_ring(pl, q, rq, kq);
    const RingGeom &P = pl->rings[rp - 1], &Q = pl->rings[rq - 1];
    const double phip = P.phi0 + (double)kp * P.dphi;
    const double phiq = Q.phi0 + (double)kq * Q.dphi;
    const double ss = P.s * Q.s;
    const double cd = std::cos(phip - phiq);
    const double zz = P.z * Q.z;
    const double sc = ss * cd;
    const double dot = zz + sc;
    return dot >= pl->dev.c;
}

sc_status run_audit(sc_plan *pl) {
    using namespace sc;
    const unsigned int cap = 1u << 20;
    unsigned long long *d_tot = nullptr, *d_unc = nullptr, *d_list = nullptr;
    unsigned int *d_err = nullptr, *d_cnt = nullptr;
    if (!cuda_ok(cudaMalloc((void **)&d_tot, 8), "cudaMalloc") || !cuda_ok(cudaMalloc((void **)&d_unc, 8), "cudaMalloc") ||
        !cuda_ok(cudaMalloc((void **)&d_err, 4), "cudaMalloc") || !cuda_ok(cudaMalloc((void **)&d_cnt, 4), "cudaMalloc") ||
        !cuda_ok(cudaMalloc((void **)&d_list, (size_t)cap * 8), "cudaMalloc"))
        return SC_ERR_ALLOC;
    sc_status st = SC_OK;
    do {
        if (!cuda_ok(cudaMemset(d_tot, 0, 8), "memset") || !cuda_ok(cudaMemset(d_unc, 0, 8), "memset") ||
            !cuda_ok(cudaMemset(d_err, 0, 4), "memset") || !cuda_ok(cudaMemset(d_cnt, 0, 4), "memset")) { st = SC_ERR_CUDA; break; }
        Audit au{d_tot, d_unc, d_err, d_list, d_cnt, cap};
        if (!cuda_ok(launch_generic_count(pl->dev, nullptr, nullptr, &au, 0), "audit launch")) { st = SC_ERR_CUDA; break; }
        if (!cuda_ok(cudaDeviceSynchronize(), "audit sync")) { st = SC_ERR_CUDA; break; }
        unsigned long long tot = 0, unc = 0; unsigned int errb = 0, n = 0;
        if (!cuda_ok(cudaMemcpy(&tot, d_tot, 8, cudaMemcpyDeviceToHost), "memcpy") ||
            !cuda_ok(cudaMemcpy(&unc, d_unc, 8, cudaMemcpyDeviceToHost), "memcpy") ||
            !cuda_ok(cudaMemcpy(&errb, d_err, 4, cudaMemcpyDeviceToHost), "memcpy") ||
            !cuda_ok(cudaMemcpy(&n, d_cnt, 4, cudaMemcpyDeviceToHost), "memcpy")) { st = SC_ERR_CUDA; break; }
        if (n > cap) { st = SC_ERR_UNSUPPORTED; break; }   // too many knife-edge pairs to list
        float errf; std::memcpy(&errf, &errb, 4);
        pl->n_uncertain = (int64_t)unc;
        pl->max_t_err = errf;
        std::vector<unsigned long long> list(n);
        if (n && !cuda_ok(cudaMemcpy(list.data(), d_list, (size_t)n * 8, cudaMemcpyDeviceToHost), "memcpy")) { st = SC_ERR_CUDA; break; }
        std::sort(list.begin(), list.end(), [](unsigned long long a, unsigned long long b) {
            return (a & ~(1ull << 63)) < (b & ~(1ull << 63)); });
        std::vector<unsigned long long> keys; std::vector<unsigned char> verdict;
        long long delta = 0;
        for (unsigned int i = 0; i < n; ++i) {
            const unsigned long long key = list[i] & ~(1ull << 63);
            if (!keys.empty() && keys.back() == key) continue;
            const bool gpu_in = (list[i] >> 63) != 0;
            const bool host_in = host_included(pl, (int64_t)(key / (unsigned long long)pl->dev.npix),
                                               (int64_t)(key % (unsigned long long)pl->dev.npix));
            keys.push_back(key); verdict.push_back(host_in ? 1 : 0);
            delta += (int)host_in - (int)gpu_in;
        }
        pl->n_knife = (int64_t)keys.size();
        pl->total_pairs = (int64_t)tot + delta;
        if (!keys.empty()) {
            if ((st = upload_owned(pl, keys, &pl->dev.ke_key)) != SC_OK) break;
            if ((st = upload_owned(pl, verdict, &pl->dev.ke_in)) != SC_OK) break;
            pl->dev.n_ke = (int)keys.size();
        }
    } while (0);
    cudaFree(d_tot); cudaFree(d_unc); cudaFree(d_err); cudaFree(d_cnt); cudaFree(d_list);
    return st;
}

}  // namespace

extern "C" {

const char *sc_status_string(sc_status s) {
    switch (s) {
        case SC_OK: return "SC_OK";
        case SC_ERR_INVALID_ARG: return "SC_ERR_INVALID_ARG";
        case SC_ERR_UNSUPPORTED: return "SC_ERR_UNSUPPORTED";
        case SC_ERR_ALLOC: return "SC_ERR_ALLOC";
        case SC_ERR_CUDA: return "SC_ERR_CUDA";
    }
    return "SC_ERR_?";
}

const char *sc_last_cuda_error(void) { return g_cuda_err.c_str(); }
const char *sc_version(void) { return "sc 0.2 (sm_100a)"; }

sc_status sc_plan_create(sc_plan **plan, int nside, int ordering, const double *ktable, int n_table,
                         double theta_max, int max_batch) {
    return sc_plan_create_zoned(plan, nside, ordering, ktable, n_table, theta_max, 0.0, max_batch);
}

sc_status sc_plan_create_zoned(sc_plan **plan, int nside, int ordering, const double *ktable, int n_table,
                               double theta_max, double zone_frac, int max_batch) {
    if (!plan || !ktable || nside < 1 || n_table < 2 || max_batch < 1) return SC_ERR_INVALID_ARG;
    if (zone_frac != 0.0 && (!(zone_frac > 0.0) || !(zone_frac < 1.0) || n_table < 4 || (n_table & 1))) return SC_ERR_INVALID_ARG;
    if (!(theta_max > 0.0) || !(theta_max <= M_PI / 2)) return SC_ERR_INVALID_ARG;
    if (ordering != SC_ORDER_RING && ordering != SC_ORDER_NESTED) return SC_ERR_INVALID_ARG;
    if (ordering == SC_ORDER_NESTED && (nside & (nside - 1))) return SC_ERR_INVALID_ARG;   // NESTED needs a power of two
    if (12LL * nside * nside >= (1LL << 31)) return SC_ERR_UNSUPPORTED;
    if (n_table > (1 << 24)) return SC_ERR_UNSUPPORTED;
    for (int i = 0; i < n_table; ++i) if (!std::isfinite(ktable[i])) return SC_ERR_INVALID_ARG;
    int ndev = 0;
    if (!cuda_ok(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount") || ndev < 1) {
        if (g_cuda_err.empty()) g_cuda_err = "no CUDA device";
        return SC_ERR_CUDA;
    }

    sc_plan *pl = new (std::nothrow) sc_plan;
    if (!pl) return SC_ERR_ALLOC;
    sc_status st = SC_OK;
    do {
        if (!cuda_ok(cudaGetDevice(&pl->device), "cudaGetDevice")) { st = SC_ERR_CUDA; break; }
        pl->max_batch = max_batch;
        pl->nested = ordering == SC_ORDER_NESTED;
        const int N = nside, nr = 4 * N - 1;
        sc::Dev &D = pl->dev;
        D.nside = N; D.nrings = nr; D.npix = 12 * N * N; D.ncap = 2 * N * (N - 1);
        D.ntab = n_table;
        D.tmax = (float)(n_table - 1);
        D.eps = 0.0625f + 4e-6f * (float)(n_table - 1);
        D.omega = (float)(4.0 * M_PI / (double)D.npix);
        D.c = std::cos(theta_max);
        const double one_minus_c = 2.0 * std::sin(0.5 * theta_max) * std::sin(0.5 * theta_max);
        D.scale = (double)(n_table - 1) / one_minus_c;
        D.ke_band = std::ldexp(1.0, -50);
        // two-zone table (R11): node index as a function of t = (1 - x) scale is the minimum of
        // two lines when the inner zone is the denser one (that is what the mode is for)
        D.zoned = 0; D.z_hm1 = 0; D.z_alpha = 1.f; D.z_gamma = 1.f; D.z_t1g = 0.f;
        if (zone_frac > 0.0) {
            const int h = n_table / 2;
            const double u1 = 2.0 * std::sin(0.5 * zone_frac * theta_max) * std::sin(0.5 * zone_frac * theta_max);
            const double t1 = u1 * D.scale, tm = (double)(n_table - 1);
            const double alpha = (double)(h - 1) / t1, gamma = (double)h / (tm - t1);
            if (!(alpha >= gamma)) { st = SC_ERR_INVALID_ARG; break; }
            D.zoned = 1; D.z_hm1 = h - 1; D.z_alpha = (float)alpha; D.z_gamma = (float)gamma; D.z_t1g = (float)(t1 * gamma);
        }
        // Steep tables: the fp32 pair geometry resolves the table coordinate to ~t 2^-23 cells, i.e. the kernel to
        // |b_j| j 2^-23 in cell j (b_j = cell slope).  If that, rms over the cells (pairs are uniform in t), exceeds 6.5e-7
        // of the table's rms, the kernels form the coordinate in fp64 (Dev::hp).  Not combined with the two-zone table.
        D.hp = 0;
        if (zone_frac == 0.0) {
            double se = 0.0, sk = 0.0;
            for (int j = 0; j + 1 < n_table; ++j) {
                const double t0 = ktable[n_table - 1 - j], t1 = ktable[n_table - 2 - j];
                const double err = (t1 - t0) * ((double)j + 0.5) * std::ldexp(1.0, -23);
                se += err * err; sk += 0.25 * (t0 + t1) * (t0 + t1);
            }
            if (sk > 0.0 && std::sqrt(se / sk) > 6.5e-7) D.hp = 1;      // leaves 3.5e-7 of the 1e-6 bar to the fp32 accumulation
            if (const char *e = std::getenv("SC_HP")) D.hp = std::atoi(e) != 0;
        }
        if (const char *e = std::getenv("SC_KNIFE_EDGE_BAND")) { const double v = std::atof(e); if (v > 0) D.ke_band = v; }

        // ring tables
        pl->rings.resize(nr);
        std::vector<double> z(nr), s(nr), phi0(nr), dphi(nr);
        std::vector<int> start(nr), npr(nr), rlo(nr), rhi(nr);
        for (int i = 1; i <= nr; ++i) {
            const RingGeom g = healpix_ring(N, i);
            pl->rings[i - 1] = g;
            z[i - 1] = g.z; s[i - 1] = g.s; phi0[i - 1] = g.phi0; dphi[i - 1] = g.dphi;
            start[i - 1] = g.start; npr[i - 1] = g.n;
        }
        // candidate input rings of an output ring: closest approach of two rings is at equal
        // azimuth, cos(theta - theta') = z z' + s s'.  Slack + one extra ring: a strict superset
        // (the kernels re-test every ring and every pixel).
        const double slack = 1e-9 + 2.0 * (double)D.eps / D.scale;
        for (int i = 1; i <= nr; ++i) {
            int lo = i, hi = i;
            while (lo > 1 && z[i - 1] * z[lo - 2] + s[i - 1] * s[lo - 2] >= D.c - slack) --lo;
            while (hi < nr && z[i - 1] * z[hi] + s[i - 1] * s[hi] >= D.c - slack) ++hi;
            if (lo > 1) --lo;
            if (hi < nr) ++hi;
            rlo[i - 1] = lo; rhi[i - 1] = hi;
        }
        pl->rlo_h = rlo; pl->rhi_h = rhi;
        // device table in the reversed coordinate t = (1 - x) (n-1)/(1-c): node j of the device
        // table is caller node n-1-j.  Cell [j, j+1): K = a_j + t b_j with b_j = T'_{j+1} - T'_j,
        // a_j = T'_j - j b_j  (fp64, rounded once).  Zero padding after the last cell.
        std::vector<float2> tab((size_t)n_table - 1 + sc::kTabPad), tabh(tab.size());
        for (int j = 0; j < n_table - 1; ++j) {
            const double t0 = ktable[n_table - 1 - j], t1 = ktable[n_table - 2 - j];
            const double b = t1 - t0, a = t0 - (double)j * b;
            tab[j] = make_float2((float)a, (float)b);
            tabh[j] = make_float2((float)(a + 0.5 * b), (float)b);
            if (zone_frac > 0.0 || D.hp) {
                // two-zone table / fp64 coordinate: cell-local form K = T_j + (tau - j) b_j (the cells of the outer zone carry
                // twice the slope at twice the index: the intercept form would lose a digit to cancellation)
                tab[j] = make_float2((float)t0, (float)b);
                tabh[j] = make_float2((float)(t0 + 0.5 * b), (float)b);      // around the cell centre
            }
        }
        for (size_t j = (size_t)n_table - 1; j < tab.size(); ++j) tab[j] = tabh[j] = make_float2(0.f, 0.f);

        if ((st = upload_owned(pl, z, &D.z)) != SC_OK) break;
        if ((st = upload_owned(pl, s, &D.s)) != SC_OK) break;
        if ((st = upload_owned(pl, phi0, &D.phi0)) != SC_OK) break;
        if ((st = upload_owned(pl, dphi, &D.dphi)) != SC_OK) break;
        if ((st = upload_owned(pl, start, &D.start)) != SC_OK) break;
        if ((st = upload_owned(pl, npr, &D.npr)) != SC_OK) break;
        if ((st = upload_owned(pl, rlo, &D.rlo)) != SC_OK) break;
        if ((st = upload_owned(pl, rhi, &D.rhi)) != SC_OK) break;
        if ((st = upload_owned(pl, tab, &D.tab)) != SC_OK) break;
        if ((st = upload_owned(pl, tabh, &D.tabh)) != SC_OK) break;
        D.ke_key = nullptr; D.ke_in = nullptr; D.n_ke = 0;

        if ((st = run_audit(pl)) != SC_OK) break;

        cudaError_t ferr = cudaSuccess;
        pl->fast = sc::fast_plan_create(D, z, s, max_batch, &pl->polar_rings, &ferr);
        if (ferr != cudaSuccess) { cuda_ok(ferr, "fast_plan_create"); st = SC_ERR_CUDA; break; }
        if (pl->nested) {                              // RING work buffers for up to max_batch (<= maps per launch) maps
            const int nm = std::min(max_batch, sc::kMaxB);
            const size_t bytes = (size_t)D.npix * 4 * nm;
            if (!cuda_ok(cudaMalloc((void **)&pl->nest_in, bytes), "cudaMalloc") ||
                !cuda_ok(cudaMalloc((void **)&pl->nest_out, bytes), "cudaMalloc")) { st = SC_ERR_ALLOC; break; }
            pl->nest_maps = nm;
        }
    } while (0);
    if (st != SC_OK) { sc_plan_destroy(pl); return st; }
    *plan = pl;
    return SC_OK;
}

sc_status sc_plan_destroy(sc_plan *plan) {
    if (!plan) return SC_OK;
    if (plan->fast) sc::fast_plan_destroy(plan->fast);
    for (void *p : plan->owned) cudaFree(p);
    if (plan->stage_in) cudaFree(plan->stage_in);
    if (plan->stage_out) cudaFree(plan->stage_out);
    if (plan->nest_in) cudaFree(plan->nest_in);
    if (plan->nest_out) cudaFree(plan->nest_out);
    if (plan->own_stream) cudaStreamDestroy(plan->own_stream);
    if (plan->comp_stream) cudaStreamDestroy(plan->comp_stream);
    if (plan->d2h_stream) cudaStreamDestroy(plan->d2h_stream);
    for (cudaEvent_t e : plan->events) cudaEventDestroy(e);
    delete plan;
    return SC_OK;
}

sc_status sc_plan_set_path(sc_plan *plan, int path) {
    if (!plan || (path != SC_PATH_AUTO && path != SC_PATH_GENERIC)) return SC_ERR_INVALID_ARG;
    plan->path = path;
    return SC_OK;
}

sc_status sc_plan_info(const sc_plan *plan, int64_t *npix, int64_t *total_pairs, double *cos_theta_max,
                       int64_t *n_knife_edge) {
    if (!plan) return SC_ERR_INVALID_ARG;
    if (npix) *npix = plan->dev.npix;
    if (total_pairs) *total_pairs = plan->total_pairs;
    if (cos_theta_max) *cos_theta_max = plan->dev.c;
    if (n_knife_edge) *n_knife_edge = plan->n_knife;
    return SC_OK;
}

sc_status sc_debug_stats(const sc_plan *plan, int64_t *n_uncertain, double *max_t_err, double *guard_band) {
    if (!plan) return SC_ERR_INVALID_ARG;
    if (n_uncertain) *n_uncertain = plan->n_uncertain;
    if (max_t_err) *max_t_err = plan->max_t_err;
    if (guard_band) *guard_band = plan->dev.eps;
    return SC_OK;
}

int sc_last_launch_count(const sc_plan *plan) { return plan ? plan->last_launches : 0; }

int sc_plan_double_coordinate(const sc_plan *plan) { return plan ? plan->dev.hp : 0; }

// Maps are N_pix floats each: no output may overlap an input or another output.
static bool maps_ok(const float *const *in_maps, float *const *out_maps, int B, size_t npix) {
    const uintptr_t bytes = (uintptr_t)npix * 4;
    auto overlap = [&](const void *a, const void *b) {
        const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
        return x < y + bytes && y < x + bytes;
    };
    for (int b = 0; b < B; ++b) {
        if (!in_maps[b] || !out_maps[b]) return false;
        if (((uintptr_t)in_maps[b] | (uintptr_t)out_maps[b]) & 15u) return false;
    }
    for (int b = 0; b < B; ++b) {
        for (int a = 0; a < B; ++a) {
            if (overlap(out_maps[b], in_maps[a])) return false;
            if (a != b && overlap(out_maps[b], out_maps[a])) return false;
        }
    }
    return true;
}

// ev (optional): 4 events recorded before the polar kernel and after each of the three kernels
static sc_status convolve_impl(const sc_plan *plan, const float *const *in_maps, float *const *out_maps, int B,
                               void *cuda_stream, cudaEvent_t *ev, float *ms) {
    if (!plan || !in_maps || !out_maps || B < 1) return SC_ERR_INVALID_ARG;
    if (!maps_ok(in_maps, out_maps, B, (size_t)plan->dev.npix)) return SC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const sc::Dev &D = plan->dev;
    int launches = 0;
    const size_t npix = (size_t)D.npix;
    // maps per launch; a NESTED plan goes through its RING work buffers, which hold nest_maps maps
    // (plans with the fp64 table coordinate, Dev::hp, have one-map kernel instances only)
    const int chunk = D.hp ? 1 : (plan->nested ? plan->nest_maps : sc::kMaxB);
    for (int b0 = 0; b0 < B; b0 += chunk) {
        const int nb = std::min(chunk, B - b0);
        sc::Maps io{};
        for (int b = 0; b < nb; ++b) { io.in[b] = in_maps[b0 + b]; io.out[b] = out_maps[b0 + b]; }
        if (plan->nested) {                                                // NESTED -> RING work buffers
            for (int b = 0; b < nb; ++b) {
                SC_CUDA(sc::reorder_f32(D.nside, 0, in_maps[b0 + b], plan->nest_in + npix * b, st));
                io.in[b] = plan->nest_in + npix * b; io.out[b] = plan->nest_out + npix * b;
            }
            launches += nb;
        }
        if (ev) SC_CUDA(cudaEventRecord(ev[0], st));
        if (plan->path == SC_PATH_GENERIC || !sc::fast_available(plan->fast, nb)) {
            SC_CUDA(sc::launch_generic_conv(D, io, nb, 0, D.npix, 0, 0, st));
            ++launches;
            if (ev) { SC_CUDA(cudaEventRecord(ev[1], st)); SC_CUDA(cudaEventRecord(ev[2], st)); SC_CUDA(cudaEventRecord(ev[3], st)); }
        } else {
            // rings next to the poles: generic kernel; everything else: fast kernels
            // (the three kernels write disjoint pixels: unless every kernel is being timed, the warp-per-pixel kernel goes
            // last and may start while the sym kernel drains)
            const int pr = plan->polar_rings;
            const int np = 2 * pr * (pr + 1);              // pixels in rings 1..pr
            const bool polar_last = !ev && !std::getenv("SC_NO_OVERLAP") &&
                                    0.5 * (double)D.npix * ((double)D.tmax / D.scale) <= 8000.0;      // discs below ~8000 pixels only: at config 6 (61000) the 36 ms polar kernel last costs +6 %
            if (pr > 0 && !polar_last) {
                SC_CUDA(sc::launch_generic_conv_warp(D, io, nb, 0, np, D.npix - np, D.npix, st));
                ++launches;
            }
            if (ev) SC_CUDA(cudaEventRecord(ev[1], st));
            int nl = 0;
            SC_CUDA(sc::fast_convolve(plan->fast, D, io, nb, st, &nl, ev ? ev + 2 : nullptr));
            launches += nl;
            if (pr > 0 && polar_last) {
                SC_CUDA(sc::launch_generic_conv_warp(D, io, nb, 0, np, D.npix - np, D.npix, st, true));
                ++launches;
            }
        }
        if (plan->nested) {                                                // RING results -> NESTED outputs
            for (int b = 0; b < nb; ++b) SC_CUDA(sc::reorder_f32(D.nside, 1, plan->nest_out + npix * b, out_maps[b0 + b], st));
            launches += nb;
        }
        if (ev) {
            SC_CUDA(cudaEventSynchronize(ev[3]));
            for (int k = 0; k < SC_K_COUNT; ++k) {
                float t = 0.f;
                SC_CUDA(cudaEventElapsedTime(&t, ev[k], ev[k + 1]));
                ms[k] += t;
            }
        }
    }
    plan->last_launches = launches;
    return SC_OK;
}

sc_status sc_convolve(const sc_plan *plan, const float *const *in_maps, float *const *out_maps, int B,
                      void *cuda_stream) {
    return convolve_impl(plan, in_maps, out_maps, B, cuda_stream, nullptr, nullptr);
}

sc_status sc_convolve_profile(const sc_plan *plan, const float *const *in_maps, float *const *out_maps, int B,
                              void *cuda_stream, float *ms) {
    if (!ms) return SC_ERR_INVALID_ARG;
    cudaEvent_t ev[SC_K_COUNT + 1] = {};
    for (int k = 0; k < SC_K_COUNT; ++k) ms[k] = 0.f;
    sc_status st = SC_OK;
    for (int k = 0; k <= SC_K_COUNT; ++k)
        if (!cuda_ok(cudaEventCreate(&ev[k]), "cudaEventCreate")) st = SC_ERR_CUDA;
    if (st == SC_OK) st = convolve_impl(plan, in_maps, out_maps, B, cuda_stream, ev, ms);
    for (int k = 0; k <= SC_K_COUNT; ++k) if (ev[k]) cudaEventDestroy(ev[k]);
    return st;
}

sc_status sc_plan_partition(const sc_plan *plan, int *polar_rings, int *first_belt_ring) {
    if (!plan) return SC_ERR_INVALID_ARG;
    const int N2 = 2 * plan->dev.nside;
    if (polar_rings) *polar_rings = plan->fast ? plan->polar_rings : N2;
    if (first_belt_ring) *first_belt_ring = plan->fast ? sc::fast_first_belt_ring(plan->fast) : N2 + 1;
    return SC_OK;
}

sc_status sc_convolve_host(sc_plan *plan, const float *const *in_maps_host, float *const *out_maps_host, int B) {
    if (!plan || !in_maps_host || !out_maps_host || B < 1) return SC_ERR_INVALID_ARG;
    for (int b = 0; b < B; ++b) if (!in_maps_host[b] || !out_maps_host[b]) return SC_ERR_INVALID_ARG;
    const size_t npix = (size_t)plan->dev.npix;
    if (plan->stage_maps < B) {
        if (plan->stage_in) cudaFree(plan->stage_in);
        if (plan->stage_out) cudaFree(plan->stage_out);
        plan->stage_in = plan->stage_out = nullptr; plan->stage_maps = 0;
        const int nm = std::max(B, plan->max_batch);
        if (!cuda_ok(cudaMalloc((void **)&plan->stage_in, npix * 4 * nm), "cudaMalloc")) return SC_ERR_ALLOC;
        if (!cuda_ok(cudaMalloc((void **)&plan->stage_out, npix * 4 * nm), "cudaMalloc")) return SC_ERR_ALLOC;
        plan->stage_maps = nm;
    }
    if (!plan->own_stream) SC_CUDA(cudaStreamCreateWithFlags(&plan->own_stream, cudaStreamNonBlocking));
    const sc::Dev &D = plan->dev;
    const int N = D.nside;
    const bool pipelined = plan->path == SC_PATH_AUTO && plan->fast && !plan->nested && sc::fast_available(plan->fast, plan->dev.hp ? 1 : std::min(B, sc::kMaxB));
    if (!pipelined) {
        std::vector<const float *> in(B); std::vector<float *> out(B);
        for (int b = 0; b < B; ++b) {
            in[b] = plan->stage_in + npix * b; out[b] = plan->stage_out + npix * b;
            SC_CUDA(cudaMemcpyAsync(plan->stage_in + npix * b, in_maps_host[b], npix * 4, cudaMemcpyHostToDevice, plan->own_stream));
        }
        sc_status st = sc_convolve(plan, in.data(), out.data(), B, plan->own_stream);
        if (st != SC_OK) return st;
        for (int b = 0; b < B; ++b)
            SC_CUDA(cudaMemcpyAsync(out_maps_host[b], out[b], npix * 4, cudaMemcpyDeviceToHost, plan->own_stream));
        SC_CUDA(cudaStreamSynchronize(plan->own_stream));
        return SC_OK;
    }

    // Pipelined over latitude chunks, from the equator towards the poles: a chunk of base rings lo .. hi
    // (and their southern mirrors) needs the input rows of rings rlo(lo) .. 4N - rlo(lo), one contiguous
    // range that grows outwards, so the copy-in stream sends two new slices per chunk, the compute
    // stream runs the chunk's tiles as soon as they have arrived, and the copy-out stream returns the
    // chunk's output rows while later chunks are still being copied in and computed.
    if (!plan->comp_stream) {
        SC_CUDA(cudaStreamCreateWithFlags(&plan->comp_stream, cudaStreamNonBlocking));
        SC_CUDA(cudaStreamCreateWithFlags(&plan->d2h_stream, cudaStreamNonBlocking));
    }
    cudaStream_t s_in = plan->own_stream, s_c = plan->comp_stream, s_out = plan->d2h_stream;
    const int N4 = 4 * N;
    auto row = [&](int ring) -> size_t { return ring <= N4 - 1 ? (size_t)plan->rings[ring - 1].start : npix; };   // first pixel of a ring
    const int pr = plan->polar_rings;
    int launches = 0;
    size_t nev = 0;
    auto next_event = [&](cudaEvent_t *ev) -> sc_status {
        if (nev == plan->events.size()) {
            cudaEvent_t e = nullptr;
            SC_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            plan->events.push_back(e);
        }
        *ev = plan->events[nev++];
        return SC_OK;
    };
    const int per_launch = D.hp ? 1 : sc::kMaxB;
    for (int b0 = 0; b0 < B; b0 += per_launch) {
        const int nb = std::min(per_launch, B - b0);
        sc::Maps io{};
        for (int b = 0; b < nb; ++b) { io.in[b] = plan->stage_in + npix * (b0 + b); io.out[b] = plan->stage_out + npix * (b0 + b); }
        auto copy_in = [&](size_t p0, size_t p1) -> sc_status {
            for (int b = 0; b < nb && p1 > p0; ++b)
                SC_CUDA(cudaMemcpyAsync((float *)io.in[b] + p0, in_maps_host[b0 + b] + p0, (p1 - p0) * 4, cudaMemcpyHostToDevice, s_in));
            return SC_OK;
        };
        auto copy_out = [&](size_t p0, size_t p1) -> sc_status {
            for (int b = 0; b < nb && p1 > p0; ++b)
                SC_CUDA(cudaMemcpyAsync(out_maps_host[b0 + b] + p0, io.out[b] + p0, (p1 - p0) * 4, cudaMemcpyDeviceToHost, s_out));
            return SC_OK;
        };
        // Pixels [in0, in1) are on the device, pixels [out0, out1) are back on the host: both ranges grow outwards from
        // the equator.  Copy boundaries are multiples of 4 KB except at the ends of the map (measured: the same
        // bidirectional traffic in copies that start and end off a page boundary takes 6 % longer): an input slice is
        // extended towards the pole, an output slice is cut short towards the equator and its remainder goes with the
        // next chunk's (those pixels are final by then; the last stage ends at 0 and N_pix).
        constexpr size_t kPage = 1024;                 // floats
        size_t in0 = 0, in1 = 0, out0 = 0, out1 = 0;
        bool have_in = false, have_out = false;
        // stage: bring rows down to ring need_lo, launch, return rows of base rings lo .. hi
        auto stage = [&](int need_lo, int kind, int chunk, int lo, int hi) -> sc_status {
            sc_status s;
            need_lo = std::max(1, std::min(need_lo, 2 * N));
            {
                const size_t a = row(need_lo) & ~(kPage - 1), b = std::min(npix, (row(N4 - need_lo + 1) + kPage - 1) & ~(kPage - 1));
                if (!have_in) {
                    if ((s = copy_in(a, b)) != SC_OK) return s;
                    in0 = a; in1 = b; have_in = true;
                } else {
                    if (a < in0) { if ((s = copy_in(a, in0)) != SC_OK) return s; in0 = a; }
                    if (b > in1) { if ((s = copy_in(in1, b)) != SC_OK) return s; in1 = b; }
                }
            }
            cudaEvent_t ev_in, ev_done;
            if ((s = next_event(&ev_in)) != SC_OK || (s = next_event(&ev_done)) != SC_OK) return s;
            SC_CUDA(cudaEventRecord(ev_in, s_in));
            SC_CUDA(cudaStreamWaitEvent(s_c, ev_in, 0));
            int nl = 0;
            if (kind == 2) {
                const int np = 2 * pr * (pr + 1);
                SC_CUDA(sc::launch_generic_conv_warp(D, io, nb, 0, np, D.npix - np, D.npix, s_c));
                nl = 1;
            } else {
                SC_CUDA(sc::fast_launch(plan->fast, D, io, nb, kind == 0 ? 1 : 2, s_c, &nl, chunk));
            }
            launches += nl;
            SC_CUDA(cudaEventRecord(ev_done, s_c));
            SC_CUDA(cudaStreamWaitEvent(s_out, ev_done, 0));
            (void)hi;
            size_t a = row(lo), b = row(N4 - lo + 1);          // everything in [a, b) is final once this chunk is done
            if (lo > 1) { a = (a + kPage - 1) & ~(kPage - 1); b = b & ~(kPage - 1); }
            if (a >= b) return SC_OK;
            if (!have_out) {
                if ((s = copy_out(a, b)) != SC_OK) return s;
                out0 = a; out1 = b; have_out = true;
                return SC_OK;
            }
            if (a < out0) { if ((s = copy_out(a, out0)) != SC_OK) return s; out0 = a; }
            if (b > out1) { if ((s = copy_out(out1, b)) != SC_OK) return s; out1 = b; }
            return SC_OK;
        };
        for (int kind = 1; kind >= 0; --kind) {        // belt chunks (equator first), then the cap chunks
            const int nch = sc::fast_chunk_count(plan->fast, nb, kind);
            for (int i = 0; i < nch; ++i) {
                int lo, hi;
                sc::fast_chunk_rings(plan->fast, nb, kind, i, &lo, &hi);
                sc_status s = stage(plan->rlo_h[lo - 1] - 1, kind, i, lo, hi);
                if (s != SC_OK) return s;
            }
        }
        if (pr > 0) { sc_status s = stage(1, 2, 0, 1, pr); if (s != SC_OK) return s; }
        if (!have_out || out0 > 0 || out1 < npix) return SC_ERR_UNSUPPORTED;   // (cannot happen: the last stage ends at ring 1)
    }
    plan->last_launches = launches;
    SC_CUDA(cudaStreamSynchronize(s_out));
    return SC_OK;
}

static void band_rows(const sc_plan *plan, int lo, int hi, int64_t *out_rows, int64_t *in_rows) {
    const int N = plan->dev.nside, N4 = 4 * N;
    const int64_t npix = plan->dev.npix;
    auto row = [&](int ring) -> int64_t { return ring <= N4 - 1 ? (int64_t)plan->rings[ring - 1].start : npix; };
    if (out_rows) {
        out_rows[0] = row(lo); out_rows[1] = row(hi + 1);
        out_rows[2] = hi >= 2 * N ? row(2 * N + 1) : row(N4 - hi); out_rows[3] = row(N4 - lo + 1);
    }
    if (in_rows) {
        const int a = std::max(1, plan->rlo_h[lo - 1] - 1), b = std::min(N4 - 1, plan->rhi_h[hi - 1] + 1);
        in_rows[0] = row(a); in_rows[1] = row(b + 1);
        in_rows[2] = row(N4 - b); in_rows[3] = row(N4 - a + 1);
        if (in_rows[2] <= in_rows[1]) { in_rows[1] = in_rows[3]; in_rows[2] = in_rows[3]; }   // merged at the equator
    }
}

sc_status sc_band_partition(const sc_plan *plan, int world, int rank, int *ring_lo, int *ring_hi,
                            int64_t *out_rows, int64_t *in_rows) {
    if (!plan) return SC_ERR_INVALID_ARG;
    const int N = plan->dev.nside;
    if (world < 1 || world > 2 * N || rank < 0 || rank >= world) return SC_ERR_INVALID_ARG;
    // base ring r stands for rings r and 4N - r: 2 n_r pixels (n_r for the equator ring 2N).  Bands get nearly equal
    // ESTIMATED TIME from per-pixel costs measured on one B200 (configs 4 and 5, round 2): with nb neighbours per pixel a
    // belt pixel costs ~5.3e-11 nb ms, a cap pixel 2.9 times that, a pixel next to the poles (warp-per-pixel kernel)
    // 6.8e-6 + 2.9e-9 nb ms, i.e. 55 + 128000 / nb belt pixels (356 at config 4, 88 at config 5).  A band boundary that
    // falls close to a hand-over between two kernels is moved onto it, so that no band pays a kernel launch (prologue:
    // the 128 KB table per CTA) for a sliver of rings.
    const int pr = plan->fast ? plan->polar_rings : 0;
    const int fb = plan->fast ? sc::fast_first_belt_ring(plan->fast) : 2 * N + 1;
    const double nb = std::max(1.0, 0.5 * (double)plan->dev.npix * ((double)plan->dev.tmax / plan->dev.scale));
    const int64_t w_polar = (int64_t)(10.0 * (55.0 + 128000.0 / nb));            // in tenths of a belt pixel
    auto weight = [&](int r) -> int64_t {
        const int64_t px = (int64_t)plan->rings[r - 1].n * (r < 2 * N ? 2 : 1);
        return px * (r <= pr ? w_polar : (r < fb ? 29 : 10));
    };
    int64_t total = 0;
    for (int r = 1; r <= 2 * N; ++r) total += weight(r);
    std::vector<int> first(world + 1, 1);            // first base ring of band k; band `world` starts at 2N + 1
    first[world] = 2 * N + 1;
    {
        int64_t cum = 0;
        int r = 1;
        for (int k = 1; k < world; ++k) {
            for (; r <= 2 * N; ++r) {
                if (cum * world >= total * k) break;
                cum += weight(r);
            }
            first[k] = r;
        }
        const int snap = std::max(2, N / 16);
        for (int k = 1; k < world; ++k) {
            if (pr > 0 && std::abs(first[k] - (pr + 1)) <= snap) first[k] = pr + 1;
            if (fb <= 2 * N && std::abs(first[k] - fb) <= snap) first[k] = fb;
        }
        for (int k = 1; k < world; ++k)              // every band keeps at least one ring
            first[k] = std::min(std::max(first[k], std::max(k + 1, first[k - 1] + 1)), 2 * N - (world - 1 - k));
    }
    auto first_ring = [&](int k) -> int { return first[std::min(std::max(k, 0), world)]; };
    const int lo = first_ring(rank), hi = first_ring(rank + 1) - 1;
    if (hi < lo) return SC_ERR_INVALID_ARG;
    if (ring_lo) *ring_lo = lo;
    if (ring_hi) *ring_hi = hi;
    band_rows(plan, lo, hi, out_rows, in_rows);
    return SC_OK;
}

sc_status sc_convolve_band(sc_plan *plan, int ring_lo, int ring_hi, const float *const *in_maps,
                           float *const *out_maps, int B, void *cuda_stream) {
    if (!plan || !in_maps || !out_maps || B < 1) return SC_ERR_INVALID_ARG;
    const sc::Dev &D = plan->dev;
    const int N = D.nside;
    if (ring_lo < 1 || ring_hi < ring_lo || ring_hi > 2 * N) return SC_ERR_INVALID_ARG;
    if (plan->nested) return SC_ERR_UNSUPPORTED;                       // bands are contiguous rows in RING order only
    if (!maps_ok(in_maps, out_maps, B, (size_t)D.npix)) return SC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int64_t orow[4];
    band_rows(plan, ring_lo, ring_hi, orow, nullptr);
    int launches = 0;
    const int per_launch = D.hp ? 1 : sc::kMaxB;
    for (int b0 = 0; b0 < B; b0 += per_launch) {
        const int nb = std::min(per_launch, B - b0);
        sc::Maps io{};
        for (int b = 0; b < nb; ++b) { io.in[b] = in_maps[b0 + b]; io.out[b] = out_maps[b0 + b]; }
        if (plan->path == SC_PATH_GENERIC || !sc::fast_available(plan->fast, nb)) {
            SC_CUDA(sc::launch_generic_conv(D, io, nb, (int)orow[0], (int)orow[1], (int)orow[2], (int)orow[3], st));
            ++launches;
            continue;
        }
        const int pr = plan->polar_rings;
        if (ring_lo <= pr) {                               // rings next to the poles
            int64_t prow[4];
            band_rows(plan, ring_lo, std::min(ring_hi, pr), prow, nullptr);
            SC_CUDA(sc::launch_generic_conv_warp(D, io, nb, (int)prow[0], (int)prow[1], (int)prow[2], (int)prow[3], st));
            ++launches;
        }
        int nl = 0;
        SC_CUDA(sc::fast_launch_band(plan->fast, D, io, nb, ring_lo, ring_hi, st, &nl));
        launches += nl;
    }
    plan->last_launches = launches;
    return SC_OK;
}

sc_status sc_cap_rows(const sc_plan *plan, int ring_hi, int64_t *out_rows, int64_t *in_rows) {
    if (!plan) return SC_ERR_INVALID_ARG;
    const int N = plan->dev.nside, N4 = 4 * N;
    if (ring_hi < 1 || ring_hi > 2 * N) return SC_ERR_INVALID_ARG;
    auto row = [&](int ring) -> int64_t { return ring <= N4 - 1 ? (int64_t)plan->rings[ring - 1].start : (int64_t)plan->dev.npix; };
    if (out_rows) { out_rows[0] = 0; out_rows[1] = row(ring_hi + 1); }
    if (in_rows) { in_rows[0] = 0; in_rows[1] = row(std::min(N4 - 1, plan->rhi_h[ring_hi - 1] + 1) + 1); }
    return SC_OK;
}

sc_status sc_convolve_cap(sc_plan *plan, int ring_hi, const float *const *in_maps, float *const *out_maps, int B,
                          void *cuda_stream) {
    if (!plan || !in_maps || !out_maps || B < 1) return SC_ERR_INVALID_ARG;
    const sc::Dev &D = plan->dev;
    const int N = D.nside;
    if (ring_hi < 1 || ring_hi > 2 * N) return SC_ERR_INVALID_ARG;
    if (plan->nested) return SC_ERR_UNSUPPORTED;                       // a cap is a contiguous block of rows in RING order only
    int64_t orow[2], irow[2];
    sc_cap_rows(plan, ring_hi, orow, irow);
    // the maps need only exist up to the last row read / written: overlap is checked on those extents
    for (int b = 0; b < B; ++b) {
        if (!in_maps[b] || !out_maps[b]) return SC_ERR_INVALID_ARG;
        if (((uintptr_t)in_maps[b] | (uintptr_t)out_maps[b]) & 15u) return SC_ERR_INVALID_ARG;
    }
    for (int b = 0; b < B; ++b)
        for (int a = 0; a < B; ++a) {
            const uintptr_t o0 = (uintptr_t)out_maps[b], o1 = o0 + (uintptr_t)orow[1] * 4;
            const uintptr_t i0 = (uintptr_t)in_maps[a], i1 = i0 + (uintptr_t)irow[1] * 4;
            if (o0 < i1 && i0 < o1) return SC_ERR_INVALID_ARG;
            const uintptr_t p0 = (uintptr_t)out_maps[a], p1 = p0 + (uintptr_t)orow[1] * 4;
            if (a != b && o0 < p1 && p0 < o1) return SC_ERR_INVALID_ARG;
        }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int launches = 0;
    for (int b = 0; b < B; ++b) {                                      // one map per launch (north-only kernel instance)
        sc::Maps io{};
        io.in[0] = in_maps[b]; io.out[0] = out_maps[b];
        if (plan->path == SC_PATH_GENERIC || !plan->fast || D.hp) {      // (no north-only instance with the fp64 coordinate)
            SC_CUDA(sc::launch_generic_conv(D, io, 1, 0, (int)orow[1], 0, 0, st));
            ++launches;
            continue;
        }
        const int pr = std::min(plan->polar_rings, ring_hi);
        if (pr > 0) {                                                  // rings next to the pole
            SC_CUDA(sc::launch_generic_conv_warp(D, io, 1, 0, 2 * pr * (pr + 1), 0, 0, st));
            ++launches;
        }
        int nl = 0;
        SC_CUDA(sc::fast_launch_cap(plan->fast, D, io, ring_hi, st, &nl));
        launches += nl;
    }
    plan->last_launches = launches;
    return SC_OK;
}

sc_status sc_debug_neighbour_counts(const sc_plan *plan, int32_t *count_dev, uint64_t *sig_dev, void *cuda_stream) {
    if (!plan || !count_dev) return SC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!plan->nested) {
        SC_CUDA(sc::launch_generic_count(plan->dev, count_dev, (unsigned long long *)sig_dev, nullptr, st));
        return SC_OK;
    }
    // NESTED plan: count in RING order into scratch, then reorder (entry p = NESTED pixel p; the signature
    // stays the sum of the neighbours' RING indices)
    const size_t npix = (size_t)plan->dev.npix;
    int *c_ring = nullptr; unsigned long long *s_ring = nullptr;
    if (!cuda_ok(cudaMalloc((void **)&c_ring, npix * 4), "cudaMalloc")) return SC_ERR_ALLOC;
    if (sig_dev && !cuda_ok(cudaMalloc((void **)&s_ring, npix * 8), "cudaMalloc")) { cudaFree(c_ring); return SC_ERR_ALLOC; }
    sc_status rs = SC_OK;
    if (!cuda_ok(sc::launch_generic_count(plan->dev, c_ring, s_ring, nullptr, st), "count") ||
        !cuda_ok(sc::reorder_i32(plan->dev.nside, 1, c_ring, count_dev, st), "reorder") ||
        (sig_dev && !cuda_ok(sc::reorder_u64(plan->dev.nside, 1, s_ring, (unsigned long long *)sig_dev, st), "reorder")) ||
        !cuda_ok(cudaStreamSynchronize(st), "sync"))
        rs = SC_ERR_CUDA;
    cudaFree(c_ring); cudaFree(s_ring);
    return rs;
}

}  // extern "C"

// internal accessors for sc_static.cu (the plan structure is private to this file)
namespace sc {
const Dev *plan_dev(const sc_plan *plan) { return plan ? &plan->dev : nullptr; }
int plan_nested(const sc_plan *plan) { return plan ? plan->nested : 0; }
int plan_device(const sc_plan *plan) { return plan ? plan->device : -1; }
void note_error(const char *what, cudaError_t e) { cuda_ok(e, what); }
void note_message(const char *msg) { g_cuda_err = msg; }
}  // namespace sc
