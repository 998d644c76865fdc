// sc_fast.cu -- the fast convolution kernel ("sym kernel") and its plan data.
//
// Design:
//  * HEALPix is invariant under phi -> phi + pi/2 and z -> -z, so the weight K(p, q) of a pair is
//    shared by its 8 images (4 quadrants x north/south).  A thread owns a BASE pixel (ring r <= 2N,
//    in-ring index k < ring_length/4), evaluates the pair geometry and the table lookup once and
//    FMA-accumulates 8 outputs (times B maps): (5 + 1 + 8 B) FMA-pipe operations per 8 B pair-maps.
//  * A CTA owns a tile of consecutive base pixels on one ring.  For each input ring within theta_max
//    it stages the needed run of map values -- the 4 quadrant images interleaved as float4, north and
//    south planes -- into shared memory with cp.async, double buffered, one __syncthreads per ring.
//  * Pair geometry in fp32 without cancellation: t = A + B (1 - cos d) with A, B per ring pair from
//    fp64, d = azimuth difference built from the INTEGER pixel offset (exact) times the ring's pixel
//    spacing; 1 - cos d by a 3-term even polynomial (|d| <= ~0.4 rad on the rings this kernel takes;
//    the few rings next to the poles go to the generic kernel).
//  * Table lookup: magic-number rounding gives the cell index; K = a_i + t b_i (one FFMA); the
//    16K-entry (a, b) table lives in shared memory (128 KB).
//  * Inclusion: t < tmax - 1 needs no test at all (fast path); the last cell and everything beyond
//    takes a branch: t > tmax + eps -> excluded, |t - tmax| <= eps -> canonical fp64 test for each
//    of the 8 images separately (bit-exact with the oracle), else included.
#include "sc_fast.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

namespace sc {

// floor(Y / d) and remainder for 0 <= Y < 2^31 with M0 = floor((2^32 - 1) / d): one multiply-high
// and one fix-up instead of an integer division
__device__ __forceinline__ int div_fast(int Y, int d, unsigned M0, int &rem) {
    int q = (int)__umulhi((unsigned)Y, M0);
    rem = Y - q * d;
    if (rem >= d) { ++q; rem -= d; }
    return q;
}

__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Exact decisions for the 8 images of one uncertain pair: bit g = 4 h + m set <=> image included.
static __device__ __noinline__ unsigned sym_exact_mask(const Dev &P, int r, int k, int ip, int rq, int kq,
                                                       int ipq, float t) {
    const int N4 = 4 * P.nside;
    const int n = 4 * ip, nq = 4 * ipq;
    unsigned mask = 0;
    kq %= nq; if (kq < 0) kq += nq;
    for (int h = 0; h < 2; ++h) {
        const int rp_i = h ? N4 - r : r, rq_i = h ? N4 - rq : rq;
        for (int m = 0; m < 4; ++m) {
            int kp_i = k + m * ip; if (kp_i >= n) kp_i -= n;
            int kq_i = kq + m * ipq; if (kq_i >= nq) kq_i -= nq;
            if (exact_included(P, rp_i, kp_i, rq_i, kq_i, t, nullptr)) mask |= 1u << (4 * h + m);
        }
    }
    return mask;
}

template <int B, int R>
__global__ void __launch_bounds__(kMaxThreads, 1)
sym_kernel(const Dev P, const FastDev F, const Maps io) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);
    float4 *stage = reinterpret_cast<float4 *>(smem_raw + (((size_t)F.ntab_s * 8 + 15) & ~(size_t)15));
    __shared__ int s_tile;
    const int tid = threadIdx.x, NT = blockDim.x;
    const int T = NT * R;
    const int N = P.nside;
    const int Lmax = F.Lmax;

    for (int i = tid; i < F.ntab_s; i += NT) tab[i] = P.tabh[i];
    const unsigned thresh = kMagicBits + (unsigned)(P.ntab - 2);
    const unsigned zero_bits = kMagicBits + (unsigned)(P.ntab - 1);
    const float tmax = P.tmax, eps = P.eps;

    while (true) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(F.counter, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= F.ntiles) break;
        const int4 tl = F.tiles[tile];
        const int r = tl.x, k0 = tl.y;
        const int ip = P.npr[r - 1] >> 2;
        const int ip2 = 2 * ip;
        const unsigned M0 = 0xFFFFFFFFu / (unsigned)ip2;
        int rem_unused;
        const int sh = (r >= N && r <= 3 * N) ? ((r - N) & 1) : 0;
        const int klast = min(k0 + T, ip) - 1;
        const int ka = min(k0 + R * tid, klast);
        const int ap = 2 * ka + 1 - sh, ap0 = 2 * k0 + 1 - sh, apl = 2 * klast + 1 - sh;
        const int e0 = F.pair_off[tl.z], e1 = F.pair_off[tl.z + 1];

        float tot[R][B][8];
#pragma unroll
        for (int rr = 0; rr < R; ++rr)
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int g = 0; g < 8; ++g) tot[rr][b][g] = 0.f;

        // stage the run of input ring entry e into buffer `buf`
        auto stage_ring = [&](int e, int buf) {
            const PairEnt pe = F.pairs[e];
            const int nq = 4 * pe.ipq;
            const int w0 = div_fast(ap0 * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) - pe.hw;
            const int L = div_fast(apl * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) + pe.hw + R - w0;
            for (int idx = tid; idx < 4 * L; idx += NT) {
                const int i = idx >> 2, m = idx & 3;
                int kq = w0 + i + m * pe.ipq + nq;
                while (kq >= nq) kq -= nq;
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    float *dn = reinterpret_cast<float *>(stage + (size_t)((buf * B + b) * 2 + 0) * Lmax + i) + m;
                    float *ds = reinterpret_cast<float *>(stage + (size_t)((buf * B + b) * 2 + 1) * Lmax + i) + m;
                    cp_async4(dn, io.in[b] + pe.start_n + kq);
                    cp_async4(ds, io.in[b] + pe.start_s + kq);
                }
            }
            cp_async_commit();
        };

        stage_ring(e0, 0);
        for (int e = e0; e < e1; ++e) {
            const int buf = (e - e0) & 1;
            cp_async_wait_all();
            __syncthreads();                       // ring e staged by everyone; ring e-1 fully consumed
            if (e + 1 < e1) stage_ring(e + 1, buf ^ 1);

            const PairEnt pe = F.pairs[e];
            const int w0 = div_fast(ap0 * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) - pe.hw;
            int rem;
            const int kc = div_fast(ap * pe.ipq + pe.shq * ip, ip2, M0, rem);
            float dc[R];
            dc[0] = (float)(ip - rem) * pe.cdc;
            if (R == 2) dc[R - 1] = (float)(ip - rem + 2 * (ip - pe.ipq)) * pe.cdc - pe.dphi;
            const float4 *pn[B], *ps[B];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                pn[b] = stage + (size_t)((buf * B + b) * 2 + 0) * Lmax + (kc - w0);
                ps[b] = stage + (size_t)((buf * B + b) * 2 + 1) * Lmax + (kc - w0);
            }
            float acc[R][B][8];
#pragma unroll
            for (int rr = 0; rr < R; ++rr)
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int g = 0; g < 8; ++g) acc[rr][b][g] = 0.f;

            const int jend = pe.hw + R - 1;
            float jf = (float)(-pe.hw);
            for (int j = -pe.hw; j <= jend; ++j, jf += 1.0f) {
                float K[R];
#pragma unroll
                for (int rr = 0; rr < R; ++rr) {
                    const float d = fmaf(jf, pe.dphi, dc[rr]);
                    const float y = d * d;
                    float h = fmaf(y, pe.c3, pe.c2);
                    h = fmaf(y, h, pe.c1);
                    const float tp = fmaf(y, h, pe.A);          // t - 0.5
                    unsigned bits = __float_as_uint(tp + kMagic);
                    if (bits >= thresh) {                        // last table cell or beyond
                        const float t = tp + 0.5f;
                        if (t >= tmax - eps) {
                            if (t <= tmax + eps) {               // decide in fp64, image by image
                                const unsigned mask = sym_exact_mask(P, r, ka + rr, ip, pe.rq, kc + j, pe.ipq, t);
                                if (mask) {
                                    const float2 el = tab[P.ntab - 2];
                                    const float Ku = fmaf(fminf(t, tmax) - 0.5f, el.y, el.x);
#pragma unroll
                                    for (int b = 0; b < B; ++b) {
                                        const float4 mn = pn[b][j], ms = ps[b][j];
                                        const float mv[8] = {mn.x, mn.y, mn.z, mn.w, ms.x, ms.y, ms.z, ms.w};
#pragma unroll
                                        for (int g = 0; g < 8; ++g)
                                            if (mask & (1u << g)) acc[rr][b][g] = fmaf(Ku, mv[g], acc[rr][b][g]);
                                    }
                                }
                            }
                            bits = zero_bits;                    // K = 0 on the common path
                        }
                    }
                    const float2 el = tab[bits - kMagicBits];
                    K[rr] = fmaf(tp, el.y, el.x);
                }
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const float4 mn = pn[b][j], ms = ps[b][j];
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) {
                        acc[rr][b][0] = fmaf(K[rr], mn.x, acc[rr][b][0]);
                        acc[rr][b][1] = fmaf(K[rr], mn.y, acc[rr][b][1]);
                        acc[rr][b][2] = fmaf(K[rr], mn.z, acc[rr][b][2]);
                        acc[rr][b][3] = fmaf(K[rr], mn.w, acc[rr][b][3]);
                        acc[rr][b][4] = fmaf(K[rr], ms.x, acc[rr][b][4]);
                        acc[rr][b][5] = fmaf(K[rr], ms.y, acc[rr][b][5]);
                        acc[rr][b][6] = fmaf(K[rr], ms.z, acc[rr][b][6]);
                        acc[rr][b][7] = fmaf(K[rr], ms.w, acc[rr][b][7]);
                    }
                }
            }
#pragma unroll
            for (int rr = 0; rr < R; ++rr)
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int g = 0; g < 8; ++g) tot[rr][b][g] += acc[rr][b][g];
        }

        // store the 8 images of every valid base pixel
        const int start_n = P.start[r - 1], start_s = P.start[4 * N - r - 1];
        const bool south = (r != 2 * N);
#pragma unroll
        for (int rr = 0; rr < R; ++rr) {
            const int k = k0 + R * tid + rr;
            if (k <= klast) {
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        io.out[b][start_n + k + m * ip] = tot[rr][b][m] * P.omega;
                        if (south) io.out[b][start_s + k + m * ip] = tot[rr][b][4 + m] * P.omega;
                    }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct BeltDev {            // mirrors sc_belt.cu
    const PairEnt *pairs;
    const int *pair_off;
    const int *woff;
    const int4 *tiles;
    int ntiles;
    int *counter;
    int Lp, pw_max, nbuf;
};
cudaError_t launch_belt(const Dev &P, const BeltDev &F, const Maps &io, int B, int threads, size_t smem, int nsm,
                        cudaStream_t st);

struct FastCfg {            // per batch size
    bool ok = false;
    int threads = 0, R = 1, Lmax = 0;
    size_t smem = 0;
    int4 *tiles = nullptr;
    int ntiles = 0;
};

struct FastPlan {
    PairEnt *pairs = nullptr;
    int *pair_off = nullptr;
    int *counter = nullptr;
    int ntab_s = 0;
    int polar = 0;
    FastCfg cfg[kMaxB + 1];
    int nsm = 148;
    // belt kernel
    bool belt_ok = false;
    BeltDev belt{};
    int belt_threads = 0;
    size_t belt_smem = 0;
    int *woff = nullptr;
    int4 *belt_tiles = nullptr;
    int *belt_counter = nullptr;
};

template <int B, int R>
static cudaError_t launch_sym(const FastPlan *fp, const FastCfg &c, const Dev &P, const Maps &io, cudaStream_t st) {
    FastDev F{fp->pairs, fp->pair_off, c.tiles, c.ntiles, fp->counter, c.Lmax, fp->ntab_s, R};
    cudaError_t e = cudaFuncSetAttribute(sym_kernel<B, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(fp->counter, 0, sizeof(int), st);
    if (e != cudaSuccess) return e;
    const int grid = std::min(fp->nsm, c.ntiles);
    if (grid <= 0) return cudaSuccess;
    sym_kernel<B, R><<<grid, c.threads, c.smem, st>>>(P, F, io);
    return cudaGetLastError();
}

cudaError_t fast_convolve(FastPlan *fp, const Dev &P, const Maps &io, int B, cudaStream_t st, int *launches) {
    *launches = 0;
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return cudaErrorInvalidValue;
    const FastCfg &c = fp->cfg[B];
    cudaError_t e;
    switch (B) {
        case 1: e = launch_sym<1, 1>(fp, c, P, io, st); break;
        case 2: e = launch_sym<2, 1>(fp, c, P, io, st); break;
        case 3: e = launch_sym<3, 1>(fp, c, P, io, st); break;
        default: e = launch_sym<4, 1>(fp, c, P, io, st); break;
    }
    if (e != cudaSuccess) return e;
    *launches = c.ntiles > 0 ? 1 : 0;
    if (fp->belt_ok) {
        e = launch_belt(P, fp->belt, io, B, fp->belt_threads, fp->belt_smem, fp->nsm, st);
        if (e == cudaSuccess) ++*launches;
    }
    return e;
}

bool fast_available(const FastPlan *fp, int B) { return fp && B >= 1 && B <= kMaxB && fp->cfg[B].ok; }

void fast_plan_destroy(FastPlan *fp) {
    if (!fp) return;
    cudaFree(fp->pairs); cudaFree(fp->pair_off); cudaFree(fp->counter);
    for (auto &c : fp->cfg) cudaFree(c.tiles);
    cudaFree(fp->woff); cudaFree(fp->belt_tiles); cudaFree(fp->belt_counter);
    delete fp;
}

FastPlan *fast_plan_create(const Dev &P, const std::vector<double> &z, const std::vector<double> &s,
                           int max_batch, int *polar_rings, cudaError_t *err) {
    *err = cudaSuccess;
    *polar_rings = 0;
    const int N = P.nside, nr = 4 * N - 1;
    const int R = 1;
    int dev = 0, smem_optin = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int ntab_s = P.ntab - 1 + kTabPad;
    const size_t tab_bytes = ((size_t)ntab_s * 8 + 15) & ~(size_t)15;
    if (tab_bytes + 8192 > (size_t)smem_optin) return nullptr;       // table does not fit: generic only

    auto ipof = [&](int r) { return r < N ? r : (r <= 3 * N ? N : 4 * N - r); };
    auto shof = [&](int r) { return (r >= N && r <= 3 * N) ? ((r - N) & 1) : 0; };
    auto startof = [&](int r) -> int {
        if (r < N) return 2 * r * (r - 1);
        if (r <= 3 * N) return 2 * N * (N - 1) + (r - N) * 4 * N;
        const int m = 4 * N - r;
        return 12 * N * N - 2 * m * (m + 1);
    };
    const double tmax = (double)(P.ntab - 1);
    // largest |d| for which the 3-term polynomial of 1 - cos d is good to 0.004 table cells
    const double dmax = std::min(0.45, std::pow(0.004 * 20160.0 / tmax, 1.0 / 6.0));

    std::vector<PairEnt> pairs;
    std::vector<int> pair_off(1, 0);
    std::vector<char> eligible(2 * N + 1, 0);
    std::vector<std::vector<PairEnt>> per_ring(2 * N + 1);
    for (int r = 1; r <= 2 * N; ++r) {
        const int ip = ipof(r);
        bool ok = true;
        std::vector<PairEnt> &lst = per_ring[r];
        const int lo = std::max(1, r - (nr)), hi = nr;
        (void)lo; (void)hi;
        // walk outwards from r in both directions while rings can hold a neighbour
        auto consider = [&](int rq) -> bool {
            double A64 = 1.0 - (z[r - 1] * z[rq - 1] + s[r - 1] * s[rq - 1]);
            if (A64 < 0) A64 = 0;
            const double Bs = s[r - 1] * s[rq - 1] * P.scale;
            const double wmax = (tmax + 2.0 * (double)P.eps + 0.01 - A64 * P.scale) / Bs;
            if (wmax < 0) return false;
            const int ipq = ipof(rq);
            const double dphi = 2.0 * M_PI / (4.0 * ipq);
            const double H = wmax >= 2.0 ? M_PI : 2.0 * std::asin(std::sqrt(0.5 * wmax));
            const double rho1 = std::fabs(1.0 - (double)ipq / ip);
            const int hw = (int)std::floor(H / dphi + 0.5 + rho1 * (R - 1) + 1e-6);
            if ((hw + 1 + R) * dphi > dmax) ok = false;
            PairEnt e;
            e.A = (float)(A64 * P.scale - 0.5);
            e.c1 = (float)(Bs / 2.0); e.c2 = (float)(-Bs / 24.0); e.c3 = (float)(Bs / 720.0);
            e.dphi = (float)dphi;
            e.cdc = (float)(M_PI / (4.0 * (double)ip * (double)ipq));
            e.rq = rq; e.hw = hw; e.ipq = ipq; e.shq = shof(rq);
            e.start_n = startof(rq); e.start_s = startof(4 * N - rq);
            lst.push_back(e);
            return true;
        };
        std::vector<PairEnt> down;
        for (int rq = r; rq >= 1; --rq) if (!consider(rq)) break;
        std::reverse(lst.begin(), lst.end());
        for (int rq = r + 1; rq <= nr; ++rq) if (!consider(rq)) break;
        // the window of a whole quadrant must not wrap onto itself
        for (const PairEnt &e : lst) if (e.ipq + 2 * e.hw + 4 >= 4 * e.ipq) ok = false;
        eligible[r] = ok;
    }
    int polar = 0;
    for (int r = 1; r <= 2 * N; ++r) if (!eligible[r]) polar = r;
    if (polar >= 2 * N) return nullptr;                            // nothing for the fast kernel
    // slots: base rings polar+1 .. 2N
    std::vector<int> slot_of(2 * N + 1, -1);
    for (int r = polar + 1; r <= 2 * N; ++r) {
        slot_of[r] = (int)pair_off.size() - 1;
        pairs.insert(pairs.end(), per_ring[r].begin(), per_ring[r].end());
        pair_off.push_back((int)pairs.size());
    }

    FastPlan *fp = new FastPlan;
    fp->ntab_s = ntab_s; fp->polar = polar; fp->nsm = nsm;
    auto fail = [&](cudaError_t e) { *err = e; fast_plan_destroy(fp); return (FastPlan *)nullptr; };
    cudaError_t e;
    if ((e = cudaMalloc((void **)&fp->pairs, std::max<size_t>(pairs.size(), 1) * sizeof(PairEnt))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc((void **)&fp->pair_off, pair_off.size() * sizeof(int))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc((void **)&fp->counter, sizeof(int))) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pairs, pairs.data(), pairs.size() * sizeof(PairEnt), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pair_off, pair_off.data(), pair_off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);

    // ---- belt kernel: base rings whose input rings all have 4N pixels ------------------------------
    std::vector<char> is_belt(2 * N + 1, 0);
    const bool no_belt = std::getenv("SC_NO_BELT") != nullptr;
    if (!no_belt && N % 128 == 0 && N >= 512) {
        const int bthreads = std::min(kMaxThreads, N / 4);
        const int T = 4 * bthreads;
        std::vector<int> woff(pairs.size(), 0);
        std::vector<int4> btiles;
        int pw_max = 0, hw_max = 0;
        for (int r = 2 * N; r > polar; --r) {
            if (ipof(r) != N) continue;
            bool all = true;
            for (const PairEnt &pe : per_ring[r]) if (pe.ipq != N) { all = false; break; }
            if (!all) continue;
            is_belt[r] = 1;
            int off = 0;
            const int base = pair_off[slot_of[r]];
            for (size_t i = 0; i < per_ring[r].size(); ++i) {
                woff[base + i] = off;
                off += 6 + 2 * per_ring[r][i].hw + 8;            // kPwPad + 2hw + 8 (sc_belt.cu)
                hw_max = std::max(hw_max, per_ring[r][i].hw);
            }
            pw_max = std::max(pw_max, off);
            for (int k0 = 0; k0 < N; k0 += T) btiles.push_back(make_int4(r, k0, slot_of[r], 0));
        }
        if (!btiles.empty()) {
            const int Lp = T - 4 + 4 * ((2 * hw_max + 4 + 3 + 3) >> 2);
            int nbuf = 0;
            size_t bsmem = 0;
            for (int nb : {3, 2}) {
                bsmem = (size_t)nb * 8 * Lp * 4 + (size_t)pw_max * 8;
                if (bsmem + 2048 <= (size_t)smem_optin) { nbuf = nb; break; }
            }
            if (nbuf) {
                if ((e = cudaMalloc((void **)&fp->woff, woff.size() * sizeof(int))) != cudaSuccess) return fail(e);
                if ((e = cudaMemcpy(fp->woff, woff.data(), woff.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
                if ((e = cudaMalloc((void **)&fp->belt_tiles, btiles.size() * sizeof(int4))) != cudaSuccess) return fail(e);
                if ((e = cudaMemcpy(fp->belt_tiles, btiles.data(), btiles.size() * sizeof(int4), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
                if ((e = cudaMalloc((void **)&fp->belt_counter, sizeof(int))) != cudaSuccess) return fail(e);
                fp->belt = BeltDev{fp->pairs, fp->pair_off, fp->woff, fp->belt_tiles, (int)btiles.size(),
                                   fp->belt_counter, Lp, pw_max, nbuf};
                fp->belt_threads = bthreads; fp->belt_smem = bsmem; fp->belt_ok = true;
            } else {
                std::fill(is_belt.begin(), is_belt.end(), 0);
            }
        }
    }

    // per batch size: threads per CTA so that table + double-buffered stage fit in shared memory
    (void)max_batch;
    for (int B = 1; B <= kMaxB; ++B) {
        FastCfg &c = fp->cfg[B];
        for (int threads : {512, 384, 256, 192, 128, 64}) {
            const int T = threads * R;
            int Lmax = 0;
            std::vector<int4> tiles;
            // larger rings first: long tiles start early, ragged small ones fill the tail
            for (int r = 2 * N; r > polar; --r) {
                if (is_belt[r]) continue;
                const int ip = ipof(r), sh = shof(r);
                for (int k0 = 0; k0 < ip; k0 += T) {
                    tiles.push_back(make_int4(r, k0, slot_of[r], 0));
                    const int klast = std::min(k0 + T, ip) - 1;
                    for (const PairEnt &pe : per_ring[r]) {
                        const int w0 = ((2 * k0 + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) - pe.hw;
                        const int L = ((2 * klast + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) + pe.hw + R - w0;
                        Lmax = std::max(Lmax, L);
                    }
                }
            }
            Lmax = (Lmax + 3) & ~3;
            const size_t smem = tab_bytes + (size_t)2 * B * 2 * Lmax * 16;
            if (smem + 1024 > (size_t)smem_optin) continue;
            c.threads = threads; c.R = R; c.Lmax = Lmax; c.smem = smem; c.ntiles = (int)tiles.size();
            if ((e = cudaMalloc((void **)&c.tiles, tiles.size() * sizeof(int4))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(c.tiles, tiles.data(), tiles.size() * sizeof(int4), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            c.ok = true;
            break;
        }
    }
    *polar_rings = polar;
    return fp;
}

}  // namespace sc
