// sc_belt.cu -- the belt kernel: output rings whose whole disc lies in the equatorial belt.
//
// In the belt every ring has 4N pixels, so the pair weight K(p, q) depends only on
// (ring r, ring r', azimuthal offset j): the convolution is a stencil with per-ring-pair taps
// (SURVEY.md 8f-1).  Per tile (one ring, T = 4 x threads consecutive base pixels of the first
// quadrant) the kernel
//   A. evaluates the taps W[r'][j] ONCE -- same fp32 geometry, table lookup and inclusion rule as
//      the sym kernel (uncertain taps are set to 0 and decided per pixel pair in fp64 afterwards) --
//      and stores them in shared memory as pairs (w[x], w[x-1]);
//   B. a dedicated producer warp stages, for every input ring, the runs of the 8 symmetric images
//      (4 quadrants x north/south) as 8 contiguous planes with TMA bulk copies (cp.async.bulk) into a
//      ring of NBUF buffers guarded by full/empty mbarriers -- no block-wide barrier per ring;
//   C. runs the stencil: a thread owns 4 consecutive pixels x 8 images = 32 accumulators, reads
//      LDS.128 (4 positions of one image, conflict free) and issues packed FFMA2 over pixel pairs:
//      (acc_k, acc_k+1) += (w[s-k], w[s-k-1]) * m[s].   One FMA per pair: 4 B of shared-memory traffic
//      per 4 pairs, no geometry in the inner loop.
#include "sc_fast.cuh"

namespace sc {

constexpr int kPwPad = 6;     // zero pairs in front of every tap array (alignment offset <= 3, pixel offset <= 3)
constexpr int kMaxExc = 32;   // uncertain taps per tile that can be listed (more -> counted, see below)

struct BeltDev {
    const PairEnt *pairs;
    const int *pair_off;
    const int *woff;          // per pair entry: offset (in float2) of its tap array within the tile's tap buffer
    const int4 *tiles;        // (ring, k0, slot, 0)
    int ntiles;
    int *counter;
    int Lp;                   // floats per staged plane (multiple of 4)
    int pw_max;               // float2 entries of the tap buffer
    int nbuf;                 // stage buffers
};

static __device__ __noinline__ unsigned belt_exact_mask(const Dev &P, int r, int k, int rq, int kq) {
    const int N = P.nside, N4 = 4 * N;
    unsigned mask = 0;
    kq %= N4; if (kq < 0) kq += N4;
    for (int h = 0; h < 2; ++h) {
        const int rp_i = h ? N4 - r : r, rq_i = h ? N4 - rq : rq;
        for (int m = 0; m < 4; ++m) {
            int kp_i = k + m * N; if (kp_i >= N4) kp_i -= N4;
            int kq_i = kq + m * N; if (kq_i >= N4) kq_i -= N4;
            if (exact_included(P, rp_i, kp_i, rq_i, kq_i, 0.f, nullptr)) mask |= 1u << (4 * h + m);
        }
    }
    return mask;
}

// One stencil tap: weight of the pair at azimuthal pixel offset j (same arithmetic as the sym kernel).
// Returns the weight (0 if excluded or uncertain); `unc` is set for taps inside the guard band, whose
// inclusion is decided per pixel pair in fp64 later; Ku is the weight such a pair gets if included.
__device__ __forceinline__ float belt_tap(const Dev &P, const PairEnt &pe, int j, float dcc, bool &unc, float &Ku) {
    const float d = fmaf((float)j, pe.dphi, dcc);
    const float y = d * d;
    float h = fmaf(y, pe.c3, pe.c2);
    h = fmaf(y, h, pe.c1);
    const float tp = fmaf(y, h, pe.A);
    const unsigned bits = __float_as_uint(tp + kMagic);
    unc = false;
    if (bits >= kMagicBits + (unsigned)(P.ntab - 2)) {
        const float t = tp + 0.5f;
        if (t >= P.tmax - P.eps) {
            if (t <= P.tmax + P.eps) {
                const float2 el = __ldg(&P.tabh[P.ntab - 2]);
                unc = true;
                Ku = fmaf(fminf(t, P.tmax) - 0.5f, el.y, el.x);
            }
            return 0.f;
        }
    }
    const float2 el = __ldg(&P.tabh[bits - kMagicBits]);
    return fmaf(tp, el.y, el.x);
}

__device__ __forceinline__ void bar_consumers(int n) { asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory"); }

// All warps run the stencil; warp 0 is also the TMA producer: after each ring it consumes it issues
// the copies of the ring NBUF-1 ahead in the (tile, map, ring) sequence (its own cursor, so it runs
// across map and tile boundaries).  Warps meet only through the full/empty mbarriers of the NBUF
// stage buffers: there is no block-wide barrier in the ring loop.
template <int NBUF>
__global__ void __launch_bounds__(kMaxThreads, 1)
belt_kernel(const Dev P, const BeltDev F, const Maps io, const int B) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, NT = blockDim.x;
    const int T = 4 * NT;
    const int N = P.nside, N4 = 4 * N;
    const int Lp = F.Lp;
    float *stage = reinterpret_cast<float *>(smem_raw);                         // [NBUF][8][Lp]
    float2 *pw = reinterpret_cast<float2 *>(smem_raw + (size_t)NBUF * 8 * Lp * 4);   // [pw_max]
    __shared__ unsigned long long full_bar[NBUF], empty_bar[NBUF];
    __shared__ int s_nexc;
    __shared__ int s_exc_e[kMaxExc], s_exc_j[kMaxExc];
    __shared__ float s_exc_k[kMaxExc];

    if (tid == 0) {
        for (int i = 0; i < NBUF; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], NT / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned it = 0;                          // rings processed so far: buffer it % NBUF, use it / NBUF

    // ---- producer cursor (meaningful in warp 0 only) ----------------------------------------------
    unsigned pit = 0;                         // rings issued so far
    int p_tile = blockIdx.x, p_b = 0, p_e = 0, p_e1 = 0, p_r = 0, p_k0 = 0;
    bool p_valid = false;
    auto produce = [&]() {                    // issue the TMA copies of the next ring, if any
        if (!p_valid) {
            if (p_tile >= F.ntiles) return;
            const int4 tl = F.tiles[p_tile];
            p_r = tl.x; p_k0 = tl.y; p_e = F.pair_off[tl.z]; p_e1 = F.pair_off[tl.z + 1]; p_b = 0;
            p_valid = true;
        }
        const int lane = tid & 31;
        const int buf = pit % NBUF;
        const unsigned use = pit / NBUF;
        const int sh = (p_r - N) & 1;
        const PairEnt pe = F.pairs[p_e];
        const int delta = (1 - sh + pe.shq) >> 1;
        const int first_pos = p_k0 + delta - pe.hw;
        const int w0a = first_pos & ~3;
        const int len = T - 4 + 4 * ((2 * pe.hw + 4 + (first_pos - w0a) + 3) >> 2);   // floats
        unsigned long long *bar = &full_bar[buf];
        mbar_wait(&empty_bar[buf], (use & 1u) ^ 1u);          // every warp has released this buffer
        if (lane == 0) mbar_expect_tx(bar, (unsigned)(8 * len * 4));
        __syncwarp();
        if (lane < 8) {                                       // one plane per lane
            const float *__restrict__ in = io.in[p_b];
            const int m = lane & 3;
            const int base = (lane < 4) ? pe.start_n : pe.start_s;
            int s0 = (w0a + m * N) % N4; if (s0 < 0) s0 += N4;
            float *dst = stage + ((size_t)buf * 8 + lane) * Lp;
            const int first = min(len, N4 - s0);
            tma_load_1d(dst, in + base + s0, (unsigned)(first * 4), bar);
            if (first < len) tma_load_1d(dst + first, in + base, (unsigned)((len - first) * 4), bar);
        }
        ++pit;
        if (++p_e == p_e1) {                                  // next map of this tile, or next tile
            if (++p_b < B) p_e = F.pair_off[F.tiles[p_tile].z];
            else { p_tile += gridDim.x; p_valid = false; }
        }
    };
    if (tid < 32) for (int i = 0; i < NBUF - 1; ++i) produce();

    // ==================================== consumers ====================================
    const int lane = tid & 31;
    for (int tile = blockIdx.x; tile < F.ntiles; tile += gridDim.x) {
        const int4 tl = F.tiles[tile];
        const int r = tl.x, k0 = tl.y;
        const int sh = (r - N) & 1;
        const int e0 = F.pair_off[tl.z], e1 = F.pair_off[tl.z + 1];

        bar_consumers(NT);                    // previous tile completely finished (taps, exception list)
        if (tid == 0) s_nexc = 0;
        bar_consumers(NT);
        // ---- A. taps ----------------------------------------------------------------------------
        for (int e = e0; e < e1; ++e) {
            const PairEnt pe = F.pairs[e];
            const int wo = F.woff[e];
            // nearest pixel of ring rq in azimuth: kc = k + delta, at angle dcc from p.  In the belt
            // Y = N (2k + 1 - sh + shq), so delta = (1 - sh + shq) >> 1 and the remainder is N or 0.
            const int Yk = 1 - sh + pe.shq;
            const float dcc = (float)(N - ((Yk & 1) ? N : 0)) * pe.cdc;
            const int nx = kPwPad + 2 * pe.hw + 8;               // x = -kPwPad .. 2hw+7
            for (int xi = tid; xi < nx; xi += NT) {
                const int x = xi - kPwPad;
                float w2[2];
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int xx = x - q;
                    float w = 0.f;
                    if (xx >= 0 && xx <= 2 * pe.hw) {
                        bool unc; float Ku;
                        w = belt_tap(P, pe, xx - pe.hw, dcc, unc, Ku);
                        if (unc && q == 0) {                              // list every uncertain tap once
                            const int slot = atomicAdd(&s_nexc, 1);
                            if (slot < kMaxExc) { s_exc_e[slot] = e; s_exc_j[slot] = xx - pe.hw; s_exc_k[slot] = Ku; }
                        }
                    }
                    w2[q] = w;
                }
                pw[wo + xi] = make_float2(w2[0], w2[1]);
            }
        }
        bar_consumers(NT);
        const int nexc = s_nexc;

        // ---- C. per map: the stencil over the staged rings ---------------------------------------
        for (int b = 0; b < B; ++b) {
            const float *__restrict__ in = io.in[b];
            float2 tot01[8], tot23[8], acc01[8], acc23[8];
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                tot01[g] = make_float2(0.f, 0.f); tot23[g] = make_float2(0.f, 0.f);
                acc01[g] = make_float2(0.f, 0.f); acc23[g] = make_float2(0.f, 0.f);
            }
            int ntaps = 0;
            for (int e = e0; e < e1; ++e, ++it) {
                const int buf = it % NBUF;
                const unsigned use = it / NBUF;
                const PairEnt pe = F.pairs[e];
                const int delta = (1 - sh + pe.shq) >> 1;
                const int first_pos = k0 + delta - pe.hw;
                const int a0 = first_pos - (first_pos & ~3);
                const int ng = (2 * pe.hw + 4 + a0 + 3) >> 2;
                const float2 *pwe = pw + F.woff[e] + kPwPad - a0;         // pwe[4 g + i] = P[4 g + i - a0]
                const float *pl = stage + (size_t)buf * 8 * Lp + 4 * tid;
                mbar_wait(&full_bar[buf], use & 1u);
                for (int g4 = 0; g4 < ng; ++g4) {
                    // pairs P[x] = (w[x], w[x-1]) for x = 4 g4 - 2 .. 4 g4 + 3 (relative to pwe)
                    float2 pwr[6];
#pragma unroll
                    for (int i = 0; i < 6; ++i) pwr[i] = pwe[4 * g4 - 2 + i];
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        float4 mv[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            mv[q] = *reinterpret_cast<const float4 *>(pl + (size_t)(half * 4 + q) * Lp + 4 * g4);
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const int g = half * 4 + q;
                            const float mm[4] = {mv[q].x, mv[q].y, mv[q].z, mv[q].w};
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const float2 m2 = make_float2(mm[i], mm[i]);
                                acc01[g] = __ffma2_rn(pwr[2 + i], m2, acc01[g]);
                                acc23[g] = __ffma2_rn(pwr[i], m2, acc23[g]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty_bar[buf]);            // this warp is done with the buffer
                if (tid < 32) produce();                                // keep NBUF-1 rings in flight
                ntaps += 2 * pe.hw + 1;
                if (ntaps >= 48 || e + 1 == e1) {
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        tot01[g].x += acc01[g].x; tot01[g].y += acc01[g].y;
                        tot23[g].x += acc23[g].x; tot23[g].y += acc23[g].y;
                        acc01[g] = make_float2(0.f, 0.f); acc23[g] = make_float2(0.f, 0.f);
                    }
                    ntaps = 0;
                }
            }

            // ---- uncertain taps: canonical fp64 decision per pixel pair and image ------------------
            if (nexc > 0) {
                float tt[4][8];
#pragma unroll
                for (int g = 0; g < 8; ++g) { tt[0][g] = tot01[g].x; tt[1][g] = tot01[g].y; tt[2][g] = tot23[g].x; tt[3][g] = tot23[g].y; }
                auto apply = [&](const PairEnt &pe, int j, float Ku) {
                    const int delta = (1 - sh + pe.shq) >> 1;
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        const int k = k0 + 4 * tid + rr;
                        const int kq = k + delta + j;
                        const unsigned mask = belt_exact_mask(P, r, k, pe.rq, kq);
                        int kqw = kq % N4; if (kqw < 0) kqw += N4;
#pragma unroll
                        for (int g = 0; g < 8; ++g) {
                            if (mask & (1u << g)) {
                                int kk = kqw + (g & 3) * N; if (kk >= N4) kk -= N4;
                                tt[rr][g] = fmaf(Ku, __ldg(in + ((g < 4) ? pe.start_n : pe.start_s) + kk), tt[rr][g]);
                            }
                        }
                    }
                };
                if (nexc <= kMaxExc) {
                    for (int i = 0; i < nexc; ++i) apply(F.pairs[s_exc_e[i]], s_exc_j[i], s_exc_k[i]);
                } else {                              // list overflow: rescan every tap (never seen in practice)
                    for (int e = e0; e < e1; ++e) {
                        const PairEnt pe = F.pairs[e];
                        const int Yk = 1 - sh + pe.shq;
                        const float dcc = (float)(N - ((Yk & 1) ? N : 0)) * pe.cdc;
                        for (int j = -pe.hw; j <= pe.hw; ++j) {
                            bool unc; float Ku;
                            belt_tap(P, pe, j, dcc, unc, Ku);
                            if (unc) apply(pe, j, Ku);
                        }
                    }
                }
#pragma unroll
                for (int g = 0; g < 8; ++g) { tot01[g] = make_float2(tt[0][g], tt[1][g]); tot23[g] = make_float2(tt[2][g], tt[3][g]); }
            }

            // ---- store: 4 consecutive pixels per image -> one 16-byte store ------------------------
            const int start_n = P.start[r - 1], start_s = P.start[N4 - r - 1];
            const bool south = (r != 2 * N);
            const int k = k0 + 4 * tid;
            float *__restrict__ out = io.out[b];
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                if (g >= 4 && !south) break;
                const float4 v = make_float4(tot01[g].x * P.omega, tot01[g].y * P.omega, tot23[g].x * P.omega, tot23[g].y * P.omega);
                *reinterpret_cast<float4 *>(out + ((g < 4) ? start_n : start_s) + k + (g & 3) * N) = v;
            }
        }
    }
}

// host ------------------------------------------------------------------------------------------
cudaError_t launch_belt(const Dev &P, const BeltDev &F, const Maps &io, int B, int threads, size_t smem, int nsm,
                        cudaStream_t st) {
    cudaError_t e;
    if (F.nbuf == 3) {
        e = cudaFuncSetAttribute(belt_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    } else {
        e = cudaFuncSetAttribute(belt_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int grid = F.ntiles < nsm ? F.ntiles : nsm;
    if (F.nbuf == 3) belt_kernel<3><<<grid, threads, smem, st>>>(P, F, io, B);
    else belt_kernel<2><<<grid, threads, smem, st>>>(P, F, io, B);
    return cudaGetLastError();
}

}  // namespace sc
