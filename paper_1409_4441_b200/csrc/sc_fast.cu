// sc_fast.cu -- the fast convolution kernel ("sym kernel") and its plan data.
//
// Design:
//  * HEALPix is invariant under phi -> phi + pi/2 and z -> -z, so the weight K(p, q) of a pair is
//    shared by its 8 images (4 quadrants x north/south).  A thread owns a BASE pixel (ring r <= 2N,
//    in-ring index k < ring_length/4), evaluates the pair geometry and the table lookup once and
//    FMA-accumulates 8 outputs (times B maps): (5 + 1 + 8 B) FMA-pipe operations per 8 B pair-maps.
//  * A persistent CTA works through tiles (runs of consecutive base pixels on one ring; several short runs
//    of the rings near the pole are packed into one tile).  It is warp-specialised: a producer warpgroup
//    stages, for every input ring within theta_max, the needed run of map values -- the 4 quadrant images
//    interleaved as float4, north and south planes -- into shared memory with cp.async, reporting to
//    full/empty mbarriers; 1-3 consumer warpgroups (setmaxnreg gives them the producers' registers) run the
//    pair loop, R adjacent base pixels per thread.  No block-wide barrier after the prologue.
//  * Pair geometry in fp32 without cancellation: t = A + B (1 - cos d) with A, B per ring pair from
//    fp64, d = azimuth difference built from the INTEGER pixel offset (exact) times the ring's pixel
//    spacing; 1 - cos d by a 4-term even polynomial (|d| <= ~0.9 rad on the rings this kernel takes;
//    the few rings next to the poles go to the generic kernel).
//  * Table lookup: magic-number rounding gives the cell index; K = a_i + t b_i (one FFMA); the
//    16K-entry (a, b) table lives in shared memory (128 KB).
//  * Inclusion: t < tmax - 1 needs no test at all (fast path); the last cell and everything beyond
//    takes a branch: t > tmax + eps -> excluded, |t - tmax| <= eps -> canonical fp64 test for each
//    of the 8 images separately (bit-exact with the oracle), else included.
//  * Sums: per-ring partial sums added to running totals (registers, or tensor memory via tcgen05.ld/st for
//    the 384-consumer variant on mid-size discs); a single set for discs of at most 700 pixels.
#include "sc_fast.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <type_traits>
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

// Shared-memory slot (16-byte unit) of staged position i.  A thread owns R adjacent base pixels, so the
// 8 lanes of a quarter warp (one LDS.128 wavefront) read positions R apart.  XOR-ing the low bits with the
// index of the 8-position block spreads such a stride over all 8 bank groups for every alignment, with no
// padding (brute-force checked: 1 wavefront per quarter warp for stride 2 and 4; stride 1 needs nothing).
template <int R> __host__ __device__ __forceinline__ int slot_of_pos(int i) {
    return R == 1 ? i : (R == 2 ? i ^ ((i >> 3) & 1) : i ^ ((i >> 3) & 3));
}

// Packed fp32 helpers (FFMA2 / FADD2 / FMUL2 on sm_100a; a scalar operand is broadcast by the hardware).
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }

constexpr int kSymProd = 128;     // producer threads per CTA (one warpgroup): they only issue cp.async
constexpr int kSymBuf = 2;        // stage buffers
constexpr int kSymChunksDflt = 5;  // latitude chunks of the cap rings for the pipelined host entry
constexpr int kBeltChunksDflt = 6; // same for the belt rings

// Tile n of this CTA: rows of gridDim.x tiles, alternate rows reversed ("snake") so that the CTAs
// get equal shares of the work-sorted tile list without a global counter.
__device__ __forceinline__ int snake_tile(int row, int G, int bid) { return row * G + ((row & 1) ? G - 1 - bid : bid); }

__device__ __forceinline__ float4 lds128(unsigned a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}

// Warp-specialised: the first blockDim.x - kSymProd threads are consumers (pair loop), the last
// kSymProd threads are producers (staging).  They meet only through the full/empty mbarriers of the
// kSymBuf stage buffers; there is no block-wide barrier after the prologue.
// TOT: per-step partial sums are added to a second accumulator set (pairwise-like summation; needed for
// discs of thousands of pixels, costs 8 R B registers).
// Z: two-zone table (lookup at tau(t), R11).  TM: the second accumulator set lives in tensor memory.
template <int B, int R, int NC, bool TOT, bool Z, bool TM>
__global__ void __launch_bounds__(NC + kSymProd, 1)
sym_kernel(const Dev P, const FastDev F, const Maps io) {
    static_assert(R == 1 || R == 2 || R == 4, "R");
    constexpr int RP = (R + 1) / 2;                      // pixel pairs per thread
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);
    const unsigned stage_sh = smem_u32(smem_raw + (((size_t)F.ntab_s * 8 + 127) & ~(size_t)127));
    __shared__ unsigned long long full_bar[kSymBuf], empty_bar[kSymBuf];
    const int tid = threadIdx.x;
    const int N = P.nside;
    const int Ltot = F.Ltot;
    const int G = gridDim.x, bid = blockIdx.x;
    const int nrows = (F.ntiles + G - 1) / G;

    for (int i = tid; i < F.ntab_s; i += blockDim.x) tab[i] = P.tabh[i];
    if (tid == 0) {
        for (int i = 0; i < kSymBuf; ++i) { mbar_init(&full_bar[i], kSymProd); mbar_init(&empty_bar[i], NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ unsigned s_tmem;
    if (TM && tid < 32) {                                  // 128 TMEM columns: warp w uses lanes 32 (w % 4) .., columns 32 (w / 4) ..
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(&s_tmem)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (TM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    unsigned it = 0;                                     // steps so far: buffer it % kSymBuf, use it / kSymBuf
    int rem_unused;

    // register budget: the launch gives every thread 65536 / (NC + 128) registers (rounded down to a
    // multiple of 8); the producer warpgroup hands most of its share to the consumer warpgroups
    if (tid >= NC) {
        // ======================================= producers =======================================
        if (NC == 256 || NC == 384) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const int pt = tid - NC;
        const int m = pt & 3;                            // quadrant image staged by this thread
        for (int row = 0; row < nrows; ++row) {
            const int tile = snake_tile(row, G, bid);
            if (tile >= F.ntiles) continue;
            const SymTile *tl = F.tiles + tile;
            const int nsub = __ldg(&tl->nsub), nsteps = __ldg(&tl->nsteps);
            for (int step = 0; step < nsteps; ++step, ++it) {
                const int buf = it % kSymBuf;
                // runs to stage for this step, worked out BEFORE waiting for the buffer so that the
                // table reads (global memory) are off the critical path
                int kq0[kMaxSub], Ls[kMaxSub], nqs[kMaxSub], sn[kMaxSub], ss[kMaxSub];
                unsigned d0[kMaxSub];
#pragma unroll
                for (int s = 0; s < kMaxSub; ++s) {
                    Ls[s] = 0;
                    if (s >= nsub) continue;
                    const int ne = __ldg(&tl->sub[s].ne);
                    if (step >= ne) continue;
                    const int r = __ldg(&tl->sub[s].r), k0 = __ldg(&tl->sub[s].k0), n = __ldg(&tl->sub[s].n);
                    const int soff = __ldg(&tl->sub[s].soff);
                    const PairEnt *pe = F.pairs + (__ldg(&tl->sub[s].e0) + step);
                    const int2 pa = __ldg(reinterpret_cast<const int2 *>(&pe->rq));       // rq, hw
                    const int2 pb = __ldg(reinterpret_cast<const int2 *>(&pe->ipq));      // ipq, shq
                    const int2 ps = __ldg(reinterpret_cast<const int2 *>(&pe->start_n));  // start_n, start_s
                    const int hw = pa.y, ipq = pb.x, shq = pb.y;
                    const int ips = r < N ? r : N;
                    const int shs = (r >= N) ? ((r - N) & 1) : 0;
                    const unsigned M0s = 0xFFFFFFFFu / (unsigned)(2 * ips);
                    const int nq = 4 * ipq;
                    const int a0s = 2 * k0 + 1 - shs, als = 2 * (k0 + n - 1) + 1 - shs;
                    const int w0 = div_fast(a0s * ipq + shq * ips, 2 * ips, M0s, rem_unused) - hw;
                    Ls[s] = div_fast(als * ipq + shq * ips, 2 * ips, M0s, rem_unused) + hw + R - w0;
                    int k = w0 + m * ipq + nq;           // in [0, 2 nq)
                    if (k >= nq) k -= nq;
                    kq0[s] = k; nqs[s] = nq; sn[s] = ps.x; ss[s] = ps.y;
                    d0[s] = stage_sh + (unsigned)((buf * B * 2) * Ltot + soff) * 16u + 4u * m;
                }
                mbar_wait_sleep(&empty_bar[buf], ((it / kSymBuf) & 1u) ^ 1u);   // every consumer warp released it
#pragma unroll
                for (int s = 0; s < kMaxSub; ++s) {
                    for (int i = pt >> 2; i < Ls[s]; i += kSymProd / 4) {
                        int kq = kq0[s] + i;             // L < nq: one wrap at most
                        if (kq >= nqs[s]) kq -= nqs[s];
                        const unsigned d = d0[s] + 16u * (unsigned)slot_of_pos<R>(i);
#pragma unroll
                        for (int b = 0; b < B; ++b) {
                            cp_async4_s(d + (unsigned)(b * 2 * Ltot) * 16u, io.in[b] + sn[s] + kq);
                            cp_async4_s(d + (unsigned)((b * 2 + 1) * Ltot) * 16u, io.in[b] + ss[s] + kq);
                        }
                    }
                }
                cp_async_mbar_arrive(&full_bar[buf]);   // arrives when this thread's copies have landed
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        return;
    }

    // ========================================= consumers =========================================
    if (NC == 256) asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    if (NC == 384) asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
    const int warp = tid >> 5, lane = tid & 31;
    const unsigned taddr = TM ? s_tmem + ((((unsigned)warp & 3u) * 32u) << 16) + ((unsigned)warp >> 2) * 32u : 0u;
    const unsigned thresh = kMagicBits + (unsigned)(P.ntab - 2);   // bits of the last table cell
    const float tmax = P.tmax, eps = P.eps;
    // shared-memory byte address of tab[0] minus 8 kMagicBits (mod 2^32): tab[bits - kMagicBits] = [tab_sh + 8 bits]
    // (kept opaque: otherwise the compiler re-derives it from the CTA's shared window inside the pair loop)
    unsigned tab_sh = smem_u32(tab) - kMagicBits * 8u;
    asm volatile("mov.u32 %0, %0;" : "+r"(tab_sh));

    for (int row = 0; row < nrows; ++row) {
        const int tile = snake_tile(row, G, bid);
        if (tile >= F.ntiles) continue;
        const SymTile *tl = F.tiles + tile;
        const int nsub = __ldg(&tl->nsub), nsteps = __ldg(&tl->nsteps);
        int si = 0;
        for (int s = 1; s < nsub; ++s) if (warp >= __ldg(&tl->sub[s].w0)) si = s;
        SubTile me;
        {
            const int4 *q = reinterpret_cast<const int4 *>(&tl->sub[si]);
            const int4 a = __ldg(q), b = __ldg(q + 1);
            me.r = a.x; me.k0 = a.y; me.n = a.z; me.e0 = a.w; me.ne = b.x; me.w0 = b.y; me.nw = b.z; me.soff = b.w;
        }
        const bool active = warp < me.w0 + me.nw;

        const int r = me.r, k0 = me.k0;
        const int ip = r < N ? r : N;                  // base rings are rings 1 .. 2N
        const int ip2 = 2 * ip;
        const unsigned M0 = 0xFFFFFFFFu / (unsigned)ip2;
        const int sh = (r >= N) ? ((r - N) & 1) : 0;
        const int klast = k0 + me.n - 1;
        const int kmine = k0 + R * (32 * (warp - me.w0) + lane);
        const int ka = min(kmine, klast);
        const int ap = 2 * ka + 1 - sh, ap0 = 2 * k0 + 1 - sh;

        float2 tot[R][B][4];
#pragma unroll
        for (int rr = 0; rr < R; ++rr)
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int g = 0; g < 4; ++g) tot[rr][b][g] = f2(0.f);
        float2 acc[R][B][4];
#pragma unroll
        for (int rr = 0; rr < R; ++rr)
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int g = 0; g < 4; ++g) acc[rr][b][g] = f2(0.f);

        bool flushed = false;                              // TM: the totals in tensor memory are valid
        PairEnt pe_next = F.pairs[me.e0];
        for (int step = 0; step < nsteps; ++step, ++it) {
            const int buf = it % kSymBuf;
            const PairEnt pe = pe_next;
            if (step + 1 < me.ne) pe_next = F.pairs[me.e0 + step + 1];       // prefetch under the pair loop
            mbar_wait(&full_bar[buf], (it / kSymBuf) & 1u);
            if (active && step < me.ne) {
                const int w0 = div_fast(ap0 * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) - pe.hw;
                int rem;
                const int kc = div_fast(ap * pe.ipq + pe.shq * ip, ip2, M0, rem);
                // azimuth of input pixel kc + j seen from base pixel ka + rr:  d = dcr[rr] + j dphi'
                float dcr[R];
#pragma unroll
                for (int rr = 0; rr < R; ++rr) dcr[rr] = (float)(ip - rem - 2 * rr * pe.ipq) * pe.cdc;
                // staged position of input pixel kc + j: i0 + j (slot_of_pos: padded against bank conflicts)
                const int i0 = kc - w0;
                unsigned pn[B];                          // shared address of this sub-tile's north plane, map b
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    pn[b] = stage_sh + (unsigned)(((buf * B + b) * 2) * Ltot + me.soff) * 16u;
                    asm volatile("mov.u32 %0, %0;" : "+r"(pn[b]));      // one register, not re-derived per position
                }
                const unsigned south = (unsigned)Ltot * 16u;

                // last table cell or the zero cell after it (rare): exact decision where needed
                auto slow = [&](int rr, float tpv, unsigned &cb, int pos) {
                    const float t = tpv + 0.5f;
                    if (t >= tmax - eps) {
                        if (t <= tmax + eps) {                   // decide in fp64, image by image
                            const unsigned mask = sym_exact_mask(P, r, ka + rr, ip, pe.rq, kc + pos - i0, pe.ipq, t);
                            if (mask) {
                                const float2 el = tab[P.ntab - 2];
                                float xk = fminf(t, tmax) - 0.5f;
                                if (Z) { int jz; zoned_cell(P, fminf(t, tmax), jz, xk); xk -= 0.5f; }   // last cell, centred form
                                const float Ku = fmaf(xk, el.y, el.x);
#pragma unroll
                                for (int b = 0; b < B; ++b) {
                                    const unsigned a = pn[b] + 16u * (unsigned)slot_of_pos<R>(pos);
                                    const float4 mn = lds128(a), ms = lds128(a + south);
                                    const float mv[8] = {mn.x, mn.y, mn.z, mn.w, ms.x, ms.y, ms.z, ms.w};
#pragma unroll
                                    for (int g = 0; g < 4; ++g) {
                                        if (mask & (1u << (2 * g))) acc[rr][b][g].x = fmaf(Ku, mv[2 * g], acc[rr][b][g].x);
                                        if (mask & (2u << (2 * g))) acc[rr][b][g].y = fmaf(Ku, mv[2 * g + 1], acc[rr][b][g].y);
                                    }
                                }
                            }
                        }
                        cb = thresh + 1u;                        // zero cell
                    }
                };

                const float2 dphi2 = f2(pe.dphi), c4 = f2(pe.c4), c3 = f2(pe.c3), c2 = f2(pe.c2), c1 = f2(pe.c1), A2 = f2(pe.A);
                // two-zone table: with t2 = t - 1/2, alpha t - 1/2 = alpha t2 + (alpha - 1)/2 and gamma (t - t1) - 1/2 = gamma t2 + gamma/2 - gamma t1 - 1/2
                const float2 za2 = f2(P.z_alpha), zao2 = f2(0.5f * P.z_alpha - 0.5f), zg2 = f2(P.z_gamma), zgo2 = f2(0.5f * P.z_gamma - P.z_t1g - 0.5f);
                const float zhm1f = (float)P.z_hm1;
                const unsigned zhm1 = (unsigned)P.z_hm1;
                float2 dc2[RP];
#pragma unroll
                for (int h = 0; h < RP; ++h) dc2[h] = f2(dcr[2 * h], dcr[R > 1 ? 2 * h + 1 : 0]);
                float2 jf = f2((float)(-pe.hw));
                const int pos0 = i0 - pe.hw, pend = i0 + pe.hw + R - 1;
                // One window position for the pixels rr in MASK (compile time).  The window of the thread is the
                // union of its R pixels' windows, which are one position apart: pixel rr can only be inside the
                // disc at positions pos0 + rr .. pend - (R - 1 - rr) (host: hw = floor(H / dphi' + 1/2 + 3 rho1),
                // |dcr0| <= dphi' / 2, pixel rr is centred rr (1 +- rho1) positions further), so the first and the
                // last R - 1 positions run bodies without the other pixels' geometry, gather and FMAs.
                auto body = [&](int pos, auto MASK) {
                    constexpr int mask = decltype(MASK)::value;
                    float tp[2 * RP], tz_[2 * RP];
                    unsigned cb[2 * RP], cz[2 * RP];
#pragma unroll
                    for (int h = 0; h < RP; ++h) {
                        if (!((mask >> (2 * h)) & 3)) continue;
                        const float2 d = __ffma2_rn(jf, dphi2, dc2[h]);
                        const float2 y = __fmul2_rn(d, d);
                        float2 p = __ffma2_rn(y, c4, c3);
                        p = __ffma2_rn(y, p, c2);
                        p = __ffma2_rn(y, p, c1);
                        const float2 t2 = __ffma2_rn(y, p, A2);          // t - 0.5
                        const float2 bb = __fadd2_rn(t2, f2(kMagic));
                        tp[2 * h] = t2.x; tp[2 * h + 1] = t2.y;
                        cb[2 * h] = __float_as_uint(bb.x); cb[2 * h + 1] = __float_as_uint(bb.y);
                        if (Z) {
                            // inner zone: alpha t - 1/2; outer zone: gamma (t - t1) - 1/2 RELATIVE to the zone start
                            // (full resolution where the kernel is steep), cell offset added to the integer bits
                            const float2 l1 = __ffma2_rn(t2, za2, zao2), l2 = __ffma2_rn(t2, zg2, zgo2);
                            const bool o0 = l2.x + zhm1f < l1.x, o1 = l2.y + zhm1f < l1.y;
                            const float2 tz = f2(o0 ? l2.x : l1.x, o1 ? l2.y : l1.y);
                            const float2 bz = __fadd2_rn(tz, f2(kMagic));
                            const float2 fz = __fadd2_rn(tz, __fadd2_rn(f2(kMagic), f2(-bz.x, -bz.y)));   // position - 1/2 in the cell
                            tz_[2 * h] = fz.x; tz_[2 * h + 1] = fz.y;
                            cz[2 * h] = __float_as_uint(bz.x) + (o0 ? zhm1 : 0u); cz[2 * h + 1] = __float_as_uint(bz.y) + (o1 ? zhm1 : 0u);
                        }
                    }
                    // cells below the last: plain lookup; beyond the zero cell: clamp onto it (weight 0);
                    // the last cell and the zero cell (t in [tmax - 1, tmax + 1)) take the branch
                    unsigned mn = 0xFFFFFFFFu;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) if ((mask >> rr) & 1) mn = min(mn, cb[rr] - thresh);
                    float *tl = Z ? tz_ : tp;                              // lookup coordinate - 0.5 and its cell bits
                    unsigned *cl = Z ? cz : cb;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) if ((mask >> rr) & 1) cl[rr] = min(cl[rr], thresh + 1u);
                    if (mn < 2u) {
#pragma unroll
                        for (int rr = 0; rr < R; ++rr)
                            if (((mask >> rr) & 1) && cb[rr] >= thresh) slow(rr, tp[rr], cl[rr], pos);
                    }
                    float K[R];
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) {
                        if (!((mask >> rr) & 1)) continue;
                        float2 el;                                  // tab[cb - kMagicBits], one LEA for the address
                        asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(el.x), "=f"(el.y) : "r"(tab_sh + cl[rr] * 8u));
                        K[rr] = fmaf(tl[rr], el.y, el.x);
                    }
                    const unsigned so = 16u * (unsigned)slot_of_pos<R>(pos);
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        const float4 mn4 = lds128(pn[b] + so), ms4 = lds128(pn[b] + so + south);
                        const float2 m01 = f2(mn4.x, mn4.y), m23 = f2(mn4.z, mn4.w), m45 = f2(ms4.x, ms4.y), m67 = f2(ms4.z, ms4.w);
#pragma unroll
                        for (int rr = 0; rr < R; ++rr) {
                            if (!((mask >> rr) & 1)) continue;
                            const float2 Kd = f2(K[rr]);
                            acc[rr][b][0] = __ffma2_rn(Kd, m01, acc[rr][b][0]);
                            acc[rr][b][1] = __ffma2_rn(Kd, m23, acc[rr][b][1]);
                            acc[rr][b][2] = __ffma2_rn(Kd, m45, acc[rr][b][2]);
                            acc[rr][b][3] = __ffma2_rn(Kd, m67, acc[rr][b][3]);
                        }
                    }
                    jf = __fadd2_rn(jf, f2(1.0f));
                };
                constexpr int kAll = (1 << R) - 1;
                int pos = pos0, plast = pend;
                const bool peel = R > 1 && 2 * pe.hw >= R - 2;       // first and last R - 1 positions do not overlap
                if (peel) {
                    body(pos++, std::integral_constant<int, 1>{});
                    if (R == 4) { body(pos++, std::integral_constant<int, 3>{}); body(pos++, std::integral_constant<int, 7>{}); }
                    plast = pend - (R - 1);
                }
#pragma unroll 2
                for (; pos <= plast; ++pos) body(pos, std::integral_constant<int, kAll>{});
                if (peel) {
                    if (R == 4) { body(pos++, std::integral_constant<int, 14 & kAll>{}); body(pos++, std::integral_constant<int, 12 & kAll>{}); }
                    body(pos++, std::integral_constant<int, (1 << (R - 1))>{});
                }
                if (TOT && TM) {                                 // totals (tensor memory) += this ring's sums
                    static_assert(!TM || (R == 4 && B == 1), "TM variant: 32 accumulators per thread");
#pragma unroll
                    for (int hh = 0; hh < 2; ++hh) {
                        float v[16], old[16];
#pragma unroll
                        for (int q = 0; q < 2; ++q)
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                float2 &a = acc[(2 * hh + q) % R][0][g];
                                v[8 * q + 2 * g] = a.x; v[8 * q + 2 * g + 1] = a.y;
                                a = f2(0.f);
                            }
                        if (flushed) {
                            tmem_ld16(taddr + 16u * hh, old);
#pragma unroll
                            for (int i = 0; i < 16; ++i) v[i] += old[i];
                        }
                        tmem_st16(taddr + 16u * hh, v);
                    }
                    tmem_wait_st();
                    flushed = true;
                } else if (TOT) {
#pragma unroll
                    for (int rr = 0; rr < R; ++rr)
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                tot[rr][b][g] = __fadd2_rn(tot[rr][b][g], acc[rr][b][g]);
                                acc[rr][b][g] = f2(0.f);
                            }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[buf]);         // this warp is done with the buffer
        }

        if (TM && flushed) {                               // totals back from tensor memory
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                float old[16];
                tmem_ld16(taddr + 16u * hh, old);
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int g = 0; g < 4; ++g) tot[(2 * hh + q) % R][0][g] = f2(old[8 * q + 2 * g], old[8 * q + 2 * g + 1]);
            }
        }
        // store the 8 images of every valid base pixel
        if (active) {
            const int start_n = P.start[r - 1], start_s = P.start[4 * N - r - 1];
            const bool south_img = (r != 2 * N);
#pragma unroll
            for (int rr = 0; rr < R; ++rr) {
                const int k = kmine + rr;
                if (k <= klast) {
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        const float2 *s = TOT ? tot[rr][b] : acc[rr][b];
                        const float v[8] = {s[0].x, s[0].y, s[1].x, s[1].y, s[2].x, s[2].y, s[3].x, s[3].y};
#pragma unroll
                        for (int m = 0; m < 4; ++m) {
                            io.out[b][start_n + k + m * ip] = v[m] * P.omega;
                            if (south_img) io.out[b][start_s + k + m * ip] = v[4 + m] * P.omega;
                        }
                    }
                }
            }
        }
    }
    if (TM) {                                              // every consumer warp is done with tensor memory
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        asm volatile("bar.sync 2, %0;" ::"r"(NC) : "memory");
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(s_tmem) : "memory");
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
size_t belt_smem_bytes(int NC, int slack, int nbuf, int ntb, int pw_max, int ne_max);
cudaError_t launch_belt(const Dev &P, const BeltDev &F, const Maps &io, int B, int threads, int slack, size_t smem, int nsm,
                        cudaStream_t st);

// Host geometry kept for building tile lists after plan creation (latitude bands)
struct HostGeo {
    int N = 0, polar = 0;
    std::vector<std::vector<PairEnt>> per_ring;   // per base ring 1 .. 2N: its input rings
    std::vector<int> slot_of, pair_off;           // base ring -> slot; slot -> first entry of `pairs`
    std::vector<char> is_belt;
    int ipof(int r) const { return r < N ? r : (r <= 3 * N ? N : 4 * N - r); }
    int shof(int r) const { return (r >= N && r <= 3 * N) ? ((r - N) & 1) : 0; }
};

// Sym-kernel tiles of the non-belt base rings r_lo .. r_hi, longest first, appended to `tiles`.  Tiles are
// packed from runs of base pixels on one ring (32 R pixels per warp): whole runs of `run` pixels first, the
// ragged remainders are bin-packed (first fit, decreasing); a tile holds at most W warps, kMaxSub runs and
// Llimit staged positions (shared memory).  Returns the staged positions the tiles need.
static int build_sym_tiles(const HostGeo &g, int R, int W, int run, int Llimit, int r_hi, int r_lo,
                           std::vector<SymTile> &tiles) {
    const int C = 32 * R;
    struct SubH { int r, k0, n, nw; int Lcap; double work; };
    auto make_sub = [&](int r, int k0, int n) {
        SubH sb{r, k0, n, (n + C - 1) / C, 0, 0.0};
        const int ip = g.ipof(r), sh = g.shof(r);
        const int klast = k0 + n - 1;
        for (const PairEnt &pe : g.per_ring[r]) {
            const int w0 = ((2 * k0 + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) - pe.hw;
            const int L = ((2 * klast + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) + pe.hw + R - w0;
            sb.Lcap = std::max(sb.Lcap, L);
            sb.work += (double)(2 * pe.hw + R);
        }
        sb.Lcap = (sb.Lcap + 7) & ~7;
        sb.work *= sb.nw;
        return sb;
    };
    std::vector<std::vector<SubH>> bins;
    std::vector<SubH> partial;
    for (int r = r_hi; r >= r_lo; --r) {
        if (r <= g.polar || g.is_belt[r]) continue;
        const int ip = g.ipof(r);
        int k0 = 0;
        for (; ip - k0 >= run; k0 += run) bins.push_back({make_sub(r, k0, run)});
        if (k0 < ip) partial.push_back(make_sub(r, k0, ip - k0));
    }
    const size_t nfull = bins.size();
    std::stable_sort(partial.begin(), partial.end(), [](const SubH &a, const SubH &b) { return a.nw > b.nw; });
    std::vector<int> used(nfull, W), lsum(nfull, 0);
    for (const SubH &sb : partial) {
        size_t i = nfull;
        for (; i < bins.size(); ++i)
            if (used[i] + sb.nw <= W && (int)bins[i].size() < kMaxSub && lsum[i] + sb.Lcap <= Llimit) break;
        if (i == bins.size()) { bins.emplace_back(); used.push_back(0); lsum.push_back(0); }
        bins[i].push_back(sb); used[i] += sb.nw; lsum[i] += sb.Lcap;
    }
    std::vector<std::pair<double, size_t>> order;
    int Lneed = 0;
    for (size_t i = 0; i < bins.size(); ++i) {
        double w = 0; int L = 0;
        for (const SubH &sb : bins[i]) { w = std::max(w, sb.work / sb.nw); L += sb.Lcap; }
        order.push_back({-w, i});
        Lneed = std::max(Lneed, L);
    }
    std::stable_sort(order.begin(), order.end());
    const size_t t0 = tiles.size();
    tiles.resize(t0 + bins.size());
    for (size_t t = 0; t < order.size(); ++t) {
        const std::vector<SubH> &bn = bins[order[t].second];
        SymTile &tl = tiles[t0 + t];
        std::memset(&tl, 0, sizeof(tl));
        tl.nsub = (int)bn.size();
        int w0 = 0, soff = 0;
        for (int i = 0; i < tl.nsub; ++i) {
            const SubH &sb = bn[i];
            const int slot = g.slot_of[sb.r];
            tl.sub[i] = SubTile{sb.r, sb.k0, sb.n, g.pair_off[slot], g.pair_off[slot + 1] - g.pair_off[slot], w0, sb.nw, soff};
            tl.nsteps = std::max(tl.nsteps, tl.sub[i].ne);
            w0 += sb.nw; soff += sb.Lcap;
        }
    }
    return Lneed;
}

struct FastCfg {            // per batch size
    bool ok = false;
    int threads = 0, R = 1, Ltot = 0;
    size_t smem = 0;
    SymTile *tiles = nullptr;     // [0, ntiles): all rings, work sorted; then the latitude chunks
    int ntiles = 0, ntiles_all = 0, run = 0;
    bool tmem = false;            // 384-consumer variant with the running totals in tensor memory (large discs)
    std::map<std::pair<int, int>, std::pair<SymTile *, int>> band_tiles;   // (ring lo, hi) -> device tile list
    std::vector<int> ch_off, ch_lo, ch_hi;   // chunk i: tiles [ch_off[i], ch_off[i+1]), base rings ch_lo[i] .. ch_hi[i]
};

struct FastPlan {
    PairEnt *pairs = nullptr;
    int ntab_s = 0;
    int polar = 0;
    int first_belt = 0;           // base rings first_belt .. 2N go to the belt kernel (2N + 1: none)
    FastCfg cfg[kMaxB + 1];
    int nsm = 148;
    // belt kernel
    bool belt_ok = false;
    BeltDev belt{};
    int belt_threads = 0;
    size_t belt_smem = 0;
    int *pair_off = nullptr;
    int *woff = nullptr;
    int4 *belt_tiles = nullptr;
    std::vector<int> bch_off, bch_lo, bch_hi;   // belt latitude chunks (tile offsets, base rings), equator first
    std::shared_ptr<HostGeo> geo;
    int belt_tiles_per_ring = 0, belt_slack = 0;
    int *grp_off = nullptr, *grp_e = nullptr;
};

template <int B, int R, int NC, bool TOT, bool Z, bool TM = false>
static cudaError_t launch_sym(const FastPlan *fp, const FastCfg &c, const Dev &P, const Maps &io, cudaStream_t st,
                              const SymTile *tiles, int nt) {
    FastDev F{fp->pairs, tiles, nt, c.Ltot, fp->ntab_s};
    static bool attr_done[64] = {};
    cudaError_t e = ensure_max_smem(sym_kernel<B, R, NC, TOT, Z, TM>, attr_done);
    if (e != cudaSuccess) return e;
    const int grid = std::min(fp->nsm, nt);
    if (grid <= 0) return cudaSuccess;
    sym_kernel<B, R, NC, TOT, Z, TM><<<grid, c.threads + kSymProd, c.smem, st>>>(P, F, io);
    return cudaGetLastError();
}

// the sym kernel instance of this batch size over a tile list
static cudaError_t dispatch_sym(const FastPlan *fp, const FastCfg &c, const Dev &P, const Maps &io, int B, cudaStream_t st,
                                const SymTile *tiles, int nt) {
    cudaError_t e = cudaErrorInvalidValue;
#define SC_SYM_CASE(BB, RR)                                                                  \
    if (B == BB && c.R == RR)                                                                \
        e = c.threads == 256 ? (P.zoned ? launch_sym<BB, RR, 256, true, true>(fp, c, P, io, st, tiles, nt)    \
                                        : launch_sym<BB, RR, 256, true, false>(fp, c, P, io, st, tiles, nt))  \
                             : (P.zoned ? launch_sym<BB, RR, 128, true, true>(fp, c, P, io, st, tiles, nt)    \
                                        : launch_sym<BB, RR, 128, true, false>(fp, c, P, io, st, tiles, nt));
    if (B == 1 && c.R == 4 && c.threads == 384 && c.tmem) {
        e = P.zoned ? launch_sym<1, 4, 384, true, true, true>(fp, c, P, io, st, tiles, nt)
                    : launch_sym<1, 4, 384, true, false, true>(fp, c, P, io, st, tiles, nt);
    } else if (B == 1 && c.R == 4 && c.threads == 384) {
        e = P.zoned ? launch_sym<1, 4, 384, false, true>(fp, c, P, io, st, tiles, nt)
                    : launch_sym<1, 4, 384, false, false>(fp, c, P, io, st, tiles, nt);
    } else {
        SC_SYM_CASE(1, 1) SC_SYM_CASE(1, 2) SC_SYM_CASE(1, 4)
        SC_SYM_CASE(2, 1) SC_SYM_CASE(2, 2) SC_SYM_CASE(2, 4)
        SC_SYM_CASE(3, 1) SC_SYM_CASE(3, 2)
        SC_SYM_CASE(4, 1) SC_SYM_CASE(4, 2)
    }
#undef SC_SYM_CASE
    return e;
}

// which: bit 0 = sym kernel, bit 1 = belt kernel (the two write disjoint pixels and may run on different
// streams); chunk < 0: all tiles (work sorted), else latitude chunk `chunk` of that kernel
cudaError_t fast_launch(FastPlan *fp, const Dev &P, const Maps &io, int B, int which, cudaStream_t st, int *launches,
                        int chunk) {
    *launches = 0;
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return cudaErrorInvalidValue;
    const FastCfg &c = fp->cfg[B];
    cudaError_t e = cudaSuccess;
    if (which & 1) {
        int t0 = 0, nt = c.ntiles;
        if (chunk >= 0) {
            if (chunk + 1 >= (int)c.ch_off.size()) return cudaErrorInvalidValue;
            t0 = c.ch_off[chunk]; nt = c.ch_off[chunk + 1] - t0;
        }
        if ((e = dispatch_sym(fp, c, P, io, B, st, c.tiles + t0, nt)) != cudaSuccess) return e;
        *launches += nt > 0 ? 1 : 0;
    }
    if ((which & 2) && fp->belt_ok) {
        BeltDev F = fp->belt;
        if (chunk >= 0) {
            if (chunk + 1 >= (int)fp->bch_off.size()) return cudaErrorInvalidValue;
            F.tiles += fp->bch_off[chunk]; F.ntiles = fp->bch_off[chunk + 1] - fp->bch_off[chunk];
        }
        if (F.ntiles > 0) {
            e = launch_belt(P, F, io, B, fp->belt_threads, fp->belt_slack, fp->belt_smem, fp->nsm, st);
            if (e == cudaSuccess) ++*launches;
        }
    }
    return e;
}

// Latitude band: the fast kernels over base rings lo .. hi only (1 <= lo <= hi <= 2N; their southern mirrors
// included).  The sym tile list of a band is built on first use and cached (synchronous the first time).
cudaError_t fast_launch_band(FastPlan *fp, const Dev &P, const Maps &io, int B, int lo, int hi, cudaStream_t st,
                             int *launches) {
    *launches = 0;
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return cudaErrorInvalidValue;
    FastCfg &c = fp->cfg[B];
    const int N = P.nside;
    cudaError_t e = cudaSuccess;
    const int s_lo = std::max(lo, fp->polar + 1), s_hi = std::min(hi, std::min(fp->first_belt - 1, 2 * N));
    if (s_lo <= s_hi) {
        auto it = c.band_tiles.find({s_lo, s_hi});
        if (it == c.band_tiles.end()) {
            std::vector<SymTile> tiles;
            const int Lneed = build_sym_tiles(*fp->geo, c.R, c.threads / 32, c.run, c.Ltot, s_hi, s_lo, tiles);
            if (Lneed > c.Ltot) return cudaErrorInvalidValue;
            SymTile *d = nullptr;
            if ((e = cudaMalloc((void **)&d, std::max<size_t>(tiles.size(), 1) * sizeof(SymTile))) != cudaSuccess) return e;
            if (!tiles.empty() && (e = cudaMemcpy(d, tiles.data(), tiles.size() * sizeof(SymTile), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
            it = c.band_tiles.emplace(std::make_pair(s_lo, s_hi), std::make_pair(d, (int)tiles.size())).first;
        }
        if (it->second.second > 0) {
            if ((e = dispatch_sym(fp, c, P, io, B, st, it->second.first, it->second.second)) != cudaSuccess) return e;
            ++*launches;
        }
    }
    const int b_lo = std::max(lo, fp->first_belt), b_hi = std::min(hi, 2 * N);
    if (fp->belt_ok && b_lo <= b_hi) {
        BeltDev F = fp->belt;                               // tile list: ring 2N first, belt_tiles_per_ring tiles per ring
        F.tiles += (2 * N - b_hi) * fp->belt_tiles_per_ring;
        F.ntiles = (b_hi - b_lo + 1) * fp->belt_tiles_per_ring;
        e = launch_belt(P, F, io, B, fp->belt_threads, fp->belt_slack, fp->belt_smem, fp->nsm, st);
        if (e == cudaSuccess) ++*launches;
    }
    return e;
}

// latitude chunks for the pipelined host entry: kind 0 = sym kernel, 1 = belt kernel
int fast_chunk_count(const FastPlan *fp, int B, int kind) {
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return 0;
    return kind == 0 ? (int)fp->cfg[B].ch_lo.size() : (fp->belt_ok ? (int)fp->bch_lo.size() : 0);
}
void fast_chunk_rings(const FastPlan *fp, int B, int kind, int i, int *lo, int *hi) {
    if (kind == 0) { *lo = fp->cfg[B].ch_lo[i]; *hi = fp->cfg[B].ch_hi[i]; }
    else { *lo = fp->bch_lo[i]; *hi = fp->bch_hi[i]; }
}

cudaError_t fast_convolve(FastPlan *fp, const Dev &P, const Maps &io, int B, cudaStream_t st, int *launches,
                          cudaEvent_t *ev) {
    int n1 = 0, n2 = 0;
    cudaError_t e = fast_launch(fp, P, io, B, 1, st, &n1, -1);
    *launches = n1;
    if (e != cudaSuccess) return e;
    if (ev && (e = cudaEventRecord(ev[0], st)) != cudaSuccess) return e;      // end of the sym kernel
    e = fast_launch(fp, P, io, B, 2, st, &n2, -1);
    *launches += n2;
    if (ev && e == cudaSuccess) e = cudaEventRecord(ev[1], st);              // end of the belt kernel
    return e;
}

int fast_first_belt_ring(const FastPlan *fp) { return fp->first_belt; }

bool fast_available(const FastPlan *fp, int B) { return fp && B >= 1 && B <= kMaxB && fp->cfg[B].ok; }

void fast_plan_destroy(FastPlan *fp) {
    if (!fp) return;
    cudaFree(fp->pairs); cudaFree(fp->pair_off);
    for (auto &c : fp->cfg) {
        cudaFree(c.tiles);
        for (auto &kv : c.band_tiles) cudaFree(kv.second.first);
    }
    cudaFree(fp->woff); cudaFree(fp->belt_tiles); cudaFree(fp->grp_off); cudaFree(fp->grp_e);
    delete fp;
}

static int env_int(const char *name, int dflt) {
    const char *e = std::getenv(name);
    return e && *e ? std::atoi(e) : dflt;
}

FastPlan *fast_plan_create(const Dev &P, const std::vector<double> &z, const std::vector<double> &s,
                           int max_batch, int *polar_rings, cudaError_t *err) {
    *err = cudaSuccess;
    *polar_rings = 0;
    const int N = P.nside, nr = 4 * N - 1;
    constexpr int Rmax = 4;                        // windows are sized for up to 4 base pixels per thread
    int dev = 0, smem_optin = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int ntab_s = P.ntab;                     // the cells and the one zero cell after them (indices are clamped)
    const size_t tab_bytes = ((size_t)ntab_s * 8 + 127) & ~(size_t)127;
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
    // largest |d| for which the 4-term polynomial of 1 - cos d is good to 0.004 table cells: the next term is
    // B scale d^10 / 3628800 with B scale <= 2 tmax / d^2 for a pair inside the disc
    const double dmax = std::min(0.9, std::pow(0.004 * 1814400.0 / tmax, 1.0 / 8.0));

    std::vector<PairEnt> pairs;
    std::vector<int> pair_off(1, 0);
    std::vector<char> eligible(2 * N + 1, 0);
    std::vector<std::vector<PairEnt>> per_ring(2 * N + 1);
    for (int r = 1; r <= 2 * N; ++r) {
        const int ip = ipof(r);
        bool ok = true;
        std::vector<PairEnt> &lst = per_ring[r];
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
            const int hw = (int)std::floor(H / dphi + 0.5 + rho1 * (Rmax - 1) + 1e-6);
            if ((hw + 1 + Rmax) * dphi > dmax) ok = false;
            PairEnt e;
            e.A = (float)(A64 * P.scale - 0.5);
            e.c1 = (float)(Bs / 2.0); e.c2 = (float)(-Bs / 24.0); e.c3 = (float)(Bs / 720.0); e.c4 = (float)(-Bs / 40320.0); e.pad_ = 0;
            e.dphi = (float)dphi;
            e.cdc = (float)(M_PI / (4.0 * (double)ip * (double)ipq));
            e.rq = rq; e.hw = hw; e.ipq = ipq; e.shq = shof(rq);
            e.start_n = startof(rq); e.start_s = startof(4 * N - rq);
            lst.push_back(e);
            return true;
        };
        for (int rq = r; rq >= 1; --rq) if (!consider(rq)) break;
        std::reverse(lst.begin(), lst.end());
        for (int rq = r + 1; rq <= nr; ++rq) if (!consider(rq)) break;
        // the window of a whole quadrant must not wrap onto itself
        for (const PairEnt &e : lst) if (e.ipq + 2 * e.hw + 2 * Rmax + 4 >= 4 * e.ipq) ok = false;
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
    fp->geo = std::make_shared<HostGeo>();
    fp->ntab_s = ntab_s; fp->polar = polar; fp->nsm = nsm;
    auto fail = [&](cudaError_t e) { *err = e; fast_plan_destroy(fp); return (FastPlan *)nullptr; };
    cudaError_t e;
    if ((e = cudaMalloc((void **)&fp->pairs, std::max<size_t>(pairs.size(), 1) * sizeof(PairEnt))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc((void **)&fp->pair_off, pair_off.size() * sizeof(int))) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pairs, pairs.data(), pairs.size() * sizeof(PairEnt), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pair_off, pair_off.data(), pair_off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);

    // ---- belt kernel: base rings whose input rings all have 4N pixels ------------------------------
    std::vector<char> is_belt(2 * N + 1, 0);
    const bool no_belt = std::getenv("SC_NO_BELT") != nullptr;
    // variants (consumer threads, slack floats per plane): tile = 4 x threads base pixels, must divide N
    struct BeltVar { int nc, slack; };
    std::vector<BeltVar> bvars;
    {
        const double mean_nb_b = 0.5 * (double)P.npix * ((double)P.tmax / P.scale);
        if (N % 2048 == 0 && mean_nb_b <= 700.0 && !std::getenv("SC_BELT_NO512")) bvars.push_back({512, 64});
        if (N % 2048 == 0 && mean_nb_b > 700.0 && !std::getenv("SC_BELT_NOTMEM")) { bvars.push_back({512, 256}); bvars.push_back({512, 512}); }
        if (N % 1024 == 0) { bvars.push_back({256, 256}); bvars.push_back({256, 512}); }
        else if (N % 512 == 0) bvars.push_back({128, 256});
    }
    for (const BeltVar &bv : bvars) {
        if (no_belt || fp->belt_ok) break;
        const int bNC = bv.nc;
        const int T = 4 * bNC;
        std::vector<int> woff(pairs.size(), 0);
        std::vector<int4> btiles;
        int pw_max = 0, ne_max = 0;
        bool fits = true;
        // The input rings of a base ring are cut into groups whose tap arrays fit one tap buffer (a few
        // hundred rings of a few hundred taps for paper-scale discs do not fit as a whole).
        const int kTapCap = 2048, kGroupRings = 96;                       // float2 entries, rings per group
        std::vector<int> grp_off(1, 0), grp_e;
        std::fill(is_belt.begin(), is_belt.end(), 0);
        for (int r = polar + 1; r <= 2 * N; ++r) {                           // slots run over base rings polar+1 .. 2N
            bool all = ipof(r) == N;
            for (const PairEnt &pe : per_ring[r]) if (pe.ipq != N) { all = false; break; }
            is_belt[r] = all;
            const int base = pair_off[slot_of[r]];
            int off = 0, cnt = 0;
            grp_e.push_back(0);
            for (size_t i = 0; i < per_ring[r].size(); ++i) {
                const int ng_max = (2 * per_ring[r][i].hw + 4 + 3 + 3) >> 2;   // chunks of 4 staged positions
                const int len = (4 * ng_max + 2 + 1) & ~1;                     // tap pairs, even count
                if (all && (4 * ng_max > bv.slack + 4 || len > kTapCap)) fits = false;   // plane = T - 4 + 4 ng floats
                if (cnt > 0 && (off + len > kTapCap || cnt >= kGroupRings)) {  // next group
                    grp_e.push_back((int)i); off = 0; cnt = 0;
                }
                woff[base + i] = off;
                off += len; ++cnt;
                if (all) { pw_max = std::max(pw_max, off); ne_max = std::max(ne_max, cnt); }
            }
            grp_e.push_back((int)per_ring[r].size());
            grp_off.push_back((int)grp_e.size());
        }
        for (int r = 2 * N; r > polar; --r) {
            if (!is_belt[r]) { for (int q = r; q > polar; --q) is_belt[q] = 0; break; }   // belt rings are contiguous from 2N down
            for (int k0 = 0; k0 < N; k0 += T) btiles.push_back(make_int4(r, k0, slot_of[r], (int)per_ring[r].size()));
        }
        int nbuf = 0, ntb = 0;
        size_t bsmem = 0;
        if (fits && !btiles.empty()) {
            const int combos[6][2] = {{2, 4}, {2, 3}, {1, 4}, {2, 2}, {1, 3}, {1, 2}};       // (tap buffers, stage buffers)
            for (const auto &cb : combos) {
                bsmem = belt_smem_bytes(bNC, bv.slack, cb[1], cb[0], pw_max, ne_max);
                if (bsmem + 2048 <= (size_t)smem_optin) { ntb = cb[0]; nbuf = cb[1]; break; }
            }
        }
        if (nbuf >= ((bNC == 512 && bv.slack == 64) ? 3 : 2)) {
            if ((e = cudaMalloc((void **)&fp->woff, woff.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->woff, woff.data(), woff.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->belt_tiles, btiles.size() * sizeof(int4))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->belt_tiles, btiles.data(), btiles.size() * sizeof(int4), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->grp_off, grp_off.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->grp_off, grp_off.data(), grp_off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->grp_e, grp_e.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->grp_e, grp_e.data(), grp_e.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            fp->belt = BeltDev{fp->pairs, fp->pair_off, fp->woff, fp->belt_tiles, fp->grp_off, fp->grp_e, (int)btiles.size(), pw_max, ne_max, nbuf, ntb};
            fp->belt_slack = bv.slack;
            fp->belt_threads = bNC; fp->belt_smem = bsmem; fp->belt_ok = true; fp->belt_tiles_per_ring = N / T;
            // latitude chunks: the tile list runs from ring 2N down to the first belt ring, N / T tiles per ring
            {
                int r_first = 2 * N + 1;
                for (int r = 2 * N; r > polar && is_belt[r]; --r) r_first = r;
                const int nrings = 2 * N - r_first + 1, per_ring_tiles = N / T;
                fp->bch_off.assign(1, 0); fp->bch_lo.clear(); fp->bch_hi.clear();
                int hi = 2 * N;
                const int nbch = std::max(1, env_int("SC_BELT_CHUNKS", kBeltChunksDflt));
                for (int cidx = 1; cidx <= nbch && hi >= r_first; ++cidx) {
                    int lo = 2 * N + 1 - (int)((long long)nrings * cidx / nbch);
                    if (cidx == nbch) lo = r_first;
                    if (lo > hi) continue;
                    fp->bch_lo.push_back(lo); fp->bch_hi.push_back(hi);
                    fp->bch_off.push_back((2 * N - lo + 1) * per_ring_tiles);
                    hi = lo - 1;
                }
            }
        } else {
            std::fill(is_belt.begin(), is_belt.end(), 0);
        }
    }

    // ---- sym kernel: per batch size pick (threads, R) so that table + double-buffered stage fit ------
    // Tiles are packed from sub-tiles (runs of base pixels on one ring, 32 R pixels per warp): whole
    // CTA-wide runs first, the ragged remainders of all rings are bin-packed (first fit, decreasing).
    (void)max_batch;
    struct Cand { int threads, R; };
    for (int B = 1; B <= kMaxB; ++B) {
        FastCfg &c = fp->cfg[B];
        std::vector<Cand> cands;
        // 384 consumer threads only come without the second accumulator set (registers): plain fp32
        // running sums, good to ~3e-7 relative rms for discs of a few hundred pixels (measured 2.7e-7 at
        // 425), so only while the mean disc holds at most 700 pixels (4.7e-7 measured at 1380 for a Gaussian, 6.9e-7 at 960 for a cancelling split kernel)
        const double mean_nb = 0.5 * (double)P.npix * ((double)P.tmax / P.scale);
        // between 700 and 6000 pixels per disc the 384-consumer variant keeps the running totals in tensor memory
        // (4-6 % faster than 256 consumers with both sets in registers; slower again for still larger discs)
        if (B == 1 && (mean_nb <= 700.0 || (mean_nb <= 6000.0 && !std::getenv("SC_SYM_NOTMEM")))) cands = {{384, 4}, {256, 4}, {256, 2}, {128, 2}};
        else if (B == 1) cands = {{256, 4}, {256, 2}, {128, 2}};
        else cands = {{256, 2}, {128, 2}, {128, 1}};
        const int fr = env_int("SC_SYM_R", 0), ft = env_int("SC_SYM_THREADS", 0);
        if (fr > 0 && ft > 0 && (fr == 1 || fr == 2 || (fr == 4 && B <= 2)) && (ft == 128 || ft == 256 || (ft == 384 && fr == 4 && B == 1)))
            cands.insert(cands.begin(), Cand{ft, fr});
        for (const Cand &cd : cands) {
            const int R = cd.R, W = cd.threads / 32, C = 32 * R;
            // full-width runs may be a little shorter than the CTA (last lanes idle) if that makes the
            // staged runs fit into shared memory
            for (int shrink = 0; shrink <= W * C / 4 && !c.ok; shrink += 16) {
            const int run = W * C - shrink;
            // a tile holds at most W warps, kMaxSub runs and Lmax staged positions (shared memory)
            const int Lmax = (int)(((size_t)smem_optin - 256 - tab_bytes) / ((size_t)2 * B * 2 * 16)) & ~7;
            HostGeo &g = *fp->geo;
            g.N = N; g.polar = polar; g.per_ring = per_ring; g.slot_of = slot_of; g.pair_off = pair_off; g.is_belt = is_belt;
            auto build = [&](int r_hi, int r_lo, std::vector<SymTile> &tl) { return build_sym_tiles(g, R, W, run, Lmax, r_hi, r_lo, tl); };
            // (1) the whole range in one work-sorted list: sc_convolve; (2) the same rings in kSymChunks
            // latitude chunks from the belt towards the pole, each sorted: the pipelined host entry
            std::vector<SymTile> tiles;
            int Ltot = build(2 * N, polar + 1, tiles);
            int sym_hi = 2 * N;
            while (sym_hi > polar && is_belt[sym_hi]) --sym_hi;
            std::vector<int> ch_off(1, (int)tiles.size()), ch_lo, ch_hi;
            {
                const long long nsymch = std::max(1, env_int("SC_SYM_CHUNKS", kSymChunksDflt));
                long long total_px = 0, acc_px = 0;
                for (int r = sym_hi; r > polar; --r) total_px += ipof(r);
                int hi = sym_hi, nch = 0;
                for (int r = sym_hi; r > polar; --r) {
                    acc_px += ipof(r);
                    if (r == polar + 1 || acc_px * nsymch >= total_px * (nch + 1)) {
                        Ltot = std::max(Ltot, build(hi, r, tiles));
                        ch_off.push_back((int)tiles.size()); ch_lo.push_back(r); ch_hi.push_back(hi);
                        hi = r - 1; ++nch;
                    }
                }
            }
            const size_t smem = tab_bytes + (size_t)2 * B * 2 * Ltot * 16;
            if (smem + 256 > (size_t)smem_optin) continue;        // 256: static shared memory (barriers)
            c.ntiles_all = ch_off[0]; c.ch_off = ch_off; c.ch_lo = ch_lo; c.ch_hi = ch_hi;
            c.threads = cd.threads; c.R = R; c.Ltot = Ltot; c.smem = smem; c.ntiles = c.ntiles_all; c.run = run;
            c.tmem = (B == 1 && cd.threads == 384 && mean_nb > 700.0);      // large discs: two-level sums, totals in TMEM
            if ((e = cudaMalloc((void **)&c.tiles, std::max<size_t>(tiles.size(), 1) * sizeof(SymTile))) != cudaSuccess) return fail(e);
            if (!tiles.empty() && (e = cudaMemcpy(c.tiles, tiles.data(), tiles.size() * sizeof(SymTile), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            c.ok = true;
            }
            if (c.ok) break;
        }
    }
    fp->first_belt = 2 * N + 1;
    for (int r = 2 * N; r > polar && is_belt[r]; --r) fp->first_belt = r;
    *polar_rings = polar;
    return fp;
}

}  // namespace sc
