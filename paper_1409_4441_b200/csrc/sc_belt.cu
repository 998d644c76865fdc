// sc_belt.cu -- the belt kernel: output rings whose whole disc lies in the equatorial belt.
//
// In the belt every ring has 4N pixels, so the pair weight K(p, q) depends only on
// (ring r, ring r', azimuthal offset j): the convolution is a stencil with per-ring-pair taps
// (SURVEY.md 8f-1).  A tile is T = 4 x NC consecutive base pixels of the first quadrant of one ring;
// its 8 symmetric images (4 quadrants x north/south) share the taps.  The CTA is warp-specialised:
//   * NC consumer threads run the stencil: a thread owns 4 consecutive pixels x 8 images = 32
//     accumulators, reads LDS.128 (4 staged positions of one image, conflict free) and issues packed
//     FFMA2 over pixel pairs: (acc_k, acc_k+1) += (w[s-k], w[s-k-1]) * m[s] -- one FMA per pair, no
//     geometry in the inner loop;
//   * one producer warp stages, ring by ring, the runs of the 8 images as 8 contiguous planes with TMA
//     bulk copies (cp.async.bulk) into a ring of NBUF buffers guarded by full/empty mbarriers;
//   * three producer warps evaluate the taps W[r'][j] of the NEXT tile -- same fp32 geometry, table
//     lookup and inclusion rule as the sym kernel (uncertain taps are set to 0 and decided per pixel
//     pair in fp64 by the consumers afterwards) -- into the other of two tap buffers; for large discs the
//     input rings are cut into groups and the tap buffers cycle through the groups.
// The first / last chunk of every input ring run bodies without the FFMA2s whose taps are zero by alignment;
// the 512-consumer large-disc variant keeps its running totals in tensor memory (tcgen05.ld/st).
// There is no block-wide barrier after the prologue.
#include "sc_fast.cuh"

#include <type_traits>


namespace sc {

constexpr int kBeltProd = 128;   // producer threads: warp 0 of them issues TMA, warps 1-3 evaluate taps
constexpr int kTapThreads = 96;
constexpr int kMaxBuf = 4;

static __device__ __noinline__ unsigned belt_exact_mask(const Dev &P, int r, int k, int rq, int kq) {
    const int N = P.nside, N4 = 4 * N;
    unsigned mask = 0;
    kq %= N4; if (kq < 0) kq += N4;
    {   // one image decides for all unless it is within kImageMargin of the threshold
        const double d0 = canonical_dot(P, r, k, rq, kq);
        if (fabs(d0 - P.c) > fmax(kImageMargin, 2.0 * P.ke_band)) return d0 >= P.c ? 0xFFu : 0u;
    }
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
// pd: the ring pair in fp64 for plans with the fp64 table coordinate (Dev::hp; dcc64 = offset to the nearest pixel), else
// unused.
__device__ __forceinline__ float belt_tap(const Dev &P, const PairEnt &pe, int j, float dcc, bool &unc, float &Ku,
                                          const PairEntD *pd = nullptr, double dcc64 = 0.0) {
    const float d = fmaf((float)j, pe.dphi, dcc);
    const float y = d * d;
    float h = fmaf(y, pe.c4, pe.c3);
    h = fmaf(y, h, pe.c2);
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
                float xk = fminf(t, P.tmax) - 0.5f;
                if (P.zoned) { int jz; zoned_cell(P, fminf(t, P.tmax), jz, xk); xk -= 0.5f; }   // last cell, centred form
                if (P.hp) xk = fminf(t, P.tmax) - (float)(P.ntab - 2) - 0.5f;                   // cell-local table
                Ku = fmaf(xk, el.y, el.x);
            }
            return 0.f;
        }
    }
    if (P.zoned) {                                   // two-zone table (t < tmax - eps here)
        int jz; float fz;
        zoned_cell(P, tp + 0.5f, jz, fz);
        const float2 el = __ldg(&P.tabh[jz]);
        return fmaf(fz - 0.5f, el.y, el.x);
    }
    if (P.hp) {                                      // fp64 coordinate -> cell + position in the cell (t < tmax - eps here)
        if (!pd) return 0.f;                         // (rescan of the uncertain taps: the weight is not used)
        const double t64 = fma(pd->Bs, one_minus_cos_poly_f64(fma((double)j, pd->dphi, dcc64)), pd->A);
        const int cell = min(__double2int_rd(t64), P.ntab - 2);
        const float2 el = __ldg(&P.tabh[cell]);
        return fmaf((float)(t64 - (double)cell) - 0.5f, el.y, el.x);
    }
    const float2 el = __ldg(&P.tabh[bits - kMagicBits]);
    return fmaf(tp, el.y, el.x);
}

__device__ __forceinline__ void bar_named(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// Window of input ring `pe` for the tile starting at base pixel k0 of a ring with shift flag sh:
// first staged position is w0a (multiple of 4), the window proper starts a0 positions later and the
// consumers walk ng chunks of 4 positions.
// PX: consecutive pixels owned by a consumer thread (4 or 8): its window is 2 hw + PX positions.
template <int PX>
__device__ __forceinline__ void belt_window(const PairEnt &pe, int sh, int k0, int &delta, int &w0a, int &a0, int &ng) {
    delta = (1 - sh + pe.shq) >> 1;
    const int first_pos = k0 + delta - pe.hw;
    w0a = first_pos & ~3;
    a0 = first_pos - w0a;
    ng = (2 * pe.hw + PX + a0 + 3) >> 2;
}

// Edge masks of the 8-pixel consumers: bit 4 p + i = the FFMA2 of pixel pair p (pixels 2p, 2p + 1) at chunk position i
// has a tap that can be non-zero.  Front chunk c (0, 1) with alignment a0: position 4c + i >= a0 + 2p.  Back chunk
// (cl = 1: the last, 0: the one before) with remq = the last chunk's last position that pixel pair 3 uses:
// i <= remq + 4 (1 - cl) - 2 (3 - p).
__host__ __device__ constexpr unsigned belt_front_mask(int c, int a0) {
    unsigned m = 0;
    for (int p = 0; p < 4; ++p)
        for (int i = 0; i < 4; ++i)
            if (4 * c + i >= a0 + 2 * p) m |= 1u << (4 * p + i);
    return m;
}
__host__ __device__ constexpr unsigned belt_back_mask(int cl, int remq) {
    unsigned m = 0;
    for (int p = 0; p < 4; ++p)
        for (int i = 0; i < 4; ++i)
            if (i <= remq + 4 * (1 - cl) - 2 * (3 - p)) m |= 1u << (4 * p + i);
    return m;
}


// SLACK: floats per staged plane beyond the tile (window + alignment); TOT: second accumulator set
// (flushed every >= 48 taps; needed for discs of thousands of pixels, costs 32 registers).
// TM: the second accumulator set lives in tensor memory (512-consumer variant for large discs).
// W8: a consumer thread owns 8 consecutive pixels x 4 images (the images of one hemisphere) instead of 4 x 8: a staged
// value then feeds 8 pixels, i.e. 4 map LDS.128 + 5 tap LDS.128 per 64 FFMA2 instead of 8 + 3.  The lanes' windows are
// then 32 bytes apart, so lanes 4-7 of every 8 read the image planes in the order (1, 0, 3, 2) and the plane stride is
// 4 floats off a multiple of 32: the 8 lanes of a quarter warp then cover all 32 banks.
template <int NC, int SLACK, bool TOT, bool TM, bool W8>
__global__ void __launch_bounds__(NC + kBeltProd, 1)
belt_kernel(const Dev P, const BeltDev F, const Maps io, const int B) {
    constexpr int PX = W8 ? 8 : 4;
    constexpr int T = 4 * NC, LP = T + SLACK + (W8 ? 4 : 0);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int N = P.nside, N4 = 4 * N;
    const int NBUF = F.nbuf, NTB = F.ntb;
    // a kernel launched behind this one with programmatic stream serialization (the sym kernel: disjoint outputs, no
    // wait on this grid) may take the SMs as this kernel's CTAs leave them
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    float *stage = reinterpret_cast<float *>(smem_raw);                           // [NBUF][8][LP]
    const TapLayout TL(F.pw_max, F.ne_max);
    unsigned char *tapbase = smem_raw + (size_t)NBUF * 8 * LP * 4;                // [NTB] tap buffers
    __shared__ unsigned long long full_bar[kMaxBuf], empty_bar[kMaxBuf], tap_full[2], tap_empty[2];

    if (tid == 0) {
        for (int i = 0; i < kMaxBuf; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], NC / 32); }
        for (int i = 0; i < 2; ++i) { mbar_init(&tap_full[i], kTapThreads); mbar_init(&tap_empty[i], NC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ unsigned s_tmem;
    if (TM && tid < 32) {                                      // 128 TMEM columns: 4 column groups x 4 lane quadrants
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(&s_tmem)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (TM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int G = gridDim.x, bid = blockIdx.x;
    const int nrows = (F.ntiles + G - 1) / G;

    if (tid >= NC) {
        if (NC == 256) asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        if (NC == 512) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (tid < NC + 32) {
            // ================================ TMA producer warp ================================
            int buf = 0; unsigned par = 0;
            for (int row = 0; row < nrows; ++row) {
                const int tile = row * G + ((row & 1) ? G - 1 - bid : bid);
                if (tile >= F.ntiles) continue;
                const int4 tl = F.tiles[tile];
                const int r = tl.x, k0 = tl.y, ne = tl.w;
                const int sh = (r - N) & 1;
                const int e0 = F.pair_off[tl.z];
                for (int b = 0; b < B; ++b) {
                    const float *__restrict__ in = io.in[b];
                    PairEnt pe_next = F.pairs[e0];
                    for (int e = 0; e < ne; ++e) {
                        const PairEnt pe = pe_next;
                        if (e + 1 < ne) pe_next = F.pairs[e0 + e + 1];      // prefetched while waiting below
                        int delta, w0a, a0, ng;
                        belt_window<PX>(pe, sh, k0, delta, w0a, a0, ng);
                        const int len = T - PX + 4 * ng;                      // floats per plane
                        unsigned long long *bar = &full_bar[buf];
                        mbar_wait_sleep(&empty_bar[buf], par ^ 1u);           // every consumer warp released it
                        if (lane == 0) mbar_expect_tx(bar, (unsigned)(8 * len * 4));
                        __syncwarp();
                        if (lane < 8) {                                       // one plane per lane
                            const int m = lane & 3;
                            const int base = (lane < 4) ? pe.start_n : pe.start_s;
                            int s0 = (w0a + m * N) % N4; if (s0 < 0) s0 += N4;
                            float *dst = stage + ((size_t)buf * 8 + lane) * LP;
                            const int first = min(len, N4 - s0);
                            tma_load_1d(dst, in + base + s0, (unsigned)(first * 4), bar);
                            if (first < len) tma_load_1d(dst + first, in + base, (unsigned)((len - first) * 4), bar);
                        }
                        if (++buf == NBUF) { buf = 0; par ^= 1u; }
                    }
                }
            }
        } else {
            // ================================ tap producer warps ================================
            const int pt = tid - NC - 32;
            int tb = 0; unsigned tpar = 0;
            for (int row = 0; row < nrows; ++row) {
                const int tile = row * G + ((row & 1) ? G - 1 - bid : bid);
                if (tile >= F.ntiles) continue;
                const int4 tl = F.tiles[tile];
                const int r = tl.x, k0 = tl.y;
                const int sh = (r - N) & 1;
                const int e0 = F.pair_off[tl.z];
                const int g0 = F.grp_off[tl.z], ngrp = F.grp_off[tl.z + 1] - g0 - 1;
                for (int b = 0; b < B; ++b)                                  // the consumers walk the groups once per map
                for (int gi = 0; gi < ngrp; ++gi) {
                unsigned char *tbuf = tapbase + (size_t)tb * TL.bytes;
                float2 *S = reinterpret_cast<float2 *>(tbuf);
                int4 *desc = reinterpret_cast<int4 *>(tbuf + TL.desc);
                int *exc_e = reinterpret_cast<int *>(tbuf + TL.exc_e), *exc_j = reinterpret_cast<int *>(tbuf + TL.exc_j);
                float *exc_k = reinterpret_cast<float *>(tbuf + TL.exc_k);
                int *nexc = reinterpret_cast<int *>(tbuf + TL.nexc);
                const int ge0 = F.grp_e[g0 + gi], ge1 = F.grp_e[g0 + gi + 1];    // input rings of this group
                mbar_wait_sleep(&tap_empty[tb], tpar ^ 1u);                   // consumers are done with this buffer
                if (pt == 0) *nexc = 0;
                bar_named(1, kTapThreads);
                for (int e = ge0; e < ge1; ++e) {
                    const PairEnt pe = F.pairs[e0 + e];
                    const int wo = F.woff[e0 + e];
                    int delta, w0a, a0, ng;
                    belt_window<PX>(pe, sh, k0, delta, w0a, a0, ng);
                    if (pt == 0) desc[e - ge0] = make_int4(ng, wo * 8, 2 * pe.hw + 1, a0);
                    // nearest pixel of ring rq in azimuth: kc = k + delta, at angle dcc from p.  In the belt
                    // Y = N (2k + 1 - sh + shq), so delta = (1 - sh + shq) >> 1 and the remainder is N or 0.
                    const int Yk = 1 - sh + pe.shq;
                    const float dcc = (float)(N - ((Yk & 1) ? N : 0)) * pe.cdc;
                    PairEntD pd{};
                    if (P.hp) pd = F.pairsd[e0 + e];
                    const double dcc64 = (double)(N - ((Yk & 1) ? N : 0)) * pd.cdc;
                    // S[i] = (w[x], w[x-1]), x = i - (PX - 2) - a0: chunk g of 4 staged positions uses S[4g .. 4g + PX + 1]
                    const int nS = 4 * ng + PX - 2;
                    for (int i = pt; i < nS; i += kTapThreads) {
                        const int x = i - (PX - 2) - a0;
                        float w2[2];
#pragma unroll
                        for (int q = 0; q < 2; ++q) {
                            const int xx = x - q;
                            float w = 0.f;
                            if (xx >= 0 && xx <= 2 * pe.hw) {
                                bool unc; float Ku;
                                w = belt_tap(P, pe, xx - pe.hw, dcc, unc, Ku, &pd, dcc64);
                                if (unc && q == 0) {                          // list every uncertain tap once
                                    const int slot = atomicAdd(nexc, 1);
                                    if (slot < kMaxExc) { exc_e[slot] = e; exc_j[slot] = xx - pe.hw; exc_k[slot] = Ku; }
                                }
                            }
                            w2[q] = w;
                        }
                        S[wo + i] = make_float2(w2[0], w2[1]);
                    }
                }
                mbar_arrive(&tap_full[tb]);
                if (++tb == NTB) { tb = 0; tpar ^= 1u; }
                }
            }
        }
        return;
    }

    // ==================================== consumers ====================================
    if (NC == 256) asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    if (NC == 512) asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
    int buf = 0; unsigned par = 0;
    int tb = 0; unsigned tpar = 0;
    const int half = W8 ? tid / (NC / 2) : 0, u8 = W8 ? tid % (NC / 2) : 0, sk = W8 ? (lane >> 2) & 1 : 0;   // (W8) hemisphere, 8-pixel group, plane order
    const unsigned taddr = TM ? s_tmem + ((((unsigned)(tid >> 5) & 3u) * 32u) << 16) + ((unsigned)tid >> 7) * 32u : 0u;
    for (int row = 0; row < nrows; ++row) {
        const int tile = row * G + ((row & 1) ? G - 1 - bid : bid);
        if (tile >= F.ntiles) continue;
        const int4 tl = F.tiles[tile];
        const int r = tl.x, k0 = tl.y;
        const int sh = (r - N) & 1;
        const int e0 = F.pair_off[tl.z];
        const int g0 = F.grp_off[tl.z], ngrp = F.grp_off[tl.z + 1] - g0 - 1;   // groups of input rings whose taps fit a buffer

        for (int b = 0; b < B; ++b) {
            const float *__restrict__ in = io.in[b];
            float2 tot01[8], tot23[8], acc01[8], acc23[8];
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                tot01[g] = make_float2(0.f, 0.f); tot23[g] = make_float2(0.f, 0.f);
                acc01[g] = make_float2(0.f, 0.f); acc23[g] = make_float2(0.f, 0.f);
            }
            int ntaps = 0;
            bool flushed = false;                                 // TM: the totals in tensor memory are valid
            for (int gi = 0; gi < ngrp; ++gi) {
            const unsigned char *tbuf = tapbase + (size_t)tb * TL.bytes;
            const int4 *desc = reinterpret_cast<const int4 *>(tbuf + TL.desc);
            const int ge0 = F.grp_e[g0 + gi], ge1 = F.grp_e[g0 + gi + 1];
            mbar_wait(&tap_full[tb], tpar);                       // taps of this group are in place
            const int nexc = *reinterpret_cast<const int *>(tbuf + TL.nexc);
            for (int e = ge0; e < ge1; ++e) {
                const int4 d = desc[e - ge0];                             // (chunks, tap offset in bytes, taps)
                const float4 *S4 = reinterpret_cast<const float4 *>(tbuf + d.y);   // S4[2 g + i] = S[4 g + 2 i .. + 1]
                mbar_wait(&full_bar[buf], par);
                if constexpr (W8) {
                // chunk g4 = 4 staged positions x 4 images: 5 LDS.128 of tap pairs (broadcast) + 4 LDS.128 of map values,
                // then 64 FFMA2.  Slot s of this thread is image 4 half + (s ^ sk); pixel pair p of slot s lives in
                // acc01[s], acc23[s], acc01[4 + s], acc23[4 + s] for p = 0 .. 3.  (A register-only loop of this
                // operand pattern -- tap pair and accumulator pair from the register file, the tap pair reused by 4 FFMA2 --
                // sustains ~105 of 128 FMA / clk / SM: sc_debug_fma_peak mode 2.)
                const float *pl0 = stage + (size_t)buf * 8 * LP + (size_t)(4 * half) * LP + 8 * u8;
                const float *pA = pl0 + sk * LP, *pB = pl0 - sk * LP;     // even / odd slots
                float4 tp[5], mv[4];
                auto load8 = [&](int g4) {
#pragma unroll
                    for (int i = 0; i < 5; ++i) tp[i] = S4[2 * g4 + i];
                    mv[0] = *reinterpret_cast<const float4 *>(pA + 4 * g4);
                    mv[1] = *reinterpret_cast<const float4 *>(pB + LP + 4 * g4);
                    mv[2] = *reinterpret_cast<const float4 *>(pA + 2 * LP + 4 * g4);
                    mv[3] = *reinterpret_cast<const float4 *>(pB + 3 * LP + 4 * g4);
                };
                auto fma8 = [&](auto MK) {
                    constexpr unsigned mk = decltype(MK)::value;
                    // pairs (w[x], w[x-1]) of the 10 tap positions this chunk touches: pixel pair p at position i uses pwr[6 - 2p + i]
                    const float2 pwr[10] = {make_float2(tp[0].x, tp[0].y), make_float2(tp[0].z, tp[0].w), make_float2(tp[1].x, tp[1].y),
                                            make_float2(tp[1].z, tp[1].w), make_float2(tp[2].x, tp[2].y), make_float2(tp[2].z, tp[2].w),
                                            make_float2(tp[3].x, tp[3].y), make_float2(tp[3].z, tp[3].w), make_float2(tp[4].x, tp[4].y),
                                            make_float2(tp[4].z, tp[4].w)};
#pragma unroll
                    for (int sl = 0; sl < 4; ++sl) {
                        const float mm[4] = {mv[sl].x, mv[sl].y, mv[sl].z, mv[sl].w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const float2 m2 = make_float2(mm[i], mm[i]);
                            if ((mk >> i) & 1) acc01[sl] = __ffma2_rn(pwr[6 + i], m2, acc01[sl]);
                            if ((mk >> (4 + i)) & 1) acc23[sl] = __ffma2_rn(pwr[4 + i], m2, acc23[sl]);
                            if ((mk >> (8 + i)) & 1) acc01[4 + sl] = __ffma2_rn(pwr[2 + i], m2, acc01[4 + sl]);
                            if ((mk >> (12 + i)) & 1) acc23[4 + sl] = __ffma2_rn(pwr[i], m2, acc23[4 + sl]);
                        }
                    }
                };
#define SC_MK(m) std::integral_constant<unsigned, (m)>{}
                const int ng = d.x, a0 = d.w;
                int g4 = 0, gend = ng;
                if (ng >= 4) {                                            // (else: every chunk with the full body, the taps are 0 there)
                    switch (a0) {
                        case 0: load8(0); fma8(SC_MK(belt_front_mask(0, 0))); load8(1); fma8(SC_MK(belt_front_mask(1, 0))); break;
                        case 1: load8(0); fma8(SC_MK(belt_front_mask(0, 1))); load8(1); fma8(SC_MK(belt_front_mask(1, 1))); break;
                        case 2: load8(0); fma8(SC_MK(belt_front_mask(0, 2))); load8(1); fma8(SC_MK(belt_front_mask(1, 2))); break;
                        default: load8(0); fma8(SC_MK(belt_front_mask(0, 3))); load8(1); fma8(SC_MK(belt_front_mask(1, 3))); break;
                    }
                    g4 = 2; gend = ng - 2;
                }
#pragma unroll 1
                for (; g4 < gend; ++g4) {
                    load8(g4);
                    fma8(SC_MK(0xFFFFu));
                }
                if (ng >= 4) {
                    const int remq = a0 + d.z + 6 - 4 * (ng - 1);         // 0 .. 3
                    switch (remq) {
                        case 0: load8(ng - 2); fma8(SC_MK(belt_back_mask(0, 0))); load8(ng - 1); fma8(SC_MK(belt_back_mask(1, 0))); break;
                        case 1: load8(ng - 2); fma8(SC_MK(belt_back_mask(0, 1))); load8(ng - 1); fma8(SC_MK(belt_back_mask(1, 1))); break;
                        case 2: load8(ng - 2); fma8(SC_MK(belt_back_mask(0, 2))); load8(ng - 1); fma8(SC_MK(belt_back_mask(1, 2))); break;
                        default: load8(ng - 2); fma8(SC_MK(belt_back_mask(0, 3))); load8(ng - 1); fma8(SC_MK(belt_back_mask(1, 3))); break;
                    }
                }
#undef SC_MK
                } else {
                const float *pl = stage + (size_t)buf * 8 * LP + 4 * tid;
                // chunk g4 = 4 staged positions x 8 images: 3 LDS.128 of tap pairs (broadcast) + 8 LDS.128 of map
                // values, then 64 FFMA2.  The loads of chunk g4 + 1 are issued before the FMAs of chunk g4.
                float4 tp[2][3], mv[2][8];
                auto load_chunk = [&](int g4, float4 (&t)[3], float4 (&m)[8]) {
#pragma unroll
                    for (int i = 0; i < 3; ++i) t[i] = S4[2 * g4 + i];
#pragma unroll
                    for (int g = 0; g < 8; ++g) m[g] = *reinterpret_cast<const float4 *>(pl + g * LP + 4 * g4);
                };
                auto fma_chunk = [&](const float4 (&t)[3], const float4 (&m)[8]) {
                    // pairs (w[x], w[x-1]) of the 6 tap positions this chunk touches
                    const float2 pwr[6] = {make_float2(t[0].x, t[0].y), make_float2(t[0].z, t[0].w), make_float2(t[1].x, t[1].y),
                                           make_float2(t[1].z, t[1].w), make_float2(t[2].x, t[2].y), make_float2(t[2].z, t[2].w)};
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        const float mm[4] = {m[g].x, m[g].y, m[g].z, m[g].w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const float2 m2 = make_float2(mm[i], mm[i]);
                            acc01[g] = __ffma2_rn(pwr[2 + i], m2, acc01[g]);
                            acc23[g] = __ffma2_rn(pwr[i], m2, acc23[g]);
                        }
                    }
                };
                // Edge chunks.  With q = 4 g4 + p - a0 the tap pair of pixels (0,1) at chunk position p is
                // non-zero only for 0 <= q <= 2hw + 1 and that of pixels (2,3) only for 2 <= q <= 2hw + 3, so
                // the first and the last chunk of a ring run a body WITHOUT the FFMA2s that would multiply two
                // zero taps (compile-time masks, selected by a warp-uniform switch on the alignment).
                auto fma_masked = [&](const float4 (&t)[3], const float4 (&m)[8], auto M01, auto M23) {
                    constexpr int k01 = decltype(M01)::value, k23 = decltype(M23)::value;
                    const float2 pwr[6] = {make_float2(t[0].x, t[0].y), make_float2(t[0].z, t[0].w), make_float2(t[1].x, t[1].y),
                                           make_float2(t[1].z, t[1].w), make_float2(t[2].x, t[2].y), make_float2(t[2].z, t[2].w)};
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        const float mm[4] = {m[g].x, m[g].y, m[g].z, m[g].w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const float2 m2 = make_float2(mm[i], mm[i]);
                            if ((k01 >> i) & 1) acc01[g] = __ffma2_rn(pwr[2 + i], m2, acc01[g]);
                            if ((k23 >> i) & 1) acc23[g] = __ffma2_rn(pwr[i], m2, acc23[g]);
                        }
                    }
                };
#define SC_MASKS(a, b) std::integral_constant<int, a>{}, std::integral_constant<int, b>{}
                const int ng = d.x, a0 = d.w;
                const int rem = a0 + d.z + 3 - 4 * (ng - 1);              // valid positions of the last chunk, 1 .. 4
                int g4 = 0, gend = ng;
                if (ng >= 2) {
                    load_chunk(0, tp[0], mv[0]);
                    switch (a0) {                                         // pixels (0,1): p >= a0; pixels (2,3): p >= a0 + 2
                        case 0: fma_masked(tp[0], mv[0], SC_MASKS(0xF, 0xC)); break;
                        case 1: fma_masked(tp[0], mv[0], SC_MASKS(0xE, 0x8)); break;
                        case 2: fma_masked(tp[0], mv[0], SC_MASKS(0xC, 0x0)); break;
                        default: fma_masked(tp[0], mv[0], SC_MASKS(0x8, 0x0)); break;
                    }
                    g4 = 1; gend = ng - 1;
                }
#pragma unroll 1
                for (; g4 < gend; ++g4) {
                    load_chunk(g4, tp[0], mv[0]);
                    fma_chunk(tp[0], mv[0]);
                }
                if (ng >= 2) {
                    load_chunk(ng - 1, tp[0], mv[0]);
                    switch (rem) {                                        // pixels (0,1): p <= rem - 3; pixels (2,3): p <= rem - 1
                        case 1: fma_masked(tp[0], mv[0], SC_MASKS(0x0, 0x1)); break;
                        case 2: fma_masked(tp[0], mv[0], SC_MASKS(0x0, 0x3)); break;
                        case 3: fma_masked(tp[0], mv[0], SC_MASKS(0x1, 0x7)); break;
                        default: fma_masked(tp[0], mv[0], SC_MASKS(0x3, 0xF)); break;
                    }
                }
#undef SC_MASKS
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty_bar[buf]);            // this warp is done with the buffer
                if (++buf == NBUF) { buf = 0; par ^= 1u; }
                ntaps += d.z;
                if (TOT && (ntaps >= 48 || e + 1 == ge1)) {
                    if (TM) {                                     // totals += partial sums, 16 columns at a time
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            float v[16], old[16];
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                v[4 * g] = acc01[4 * hh + g].x; v[4 * g + 1] = acc01[4 * hh + g].y;
                                v[4 * g + 2] = acc23[4 * hh + g].x; v[4 * g + 3] = acc23[4 * hh + g].y;
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
#pragma unroll
                        for (int g = 0; g < 8; ++g) { acc01[g] = make_float2(0.f, 0.f); acc23[g] = make_float2(0.f, 0.f); }
                    } else {
#pragma unroll
                        for (int g = 0; g < 8; ++g) {
                            tot01[g] = __fadd2_rn(tot01[g], acc01[g]); tot23[g] = __fadd2_rn(tot23[g], acc23[g]);
                            acc01[g] = make_float2(0.f, 0.f); acc23[g] = make_float2(0.f, 0.f);
                        }
                    }
                    ntaps = 0;
                }
            }

            // ---- uncertain taps of this group: canonical fp64 decision per pixel pair and image -----
            if (nexc > 0) {
                float2 *s01 = (TOT && !TM) ? tot01 : acc01, *s23 = (TOT && !TM) ? tot23 : acc23;   // a set that is in registers now
                float tt[4][8];
#pragma unroll
                for (int g = 0; g < 8; ++g) { tt[0][g] = s01[g].x; tt[1][g] = s01[g].y; tt[2][g] = s23[g].x; tt[3][g] = s23[g].y; }
                auto apply = [&](const PairEnt &pe, int j, float Ku) {
                    const int delta = (1 - sh + pe.shq) >> 1;
                    if constexpr (W8) {
                        // pixel rr8 of this thread, slot sl: tt[rr8 & 3][4 (rr8 >> 2) + sl], image 4 half + (sl ^ sk)
#pragma unroll
                        for (int rr8 = 0; rr8 < 8; ++rr8) {
                            const int k = k0 + 8 * u8 + rr8;
                            const int kq = k + delta + j;
                            const unsigned mask = belt_exact_mask(P, r, k, pe.rq, kq);
                            int kqw = kq % N4; if (kqw < 0) kqw += N4;
#pragma unroll
                            for (int sl = 0; sl < 4; ++sl) {
                                const int g = 4 * half + (sl ^ sk);
                                if (mask & (1u << g)) {
                                    int kk = kqw + (g & 3) * N; if (kk >= N4) kk -= N4;
                                    tt[rr8 & 3][4 * (rr8 >> 2) + sl] =
                                        fmaf(Ku, __ldg(in + (half ? pe.start_s : pe.start_n) + kk), tt[rr8 & 3][4 * (rr8 >> 2) + sl]);
                                }
                            }
                        }
                    } else {
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
                    }
                };
                if (nexc <= kMaxExc) {
                    const int *exc_e = reinterpret_cast<const int *>(tbuf + TL.exc_e), *exc_j = reinterpret_cast<const int *>(tbuf + TL.exc_j);
                    const float *exc_k = reinterpret_cast<const float *>(tbuf + TL.exc_k);
                    for (int i = 0; i < nexc; ++i) apply(F.pairs[e0 + exc_e[i]], exc_j[i], exc_k[i]);
                } else {                              // list overflow: rescan every tap (never seen in practice)
                    for (int e = ge0; e < ge1; ++e) {
                        const PairEnt pe = F.pairs[e0 + e];
                        const int Yk = 1 - sh + pe.shq;
                        const float dcc = (float)(N - ((Yk & 1) ? N : 0)) * pe.cdc;
                        for (int j = -pe.hw; j <= pe.hw; ++j) {
                            bool unc; float Ku;
                            belt_tap(P, pe, j, dcc, unc, Ku);                     // (only `unc` and Ku are used: no fp64 needed)
                            if (unc) apply(pe, j, Ku);
                        }
                    }
                }
#pragma unroll
                for (int g = 0; g < 8; ++g) { s01[g] = make_float2(tt[0][g], tt[1][g]); s23[g] = make_float2(tt[2][g], tt[3][g]); }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&tap_empty[tb]);                   // tap buffer may be refilled
            if (++tb == NTB) { tb = 0; tpar ^= 1u; }
            }
            if (!TOT) {
#pragma unroll
                for (int g = 0; g < 8; ++g) { tot01[g] = acc01[g]; tot23[g] = acc23[g]; }
            }
            if (TM) {                                             // totals from tensor memory + what the exact pairs added
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    float old[16];
                    tmem_ld16(taddr + 16u * hh, old);
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        tot01[4 * hh + g] = make_float2(old[4 * g] + acc01[4 * hh + g].x, old[4 * g + 1] + acc01[4 * hh + g].y);
                        tot23[4 * hh + g] = make_float2(old[4 * g + 2] + acc23[4 * hh + g].x, old[4 * g + 3] + acc23[4 * hh + g].y);
                    }
                }
            }

            // ---- store: 4 consecutive pixels per image -> one 16-byte store ------------------------
            const int start_n = P.start[r - 1], start_s = P.start[N4 - r - 1];
            const bool south = (r != 2 * N);
            const int k = k0 + 4 * tid;
            float *__restrict__ out = io.out[b];
            if constexpr (W8) {                                   // 8 consecutive pixels per image -> two 16-byte stores
                if (!half || south) {
#pragma unroll
                    for (int sl = 0; sl < 4; ++sl) {
                        const int g = sl ^ sk;
                        float *o = out + (half ? start_s : start_n) + k0 + 8 * u8 + g * N;
                        *reinterpret_cast<float4 *>(o) = make_float4(tot01[sl].x * P.omega, tot01[sl].y * P.omega,
                                                                     tot23[sl].x * P.omega, tot23[sl].y * P.omega);
                        *reinterpret_cast<float4 *>(o + 4) = make_float4(tot01[4 + sl].x * P.omega, tot01[4 + sl].y * P.omega,
                                                                         tot23[4 + sl].x * P.omega, tot23[4 + sl].y * P.omega);
                    }
                }
            } else {
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                if (g >= 4 && !south) break;
                const float4 v = make_float4(tot01[g].x * P.omega, tot01[g].y * P.omega, tot23[g].x * P.omega, tot23[g].y * P.omega);
                *reinterpret_cast<float4 *>(out + ((g < 4) ? start_n : start_s) + k + (g & 3) * N) = v;
            }
            }
        }
    }
    if (TM) {                                                      // all consumer warps are done with tensor memory
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        bar_named(2, NC);
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(s_tmem) : "memory");
    }
}

// host ------------------------------------------------------------------------------------------
size_t belt_smem_bytes(int NC, int slack, int px, int nbuf, int ntb, int pw_max, int ne_max) {
    return (size_t)nbuf * 8 * (4 * NC + slack + (px == 8 ? 4 : 0)) * 4 + (size_t)ntb * TapLayout(pw_max, ne_max).bytes;
}

template <int NC, int SLACK, bool TOT, bool TM, bool W8>
static cudaError_t launch_belt_nc(const Dev &P, const BeltDev &F, const Maps &io, int B, size_t smem, int nsm, cudaStream_t st) {
    static bool attr_done[64] = {};
    cudaError_t e = ensure_max_smem(belt_kernel<NC, SLACK, TOT, TM, W8>, attr_done);
    if (e != cudaSuccess) return e;
    const int grid = F.ntiles < nsm ? F.ntiles : nsm;
    belt_kernel<NC, SLACK, TOT, TM, W8><<<grid, NC + kBeltProd, smem, st>>>(P, F, io, B);
    return cudaGetLastError();
}

// variants: (512 consumer threads, slack 64, single accumulator set) for small discs on Nside % 2048 == 0;
// (256 | 128, slack 256 or 512, two accumulator sets) otherwise
cudaError_t launch_belt(const Dev &P, const BeltDev &F, const Maps &io, int B, int threads, int slack, int px, size_t smem,
                        int nsm, cudaStream_t st) {
#define SC_BELT(nc, sl, tot, tm)                                                                                          \
    if (threads == nc && slack == sl)                                                                                     \
        return px == 8 ? launch_belt_nc<nc, sl, tot, tm, true>(P, F, io, B, smem, nsm, st)                                \
                       : launch_belt_nc<nc, sl, tot, tm, false>(P, F, io, B, smem, nsm, st);
    SC_BELT(512, 64, false, false)
    SC_BELT(512, 256, true, true)
    SC_BELT(512, 512, true, true)
    SC_BELT(256, 256, true, false)
    SC_BELT(256, 512, true, false)
    SC_BELT(128, 256, true, false)
#undef SC_BELT
    return cudaErrorInvalidValue;
}

}  // namespace sc
