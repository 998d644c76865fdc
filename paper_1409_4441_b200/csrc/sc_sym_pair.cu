// sc_sym_pair.cu -- the lane-pair instance of the sym kernel (polar caps and the cap/belt transition), one map per
// launch: 16 images per pair geometry with twice the warps of the one-thread-per-pixel-group layout.
//
// The weight K(p, q) of a pair is shared by 16 image pairs (4 rotations x north/south x the reflection phi -> pi/2 - phi,
// see sc_sym.cuh).  Sixteen accumulators per base pixel and 4 base pixels per thread would leave room for 6-8 warps per SM,
// too few to cover the shared-memory latency.  Here TWO ADJACENT LANES share a group of 4 adjacent base pixels:
//   * lane h = 0 accumulates the direct images (planes N, S), lane h = 1 the reflected images (planes NM, SM):
//     4 pixels x 8 images = 32 accumulators per lane;
//   * each lane evaluates the pair geometry and the table lookup for TWO of the four pixels (pixels 2h, 2h + 1, one packed
//     FFMA2 chain and two LDS.64 gathers) and receives the other two weights from its partner with two SHFL.BFLY;
//   * each lane reads its own two planes of the staged position (two LDS.128) and issues 16 FFMA2.
// Per 64 pair-images that is 4 gathers + 4 LDS.128 + 4 SHFL, the same shared-memory traffic as one thread with 64
// accumulators, at half the registers -- 12 consumer warps of 128 registers instead of 6 of 255.
//
// Producers (4 warps): every thread fetches, for a staged position, the 4 rotation images of each plane with coalesced
// 4-byte loads (the image runs are misaligned against each other and the reflected runs are reversed, which rules out
// TMA) and writes them as ONE 16-byte shared-memory store per plane -- a quarter of the shared-memory wavefronts that
// 4-byte cp.async writes of the same data cost -- then arrives on the stage's `full` mbarrier.
//
// Inclusion is decided exactly as in the other kernels: cells below the last need no
// test, beyond tmax + eps the pair is excluded, inside the guard band every image is decided by the canonical fp64 test;
// the two lanes of a pair exchange the (rare) guard-band coordinates so that each applies the verdicts of its own images.
#include "sc_sym.cuh"

namespace sc {

__device__ __forceinline__ float ldg_f32(const float *base, unsigned idx) {
    float v;
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(elem_ptr(base, idx)));   // (.nc.L1::no_allocate: 30 % slower)
    return v;
}
__device__ __forceinline__ void sts128(unsigned a, float x, float y, float z, float w) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

// What the producers hand to everybody for one step (= one input ring) of one sub-tile, through shared memory: the ring
// pair's constants, the staged run and the sub-tile's place on its base ring.  Six 16-byte words.
struct StepInfo {
    float A, c1, c2, c3;            // PairEnt: table coordinate t - 1/2 = A + y (c1 + y (c2 + y (c3 + y c4))), y = d^2
    float dphi, cdc, c4; int w0;    // pixel spacing of the input ring, pi / (4 ip ip'); first staged input pixel (may be < 0)
    int rq, hw, ipq, shq;           // input ring, half window, pixels per quadrant, shift flag
    int start_n, start_s, L, soff;  // ring starts (north, southern mirror); staged positions (0: sub-tile idle), slot offset
    int kq0, km0; unsigned M0; int nw;   // first staged pixel in [0, 4 ipq), its reflected image; floor((2^32 - 1) / (2 ip)); warps
    int r, k0, n, w0s;              // sub-tile: base ring, first base pixel, base pixels, first warp
};
constexpr int kInfoRing = 4;        // entries are written one step ahead and read until the step's buffer is released

// NCW consumer warps + NPW producer warps, 128 registers each.  TOT: per-ring partial sums added to running totals (discs
// of more than ~700 pixels).  Z: two-zone table.  SOUTH: z -> -z images as well (false: north cap only, planes N and NM).
template <int NCW, int NPW, bool TOT, bool Z, bool SOUTH>
__global__ void __launch_bounds__(32 * (NCW + NPW), 1)
sym_pair_kernel(const Dev P, const FastDev F, const Maps io) {
    constexpr int R = 4;                                 // base pixels per lane pair
    constexpr int NC = 32 * NCW, NP = 32 * NPW;
    constexpr int NPLL = SOUTH ? 2 : 1;                  // planes per lane
    constexpr int NPL = 2 * NPLL;                        // staged planes per position: N, (S,) NM(, SM)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);
    const unsigned stage_sh = smem_u32(smem_raw + (((size_t)F.ntab_s * 8 + 127) & ~(size_t)127));
    __shared__ unsigned long long full_bar[kSymBuf], empty_bar[kSymBuf];
    __shared__ __align__(16) StepInfo info[kInfoRing][kMaxSub];
    __shared__ __align__(16) PairEnt pre_pe[kMaxSub];    // publishing threads: ring pair fetched one step early
    __shared__ int4 pub_sf[kMaxSub][2], pub_m[kMaxSub], pub_hd;   // ... their tile, its sub-tile fields and header
    __shared__ int4 head[kInfoRing];                     // per step: first warps of sub-tiles 1 .. 3 (absent: huge), 1 = last step of its tile
    const int tid = threadIdx.x;
    const int N = P.nside;
    const int Ltot = F.Ltot;
    const int GS = gridDim.x, bid = blockIdx.x;
    const int nrows = (F.ntiles + GS - 1) / GS;
    const unsigned plane = (unsigned)Ltot * 16u;

    for (int i = tid; i < F.ntab_s; i += blockDim.x) tab[i] = P.tabh[i];
    if (tid == 0) {
        for (int i = 0; i < kSymBuf; ++i) { mbar_init(&full_bar[i], NP); mbar_init(&empty_bar[i], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned it = 0;                                     // steps so far: buffer it % kSymBuf, use it / kSymBuf
    int rem_unused;

    if (tid >= NC) {
        // ======================================= producers =======================================
        // A producer WARP owns 1 / NPW of the tile's staged slots; a lane takes every 32nd slot of its warp's part, four
        // slots per batch.  The step's runs (one per sub-tile) are worked out ONE STEP AHEAD by the first kMaxSub producer
        // threads and published in `info`, so that nobody walks the dependent loads tile -> ring pair -> pixels in sequence;
        // the loads of a step's first batch are issued BEFORE the wait for the stage buffer, so their latency hides behind
        // the consumers' work on the previous step.
        const int pt = tid - NC, pw = pt >> 5, lane = tid & 31;
        const float *in = io.in[0];
        constexpr int NB = 4;                                // slots per batch and lane
        // A publishing thread (pt < kMaxSub: sub-tile pt) keeps its state in shared memory, not in registers (the producers'
        // registers hold the loads in flight): the tile it last published for with that sub-tile's fields, and the ring pair of
        // the step after the one it published last, fetched one step early with cp.async.
        auto publish = [&](int tile, int step, int s, int slot) {          // -> info[slot][s]
            const SymTile *tl = F.tiles + tile;
            int4 m = pub_m[s];                               // tile, sub-tiles, steps, ring pair prefetched
            if (m.x != tile) {                               // first step of a tile: its fields (dependent loads, once per tile)
                const int4 *q = reinterpret_cast<const int4 *>(&tl->sub[s]);
                pub_sf[s][0] = __ldg(q); pub_sf[s][1] = __ldg(q + 1);
                m = make_int4(tile, __ldg(&tl->nsub), __ldg(&tl->nsteps), 0);
                if (s == 0)
                    pub_hd = make_int4(m.y > 1 ? __ldg(&tl->sub[1].w0) : 0x7fffffff, m.y > 2 ? __ldg(&tl->sub[2].w0) : 0x7fffffff,
                                       m.y > 3 ? __ldg(&tl->sub[3].w0) : 0x7fffffff, 0);
            }
            const int4 sa = pub_sf[s][0], sb = pub_sf[s][1];     // r, k0, n, e0 | ne, w0, nw, soff
            StepInfo o{};
            if (s < m.y) {
                const int r = sa.x, k0 = sa.y, n = sa.z;
                o.r = r; o.k0 = k0; o.n = n; o.w0s = sb.y; o.nw = sb.z;        // also on idle steps (the store needs them)
                if (step < sb.x) {
                    PairEnt pe;
                    if (m.w) {
                        asm volatile("cp.async.wait_all;" ::: "memory");
                        pe = pre_pe[s];
                    } else pe = F.pairs[sa.w + step];
                    const int hw = pe.hw, ipq = pe.ipq, shq = pe.shq, nq = 4 * ipq;
                    const int ips = r < N ? r : N;
                    const int shs = (r >= N) ? ((r - N) & 1) : 0;
                    const unsigned M0s = 0xFFFFFFFFu / (unsigned)(2 * ips);
                    const int a0s = 2 * k0 + 1 - shs, als = 2 * (k0 + n - 1) + 1 - shs;
                    const int w0 = div_fast(a0s * ipq + shq * ips, 2 * ips, M0s, rem_unused) - hw;
                    const int L = div_fast(als * ipq + shq * ips, 2 * ips, M0s, rem_unused) + hw + R - w0;
                    int kq0 = w0 + nq;                    // in [0, 2 nq): w0 >= -hw - 1 > -nq
                    if (kq0 >= nq) kq0 -= nq;
                    // reflected image of position i: pixel ipq - 1 + shq - (w0 + i), walking backwards
                    int km0 = (ipq - 1 + shq - w0) % nq;
                    if (km0 < 0) km0 += nq;
                    o.A = pe.A; o.c1 = pe.c1; o.c2 = pe.c2; o.c3 = pe.c3; o.dphi = pe.dphi; o.cdc = pe.cdc; o.c4 = pe.c4; o.w0 = w0;
                    o.rq = pe.rq; o.hw = hw; o.ipq = ipq; o.shq = shq;
                    o.start_n = pe.start_n; o.start_s = pe.start_s; o.L = L; o.soff = sb.w;
                    o.kq0 = kq0; o.km0 = km0; o.M0 = M0s;
                }
                m.w = step + 1 < sb.x;
                if (m.w) {                                   // the ring pair of the next step, used when that step is published
                    const float *src = reinterpret_cast<const float *>(F.pairs + (sa.w + step + 1));
                    const unsigned dstp = smem_u32(&pre_pe[s]);
#pragma unroll
                    for (int k = 0; k < (int)(sizeof(PairEnt) / 4); ++k) cp_async4_s(dstp + 4u * k, src + k);
                }
            }
            pub_m[s] = m;
            int4 *dst = reinterpret_cast<int4 *>(&info[slot][s]);
            const int4 *src4 = reinterpret_cast<const int4 *>(&o);
#pragma unroll
            for (int k = 0; k < 6; ++k) dst[k] = src4[k];
            if (s == 0) { const int4 hh = pub_hd; head[slot] = make_int4(hh.x, hh.y, hh.z, step + 1 == m.z ? 1 : 0); }
        };
        if (pt < kMaxSub) pub_m[pt] = make_int4(-1, 0, 0, 0);
        int row = 0;
        while (row < nrows && snake_tile(row, GS, bid) >= F.ntiles) ++row;
        if (row < nrows && pt < kMaxSub) publish(snake_tile(row, GS, bid), 0, pt, 0);
        asm volatile("bar.sync 1, %0;" ::"n"(NP) : "memory");
        for (; row < nrows; ++row) {
            const int tile = snake_tile(row, GS, bid);
            if (tile >= F.ntiles) continue;
            const SymTile *tl = F.tiles + tile;
            const int nsub = __ldg(&tl->nsub), nsteps = __ldg(&tl->nsteps);
            const int Ltile = __ldg(&tl->pad0);              // staged slots of the tile (sum of the runs' capacities)
            const int wlo = (Ltile * pw) / NPW, whi = (Ltile * (pw + 1)) / NPW;
            const int so1 = nsub > 1 ? __ldg(&tl->sub[1].soff) : 0x7fffffff, so2 = nsub > 2 ? __ldg(&tl->sub[2].soff) : 0x7fffffff,
                      so3 = nsub > 3 ? __ldg(&tl->sub[3].soff) : 0x7fffffff;
            int nrow = row + 1;                              // the tile after this one
            while (nrow < nrows && snake_tile(nrow, GS, bid) >= F.ntiles) ++nrow;
            for (int step = 0; step < nsteps; ++step, ++it) {
                const int buf = it % kSymBuf;
                const StepInfo *cur = info[it % kInfoRing];
                bool waited = false;
                const unsigned empty_par = ((it / kSymBuf) & 1u) ^ 1u;
                unsigned dst[NB];
                float v[NB][NPL][4];
                // one staged slot: 4 rotation images of every plane -> one 16-byte store per plane
                auto fetch = [&](int q, unsigned &d, float (&w)[NPL][4]) {
                    const int sq = (q >= so1) + (q >= so2) + (q >= so3);
                    const int4 a = *reinterpret_cast<const int4 *>(&cur[sq].start_n);     // start_n, start_s, L, soff
                    const int i = q - a.w;
                    d = 0u;
                    if (q >= whi || i >= a.z || (F.dbg & 2)) return;
                    const int2 k2 = *reinterpret_cast<const int2 *>(&cur[sq].kq0);
                    const unsigned ipq = (unsigned)cur[sq].ipq, nq = 4u * ipq;
                    const float *gn = in + a.x, *gs = in + a.y;
                    unsigned kq = (unsigned)k2.x + (unsigned)i; if (kq >= nq) kq -= nq;
                    int kmi = k2.y - i; if (kmi < 0) kmi += (int)nq;
                    unsigned km = (unsigned)kmi;
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        w[0][m] = ldg_f32(gn, kq);
                        if (SOUTH) w[1][m] = ldg_f32(gs, kq);
                        w[NPLL][m] = ldg_f32(gn, km);
                        if (SOUTH) w[NPLL + 1][m] = ldg_f32(gs, km);
                        kq += ipq; if (kq >= nq) kq -= nq;
                        km += ipq; if (km >= nq) km -= nq;
                    }
                    d = stage_sh + (unsigned)((buf * NPL) * Ltot + a.w) * 16u + 16u * (unsigned)slot_of_pos<R>(i);
                };
                auto put = [&](unsigned d, const float (&w)[NPL][4]) {
                    if (!d) return;
#pragma unroll
                    for (int pl = 0; pl < NPL; ++pl)         // reflected planes: slot ^ 2 (bank groups disjoint from the direct lanes')
                        sts128((pl >= NPLL ? d ^ 32u : d) + pl * plane, w[pl][0], w[pl][1], w[pl][2], w[pl][3]);
                };
                auto ahead = [&]() {     // the runs of the next step (of this tile or of the next one)
                    if (pt < kMaxSub) {
                        if (step + 1 < nsteps) publish(tile, step + 1, pt, (it + 1) % kInfoRing);
                        else if (nrow < nrows) publish(snake_tile(nrow, GS, bid), 0, pt, (it + 1) % kInfoRing);
                    }
                };
                for (int q = wlo + lane; q < whi; q += 32 * NB) {
#pragma unroll
                    for (int u = 0; u < NB; ++u) fetch(q + 32 * u, dst[u], v[u]);
                    if (!waited) {
                        ahead();                                                 // under the latency of the loads just issued
                        mbar_wait_sleep(&empty_bar[buf], empty_par);             // every consumer warp released the buffer
                        waited = true;
                    }
#pragma unroll
                    for (int u = 0; u < NB; ++u) put(dst[u], v[u]);
                }
                if (!waited) {
                    ahead();
                    mbar_wait_sleep(&empty_bar[buf], empty_par);                 // stay in step with the buffer's phases
                }
                mbar_arrive(&full_bar[buf]);             // release: this thread's stores are visible to the waiters
                asm volatile("bar.sync 1, %0;" ::"n"(NP) : "memory");           // the next step's runs are in place
            }
        }
        return;
    }

    // ========================================= consumers =========================================
    const int warp = tid >> 5, lane = tid & 31;
    const int h = lane & 1;                              // 0: direct images, 1: reflected images
    const unsigned thresh = kMagicBits + (unsigned)(P.ntab - 2);   // bits of the last table cell
    const float tmax = P.tmax, eps = P.eps;
    unsigned tab_sh = smem_u32(tab) - kMagicBits * 8u;   // tab[bits - kMagicBits] = [tab_sh + 8 bits]
    asm volatile("mov.u32 %0, %0;" : "+r"(tab_sh));

    // Everything a consumer needs for a step comes from the producers' step records (shared memory): it keeps no per-tile
    // state in registers besides the accumulators -- with nearly all of the SM's L1 configured as shared memory a register
    // spill costs an L2 round trip per step.
    unsigned nit = 0;                                    // steps of all tiles of this CTA
    for (int row = 0; row < nrows; ++row) {
        const int tile = snake_tile(row, GS, bid);
        if (tile < F.ntiles) nit += (unsigned)__ldg(&F.tiles[tile].nsteps);
    }
    // accumulators: [a][plane of this lane][rotation pair]; a = 0, 1: this lane's own pixels 2h, 2h + 1,
    // a = 2, 3: the partner's pixels 2(1 - h), 2(1 - h) + 1
    float2 acc[4][NPLL][2], tot[TOT ? 4 : 1][NPLL][2];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int pl = 0; pl < NPLL; ++pl) {
            acc[a][pl][0] = acc[a][pl][1] = f2(0.f);
            if (TOT) tot[a][pl][0] = tot[a][pl][1] = f2(0.f);
        }

    {
#pragma unroll 1
        for (; it < nit; ++it) {
            const int buf = it % kSymBuf;
            mbar_wait(&full_bar[buf], (it / kSymBuf) & 1u);
            const int4 hd = head[it % kInfoRing];
            const int si = (warp >= hd.x) + (warp >= hd.y) + (warp >= hd.z);      // this warp's sub-tile
            // this step's ring pair and run, published by the producers
            const StepInfo *inf = &info[it % kInfoRing][si];
            const int4 q2 = *reinterpret_cast<const int4 *>(&inf->rq);               // rq, hw, ipq, shq
            const int4 q5 = *reinterpret_cast<const int4 *>(&inf->r);                // r, k0, n, first warp
            if (warp < q5.w + inf->nw && inf->L > 0 && !(F.dbg & 1)) {
                const float4 q0 = *reinterpret_cast<const float4 *>(&inf->A);        // A, c1, c2, c3
                const float4 q1 = *reinterpret_cast<const float4 *>(&inf->dphi);     // dphi, cdc, c4, (w0)
                const int hw = q2.y, ipq = q2.z;
                // this lane pair's pixel group: first pixel ka (clamped to the run's last), 2 ka + 1 - shift
                const int ip = q5.x < N ? q5.x : N;
                const int ap = 2 * min(q5.y + R * (16 * (warp - q5.w) + (lane >> 1)), q5.y + q5.z - 1) + 1 - ((q5.x >= N) ? ((q5.x - N) & 1) : 0);
                const int ip2 = 2 * ip;
                int rem;
                const int kc = div_fast(ap * ipq + q2.w * ip, ip2, inf->M0, rem);
                // azimuth of input pixel kc + j seen from base pixel ka + rr:  d = (ip - rem - 2 rr ipq) cdc + j dphi'
                const int rr0 = 2 * h;
                const float2 dc = f2((float)(ip - rem - 2 * rr0 * ipq) * q1.y, (float)(ip - rem - 2 * (rr0 + 1) * ipq) * q1.y);
                const int i0 = kc - inf->w0;             // staged position of input pixel kc + j: i0 + j
                // this lane's first plane of the sub-tile's staged run
                unsigned pn = stage_sh + (unsigned)((buf * NPL + h * NPLL) * Ltot + inf->soff) * 16u;
                asm volatile("mov.u32 %0, %0;" : "+r"(pn));

                const float2 dphi2 = f2(q1.x), c4 = f2(q1.z), c3 = f2(q0.w), c2 = f2(q0.z), c1 = f2(q0.y), A2 = f2(q0.x);
                const float2 za2 = f2(P.z_alpha), zao2 = f2(0.5f * P.z_alpha - 0.5f), zg2 = f2(P.z_gamma), zgo2 = f2(0.5f * P.z_gamma - P.z_t1g - 0.5f);
                const float zhm1f = (float)P.z_hm1;
                const unsigned zhm1 = (unsigned)P.z_hm1;

                // One window position: the geometry of this lane's two pixels (one packed chain) -> lookup coordinate
                // - 1/2 and table cell bits.  Cells below the last: plain lookup; from tmax - eps on: the zero cell after the
                // table (weight 0) -- pairs inside the guard band |t - tmax| <= eps are decided exactly in a second pass.
                const float tzh = tmax - eps - 0.5f, tch = tmax - 0.5f;
                auto geom = [&](float2 jf, float2 &gt, unsigned &gc0, unsigned &gc1, float2 &t2) {
                    const float2 d = __ffma2_rn(jf, dphi2, dc);
                    const float2 y = __fmul2_rn(d, d);
                    float2 p = __ffma2_rn(y, c4, c3);
                    p = __ffma2_rn(y, p, c2);
                    p = __ffma2_rn(y, p, c1);
                    t2 = __ffma2_rn(y, p, A2);                           // t - 1/2
                    // t >= tmax - eps -> far beyond the table (clamped onto the zero cell below)
                    const float2 ts = f2(t2.x >= tzh ? 3.0e6f : t2.x, t2.y >= tzh ? 3.0e6f : t2.y);
                    const float2 bb = __fadd2_rn(ts, f2(kMagic));
                    gt = t2;
                    gc0 = __float_as_uint(bb.x); gc1 = __float_as_uint(bb.y);
                    if (Z) {
                        // inner zone: alpha t - 1/2; outer zone: gamma (t - t1) - 1/2 RELATIVE to the zone start
                        const float2 l1 = __ffma2_rn(t2, za2, zao2), l2 = __ffma2_rn(t2, zg2, zgo2);
                        const bool o0 = l2.x + zhm1f < l1.x, o1 = l2.y + zhm1f < l1.y;
                        const float2 tz = f2(o0 ? l2.x : l1.x, o1 ? l2.y : l1.y);
                        const float2 bz = __fadd2_rn(tz, f2(kMagic));
                        const float2 fz = __fadd2_rn(tz, __fadd2_rn(f2(kMagic), f2(-bz.x, -bz.y)));   // position - 1/2 in the cell
                        gt = fz;
                        const unsigned z0 = __float_as_uint(bz.x) + (o0 ? zhm1 : 0u), z1 = __float_as_uint(bz.y) + (o1 ? zhm1 : 0u);
                        gc0 = t2.x >= tzh ? thresh + 1u : z0; gc1 = t2.y >= tzh ? thresh + 1u : z1;
                    }
                    gc0 = min(gc0, thresh + 1u); gc1 = min(gc1, thresh + 1u);
                };

                const int pend = i0 + hw + R - 1;
                const unsigned hx = 2u * (unsigned)h;                    // reflected planes are staged at slot ^ 2
                float2 jf = f2((float)(-hw));
                float2 near = f2(1.0e30f);                               // min |t - tmax| over the window, per pixel
#pragma unroll 2
                for (int pos = i0 - hw; pos <= pend; ++pos) {
                    float2 gt, t2;
                    unsigned gc0, gc1;
                    geom(jf, gt, gc0, gc1, t2);
                    const float2 dt = __fadd2_rn(t2, f2(-tch));
                    near = f2(fminf(near.x, fabsf(dt.x)), fminf(near.y, fabsf(dt.y)));
                    // ---- table cells of the two pixels, the staged values of this lane's planes
                    float2 el0, el1;
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(el0.x), "=f"(el0.y) : "r"(tab_sh + gc0 * 8u));
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(el1.x), "=f"(el1.y) : "r"(tab_sh + gc1 * 8u));
                    const unsigned ad = pn + 16u * ((unsigned)slot_of_pos<R>(pos) ^ hx);
                    float4 mv[NPLL];
#pragma unroll
                    for (int pl = 0; pl < NPLL; ++pl) mv[pl] = lds128(ad + pl * plane);
                    // ---- weights: two of my own, two from the partner lane
                    float K[4];
                    K[0] = fmaf(gt.x, el0.y, el0.x);
                    K[1] = fmaf(gt.y, el1.y, el1.x);
                    K[2] = __shfl_xor_sync(0xFFFFFFFFu, K[0], 1);
                    K[3] = __shfl_xor_sync(0xFFFFFFFFu, K[1], 1);
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int pl = 0; pl < NPLL; ++pl) {
                            acc[a][pl][0] = __ffma2_rn(f2(K[a]), f2(mv[pl].x, mv[pl].y), acc[a][pl][0]);
                            acc[a][pl][1] = __ffma2_rn(f2(K[a]), f2(mv[pl].z, mv[pl].w), acc[a][pl][1]);
                        }
                    jf = __fadd2_rn(jf, f2(1.0f));
                }

                // ---- second pass (rare): some pair of this warp lies inside the guard band.  Same arithmetic -> same t;
                // every image of such a pair is decided by the canonical fp64 test, each lane applies those of its planes.
                if (__any_sync(0xFFFFFFFFu, fminf(near.x, near.y) <= eps)) {
                    // (what this pass needs is derived again from the step counter and the step record rather than kept in
                    // registers across the pair loop)
                    unsigned itb = it;
                    asm volatile("mov.u32 %0, %0;" : "+r"(itb));
                    const int4 h2 = head[itb % kInfoRing];
                    const StepInfo *in2 = &info[itb % kInfoRing][(warp >= h2.x) + (warp >= h2.y) + (warp >= h2.z)];
                    const int4 s2 = *reinterpret_cast<const int4 *>(&in2->rq), s5 = *reinterpret_cast<const int4 *>(&in2->r);
                    struct { int r, ip, sh, ka; } g;
                    g.r = s5.x; g.ip = s5.x < N ? s5.x : N; g.sh = (s5.x >= N) ? ((s5.x - N) & 1) : 0;
                    g.ka = min(s5.y + R * (16 * (warp - s5.w) + (lane >> 1)), s5.y + s5.z - 1);
                    const int hw = s2.y, ipq = s2.z;
                    int rem2;
                    const int kc = div_fast((2 * g.ka + 1 - g.sh) * ipq + s2.w * g.ip, 2 * g.ip, in2->M0, rem2);
                    const int i0 = kc - in2->w0, pend = i0 + hw + R - 1;
                    const int4 q2 = s2;
                    const unsigned pn = stage_sh + (unsigned)(((itb % kSymBuf) * NPL + h * NPLL) * Ltot + in2->soff) * 16u;
                    const float2 el = tab[P.ntab - 2];
                    auto apply_exact = [&](int rr, int a, float t, int pos) {
                        const unsigned mask = sym_exact_mask(P, g.r, g.ka + rr, g.ip, g.sh, q2.x, kc + pos - i0, ipq, q2.w, t, SOUTH ? 1 : 0, 1);
                        const unsigned mine = mask >> (4 * NPLL * h);
                        if (!(mine & (SOUTH ? 0xFFu : 0xFu))) return;
                        float xk = fminf(t, tmax) - 0.5f;
                        if (Z) { int jz; zoned_cell(P, fminf(t, tmax), jz, xk); xk -= 0.5f; }      // last cell, centred form
                        const float Ku = fmaf(xk, el.y, el.x);
                        const unsigned ad = pn + 16u * ((unsigned)slot_of_pos<R>(pos) ^ hx);
#pragma unroll
                        for (int pl = 0; pl < NPLL; ++pl) {
                            const float4 mq = lds128(ad + pl * plane);
                            const unsigned mk = mine >> (4 * pl);
                            if (mk & 1u) acc[a][pl][0].x = fmaf(Ku, mq.x, acc[a][pl][0].x);
                            if (mk & 2u) acc[a][pl][0].y = fmaf(Ku, mq.y, acc[a][pl][0].y);
                            if (mk & 4u) acc[a][pl][1].x = fmaf(Ku, mq.z, acc[a][pl][1].x);
                            if (mk & 8u) acc[a][pl][1].y = fmaf(Ku, mq.w, acc[a][pl][1].y);
                        }
                    };
                    float2 jg = f2((float)(-hw));
#pragma unroll 1
                    for (int pos = i0 - hw; pos <= pend; ++pos) {
                        float2 gt, t2;
                        unsigned gc0, gc1;
                        geom(jg, gt, gc0, gc1, t2);
                        jg = __fadd2_rn(jg, f2(1.0f));
                        const float ta = t2.x + 0.5f, tb = t2.y + 0.5f;
                        const int ea = (ta >= tmax - eps && ta <= tmax + eps) ? 1 : 0, eb = (tb >= tmax - eps && tb <= tmax + eps) ? 1 : 0;
                        if (!__any_sync(0xFFFFFFFFu, ea | eb)) continue;
                        const float tpa = __shfl_xor_sync(0xFFFFFFFFu, ta, 1), tpb = __shfl_xor_sync(0xFFFFFFFFu, tb, 1);
                        const int epa = __shfl_xor_sync(0xFFFFFFFFu, ea, 1), epb = __shfl_xor_sync(0xFFFFFFFFu, eb, 1);
                        if (ea) apply_exact(rr0, 0, ta, pos);
                        if (eb) apply_exact(rr0 + 1, 1, tb, pos);
                        if (epa) apply_exact(2 - rr0, 2, tpa, pos);
                        if (epb) apply_exact(3 - rr0, 3, tpb, pos);
                    }
                }
                if (TOT) {
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int pl = 0; pl < NPLL; ++pl) {
                            tot[a][pl][0] = __fadd2_rn(tot[a][pl][0], acc[a][pl][0]); acc[a][pl][0] = f2(0.f);
                            tot[a][pl][1] = __fadd2_rn(tot[a][pl][1], acc[a][pl][1]); acc[a][pl][1] = f2(0.f);
                        }
                }
            }
            // what the store of a tile's last step needs, read before the buffer (and with it the step record) is released
            unsigned itc = it;
            asm volatile("mov.u32 %0, %0;" : "+r"(itc));
            const int4 h3 = head[itc % kInfoRing];
            const int last = h3.w;
            int4 g5 = make_int4(0, 0, 0, 0);
            int gnw = 0;
            if (last) {
                const StepInfo *in3 = &info[itc % kInfoRing][(warp >= h3.x) + (warp >= h3.y) + (warp >= h3.z)];
                g5 = *reinterpret_cast<const int4 *>(&in3->r); gnw = in3->nw;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[itc % kSymBuf]);       // this warp is done with the buffer

            // last step of the tile: store the images of every valid base pixel (lane 0 of the pair the direct ones, lane 1
            // the reflected ones) and clear the sums
            if (last) {
                if (warp < g5.w + gnw) {
                    const int r = g5.x;
                    const int ip = r < N ? r : N, sh = (r >= N) ? ((r - N) & 1) : 0;
                    const int klast = g5.y + g5.z - 1;
                    const int kmine = g5.y + R * (16 * (warp - g5.w) + (lane >> 1));
                    const int start_n = P.start[r - 1], start_s = P.start[4 * N - r - 1];
                    const bool south_img = (r != 2 * N);
#pragma unroll
                    for (int a = 0; a < 4; ++a) {
                        const int rr = a < 2 ? 2 * h + a : 2 * (1 - h) + (a - 2);
                        const int k = kmine + rr;
                        if (k > klast) continue;
                        // reflected base pixel; a pixel on the mirror axis (or at phi = 0 of a shifted ring, whose reflection
                        // is its own rotation image) is its own mirror image: stored once, by the direct lane
                        const int km = ip - 1 + sh - k;
                        if (h && ((2 * k == ip - 1 + sh) || (sh && k == 0))) continue;
#pragma unroll
                        for (int pl = 0; pl < NPLL; ++pl) {
                            if (pl == 1 && !south_img) continue;
                            const float2 *sm = TOT ? tot[TOT ? a : 0][pl] : acc[a][pl];
                            const float v[4] = {sm[0].x, sm[0].y, sm[1].x, sm[1].y};
                            const int base = (pl ? start_s : start_n) + (h ? km : k);
#pragma unroll
                            for (int m = 0; m < 4; ++m) io.out[0][base + m * ip] = v[m] * P.omega;
                        }
                    }
                }
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int pl = 0; pl < NPLL; ++pl) {
                        acc[a][pl][0] = acc[a][pl][1] = f2(0.f);
                        if (TOT) tot[a][pl][0] = tot[a][pl][1] = f2(0.f);
                    }
            }
        }
    }
}

template <int NCW, int NPW, bool TOT, bool Z, bool SOUTH>
static cudaError_t launch_pair(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st) {
    const char *dbg = std::getenv("SC_DBG");
    FastDev F{L.pairs, L.tiles, L.ntiles, L.Ltot, L.ntab_s, dbg ? std::atoi(dbg) : 0, nullptr, nullptr};
    static bool attr_done[64] = {};
    cudaError_t e = ensure_max_smem(sym_pair_kernel<NCW, NPW, TOT, Z, SOUTH>, attr_done);
    if (e != cudaSuccess) return e;
    const int grid = std::min(L.nsm, L.ntiles);
    if (grid <= 0) return cudaSuccess;
    sym_pair_kernel<NCW, NPW, TOT, Z, SOUTH><<<grid, 32 * (NCW + NPW), L.smem, st>>>(P, F, io);
    return cudaGetLastError();
}

// L.threads = consumer threads: 384 (12 warps + 4 producer warps) or 320 (10 + 6): 512 threads of 128 registers
cudaError_t dispatch_sym_pair(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st) {
    const bool z = P.zoned != 0;
#define SC_GO(NCW, NPW, TOT, SOUTH) \
    return z ? launch_pair<NCW, NPW, TOT, true, SOUTH>(L, P, io, st) : launch_pair<NCW, NPW, TOT, false, SOUTH>(L, P, io, st)
    if (L.R != 4 || !L.mirror) return cudaErrorInvalidValue;
    if (L.south) {
        if (L.threads == 384 && !L.tot) { SC_GO(12, 4, false, true); }
        if (L.threads == 320 && !L.tot) { SC_GO(10, 6, false, true); }
        if (L.threads == 256 && L.tot) { SC_GO(8, 4, true, true); }
    } else {
        if (L.threads == 384 && !L.tot) { SC_GO(12, 4, false, false); }
        if (L.threads == 384 && L.tot) { SC_GO(12, 4, true, false); }
    }
#undef SC_GO
    return cudaErrorInvalidValue;
}

}  // namespace sc
