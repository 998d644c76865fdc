// sc_sym.cuh -- the sym kernel (polar caps and the cap/belt transition) and its launcher template.
// Included by the translation units that instantiate it (sc_sym_b1.cu: one map per launch; sc_sym_bn.cu: batches).
//
// Design:
//  * HEALPix RING is invariant under phi -> phi + pi/2, z -> -z and the reflection phi -> pi/2 - phi, so the
//    weight K(p, q) of a pair is shared by up to 16 image pairs (4 rotations x north/south x mirror).  A thread
//    owns R adjacent BASE pixels (ring r <= 2N; in-ring index k in the first quadrant, or in its first half when
//    the mirror images are used), evaluates the pair geometry and the table lookup once per (base pixel, input
//    pixel) and FMA-accumulates one output per image and map with packed FFMA2.
//    Template flags: SOUTH = z -> -z images, MIRROR = reflected images; staged planes per position
//    NPL = (1 + SOUTH)(1 + MIRROR), each plane holding the 4 rotation images as one float4.
//  * A persistent CTA works through tiles (runs of consecutive base pixels on one ring; several short runs
//    of the rings near the pole are packed into one tile).  It is warp-specialised: producer warps stage, for every
//    input ring within theta_max, the needed run of map values of every image into shared memory, reporting to
//    full/empty mbarriers; the consumer warps (setmaxnreg gives them the producers' registers) run the pair loop.
//    No block-wide barrier after the prologue.  Two stage layouts: the 4 rotation images of a position interleaved
//    as one float4, written with 4-byte cp.async (the image runs are 4-byte-misaligned against each other and the
//    mirrored runs are reversed, which rules out TMA for this layout); or PLANAR (flag PLN, sc_sym_pl.cu: one map,
//    small discs) -- one plane per image, filled by TMA bulk copies of 16-byte-aligned ring pieces, read with LDS.32
//    by lanes kept exactly R positions apart (lane skew), two positions per straight-line block.
//  * Pair geometry in fp32 without cancellation: t = A + B (1 - cos d) with A, B per ring pair from
//    fp64, d = azimuth difference built from the INTEGER pixel offset (exact) times the ring's pixel
//    spacing; 1 - cos d by a 4-term even polynomial (|d| <= ~0.9 rad on the rings this kernel takes;
//    the few rings next to the poles go to the generic kernel).  The mirrored pair has d' = -d: same t.
//  * Table lookup: magic-number rounding gives the cell index; K = a_i + t b_i (one FFMA); the
//    16K-entry (a, b) table lives in shared memory (128 KB).
//  * Inclusion: t < tmax - 1 needs no test at all (fast path); the last cell and everything beyond
//    takes a branch: t > tmax + eps -> excluded, |t - tmax| <= eps -> canonical fp64 test for each
//    of the images separately (bit-exact with the oracle), else included.
//  * Sums: per-ring partial sums added to running totals (registers, or tensor memory via tcgen05.ld/st for
//    the 384-consumer variant on mid-size discs); a single set for discs of at most 700 pixels.
#pragma once
#include "sc_fast.cuh"

#include <algorithm>
#include <cstdlib>
#include <type_traits>

namespace sc {

// floor(Y / d) and remainder for 0 <= Y < 2^31 with M0 = floor((2^32 - 1) / d): one multiply-high
// and one fix-up instead of an integer division
__device__ __forceinline__ int div_fast(int Y, int d, unsigned M0, int &rem) {
    int q = (int)__umulhi((unsigned)Y, M0);
    rem = Y - q * d;
    if (rem >= d) { ++q; rem -= d; }
    return q;
}

// Exact decisions for the images of one uncertain pair: bit 4 pl + m set <=> rotation m of plane pl included;
// planes are ordered north, south (if `south`), north mirrored, south mirrored (if `mirror`).
// (k, sh) / (kq, shq): in-ring index and shift flag of the base pixel / the input pixel.
static __device__ __noinline__ unsigned sym_exact_mask(const Dev &P, int r, int k, int ip, int sh, int rq, int kq,
                                                       int ipq, int shq, float t, int south, int mirror) {
    const int N4 = 4 * P.nside;
    const int n = 4 * ip, nq = 4 * ipq;
    unsigned mask = 0;
    kq %= nq; if (kq < 0) kq += nq;
    {   // one image decides for all unless it is within kImageMargin of the threshold
        const double d0 = canonical_dot(P, r, k, rq, kq);
        if (fabs(d0 - P.c) > fmax(kImageMargin, 2.0 * P.ke_band)) return d0 >= P.c ? (1u << (4 * (1 + south) * (1 + mirror))) - 1u : 0u;
    }
    int pl = 0;
    for (int mi = 0; mi <= mirror; ++mi) {
        // reflection phi -> pi/2 - phi: (2 k' + 1 - sh) = 2 ip - (2 k + 1 - sh)
        int kb = mi ? ip - 1 + sh - k : k;
        int kqb = mi ? ipq - 1 + shq - kq : kq;
        if (kb < 0) kb += n;
        if (kqb < 0) kqb += nq;
        for (int h = 0; h <= south; ++h, ++pl) {
            const int rp_i = h ? N4 - r : r, rq_i = h ? N4 - rq : rq;
            for (int m = 0; m < 4; ++m) {
                int kp_i = kb + m * ip; if (kp_i >= n) kp_i -= n;
                int kq_i = kqb + m * ipq; if (kq_i >= nq) kq_i -= nq;
                if (exact_included(P, rp_i, kp_i, rq_i, kq_i, t, nullptr)) mask |= 1u << (4 * pl + m);
            }
        }
    }
    return mask;
}

// Shared-memory slot (16-byte unit) of staged position i.  A thread owns R adjacent base pixels, so the
// 8 lanes of a quarter warp (one LDS.128 wavefront) read positions R apart.  XOR-ing the low bits with the
// index of the 8-position block spreads such a stride over all 8 bank groups for every alignment, with no
// padding (brute-force checked: 1 wavefront per quarter warp for stride 2 and 4; stride 1 needs nothing).
template <int R> __host__ __device__ __forceinline__ int slot_of_pos(int i) {
    return (R == 1 || R == 3) ? i : (R == 2 ? i ^ ((i >> 3) & 1) : i ^ ((i >> 3) & 3));     // stride 3 is coprime with the 8 bank groups
}

// Packed fp32 helpers (FFMA2 / FADD2 / FMUL2 on sm_100a; a scalar operand is broadcast by the hardware).
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }

// &base[idx] with one IMAD.WIDE.U32
__device__ __forceinline__ const float *elem_ptr(const float *base, unsigned idx) {
    unsigned long long a;
    asm("mad.wide.u32 %0, %1, 4, %2;" : "=l"(a) : "r"(idx), "l"(base));
    return reinterpret_cast<const float *>(a);
}

constexpr int kSymBuf = 2;        // stage buffers
// Producer threads per CTA: they only issue cp.async.  One warpgroup, except in the 192-consumer variant (mirror
// images: twice the staged bytes per base pixel, so half the base pixels fit): 6 consumer + 2 producer warps, i.e. two
// warps on every scheduler, 256 threads that keep the compiler's register count (no setmaxnreg).
#ifndef SC_L192
#define SC_L192 1
#endif
#ifndef SC_R3_PIPE
#define SC_R3_PIPE 0
#endif
// lane skew in every instance (0: only the planar and the batch instances)
#ifndef SC_SKEW_ALL
#define SC_SKEW_ALL 1
#endif
#ifndef SC_SYM_BATCH
#define SC_SYM_BATCH 1
#endif
#ifndef SC_PLN_BATCH
#define SC_PLN_BATCH 1           // planar instances: two positions per straight-line block (one branch for the exact path)
#endif
#ifndef SC_PLN_UNROLL
#define SC_PLN_UNROLL 2          // positions per iteration of the planar instances' main loop (2 or 4; 4 measured slower)
#endif
__host__ __device__ constexpr int sym_nprod(int NC) { return (NC == 192 && SC_L192 == 1) ? 64 : 128; }
// SC_L192 == 0 (A/B layout): warps 0-5 = consumers, 6-7 = idle (they exit after the register hand-over of their
// warpgroup: setmaxnreg works on whole warpgroups), 8-11 = producers.
__host__ __device__ constexpr int sym_prod0(int NC) { return (NC == 192 && SC_L192 == 0) ? 256 : NC; }     // first producer thread
__host__ __device__ constexpr int sym_threads(int NC) { return sym_prod0(NC) + sym_nprod(NC); }
__host__ __device__ constexpr int sym_planes(bool south, bool mirror) { return (south ? 2 : 1) * (mirror ? 2 : 1); }
__host__ __device__ constexpr int sym_tmem_cols(int NC, int per_thread) {
    int need = ((NC / 32 + 3) / 4) * per_thread, c = 32;
    while (c < need) c *= 2;
    return c;
}

// Per-position state of the pair loop: lookup coordinate - 1/2 and table cell bits of the R pixels (geometry stage),
// table cells and map values (load stage)
// (tp, cb: coordinate - 1/2 and cell bits before the two-zone / fp64 / clamping steps, for the exact path)
template <int R> struct SymGeo { float t[2 * ((R + 1) / 2)]; unsigned c[2 * ((R + 1) / 2)]; float tp[2 * ((R + 1) / 2)]; unsigned cb[2 * ((R + 1) / 2)]; };
template <int R, int B, int NPL> struct SymLd { float2 el[R]; float4 mv[B][NPL]; };

// Tile n of this CTA: rows of gridDim.x tiles, alternate rows reversed ("snake") so that the CTAs
// get equal shares of the work-sorted tile list without a global counter.
__device__ __forceinline__ int snake_tile(int row, int G, int bid) { return row * G + ((row & 1) ? G - 1 - bid : bid); }

// 4 bytes at shared address a + IMM (IMM: compile-time plane offset, folded into the instruction)
template <int IMM> __device__ __forceinline__ float lds32(unsigned a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(IMM));
    return v;
}

// Planar staging (template flag PLN; R = 3, one map): every image has a plane of its own (4 NPL planes of kLp floats per
// stage buffer), filled by TMA bulk copies of 16-byte-aligned pieces of the input rings -- the run of an image starts 0-3
// floats into its plane (its alignment in the ring; ring starts and lengths are multiples of 4 pixels), the reflected
// images are staged in ring order and read backwards.  The consumers read one float per image and position (LDS.32:
// lanes 3 positions apart hit 32 different banks) instead of one float4 per plane of 4 interleaved rotation images.
constexpr int kLp = kPlanarPlane;          // floats per plane: 2 buffers x 16 planes x 784 x 4 B = 98 KB next to the 128 KB table

__device__ __forceinline__ float4 lds128(unsigned a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}

// Warp-specialised: the first NC threads are consumers (pair loop), the last sym_nprod(NC) threads are producers
// (staging).  They meet only through the full/empty mbarriers of the kSymBuf stage buffers; there is no block-wide
// barrier after the prologue.
// TOT: per-step partial sums are added to a second accumulator set (pairwise-like summation; needed for
// discs of thousands of pixels, costs as many registers again).
// Z: two-zone table (lookup at tau(t), R11).  TM: the second accumulator set lives in tensor memory.
// HP: table coordinate in fp64 (Dev::hp, steep tables), split into cell + position in the cell; cell-local table.
template <int B, int R, int NC, bool TOT, bool Z, bool TM, bool SOUTH, bool MIRROR, bool HP = false, bool PLN = false>
__global__ void __launch_bounds__(sym_threads(NC), 1)
sym_kernel(const Dev P, const FastDev F, const Maps io) {
    static_assert(!(HP && Z), "the fp64 coordinate is not combined with the two-zone table");
    static_assert(!PLN || (B == 1 && (R == 3 || R == 1)), "planar staging: one map, lanes 3 positions (or 1) apart");
    static_assert(R >= 1 && R <= 4, "R");
    constexpr int RP = (R + 1) / 2;                      // pixel pairs per thread
    constexpr int NPROD = sym_nprod(NC), PROD0 = sym_prod0(NC);
    constexpr int NPL = sym_planes(SOUTH, MIRROR);       // staged planes per position, 4 rotation images each
    constexpr int G = 2 * NPL;                           // float2 accumulators per base pixel and map
    constexpr int TMC = sym_tmem_cols(NC, R * G * 2);
    constexpr int NPD = SOUTH ? 2 : 1;                   // planes of direct images (the others: reflected)
    constexpr bool SKEW = SC_SKEW_ALL || PLN || B > 1;                  // lane skew (see the consumers): runs staged PairEnt.ex positions further on both sides
    constexpr int NTASK = PLN ? 4 * NPL * kMaxSub : 0;   // planar staging: bulk-copy tasks (sub-tile, image) = producer threads that arrive
    static_assert(NTASK <= NPROD, "one producer thread per (sub-tile, image)");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);
    const unsigned stage_sh = smem_u32(smem_raw + (((size_t)F.ntab_s * 8 + 127) & ~(size_t)127));
    __shared__ unsigned long long full_bar[kSymBuf], empty_bar[kSymBuf];
    __shared__ int s_tile[4];                            // tiles taken by this CTA (ring): written by producer 0, -1 = no more
    __shared__ int4 s_run[2][kMaxSub][2];                // producers: the runs of a step {kq0, km0, L, nq}, {start_n, start_s, soff, -}
    const int tid = threadIdx.x;
    const int N = P.nside;
    const int Ltot = F.Ltot;

    // a kernel launched behind this one with programmatic stream serialization (the warp-per-pixel kernel: disjoint outputs,
    // no wait on this grid) may take the SMs as this kernel's CTAs leave them
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // the table: one bulk copy (the consumers wait for it before their first tile), an odd last cell by hand -- in the
    // small-disc instances, whose launches are short enough for the prologue to count (config 3: -1.7 %, config 4: -0.9 %);
    // the large-disc instances keep the load loop (with the bulk copy their pair loop came out 1.5 % slower, config 5)
    constexpr bool BULK = !TOT;
    __shared__ unsigned long long tab_bar;
    if (!BULK)
        for (int i = tid; i < F.ntab_s; i += blockDim.x) tab[i] = P.tabh[i];
    if (tid == 0) {
        for (int i = 0; i < kSymBuf; ++i) { mbar_init(&full_bar[i], PLN ? NTASK : NPROD); mbar_init(&empty_bar[i], NC / 32); }
        if (BULK) mbar_init(&tab_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (BULK) {
            const unsigned bytes = ((unsigned)F.ntab_s * 8u) & ~15u;
            mbar_expect_tx(&tab_bar, bytes);
            if (bytes) tma_load_1d(tab, P.tabh, bytes, &tab_bar);
        }
    }
    if (BULK && tid == 32 && (F.ntab_s & 1)) tab[F.ntab_s - 1] = P.tabh[F.ntab_s - 1];
    __shared__ unsigned s_tmem;
    if (TM && tid < 32) {                                  // warp w uses TMEM lanes 32 (w % 4) .., columns (R G 2) (w / 4) ..
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TMC) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (TM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    unsigned it = 0;                                     // steps so far: buffer it % kSymBuf, use it / kSymBuf
    int rem_unused;

    // register budget: the launch gives every thread 65536 / blockDim.x registers (rounded down to a
    // multiple of 8); the producer warpgroup hands most of its share to the consumer warpgroups
    if (tid >= PROD0) {
        // ======================================= producers =======================================
        if (NC == 256 || NC == 384 || (NC == 192 && SC_L192 == 0)) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const int pt = tid - PROD0;
        const int m = pt & 3;                            // quadrant image staged by this thread
        // the run of sub-tile s at a step: first staged input pixel (rotation 0) and its reflected image, length, ring starts
        auto run_of = [&](const SymTile *tl, int step, int s, int par) {
            int4 ra = make_int4(0, 0, 0, 4), rb = make_int4(0, 0, 0, 0);
            if (s < __ldg(&tl->nsub) && step < __ldg(&tl->sub[s].ne)) {
                const int r = __ldg(&tl->sub[s].r), k0 = __ldg(&tl->sub[s].k0), n = __ldg(&tl->sub[s].n);
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
                const int ex = SKEW ? __ldg(&pe->ex) : 0;     // extra positions on both sides (lane skew of the consumers)
                const int w0 = div_fast(a0s * ipq + shq * ips, 2 * ips, M0s, rem_unused) - hw - ex;
                const int L = div_fast(als * ipq + shq * ips, 2 * ips, M0s, rem_unused) + hw + R + ex - w0;
                int k = w0 + nq;                          // in [0, 2 nq): w0 >= -hw - 1 > -nq
                if (k >= nq) k -= nq;
                // mirror image of position i: pixel ipq - 1 + shq - (w0 + i), walking backwards
                int km = (ipq - 1 + shq - w0) % nq;
                if (km < 0) km += nq;
                ra = make_int4(k, km, L, nq);
                rb = make_int4(ps.x, ps.y, __ldg(&tl->sub[s].soff), 0);
            }
            s_run[par][s][0] = ra; s_run[par][s][1] = rb;
        };
        // Dynamic schedule: the tile list is sorted by decreasing work and a CTA takes the next tile when it is done with
        // its last one (one atomicAdd per tile by producer 0, handed to the other threads through s_tile).
        for (int n = 0;; ++n) {
            if (pt == 0) { const int t = atomicAdd(F.tile_ctr, 1); s_tile[n & 3] = t < F.ntiles ? t : -1; }
            asm volatile("bar.sync 1, %0;" ::"n"(NPROD) : "memory");
            const int tile = *(volatile int *)&s_tile[n & 3];
            if (tile < 0) {                              // no more tiles: wake the consumers with one empty step
                mbar_wait_sleep(&empty_bar[it % kSymBuf], ((it / kSymBuf) & 1u) ^ 1u);
                if (!PLN) cp_async_mbar_arrive(&full_bar[it % kSymBuf]);
                else if (pt < NTASK) mbar_arrive(&full_bar[it % kSymBuf]);
                break;
            }
            const SymTile *tl = F.tiles + tile;
            const int nsteps = __ldg(&tl->nsteps);
            if (pt < kMaxSub) run_of(tl, 0, pt, it & 1);    // (the tile's first step: its runs are not known earlier)
            for (int step = 0; step < nsteps; ++step, ++it) {
                const int buf = it % kSymBuf;
                asm volatile("bar.sync 1, %0;" ::"n"(NPROD) : "memory");        // this step's runs are in s_run[it & 1]
                if constexpr (PLN) {
                    // one producer thread per (sub-tile, image): the image's run as one or two (wrap) 16-byte-aligned bulk copies
                    mbar_wait_sleep(&empty_bar[buf], ((it / kSymBuf) & 1u) ^ 1u);   // every consumer warp released it
                    if (pt < NTASK) {
                        const int s = pt / (4 * NPL), img = pt % (4 * NPL), pl = img >> 2, mr = img & 3;
                        const int4 ra = s_run[it & 1][s][0], rb = s_run[it & 1][s][1];
                        const int L = ra.z, nq = ra.w;
                        unsigned long long *bar = &full_bar[buf];
                        if (L > 0 && !(F.dbg & 2)) {
                            int first = (pl < NPD ? ra.x : ra.y - (L - 1)) + mr * (nq >> 2);   // first pixel in ring order
                            first %= nq; if (first < 0) first += nq;
                            const int a = first & ~3, n4 = ((first & 3) + L + 3) & ~3;            // aligned piece: pixels a .. a + n4
                            const bool sth = SOUTH && ((pl < NPD ? pl : pl - NPD) & 1);
                            const float *ring = io.in[0] + (sth ? rb.y : rb.x);
                            float *dst = reinterpret_cast<float *>(smem_raw + (((size_t)F.ntab_s * 8 + 127) & ~(size_t)127)) +
                                         (size_t)(buf * 4 * NPL + img) * kLp + rb.z;
                            const int n1 = min(n4, nq - a);
                            mbar_expect_tx(bar, (unsigned)n4 * 4u);
                            tma_load_1d(dst, ring + a, (unsigned)n1 * 4u, bar);
                            if (n1 < n4) tma_load_1d(dst + n1, ring, (unsigned)(n4 - n1) * 4u, bar);
                        } else {
                            mbar_arrive(bar);
                        }
                    }
                    if (pt < kMaxSub && step + 1 < nsteps) run_of(tl, step + 1, pt, (it + 1) & 1);
                    continue;
                }
                // The runs to stage for this step (one per sub-tile) were worked out by producer threads 0 .. kMaxSub - 1 during
                // the PREVIOUS step (run_of below) and handed over through s_run: nobody walks the dependent loads
                // tile -> ring pair in every thread, and they are off the critical path.
                int kq0[kMaxSub], km0[kMaxSub], Ls[kMaxSub], nqs[kMaxSub], sn[kMaxSub], ss[kMaxSub];
                unsigned d0[kMaxSub];
#pragma unroll
                for (int s = 0; s < kMaxSub; ++s) {
                    const int4 ra = s_run[it & 1][s][0], rb = s_run[it & 1][s][1];
                    Ls[s] = ra.z; nqs[s] = ra.w; sn[s] = rb.x; ss[s] = rb.y;
                    int k = ra.x + m * (ra.w >> 2);           // rotation m of the first staged pixel
                    if (k >= ra.w) k -= ra.w;
                    kq0[s] = k;
                    int km = ra.y + m * (ra.w >> 2);
                    if (km >= ra.w) km -= ra.w;
                    km0[s] = km;
                    d0[s] = stage_sh + (unsigned)((buf * B * NPL) * Ltot + rb.z) * 16u + 4u * m;
                }
                mbar_wait_sleep(&empty_bar[buf], ((it / kSymBuf) & 1u) ^ 1u);   // every consumer warp released it
#pragma unroll
                for (int s = 0; s < kMaxSub; ++s) {
                    if (F.dbg & 2) break;
                    // this thread's positions i = pt / 4 + j NPROD / 4: input pixel kq walks forwards, its mirror
                    // image km backwards, both with at most one wrap (L < nq); unsigned 32-bit indices added to
                    // the ring's base pointer keep the address arithmetic to one instruction per copy
                    const unsigned nq = (unsigned)nqs[s];
                    int i = pt >> 2;
                    unsigned kq = (unsigned)(kq0[s] + i); if (kq >= nq) kq -= nq;
                    int km = km0[s] - i; if (km < 0) km += (int)nq;
                    const unsigned plane = (unsigned)Ltot * 16u;
                    const float *gn[B], *gs[B];              // first pixel of the input ring and of its southern mirror
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        gn[b] = io.in[b] + sn[s]; gs[b] = io.in[b] + ss[s];
                        asm volatile("" : "+l"(gn[b]), "+l"(gs[b]));     // kept as 64-bit registers
                    }
                    // positions 32 apart share the swizzle term of slot_of_pos: the destinations advance by 512 bytes per
                    // iteration; a thread takes PPI positions (NPROD / 4 apart) per iteration
                    constexpr int PPI = 32 / (NPROD / 4);
                    static_assert(PPI == 1 || PPI == 2, "positions per producer iteration");
                    unsigned d = d0[s] + 16u * (unsigned)slot_of_pos<R>(i);
                    const unsigned d2off = 16u * (unsigned)slot_of_pos<R>(i + NPROD / 4) - 16u * (unsigned)slot_of_pos<R>(i);
                    const int L = Ls[s];
#pragma unroll 2
                    for (; i < L; i += 32, d += 512u) {
#pragma unroll
                        for (int u = 0; u < PPI; ++u) {
                            if (u == 1 && i + NPROD / 4 >= L) break;
#pragma unroll
                            for (int b = 0; b < B; ++b) {
                                unsigned dd = d + (u ? d2off : 0u) + (unsigned)(b * NPL) * plane;
                                cp_async4_s(dd, elem_ptr(gn[b], kq));
                                if (SOUTH) { dd += plane; cp_async4_s(dd, elem_ptr(gs[b], kq)); }
                                if (MIRROR) {
                                    dd += plane; cp_async4_s(dd, elem_ptr(gn[b], (unsigned)km));
                                    if (SOUTH) { dd += plane; cp_async4_s(dd, elem_ptr(gs[b], (unsigned)km)); }
                                }
                            }
                            kq += NPROD / 4; if (kq >= nq) kq -= nq;
                            km -= NPROD / 4; if (km < 0) km += (int)nq;
                        }
                    }
                }
                cp_async_mbar_arrive(&full_bar[buf]);   // arrives when this thread's copies have landed
                // ... and the runs of the next step, while the copies are in flight (of this tile: the first step of the next
                // tile is done at its start)
                if (pt < kMaxSub && step + 1 < nsteps) run_of(tl, step + 1, pt, (it + 1) & 1);
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        return;
    }

    // ========================================= consumers =========================================
    if (NC == 256) asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    if (NC == 384) asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
    if (NC == 192 && SC_L192 == 0) {                       // 384 threads x 168 registers = 256 x 224 + 128 x 56
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        if (tid >= NC) return;                             // warps 6-7 only complete the warpgroup
    }
    if (BULK) mbar_wait(&tab_bar, 0);                      // the table is in shared memory
    const int warp = tid >> 5, lane = tid & 31;
    const unsigned taddr = TM ? s_tmem + ((((unsigned)warp & 3u) * 32u) << 16) + ((unsigned)warp >> 2) * (unsigned)(R * G * 2) : 0u;
    const unsigned thresh = kMagicBits + (unsigned)(P.ntab - 2);   // bits of the last table cell
    const float tmax = P.tmax, eps = P.eps;
    // shared-memory byte address of tab[0] minus 8 kMagicBits (mod 2^32): tab[bits - kMagicBits] = [tab_sh + 8 bits]
    // (kept opaque: otherwise the compiler re-derives it from the CTA's shared window inside the pair loop)
    unsigned tab_sh = smem_u32(tab) - kMagicBits * 8u;
    asm volatile("mov.u32 %0, %0;" : "+r"(tab_sh));

    for (int n = 0;; ++n) {
        // the tile's number is valid once the producers have filled (arrived on) the buffer of its first step
        mbar_wait(&full_bar[it % kSymBuf], (it / kSymBuf) & 1u);
        const int tile = *(volatile int *)&s_tile[n & 3];
        if (tile < 0) break;
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

        float2 tot[TOT && !TM ? R : 1][B][G];
#pragma unroll
        for (int rr = 0; rr < (TOT && !TM ? R : 1); ++rr)
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int g = 0; g < G; ++g) tot[rr][b][g] = f2(0.f);
        float2 acc[R][B][G];
#pragma unroll
        for (int rr = 0; rr < R; ++rr)
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int g = 0; g < G; ++g) acc[rr][b][g] = f2(0.f);

        bool flushed = false;                              // TM: the totals in tensor memory are valid
        PairEnt pe_next = F.pairs[me.e0];
        for (int step = 0; step < nsteps; ++step, ++it) {
            const int buf = it % kSymBuf;
            const PairEnt pe = pe_next;
            if (step + 1 < me.ne) pe_next = F.pairs[me.e0 + step + 1];       // prefetch under the pair loop
            mbar_wait(&full_bar[buf], (it / kSymBuf) & 1u);
            if (active && step < me.ne && !(F.dbg & 1)) {
                const int ex = SKEW ? pe.ex : 0;
                const int w0 = div_fast(ap0 * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) - pe.hw - ex;
                int rem;
                const int kc = div_fast(ap * pe.ipq + pe.shq * ip, ip2, M0, rem);
                // azimuth of input pixel kc + j seen from base pixel ka + rr:  d = dcr[rr] + j dphi'
                float dcr[R];
#pragma unroll
                for (int rr = 0; rr < R; ++rr) dcr[rr] = (float)(ip - rem - 2 * rr * pe.ipq) * pe.cdc;
                // fp64 coordinate (HP): the same ring pair in double
                PairEntD pd{};
                double dcr64[HP ? R : 1], jd = -(double)pe.hw;
                if (HP) {
                    pd = F.pairsd[me.e0 + step];
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) dcr64[rr] = (double)(ip - rem - 2 * rr * pe.ipq) * pd.cdc;
                }
                // staged position of input pixel kc + j: i0 + j (slot_of_pos: padded against bank conflicts)
                const int i0 = kc - w0;
                unsigned pn[B];                          // shared address of this sub-tile's first plane, map b
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    pn[b] = stage_sh + (unsigned)(((buf * B + b) * NPL) * Ltot + me.soff) * 16u;
                    asm volatile("mov.u32 %0, %0;" : "+r"(pn[b]));      // one register, not re-derived per position
                }
                const unsigned plane = (unsigned)Ltot * 16u;
                // planar staging: shared address of position 0 of the 4 direct rotation images (north plane; position i at
                // +4 i) and of the 4 reflected ones (position i at -4 i); the southern planes lie 4 kLp floats further
                unsigned ad[PLN ? 4 : 1], am[PLN ? 4 : 1];
                if constexpr (PLN) {
                    const int Lrun = div_fast((2 * klast + 1 - sh) * pe.ipq + pe.shq * ip, ip2, M0, rem_unused) + pe.hw + R + ex - w0;
                    const unsigned b0 = stage_sh + (unsigned)(buf * 4 * NPL * kLp + me.soff) * 4u;
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const int fd = w0 + m * pe.ipq;                                   // first staged pixel (mod 4 = mod-nq value mod 4)
                        const int fm = pe.ipq - 1 + pe.shq - w0 + m * pe.ipq - (Lrun - 1);   // reflected run: first pixel in ring order
                        ad[m] = b0 + (unsigned)(m * kLp + (fd & 3)) * 4u;
                        am[m] = b0 + (unsigned)((4 * NPD + m) * kLp + (fm & 3) + Lrun - 1) * 4u;
                    }
                }
                // the 4 rotation images of plane pl at staged position pos (planar: ad / am point at position pos - U, with
                // U a compile-time constant: the unrolled main loop advances the 8 addresses once per kUn positions)
                auto ldmap = [&](int b, auto PLc, int pos, auto Uc) -> float4 {
                    constexpr int pl = decltype(PLc)::value;
                    if constexpr (PLN) {
                        constexpr int U = decltype(Uc)::value;
                        constexpr int off = (pl < NPD ? pl : pl - NPD) * 4 * kLp * 4;
                        if constexpr (pl < NPD)
                            return make_float4(lds32<off + 4 * U>(ad[0]), lds32<off + 4 * U>(ad[1]), lds32<off + 4 * U>(ad[2]), lds32<off + 4 * U>(ad[3]));
                        else
                            return make_float4(lds32<off - 4 * U>(am[0]), lds32<off - 4 * U>(am[1]), lds32<off - 4 * U>(am[2]), lds32<off - 4 * U>(am[3]));
                    } else {
                        return lds128(pn[b] + 16u * (unsigned)slot_of_pos<R>(pos) + pl * plane);
                    }
                };

                // last table cell or the zero cell after it (rare): exact decision where needed
                auto slow = [&](int rr, float tpv, unsigned &cb, int pos, auto Uc) {
                    const float t = tpv + 0.5f;
                    if (t >= tmax - eps) {
                        if (t <= tmax + eps) {                   // decide in fp64, image by image
                            const unsigned mask = sym_exact_mask(P, r, ka + rr, ip, sh, pe.rq, kc + pos - i0, pe.ipq, pe.shq, t,
                                                                 SOUTH ? 1 : 0, MIRROR ? 1 : 0);
                            if (mask) {
                                const float2 el = tab[P.ntab - 2];
                                float xk = fminf(t, tmax) - 0.5f;
                                if (Z) { int jz; zoned_cell(P, fminf(t, tmax), jz, xk); xk -= 0.5f; }   // last cell, centred form
                                if (HP) xk = fminf(t, tmax) - (float)(P.ntab - 2) - 0.5f;               // cell-local table
                                const float Ku = fmaf(xk, el.y, el.x);
#pragma unroll
                                for (int b = 0; b < B; ++b) {
                                    auto one = [&](auto PLc) {
                                        constexpr int pl = decltype(PLc)::value;
                                        if constexpr (pl < NPL) {
                                            const float4 mq = ldmap(b, PLc, pos, Uc);
                                            const unsigned mk = mask >> (4 * pl);
                                            if (mk & 1u) acc[rr][b][2 * pl].x = fmaf(Ku, mq.x, acc[rr][b][2 * pl].x);
                                            if (mk & 2u) acc[rr][b][2 * pl].y = fmaf(Ku, mq.y, acc[rr][b][2 * pl].y);
                                            if (mk & 4u) acc[rr][b][2 * pl + 1].x = fmaf(Ku, mq.z, acc[rr][b][2 * pl + 1].x);
                                            if (mk & 8u) acc[rr][b][2 * pl + 1].y = fmaf(Ku, mq.w, acc[rr][b][2 * pl + 1].y);
                                        }
                                    };
                                    one(std::integral_constant<int, 0>{}); one(std::integral_constant<int, 1>{});
                                    one(std::integral_constant<int, 2>{}); one(std::integral_constant<int, 3>{});
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
                for (int h = 0; h < RP; ++h) dc2[h] = f2(dcr[2 * h], dcr[2 * h + 1 < R ? 2 * h + 1 : 2 * h]);
                // Lane skew (planar and batch instances): on an input ring with another pixel count the lanes' positions, R apart
                // on the base ring, drift apart by up to ex and their loads would collide in the banks.  A lane whose position is
                // `skew` ahead of the grid (first valid lane's position + R per lane, shifted to the smallest) starts its walk
                // `skew` positions early and all lanes walk 2 hw + R + wd positions (wd = the largest skew of the warp): at
                // every step the valid lanes are exactly R positions apart.  The extra positions lie outside the disc (weight
                // 0) and inside the staged run (extended by ex on both sides).
                int skew = 0, wd = 0;
                if (SKEW && ex > 0) {
                    const bool valid = kmine <= klast;
                    const int q = i0 - R * lane;
                    const int mn = __reduce_min_sync(0xFFFFFFFFu, valid ? q : 0x7FFFFFFF);
                    const int mx = __reduce_max_sync(0xFFFFFFFFu, valid ? q : (int)0x80000000);
                    if (mx - mn <= ex) {                          // (always, by the choice of ex; else: no skew, the run is not that long)
                        skew = valid ? q - mn : 0;
                        wd = mx - mn;
                    }
                }
                if (HP) jd = -(double)(pe.hw + skew);
                float2 jf = f2((float)(-pe.hw - skew));
                const int pos0 = i0 - pe.hw - skew, pend = i0 + pe.hw + R - 1 + wd - skew;
                // One window position for the pixels rr in MASK (compile time).  The window of the thread is the
                // union of its R pixels' windows, which are one position apart: pixel rr can only be inside the
                // disc at positions pos0 + rr .. pend - (R - 1 - rr) (host: hw = floor(H / dphi' + 1/2 + 3 rho1),
                // |dcr0| <= dphi' / 2, pixel rr is centred rr (1 +- rho1) positions further), so the first and the
                // last R - 1 positions run bodies without the other pixels' geometry, gather and FMAs.
                // The work of one position in three stages, so that the main loop can be software-pipelined (with only
                // 6-12 consumer warps per SM the shared-memory latency must be covered inside the warp):
                //   geom: pair geometry -> lookup coordinate - 1/2 (gt) and table cell bits (gc) of the R pixels,
                //         exact fp64 decisions for the rare cells next to theta_max (slow);
                //   load: the table cells (one LDS.64 gather per pixel) and the map values of this position;
                //   fma:  K = a + t b and the accumulation into the images.
                // (geomA: the arithmetic, returns the distance of the nearest cell to the last table cell -- < 2 means some pixel
                // needs geomS, the exact decisions; two positions can run geomA back to back before one shared branch)
                auto geomA = [&](auto MASK, SymGeo<R> &ge) -> unsigned {
                    float *gt = ge.t;
                    unsigned *gc = ge.c;
                    constexpr int mask = decltype(MASK)::value;
                    float *tp = ge.tp;
                    unsigned *cb = ge.cb;
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
                        gt[2 * h] = t2.x; gt[2 * h + 1] = t2.y;
                        gc[2 * h] = cb[2 * h]; gc[2 * h + 1] = cb[2 * h + 1];
                        if (Z) {
                            // inner zone: alpha t - 1/2; outer zone: gamma (t - t1) - 1/2 RELATIVE to the zone start
                            // (full resolution where the kernel is steep), cell offset added to the integer bits
                            const float2 l1 = __ffma2_rn(t2, za2, zao2), l2 = __ffma2_rn(t2, zg2, zgo2);
                            const bool o0 = l2.x + zhm1f < l1.x, o1 = l2.y + zhm1f < l1.y;
                            const float2 tz = f2(o0 ? l2.x : l1.x, o1 ? l2.y : l1.y);
                            const float2 bz = __fadd2_rn(tz, f2(kMagic));
                            const float2 fz = __fadd2_rn(tz, __fadd2_rn(f2(kMagic), f2(-bz.x, -bz.y)));   // position - 1/2 in the cell
                            gt[2 * h] = fz.x; gt[2 * h + 1] = fz.y;
                            gc[2 * h] = __float_as_uint(bz.x) + (o0 ? zhm1 : 0u); gc[2 * h + 1] = __float_as_uint(bz.y) + (o1 ? zhm1 : 0u);
                        }
                    }
                    if (HP) {
                        // the coordinate again in fp64: cell and position in the cell from it (the fp32 value above only
                        // serves the guard-band logic, whose band is far wider than its error)
#pragma unroll
                        for (int rr = 0; rr < R; ++rr) {
                            if (!((mask >> rr) & 1)) continue;
                            const double t64 = fma(pd.Bs, one_minus_cos_poly_f64(fma(jd, pd.dphi, dcr64[rr])), pd.A);
                            const int cell = min(__double2int_rd(t64), 0x3FFFFF);
                            gt[rr] = (float)(t64 - (double)cell) - 0.5f;
                            gc[rr] = kMagicBits + (unsigned)cell;
                            cb[rr] = gc[rr];
                        }
                        jd += 1.0;
                    }
                    // cells below the last: plain lookup; beyond the zero cell: clamp onto it (weight 0);
                    // the last cell and the zero cell (t in [tmax - 1, tmax + 1)) take the branch
                    unsigned mn = 0xFFFFFFFFu;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) if ((mask >> rr) & 1) mn = min(mn, cb[rr] - thresh);
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) if ((mask >> rr) & 1) gc[rr] = min(gc[rr], thresh + 1u);
                    jf = __fadd2_rn(jf, f2(1.0f));
                    return mn;
                };
                auto geomS = [&](int pos, auto MASK, SymGeo<R> &ge, auto Uc) {
                    constexpr int mask = decltype(MASK)::value;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr)
                        if (((mask >> rr) & 1) && ge.cb[rr] >= thresh) slow(rr, ge.tp[rr], ge.c[rr], pos, Uc);
                };
                auto geom = [&](int pos, auto MASK, SymGeo<R> &ge, auto Uc) {
                    if (geomA(MASK, ge) < 2u) geomS(pos, MASK, ge, Uc);
                };
                auto load = [&](int pos, auto MASK, const SymGeo<R> &ge, SymLd<R, B, NPL> &ld, auto Uc) {
                    const unsigned *gc = ge.c;
                    float2 *el = ld.el;
                    float4 (*mv)[NPL] = ld.mv;
                    constexpr int mask = decltype(MASK)::value;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) {
                        if (!((mask >> rr) & 1)) continue;          // tab[gc - kMagicBits], one LEA for the address
                        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(el[rr].x), "=f"(el[rr].y) : "r"(tab_sh + gc[rr] * 8u));
                    }
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        mv[b][0] = ldmap(b, std::integral_constant<int, 0>{}, pos, Uc);
                        if constexpr (NPL > 1) mv[b][1] = ldmap(b, std::integral_constant<int, 1>{}, pos, Uc);
                        if constexpr (NPL > 2) {
                            mv[b][2] = ldmap(b, std::integral_constant<int, 2>{}, pos, Uc);
                            mv[b][3] = ldmap(b, std::integral_constant<int, 3>{}, pos, Uc);
                        }
                    }
                };
                auto fma = [&](auto MASK, const SymGeo<R> &ge, const SymLd<R, B, NPL> &ld) {
                    const float *gt = ge.t;
                    const float2 *el = ld.el;
                    const float4 (*mv)[NPL] = ld.mv;
                    constexpr int mask = decltype(MASK)::value;
#pragma unroll
                    for (int rr = 0; rr < R; ++rr) {
                        if (!((mask >> rr) & 1)) continue;
                        const float2 Kd = f2(fmaf(gt[rr], el[rr].y, el[rr].x));
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int pl = 0; pl < NPL; ++pl) {
                                acc[rr][b][2 * pl] = __ffma2_rn(Kd, f2(mv[b][pl].x, mv[b][pl].y), acc[rr][b][2 * pl]);
                                acc[rr][b][2 * pl + 1] = __ffma2_rn(Kd, f2(mv[b][pl].z, mv[b][pl].w), acc[rr][b][2 * pl + 1]);
                            }
                    }
                };
                SymGeo<R> geA, geB;
                SymLd<R, B, NPL> ldA, ldB;
                const auto U0 = std::integral_constant<int, 0>{};
                auto bodyu = [&](int pos, auto MASK, auto Uc) {   // one position, not pipelined
                    geom(pos, MASK, geA, Uc);
                    load(pos, MASK, geA, ldA, Uc);
                    fma(MASK, geA, ldA);
                };
                auto adv = [&](int n) {                           // planar: the image addresses move on by n positions
                    if constexpr (PLN) {
#pragma unroll
                        for (int m = 0; m < 4; ++m) { ad[m] += 4u * (unsigned)n; am[m] -= 4u * (unsigned)n; }
                    }
                };
                auto body = [&](int pos, auto MASK) {             // (window edges)
                    bodyu(pos, MASK, U0);
                    adv(1);
                };
                constexpr int kAll = (1 << R) - 1;
                const auto ALL = std::integral_constant<int, kAll>{};
                int pos = pos0, plast = pend;
                if constexpr (PLN) {                              // ad / am: position pos0 from here on
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        ad[m] += 4u * (unsigned)pos0; am[m] -= 4u * (unsigned)pos0;
                        asm volatile("mov.u32 %0, %0;" : "+r"(ad[m]));      // registers, not re-derived per position
                        asm volatile("mov.u32 %0, %0;" : "+r"(am[m]));
                    }
                }
                const bool peel = R > 1 && 2 * pe.hw >= R - 2;       // first and last R - 1 positions do not overlap
                if (peel) {
                    body(pos++, std::integral_constant<int, 1>{});
                    if (R >= 3) body(pos++, std::integral_constant<int, 3>{});
                    if (R == 4) body(pos++, std::integral_constant<int, 7>{});
                    plast = pend - (R - 1);
                }
                // Main positions (all R pixels), software-pipelined over two register sets: the loads of position
                // i + 1 are issued before the FMAs of position i, the geometry of position i + 2 after them.  The
                // number of positions is the same for all lanes (2 hw + R - 2 (R - 1) or 2 hw + R).
                int left = plast - pos + 1;
                constexpr bool PIPE = NC == 192 || (R == 3 && SC_R3_PIPE);                     // only the 6-warp instance needs it (elsewhere: spills, slower)
                if (PLN) {
                    constexpr int kUn = SC_PLN_UNROLL;
                    const std::integral_constant<int, 1> U1{};
#pragma unroll 1
                    for (; pos + kUn - 1 <= plast; pos += kUn) {
                        if constexpr (SC_PLN_BATCH && kUn == 2) {
                            // two positions as one straight-line block: both geometries, one branch for the rare exact
                            // decisions, both sets of loads, both accumulations (the compiler cannot move position n + 1's
                            // geometry across position n's branch by itself)
                            const unsigned mA = geomA(ALL, geA), mB = geomA(ALL, geB);
                            if (min(mA, mB) < 2u) {
                                if (mA < 2u) geomS(pos, ALL, geA, U0);
                                if (mB < 2u) geomS(pos + 1, ALL, geB, U1);
                            }
                            load(pos, ALL, geA, ldA, U0);
                            load(pos + 1, ALL, geB, ldB, U1);
                            fma(ALL, geA, ldA);
                            fma(ALL, geB, ldB);
                        } else {
                            bodyu(pos, ALL, U0);
                            bodyu(pos + 1, ALL, U1);
                            if constexpr (kUn == 4) {
                                bodyu(pos + 2, ALL, std::integral_constant<int, 2>{});
                                bodyu(pos + 3, ALL, std::integral_constant<int, 3>{});
                            }
                        }
                        adv(kUn);
                    }
#pragma unroll 1
                    for (; pos <= plast; ++pos) body(pos, ALL);
                } else if (!PIPE && SC_SYM_BATCH && B > 1) {   // the same two-position blocks in the batch instances (config 5: sym 25.0 -> 23.8 ms; one map, tensor-memory totals: 1-2 % slower, left as it was)
#pragma unroll 1
                    for (; pos + 1 <= plast; pos += 2) {
                        const unsigned mA = geomA(ALL, geA), mB = geomA(ALL, geB);
                        if (min(mA, mB) < 2u) {
                            if (mA < 2u) geomS(pos, ALL, geA, U0);
                            if (mB < 2u) geomS(pos + 1, ALL, geB, U0);
                        }
                        load(pos, ALL, geA, ldA, U0);
                        load(pos + 1, ALL, geB, ldB, U0);
                        fma(ALL, geA, ldA);
                        fma(ALL, geB, ldB);
                    }
                    if (pos <= plast) body(pos++, ALL);
                } else if (!PIPE) {
#pragma unroll 2
                    for (; pos <= plast; ++pos) body(pos, ALL);
                } else if (left > 0) {
                    geom(pos, ALL, geA, U0);
                    load(pos, ALL, geA, ldA, U0);
                    if (left > 1) geom(pos + 1, ALL, geB, U0);
                    while (true) {
                        if (left > 1) load(pos + 1, ALL, geB, ldB, U0);
                        fma(ALL, geA, ldA);
                        if (left > 2) geom(pos + 2, ALL, geA, U0);
                        ++pos;
                        if (--left == 0) break;
                        if (left > 1) load(pos + 1, ALL, geA, ldA, U0);
                        fma(ALL, geB, ldB);
                        if (left > 2) geom(pos + 2, ALL, geB, U0);
                        ++pos;
                        if (--left == 0) break;
                    }
                }
                if (peel) {
                    if (R == 4) body(pos++, std::integral_constant<int, 14 & kAll>{});
                    if (R >= 3) body(pos++, std::integral_constant<int, (3 << (R >= 2 ? R - 2 : 0)) & kAll>{});
                    body(pos++, std::integral_constant<int, (1 << (R - 1))>{});
                }
                if (TOT && TM) {                                 // totals (tensor memory) += this ring's sums
                    static_assert(!TM || B == 1, "TM variant: one map");
                    static_assert(!TM || (R * G) % 8 == 0, "TM variant: 16 columns at a time");
#pragma unroll
                    for (int hh = 0; hh < R * G / 8; ++hh) {
                        float v[16], old[16];
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            float2 &a = acc[(hh * 8 + j) / G][0][(hh * 8 + j) % G];
                            v[2 * j] = a.x; v[2 * j + 1] = a.y;
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
                            for (int g = 0; g < G; ++g) {
                                tot[TM ? 0 : rr][b][g] = __fadd2_rn(tot[TM ? 0 : rr][b][g], acc[rr][b][g]);
                                acc[rr][b][g] = f2(0.f);
                            }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[buf]);         // this warp is done with the buffer
        }

        if (TM && flushed) {                               // totals back from tensor memory (into the accumulator registers)
#pragma unroll
            for (int hh = 0; hh < R * G / 8; ++hh) {
                float old[16];
                tmem_ld16(taddr + 16u * hh, old);
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[(hh * 8 + j) / G][0][(hh * 8 + j) % G] = f2(old[2 * j], old[2 * j + 1]);
            }
        }
        // store the images of every valid base pixel
        if (active) {
            const int start_n = P.start[r - 1], start_s = P.start[4 * N - r - 1];
            const bool south_img = (r != 2 * N);
#pragma unroll
            for (int rr = 0; rr < R; ++rr) {
                const int k = kmine + rr;
                if (k <= klast) {
                    // reflected base pixel; a pixel on the mirror axis (or at phi = 0 of a shifted ring, whose
                    // reflection is its own rotation image) is its own mirror image: stored once
                    const int km = ip - 1 + sh - k;
                    const bool mir_img = MIRROR && (2 * k != ip - 1 + sh) && !(sh && k == 0);
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        const float2 *s = (TOT && !TM) ? tot[TOT && !TM ? rr : 0][b] : acc[rr][b];
#pragma unroll
                        for (int pl = 0; pl < NPL; ++pl) {
                            const bool is_s = SOUTH && (pl & 1), is_m = MIRROR && (pl >= (SOUTH ? 2 : 1));
                            if ((is_s && !south_img) || (is_m && !mir_img)) continue;
                            const float v[4] = {s[2 * pl].x, s[2 * pl].y, s[2 * pl + 1].x, s[2 * pl + 1].y};
                            const int base = (is_s ? start_s : start_n) + (is_m ? km : k);
#pragma unroll
                            for (int m = 0; m < 4; ++m) io.out[b][base + m * ip] = v[m] * P.omega;
                        }
                    }
                }
            }
        }
    }
    if (TM) {                                              // every consumer warp is done with tensor memory
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        asm volatile("bar.sync 2, %0;" ::"r"(NC) : "memory");
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "n"(TMC) : "memory");
    }
}

template <int B, int R, int NC, bool TOT, bool Z, bool TM, bool SOUTH, bool MIRROR, bool HP = false, bool PLN = false>
static cudaError_t launch_sym(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st) {
    const char *dbg = std::getenv("SC_DBG");
    FastDev F{L.pairs, L.tiles, L.ntiles, L.Ltot, L.ntab_s, dbg ? std::atoi(dbg) : 0, L.pairsd, L.tile_ctr};
    static bool attr_done[64] = {};
    cudaError_t e = ensure_max_smem(sym_kernel<B, R, NC, TOT, Z, TM, SOUTH, MIRROR, HP, PLN>, attr_done);
    if (e != cudaSuccess) return e;
    const int grid = std::min(L.nsm, L.ntiles);
    if (grid <= 0) return cudaSuccess;
    if (L.overlap) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(sym_threads(NC)); cfg.dynamicSmemBytes = L.smem; cfg.stream = st;
        cudaLaunchAttribute at{};
        at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at.val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, sym_kernel<B, R, NC, TOT, Z, TM, SOUTH, MIRROR, HP, PLN>, P, F, io);
    }
    if ((e = cudaMemsetAsync(L.tile_ctr, 0, sizeof(int), st)) != cudaSuccess) return e;      // the launch's tile counter
    sym_kernel<B, R, NC, TOT, Z, TM, SOUTH, MIRROR, HP, PLN><<<grid, sym_threads(NC), L.smem, st>>>(P, F, io);
    return cudaGetLastError();
}

}  // namespace sc
