// sc_fast.cuh -- plan data shared by the fast kernels (sym kernel: sc_fast.cu, belt kernel: sc_belt.cu).
#pragma once
#include "sc_internal.cuh"

namespace sc {

constexpr int kMaxThreads = 512;
constexpr float kMagic = 12582912.0f;             // 1.5 * 2^23: low mantissa bits = round(x)
constexpr unsigned kMagicBits = 0x4B400000u;

struct PairEnt {            // uniform per (base ring, input ring); 56 bytes
    float A;                // A * scale - 0.5   (table coordinate shifted by half a cell)
    float c1, c2, c3;       // B * scale * {1/2, -1/24, 1/720}
    float dphi;             // azimuthal pixel spacing of the input ring
    float cdc;              // pi / (4 ip ip')
    int rq, hw, ipq, shq;   // input ring, half window (pixels), pixels per quadrant, shift flag
    int start_n, start_s;   // first pixel of the input ring and of its southern mirror
    float c4;               // B * scale * (-1/40320): fourth term of 1 - cos d
    int ex;                 // planar sym instances: positions staged beyond the window on both sides (>= the drift of 32 lanes
                            // 3 base pixels apart against this ring's pixel spacing); 0 = no lane skew on this ring pair
};

// The same ring pair in fp64 for plans with Dev::hp (steep tables): t = A + Bs (1 - cos d), d = (integer offset) cdc + j dphi
struct PairEntD { double A, Bs, dphi, cdc; };

// A tile of the sym kernel is a set of up to kMaxSub sub-tiles, each a run of base pixels on one ring that
// is worked on by `nw` consecutive warps (32 R pixels per warp).  Packing several short runs into one
// tile keeps all warps of the CTA busy on the short rings of the polar caps.
constexpr int kMaxSub = 4;
struct SubTile {
    int r, k0, n;           // base ring, first base pixel, number of base pixels
    int e0, ne;             // its input rings: pairs[e0 .. e0 + ne)
    int w0, nw;             // first warp, number of warps
    int soff;               // offset (positions) of its staged runs within a stage plane
};
struct SymTile {
    int nsub, nsteps, pad0, pad1;   // nsteps = max ne over the sub-tiles
    SubTile sub[kMaxSub];
};

struct FastDev {
    const PairEnt *pairs;
    const SymTile *tiles;
    int ntiles;
    int Ltot;               // staged positions per plane
    int ntab_s;             // entries of the shared-memory table
    int dbg;                // measurement only (SC_DBG): 1 = consumers skip the pair loop, 2 = producers skip the copies
    const PairEntD *pairsd; // fp64 ring pairs (Dev::hp), same index as pairs; else nullptr
    int *tile_ctr;          // sym kernel: tile counter of the launch (zeroed before it): CTAs take tiles in list order as they finish
};

// What a launch of the sym kernel needs from the plan (host); the instantiations live in sc_sym_b1.cu (one map per
// launch: 8 images, 16 images with the mirror symmetry, north-only) and sc_sym_bn.cu (batches of 2-4 maps)
struct SymLaunch {
    const PairEnt *pairs;
    const SymTile *tiles;
    int ntiles, Ltot, ntab_s, nsm;
    int threads, R;             // consumer threads, base pixels per thread
    size_t smem;
    bool tot, tmem, mirror, south;
    bool pair;                  // lane-pair instance (sc_sym_pair.cu): two lanes share a group of R base pixels
    int *tile_ctr;              // plan-owned device counter for the dynamic tile schedule
    const PairEntD *pairsd;     // fp64 ring pairs of a Dev::hp plan
    bool overlap;               // launch with programmatic stream serialization: the CTAs may start while the previous kernel of
                                // the stream (the belt kernel: disjoint outputs) drains; the tile counter was zeroed before that kernel
    bool planar = false;        // planar staging by TMA bulk copies (sc_sym_pl.cu): one plane per image instead of float4-interleaved rotations
};
cudaError_t dispatch_sym_pair(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st);
cudaError_t dispatch_sym_b1(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st);
cudaError_t dispatch_sym_pl(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st);
constexpr int kPlanarPlane = 784;   // floats per image plane of the planar instances (kLp in sc_sym.cuh)
constexpr int kPlanarPad = 8;       // extra staged floats per run: 0-3 in front (alignment in the ring), rounded up to 4 behind
cudaError_t dispatch_sym_bn(const SymLaunch &L, const Dev &P, const Maps &io, int B, cudaStream_t st);

constexpr int kMaxExc = 32;      // uncertain taps per belt tile that can be listed (more -> rescan)

struct BeltDev {
    const PairEnt *pairs;
    const int *pair_off;
    const int *woff;          // per pair entry: offset (in float2, even) of its tap array within a tap buffer
    const int4 *tiles;        // (ring, k0, slot, number of input rings)
    const int *grp_off;       // per slot: its group boundaries are grp_e[grp_off[slot] .. grp_off[slot + 1])
    const int *grp_e;         // entry indices (relative to the ring's first entry) where the groups begin, then the end
    int ntiles;
    int pw_max;               // float2 entries of a tap buffer
    int ne_max;               // input rings per group, at most
    int nbuf;                 // stage buffers
    int ntb;                  // tap buffers (1 or 2)
    const PairEntD *pairsd;   // fp64 ring pairs (Dev::hp), same index as pairs; else nullptr
};

// Layout of one tap buffer in shared memory (bytes): taps | ring descriptors | exception list
struct TapLayout {
    unsigned desc, exc_e, exc_j, exc_k, nexc, bytes;
    __host__ __device__ TapLayout(int pw_max, int ne_max) {
        desc = (unsigned)pw_max * 8u;
        exc_e = desc + (unsigned)ne_max * 16u;
        exc_j = exc_e + kMaxExc * 4u;
        exc_k = exc_j + kMaxExc * 4u;
        nexc = exc_k + kMaxExc * 4u;
        bytes = (nexc + 16u + 15u) & ~15u;
    }
};

// Host: opt a kernel instance in to the device's maximum dynamic shared memory ONCE per device instead of on every
// launch.  `done` is a per-instantiation flag array owned by the calling launcher template.
template <class K> inline cudaError_t ensure_max_smem(K kernel, bool (&done)[64]) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
    int optin = 0;
    cudaFuncAttributes fa{};
    if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return e;
    if ((e = cudaFuncGetAttributes(&fa, kernel)) != cudaSuccess) return e;
    // the opt-in limit covers static + dynamic shared memory
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes)) != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) done[dev] = true;
    return cudaSuccess;
}

// ---- mbarrier / TMA bulk copy -------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    unsigned ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// same for producer warps that may wait long: back off so the spin does not take issue slots
__device__ __forceinline__ void mbar_wait_sleep(unsigned long long *bar, unsigned parity) {
    unsigned ok;
    while (true) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (ok) break;
        __nanosleep(32);
    }
}
__device__ __forceinline__ void tma_load_1d(void *smem_dst, const void *gsrc, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// ---- tensor memory (TMEM) as accumulator storage -------------------------------------------------------------
// With three or four consumer warpgroups a thread has 104-152 registers: the running totals (32 floats per
// thread) of the two-accumulator summation do not fit next to the 32 per-ring accumulators, so they live in
// tensor memory:
// a warp owns the 32 TMEM lanes of its quadrant (warp % 4) and 32 columns (warp / 4); tcgen05.ld / st with the
// 32x32b shape move one row (lane) x 16 columns per thread.
__device__ __forceinline__ void tmem_st16(unsigned taddr, const float (&v)[16]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 :: "r"(taddr), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]),
                    "f"(v[8]), "f"(v[9]), "f"(v[10]), "f"(v[11]), "f"(v[12]), "f"(v[13]), "f"(v[14]), "f"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_ld16(unsigned taddr, float (&v)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]),
                   "=f"(v[8]), "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// cp.async (LDGSTS) of 4 bytes; completion is reported to an mbarrier with cp_async_mbar_arrive
__device__ __forceinline__ void cp_async4_s(unsigned smem_dst, const void *gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_dst), "l"(gsrc) : "memory");
}
// one arrival on `bar` (already counted in its init count) once all prior cp.async of this thread landed
__device__ __forceinline__ void cp_async_mbar_arrive(unsigned long long *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace sc
