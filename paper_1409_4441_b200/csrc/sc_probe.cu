// sc_probe.cu -- measurement only: the sustained FP32 FMA rate of the device, the denominator of the roofline
// that bench.py reports ("report against (i) the nominal figure and (ii) a sustained FFMA
// microbenchmark run in the same job").  Register-only loops of independent FMA chains: scalar FFMA or packed
// FFMA2 (fma.rn.f32x2, the instruction the convolution kernels accumulate with), and a third loop with the OPERAND
// PATTERN of the belt kernel's accumulation -- acc_pair += tap_pair * map_value, the tap pair shared by 4 FFMA2 and a
// fresh map value and accumulator pair each time: what the register file sustains for it (measured ~105 against ~125
// FMA / clk / SM with constant operands; an arrangement whose tap pairs are not aligned register pairs drops to 83).
#include "../../include/sc.h"
#include <cuda_runtime.h>

namespace {

constexpr int kChains = 16;          // independent fp32 accumulators per thread (8 float2 in the packed loop)

template <bool PACKED>
__global__ void __launch_bounds__(1024, 1)
fma_probe_kernel(float *out, int iters, float a, float b) {
    float2 acc[kChains / 2];
#pragma unroll
    for (int j = 0; j < kChains / 2; ++j) acc[j] = make_float2((float)threadIdx.x + j, (float)j - 0.5f);
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int j = 0; j < kChains / 2; ++j) {
                if (PACKED) acc[j] = __ffma2_rn(acc[j], a2, b2);
                else { acc[j].x = fmaf(acc[j].x, a, b); acc[j].y = fmaf(acc[j].y, a, b); }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kChains / 2; ++j) s += acc[j].x + acc[j].y;
    if (s == 123.456f) out[0] = s;       // never true in practice: keeps the loop alive
}

// acc[p][s] += tap[6 - 2p + i] * m[s][i]: the belt kernel's chunk (8 pixels = 4 pairs p, 4 images s, 4 positions i) with
// its register layout -- tap pairs and map values as they come out of LDS.128 (float4), so that every tap pair is an
// aligned register pair -- register only, the operands changing a little every iteration so that nothing is hoisted
__global__ void __launch_bounds__(512, 1)
fma_pattern_kernel(float *out, const float *in, int iters) {
    float2 acc[16];
    float4 tp[5], mv[4];
#pragma unroll
    for (int j = 0; j < 16; ++j) acc[j] = make_float2((float)threadIdx.x + j, (float)j - 0.5f);
#pragma unroll
    for (int j = 0; j < 5; ++j) tp[j] = make_float4(in[4 * j], in[4 * j + 1], in[4 * j + 2], in[4 * j + 3]);
#pragma unroll
    for (int j = 0; j < 4; ++j) mv[j] = make_float4(in[32 + 4 * j], in[33 + 4 * j], in[34 + 4 * j], in[35 + 4 * j]);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
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
#pragma unroll
                for (int p = 0; p < 4; ++p) acc[4 * p + sl] = __ffma2_rn(pwr[6 - 2 * p + i], m2, acc[4 * p + sl]);
            }
        }
        tp[0].x += 1e-9f; mv[0].x += 1e-9f; mv[1].y += 1e-9f; mv[2].z += 1e-9f; mv[3].w += 1e-9f;
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 16; ++j) s += acc[j].x + acc[j].y;
    if (s == 123.456f) out[0] = s;
}

}  // namespace

extern "C" sc_status sc_debug_fma_peak(int packed, double *fma_per_s, double *elapsed_ms) {
    if (!fma_per_s) return SC_ERR_INVALID_ARG;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return SC_ERR_CUDA;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) return SC_ERR_CUDA;
    if (packed < 0 || packed > 2) return SC_ERR_INVALID_ARG;
    float *d = nullptr;
    if (cudaMalloc((void **)&d, 256) != cudaSuccess) return SC_ERR_ALLOC;
    if (cudaMemset(d, 0, 256) != cudaSuccess) { cudaFree(d); return SC_ERR_CUDA; }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    sc_status st = SC_OK;
    double best = 0.0, best_ms = 0.0;
    do {
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { st = SC_ERR_CUDA; break; }
        const int blocks = packed == 2 ? nsm : 2 * nsm, threads = packed == 2 ? 512 : 1024, iters = packed == 2 ? 20000 : 12000;   // ~ 6 ms at 128 FMA / clk / SM
        const double fmas = packed == 2 ? (double)blocks * threads * (double)iters * 128.0
                                        : (double)blocks * threads * (double)iters * 4.0 * kChains;
        for (int rep = 0; rep < 4 && st == SC_OK; ++rep) {               // first repetition = warm-up
            cudaEventRecord(e0, 0);
            if (packed == 2) fma_pattern_kernel<<<blocks, threads>>>(d + 32, d, iters);
            else if (packed) fma_probe_kernel<true><<<blocks, threads>>>(d, iters, 1.000001f, 1e-7f);
            else fma_probe_kernel<false><<<blocks, threads>>>(d, iters, 1.000001f, 1e-7f);
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { st = SC_ERR_CUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms > 0.f && fmas / (ms * 1e-3) > best) { best = fmas / (ms * 1e-3); best_ms = ms; }
        }
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d);
    if (st != SC_OK) return st;
    *fma_per_s = best;
    if (elapsed_ms) *elapsed_ms = best_ms;
    return SC_OK;
}
