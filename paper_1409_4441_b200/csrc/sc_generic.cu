// sc_generic.cu -- the simple kernel: one thread per output pixel, every ring geometry handled
// (pole-containing discs, whole-ring windows, wrap through phi = 0).  It is
//   * the path for the few rings next to the poles that the fast kernels leave out,
//   * the whole-sphere path when SC_PATH_GENERIC is selected,
//   * the neighbour count / audit pass (MODE_COUNT).
//
// Per pair (BASELINE.json north_star "pair loop"):
//   u = 1 - cos(theta_pq) = A + B (1 - cos dphi),  A = 1 - cos(theta_r - theta_r'),  B = s_r s_r'
//   t = u * (n-1)/(1-c)             table coordinate, 0 at theta = 0, n-1 at theta_max
//   K = tab[floor t].x + t * tab[floor t].y
// A and B come from fp64 ring tables and are rounded once to fp32; dphi is formed from the integer
// pixel offset so no large angles are subtracted in fp32.
// Inclusion: t < tmax - eps -> in; t > tmax + eps -> out; otherwise the canonical fp64 test.
#include "sc_internal.cuh"

namespace sc {

enum { MODE_CONV = 0, MODE_COUNT = 1 };

template <int B, int MODE, bool HP>
__global__ void __launch_bounds__(128)
generic_kernel(const Dev P, const Maps io, int a0, int a1, int b0, int b1,
               int *__restrict__ count_out, unsigned long long *__restrict__ sig_out, Audit au,
               int audit) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int na = a1 - a0;
    int p;
    bool active = true;
    if (tid < na) p = a0 + tid;
    else if (tid - na < b1 - b0) p = b0 + (tid - na);
    else { p = 0; active = false; }

    unsigned long long cnt = 0, sig = 0;
    float tot[B > 0 ? B : 1];
#pragma unroll
    for (int b = 0; b < B; ++b) tot[b] = 0.f;

    if (active) {
        int kp;
        const int rp = ring_of_pixel(P, p, kp);
        const double zp = P.z[rp - 1], sp = P.s[rp - 1];
        const double phip = P.phi0[rp - 1] + (double)kp * P.dphi[rp - 1];
        const int r_lo = P.rlo[rp - 1], r_hi = P.rhi[rp - 1];
        const Audit *aup = audit ? &au : nullptr;

        for (int rq = r_lo; rq <= r_hi; ++rq) {
            const double zq = P.z[rq - 1], sq = P.s[rq - 1];
            double A64 = 1.0 - (zp * zq + sp * sq);
            if (A64 < 0.0) A64 = 0.0;
            const float Af = (float)(A64 * P.scale);
            const float Bf = (float)(sp * sq * P.scale);
            const float wmax = (P.tmax + P.eps - Af) / Bf;
            if (!(wmax >= 0.f)) continue;                    // whole ring beyond theta_max
            const int nq = P.npr[rq - 1];
            const int startq = P.start[rq - 1];
            const double dphiq = P.dphi[rq - 1];
            const float dphiq_f = (float)dphiq;
            // nearest pixel of ring rq in azimuth and the (small) offset to it
            const double xq = (phip - P.phi0[rq - 1]) / dphiq;
            int kc = (int)rint(xq);
            const double dc64 = (P.phi0[rq - 1] + (double)kc * dphiq) - phip;   // (kept in fp64 only if HP)
            const float dc = (float)dc64;
            kc %= nq; if (kc < 0) kc += nq;
            int jlo, jcnt;
            if (wmax >= 2.f) { jlo = -(nq / 2); jcnt = nq; }
            else {
                const float H = 2.f * asinf(sqrtf(0.5f * wmax));
                const int hw = (int)(H / dphiq_f * 1.0001f + 1.5f) + 1;
                if (2 * hw + 1 >= nq) { jlo = -(nq / 2); jcnt = nq; }
                else { jlo = -hw; jcnt = 2 * hw + 1; }
            }
            float racc[B > 0 ? B : 1];
#pragma unroll
            for (int b = 0; b < B; ++b) racc[b] = 0.f;
            for (int jj = 0; jj < jcnt; ++jj) {
                const int j = jlo + jj;
                int kq = kc + j;
                if (kq < 0) kq += nq; else if (kq >= nq) kq -= nq;
                const float d = fmaf((float)j, dphiq_f, dc);
                const float sh = sinf(0.5f * d);
                const float w = 2.f * sh * sh;
                const float t = fmaf(Bf, w, Af);
                bool in = t < P.tmax - P.eps;
                float tt = t;
                if (!in && t <= P.tmax + P.eps) {
                    in = exact_included(P, rp, kp, rq, kq, t, aup);
                    tt = fminf(t, P.tmax);
                }
                if (in) {
                    if (MODE == MODE_COUNT) {
                        ++cnt; sig += (unsigned long long)(startq + kq);
                    } else {
                        int i = (int)tt;
                        float xk = tt;                                  // K = tab[i].x + xk tab[i].y
                        if (P.zoned) zoned_cell(P, tt, i, xk);
                        else if (HP) {                                  // fp64 coordinate -> cell + position in the cell
                            const double t64 = fmin(fma(sp * sq * P.scale, one_minus_cos_f64(fma((double)j, dphiq, dc64)), A64 * P.scale), (double)P.tmax);
                            i = min((int)t64, P.ntab - 2);
                            xk = (float)(t64 - (double)i);
                        }
                        else if (i > P.ntab - 2) i = P.ntab - 2;
                        const float2 e = __ldg(&P.tab[i]);
                        const float K = fmaf(xk, e.y, e.x);
#pragma unroll
                        for (int b = 0; b < B; ++b) racc[b] = fmaf(K, __ldg(&io.in[b][startq + kq]), racc[b]);
                    }
                }
            }
#pragma unroll
            for (int b = 0; b < B; ++b) tot[b] += racc[b];
        }
        if (MODE == MODE_CONV) {
#pragma unroll
            for (int b = 0; b < B; ++b) io.out[b][p] = tot[b] * P.omega;
        } else {
            if (count_out) count_out[p] = (int)cnt;
            if (sig_out) sig_out[p] = sig;
        }
    }
    if (MODE == MODE_COUNT && audit) {
        // block total -> one atomic
        __shared__ unsigned long long sh_tot;
        if (threadIdx.x == 0) sh_tot = 0;
        __syncthreads();
        unsigned long long v = cnt;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sh_tot, v);
        __syncthreads();
        if (threadIdx.x == 0 && sh_tot) atomicAdd(au.total_pairs, sh_tot);
    }
}

// Same arithmetic with one WARP per output pixel: 4 groups of 8 lanes take every 4th input ring, the 8
// lanes of a group share its azimuthal window, and the partial sums are combined with warp shuffles.  Used for the few thousand pixels next to
// the poles, where one thread per pixel leaves the GPU almost empty (latency bound).
template <int B, bool HP>
__global__ void __launch_bounds__(128)
generic_warp_kernel(const Dev P, const Maps io, int a0, int a1, int b0, int b1) {
    const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int na = a1 - a0;
    int p;
    if (wid < na) p = a0 + wid;
    else if (wid - na < b1 - b0) p = b0 + (wid - na);
    else return;                                             // whole warp
    const int grp = lane >> 3, gl = lane & 7;

    float tot[B];
#pragma unroll
    for (int b = 0; b < B; ++b) tot[b] = 0.f;
    int kp;
    const int rp = ring_of_pixel(P, p, kp);
    const double zp = P.z[rp - 1], sp = P.s[rp - 1];
    const double phip = P.phi0[rp - 1] + (double)kp * P.dphi[rp - 1];
    const int r_lo = P.rlo[rp - 1], r_hi = P.rhi[rp - 1];

    for (int rq = r_lo + grp; rq <= r_hi; rq += 4) {
        const double zq = P.z[rq - 1], sq = P.s[rq - 1];
        double A64 = 1.0 - (zp * zq + sp * sq);
        if (A64 < 0.0) A64 = 0.0;
        const float Af = (float)(A64 * P.scale);
        const float Bf = (float)(sp * sq * P.scale);
        const float wmax = (P.tmax + P.eps - Af) / Bf;
        if (!(wmax >= 0.f)) continue;                        // whole ring beyond theta_max
        const int nq = P.npr[rq - 1];
        const int startq = P.start[rq - 1];
        const double dphiq = P.dphi[rq - 1];
        const float dphiq_f = (float)dphiq;
        const double xq = (phip - P.phi0[rq - 1]) / dphiq;
        int kc = (int)rint(xq);
        const double dc64 = (P.phi0[rq - 1] + (double)kc * dphiq) - phip;
        const float dc = (float)dc64;
        kc %= nq; if (kc < 0) kc += nq;
        int jlo, jcnt;
        if (wmax >= 2.f) { jlo = -(nq / 2); jcnt = nq; }
        else {
            const float H = 2.f * asinf(sqrtf(0.5f * wmax));
            const int hw = (int)(H / dphiq_f * 1.0001f + 1.5f) + 1;
            if (2 * hw + 1 >= nq) { jlo = -(nq / 2); jcnt = nq; }
            else { jlo = -hw; jcnt = 2 * hw + 1; }
        }
        float racc[B];
#pragma unroll
        for (int b = 0; b < B; ++b) racc[b] = 0.f;
        for (int jj = gl; jj < jcnt; jj += 8) {
            const int j = jlo + jj;
            int kq = kc + j;
            if (kq < 0) kq += nq; else if (kq >= nq) kq -= nq;
            const float d = fmaf((float)j, dphiq_f, dc);
            const float sh = sinf(0.5f * d);
            const float w = 2.f * sh * sh;
            const float t = fmaf(Bf, w, Af);
            bool in = t < P.tmax - P.eps;
            float tt = t;
            if (!in && t <= P.tmax + P.eps) {
                in = exact_included(P, rp, kp, rq, kq, t, nullptr);
                tt = fminf(t, P.tmax);
            }
            if (in) {
                int i = (int)tt;
                float xk = tt;                                  // K = tab[i].x + xk tab[i].y
                if (P.zoned) zoned_cell(P, tt, i, xk);
                else if (HP) {                                  // fp64 coordinate -> cell + position in the cell
                    const double t64 = fmin(fma(sp * sq * P.scale, one_minus_cos_f64(fma((double)j, dphiq, dc64)), A64 * P.scale), (double)P.tmax);
                    i = min((int)t64, P.ntab - 2);
                    xk = (float)(t64 - (double)i);
                }
                else if (i > P.ntab - 2) i = P.ntab - 2;
                const float2 e = __ldg(&P.tab[i]);
                const float K = fmaf(xk, e.y, e.x);
#pragma unroll
                for (int b = 0; b < B; ++b) racc[b] = fmaf(K, __ldg(&io.in[b][startq + kq]), racc[b]);
            }
        }
#pragma unroll
        for (int b = 0; b < B; ++b) tot[b] += racc[b];
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
        float v = tot[b];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) io.out[b][p] = v * P.omega;
    }
}

// host launchers -----------------------------------------------------------------------------
cudaError_t launch_generic_conv(const Dev &P, const Maps &io, int B, int a0, int a1, int b0, int b1,
                                cudaStream_t st) {
    const int n = (a1 - a0) + (b1 - b0);
    if (n <= 0) return cudaSuccess;
    const int threads = 128, blocks = (n + threads - 1) / threads;
    Audit au{};
    if (P.hp) {                                              // fp64 table coordinate: one map per launch (sc_plan.cu)
        if (B != 1) return cudaErrorInvalidValue;
        generic_kernel<1, MODE_CONV, true><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1, nullptr, nullptr, au, 0);
        return cudaGetLastError();
    }
    switch (B) {
        case 1: generic_kernel<1, MODE_CONV, false><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1, nullptr, nullptr, au, 0); break;
        case 2: generic_kernel<2, MODE_CONV, false><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1, nullptr, nullptr, au, 0); break;
        case 3: generic_kernel<3, MODE_CONV, false><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1, nullptr, nullptr, au, 0); break;
        case 4: generic_kernel<4, MODE_CONV, false><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1, nullptr, nullptr, au, 0); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// overlap: launched with programmatic stream serialization -- the blocks may start while the previous kernel of the stream
// (a fast kernel: disjoint outputs, same inputs) drains
template <int B, bool HP>
static cudaError_t launch_warp(const Dev &P, const Maps &io, int a0, int a1, int b0, int b1, int blocks, int threads, cudaStream_t st,
                               bool overlap) {
    if (!overlap) {
        generic_warp_kernel<B, HP><<<blocks, threads, 0, st>>>(P, io, a0, a1, b0, b1);
        return cudaGetLastError();
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(blocks); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at{};
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, generic_warp_kernel<B, HP>, P, io, a0, a1, b0, b1);
}

cudaError_t launch_generic_conv_warp(const Dev &P, const Maps &io, int B, int a0, int a1, int b0, int b1,
                                     cudaStream_t st, bool overlap) {
    const int n = (a1 - a0) + (b1 - b0);
    if (n <= 0) return cudaSuccess;
    const int threads = 128, blocks = (n + 3) / 4;
    if (P.hp) return B == 1 ? launch_warp<1, true>(P, io, a0, a1, b0, b1, blocks, threads, st, overlap) : cudaErrorInvalidValue;
    switch (B) {
        case 1: return launch_warp<1, false>(P, io, a0, a1, b0, b1, blocks, threads, st, overlap);
        case 2: return launch_warp<2, false>(P, io, a0, a1, b0, b1, blocks, threads, st, overlap);
        case 3: return launch_warp<3, false>(P, io, a0, a1, b0, b1, blocks, threads, st, overlap);
        case 4: return launch_warp<4, false>(P, io, a0, a1, b0, b1, blocks, threads, st, overlap);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_generic_count(const Dev &P, int *count_dev, unsigned long long *sig_dev,
                                 const Audit *au, cudaStream_t st) {
    const int n = P.npix;
    const int threads = 128, blocks = (n + threads - 1) / threads;
    Maps io{};
    Audit a{};
    if (au) a = *au;
    generic_kernel<0, MODE_COUNT, false><<<blocks, threads, 0, st>>>(P, io, 0, n, 0, 0, count_dev, sig_dev, a, au ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace sc
