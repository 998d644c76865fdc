// sc_nested.cu -- NESTED <-> RING reordering for plans created with SC_ORDER_NESTED.
// The convolution kernels work on RING-ordered maps; a NESTED plan scatters every input map into a
// plan-owned RING buffer, convolves there and gathers the result back.  Both directions use the same index
// map nest -> ring (HEALPix nested scheme, Gorski et al. 2005, which the paper only cites):
//   p = face * nside^2 + interleave(ix, iy)   (ix on the even bits), nside a power of two;
//   ring number (1-based)   jr = jrll[face] * nside - ix - iy - 1,  jrll = 2,2,2,2,3,3,3,3,4,4,4,4;
//   pixels per quadrant nr and pixels before the ring from the RING layout; shifted belt rings have kshift = 1;
//   position in ring (1-based)  jp = (jpll[face] * nr + ix - iy + 1 + kshift) / 2, wrapped into 1 .. 4 nr,
//   jpll = 1,3,5,7,0,2,4,6,1,3,5,7.
#include "sc_internal.cuh"

namespace sc {

__device__ __forceinline__ unsigned even_bits(unsigned x) {            // bits 0, 2, 4, ... packed together
    x &= 0x55555555u;
    x = (x | (x >> 1)) & 0x33333333u;
    x = (x | (x >> 2)) & 0x0f0f0f0fu;
    x = (x | (x >> 4)) & 0x00ff00ffu;
    x = (x | (x >> 8)) & 0x0000ffffu;
    return x;
}

__device__ __forceinline__ int nest_to_ring(int nside, int order, int p) {
    const int face = p >> (2 * order);
    const unsigned pf = (unsigned)p & ((1u << (2 * order)) - 1u);
    const int ix = (int)even_bits(pf), iy = (int)even_bits(pf >> 1);
    const int jr = (face / 4 + 2) * nside - ix - iy - 1;
    int nr, before, kshift = 0;
    if (jr < nside) { nr = jr; before = 2 * nr * (nr - 1); }
    else if (jr > 3 * nside) { nr = 4 * nside - jr; before = 12 * nside * nside - 2 * (nr + 1) * nr; }
    else { nr = nside; before = 2 * nside * (nside - 1) + (jr - nside) * 4 * nside; kshift = (jr - nside) & 1; }
    const int jpll = 2 * (face & 3) + ((face >> 2) == 1 ? 0 : 1);
    int jp = (jpll * nr + ix - iy + 1 + kshift) / 2;
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    return before + jp - 1;
}

// DIR 0: ring[n2r(p)] = nest[p] (scatter);  DIR 1: nest[p] = ring[n2r(p)] (gather)
template <class T, int DIR>
__global__ void reorder_kernel(int nside, int order, int npix, const T *__restrict__ src, T *__restrict__ dst) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    const int q = nest_to_ring(nside, order, p);
    if (DIR == 0) dst[q] = src[p]; else dst[p] = src[q];
}

template <class T>
static cudaError_t reorder(int nside, int dir, const T *src, T *dst, cudaStream_t st) {
    int order = 0;
    while ((1 << order) < nside) ++order;
    const int npix = 12 * nside * nside, threads = 256, blocks = (npix + threads - 1) / threads;
    if (dir == 0) reorder_kernel<T, 0><<<blocks, threads, 0, st>>>(nside, order, npix, src, dst);
    else reorder_kernel<T, 1><<<blocks, threads, 0, st>>>(nside, order, npix, src, dst);
    return cudaGetLastError();
}

cudaError_t reorder_f32(int nside, int dir, const float *src, float *dst, cudaStream_t st) { return reorder<float>(nside, dir, src, dst, st); }
cudaError_t reorder_i32(int nside, int dir, const int *src, int *dst, cudaStream_t st) { return reorder<int>(nside, dir, src, dst, st); }
cudaError_t reorder_u64(int nside, int dir, const unsigned long long *src, unsigned long long *dst, cudaStream_t st) {
    return reorder<unsigned long long>(nside, dir, src, dst, st);
}

}  // namespace sc
