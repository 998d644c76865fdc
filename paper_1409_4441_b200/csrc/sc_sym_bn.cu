// sc_sym_bn.cu -- sym kernel instances for batches of 2-4 maps per launch (8 images: rotations x north/south; two
// accumulator sets in registers) and their dispatch.
#include "sc_sym.cuh"

namespace sc {

cudaError_t dispatch_sym_bn(const SymLaunch &L, const Dev &P, const Maps &io, int B, cudaStream_t st) {
    if (!L.south || L.mirror || L.tmem || !L.tot) return cudaErrorInvalidValue;
    const bool z = P.zoned != 0;
#define SC_CASE(BB, RR, NC) \
    if (B == BB && L.R == RR && L.threads == NC) \
        return z ? launch_sym<BB, RR, NC, true, true, false, true, false>(L, P, io, st) : launch_sym<BB, RR, NC, true, false, false, true, false>(L, P, io, st);
    SC_CASE(2, 1, 256) SC_CASE(2, 2, 256) SC_CASE(2, 4, 256) SC_CASE(2, 1, 128) SC_CASE(2, 2, 128) SC_CASE(2, 4, 128)
    SC_CASE(3, 1, 256) SC_CASE(3, 2, 256) SC_CASE(3, 1, 128) SC_CASE(3, 2, 128)
    SC_CASE(4, 1, 256) SC_CASE(4, 2, 256) SC_CASE(4, 1, 128) SC_CASE(4, 2, 128)
#undef SC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace sc
