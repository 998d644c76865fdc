// sc_sym_pl.cu -- sym kernel instances with PLANAR staging (template flag PLN of sc_sym.cuh): 16 images, one map per
// launch, 256 consumer threads x 3 base pixels (single accumulator set for discs of at most 700 pixels, totals in tensor
// memory up to 2500); every image has a stage plane of its own, filled by TMA bulk copies.
#include "sc_sym.cuh"

namespace sc {

cudaError_t dispatch_sym_pl(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st) {
    if (!L.planar || !L.south || !L.mirror || L.threads != 256 || L.R != 3 || P.hp || L.tot != L.tmem) return cudaErrorInvalidValue;
    const bool z = P.zoned != 0;
    if (L.tot) return z ? launch_sym<1, 3, 256, true, true, true, true, true, false, true>(L, P, io, st)
                        : launch_sym<1, 3, 256, true, false, true, true, true, false, true>(L, P, io, st);
    return z ? launch_sym<1, 3, 256, false, true, false, true, true, false, true>(L, P, io, st)
             : launch_sym<1, 3, 256, false, false, false, true, true, false, true>(L, P, io, st);
}

}  // namespace sc
