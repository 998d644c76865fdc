// sc_sym_b1.cu -- sym kernel instances for ONE map per launch (the headline path) and their dispatch.
//   16 images (rotations x north/south x mirror): 192 consumer threads, 4 base pixels per thread;
//    8 images (rotations x north/south):          384 / 256 / 128 consumer threads (fallbacks; tensor-memory totals);
//    8 images north only (rotations x mirror):    sc_convolve_cap (partial-sky maps in the polar cap).
#include "sc_sym.cuh"

namespace sc {

cudaError_t dispatch_sym_b1(const SymLaunch &L, const Dev &P, const Maps &io, cudaStream_t st) {
    const bool z = P.zoned != 0;
#define SC_GO(R, NC, TOT, TM, SOUTH, MIRROR) \
    return z ? launch_sym<1, R, NC, TOT, true, TM, SOUTH, MIRROR>(L, P, io, st) : launch_sym<1, R, NC, TOT, false, TM, SOUTH, MIRROR>(L, P, io, st)
    if (P.hp) {                                         // fp64 table coordinate (steep tables), full-sphere instances only
        if (!L.south || z || !L.pairsd) return cudaErrorInvalidValue;
        if (L.mirror && L.threads == 256 && L.R == 3) {
            if (L.tot && L.tmem) return launch_sym<1, 3, 256, true, false, true, true, true, true>(L, P, io, st);
            if (!L.tot && !L.tmem) return launch_sym<1, 3, 256, false, false, false, true, true, true>(L, P, io, st);
            return cudaErrorInvalidValue;
        }
        if (L.mirror) {
            if (L.threads != 192 || L.R != 4) return cudaErrorInvalidValue;
            if (L.tot && L.tmem) return launch_sym<1, 4, 192, true, false, true, true, true, true>(L, P, io, st);
            if (!L.tot && !L.tmem) return launch_sym<1, 4, 192, false, false, false, true, true, true>(L, P, io, st);
            return cudaErrorInvalidValue;
        }
        if (!L.tot || L.tmem) return cudaErrorInvalidValue;      // large discs whose runs do not fit the 16-image tiles
        if (L.threads == 256 && L.R == 4) return launch_sym<1, 4, 256, true, false, false, true, false, true>(L, P, io, st);
        if (L.threads == 256 && L.R == 2) return launch_sym<1, 2, 256, true, false, false, true, false, true>(L, P, io, st);
        if (L.threads == 128 && L.R == 2) return launch_sym<1, 2, 128, true, false, false, true, false, true>(L, P, io, st);
        return cudaErrorInvalidValue;
    }
    if (L.south && L.mirror) {                          // 16 images
        if (L.threads == 256 && L.R == 3 && L.tot && L.tmem) { SC_GO(3, 256, true, true, true, true); }
        if (L.threads == 256 && L.R == 3 && !L.tot && !L.tmem) { SC_GO(3, 256, false, false, true, true); }
        if (L.threads == 192 && L.R == 4 && L.tot && L.tmem) { SC_GO(4, 192, true, true, true, true); }
        if (L.threads == 192 && L.R == 4 && !L.tot && !L.tmem) { SC_GO(4, 192, false, false, true, true); }
        return cudaErrorInvalidValue;
    }
    if (!L.south && L.mirror) {                         // north only, 8 images
        if (L.threads == 384 && L.R == 4 && !L.tmem && !L.tot) { SC_GO(4, 384, false, false, false, true); }
        if (L.threads == 256 && L.R == 4 && !L.tmem && L.tot) { SC_GO(4, 256, true, false, false, true); }
        if (L.threads == 128 && L.R == 2 && !L.tmem && L.tot) { SC_GO(2, 128, true, false, false, true); }
        return cudaErrorInvalidValue;
    }
    if (!L.south) return cudaErrorInvalidValue;
    if (L.threads == 384 && L.R == 4 && L.tmem) { SC_GO(4, 384, true, true, true, false); }
    if (L.threads == 384 && L.R == 4 && !L.tot) { SC_GO(4, 384, false, false, true, false); }
    if (!L.tot || L.tmem) return cudaErrorInvalidValue;
    if (L.threads == 256 && L.R == 4) { SC_GO(4, 256, true, false, true, false); }
    if (L.threads == 256 && L.R == 2) { SC_GO(2, 256, true, false, true, false); }
    if (L.threads == 256 && L.R == 1) { SC_GO(1, 256, true, false, true, false); }
    if (L.threads == 128 && L.R == 4) { SC_GO(4, 128, true, false, true, false); }
    if (L.threads == 128 && L.R == 2) { SC_GO(2, 128, true, false, true, false); }
    if (L.threads == 128 && L.R == 1) { SC_GO(1, 128, true, false, true, false); }
#undef SC_GO
    return cudaErrorInvalidValue;
}

}  // namespace sc
