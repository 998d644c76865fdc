// sc_fast.cuh -- plan data shared by the fast kernels (sym kernel: sc_fast.cu, belt kernel: sc_belt.cu).
#pragma once
#include "sc_internal.cuh"

namespace sc {

constexpr int kMaxThreads = 512;
constexpr float kMagic = 12582912.0f;             // 1.5 * 2^23: low mantissa bits = round(x)
constexpr unsigned kMagicBits = 0x4B400000u;

struct PairEnt {            // uniform per (base ring, input ring); 48 bytes
    float A;                // A * scale - 0.5   (table coordinate shifted by half a cell)
    float c1, c2, c3;       // B * scale * {1/2, -1/24, 1/720}
    float dphi;             // azimuthal pixel spacing of the input ring
    float cdc;              // pi / (4 ip ip')
    int rq, hw, ipq, shq;   // input ring, half window (pixels), pixels per quadrant, shift flag
    int start_n, start_s;   // first pixel of the input ring and of its southern mirror
};

struct FastDev {
    const PairEnt *pairs;
    const int *pair_off;    // [nslots + 1]
    const int4 *tiles;      // (ring, k0, slot, 0)
    int ntiles;
    int *counter;
    int Lmax;               // staged positions per plane
    int ntab_s;             // entries of the shared-memory table
    int R;
};

}  // namespace sc
