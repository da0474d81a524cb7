// k3d_pk_m0.cu -- instantiations of recon3d_pk_kernel<CPL, GZP, 0> (axial+z LRFs, 3-D search, level pairs packed)
#include "recon3d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_3d_pk_m0(int cpl, int gzp, int cross) {
    // an odd grid with two columns per lane (G = 7) packs its top level across the lane's columns (CROSS)
    if (cross) return cpl == 2 && gzp == 4 ? (const void *)recon3d_pk_kernel<2, 4, 0, true> : nullptr;
#define ANTS_K3(C, Z) if (cpl == C && gzp == Z) return (const void *)recon3d_pk_kernel<C, Z, 0>
    // GZP = the grid's level pairs exactly, (G + 1) / 2; one column per lane up to G = 5, two for G = 6 .. 8
    ANTS_K3(1, 1); ANTS_K3(1, 2); ANTS_K3(1, 3); ANTS_K3(2, 3); ANTS_K3(2, 4);
#undef ANTS_K3
    return nullptr;
}
}  // namespace ants
