// k3d_m0.cu -- instantiations of recon3d_kernel<CPL, GZM, 0> (axial+z LRFs)
#include "recon3d.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_3d_m0(int cpl, int gzm) {
#define ANTS_K3(C, Z) if (cpl == C && gzm == Z) return (const void *)recon3d_kernel<C, Z, 0>
    ANTS_K3(1, 1); ANTS_K3(2, 1); ANTS_K3(3, 1); ANTS_K3(4, 1); ANTS_K3(8, 1);
    ANTS_K3(1, 4); ANTS_K3(2, 4); ANTS_K3(1, 8); ANTS_K3(2, 8);
#undef ANTS_K3
    return nullptr;
}
}  // namespace ants
