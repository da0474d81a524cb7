// k2d_gen_m0.cu -- instantiations of recon2d_kernel<NPT, 0, false> (LRFs that are not positive everywhere)
#include "recon2d.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_gen_m0(int npt) {
    switch (npt) {
        case 1: return (const void *)recon2d_kernel<1, 0, false>;
        case 2: return (const void *)recon2d_kernel<2, 0, false>;
        case 3: return (const void *)recon2d_kernel<3, 0, false>;
        case 4: return (const void *)recon2d_kernel<4, 0, false>;
        case 8: return (const void *)recon2d_kernel<8, 0, false>;
    }
    return nullptr;
}
}  // namespace ants
