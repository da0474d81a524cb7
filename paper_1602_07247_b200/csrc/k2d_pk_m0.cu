// k2d_pk_m0.cu -- instantiations of recon2d_pk_kernel<NPT, 0> (one translation unit per method: parallel build)
#include "recon2d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_pk_m0(int npt) {
    switch (npt) {
        case 1: return (const void *)recon2d_pk_kernel<1, 0>;
        case 2: return (const void *)recon2d_pk_kernel<2, 0>;
        case 3: return (const void *)recon2d_pk_kernel<3, 0>;
        case 4: return (const void *)recon2d_pk_kernel<4, 0>;
        case 8: return (const void *)recon2d_pk_kernel<8, 0>;
    }
    return nullptr;
}
}  // namespace ants
