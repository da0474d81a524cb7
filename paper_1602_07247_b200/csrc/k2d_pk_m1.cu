// k2d_pk_m1.cu -- instantiations of recon2d_pk_kernel<NPT, 1> (one translation unit per method: parallel build)
#include "recon2d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_pk_m1(int npt) {
    switch (npt) {
        case 1: return (const void *)recon2d_pk_kernel<1, 1>;
        case 2: return (const void *)recon2d_pk_kernel<2, 1>;
        case 3: return (const void *)recon2d_pk_kernel<3, 1>;
        case 4: return (const void *)recon2d_pk_kernel<4, 1>;
        case 8: return (const void *)recon2d_pk_kernel<8, 1>;
    }
    return nullptr;
}
}  // namespace ants
