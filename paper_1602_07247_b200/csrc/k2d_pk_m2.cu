// k2d_pk_m2.cu -- instantiations of recon2d_pk_kernel<NPT, 2> (one translation unit per method: parallel build)
#include "recon2d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_pk_m2(int npt) {
    switch (npt) {
        case 1: return (const void *)recon2d_pk_kernel<1, 2>;
        case 2: return (const void *)recon2d_pk_kernel<2, 2>;
        case 3: return (const void *)recon2d_pk_kernel<3, 2>;
        case 4: return (const void *)recon2d_pk_kernel<4, 2>;
        case 8: return (const void *)recon2d_pk_kernel<8, 2>;
    }
    return nullptr;
}
}  // namespace ants
