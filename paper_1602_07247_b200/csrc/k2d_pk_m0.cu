// k2d_pk_m0.cu -- instantiations of recon2d_pk_kernel<NPT, 0, REUSE, LOCKSTEP> (one translation unit per method: parallel build)
#include "recon2d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_pk_m0(int npt, int reuse) {
#define ANTS_K2(NP)                                                                    \
    if (npt == NP)                                                                     \
        return reuse == 2   ? (const void *)recon2d_pk_kernel<NP, 0, true, true>         \
               : reuse == 1 ? (const void *)recon2d_pk_kernel<NP, 0, true, false>        \
                            : (const void *)recon2d_pk_kernel<NP, 0, false, false>
    ANTS_K2(1); ANTS_K2(2); ANTS_K2(3); ANTS_K2(4); ANTS_K2(8);
#undef ANTS_K2
    return nullptr;
}
}  // namespace ants
