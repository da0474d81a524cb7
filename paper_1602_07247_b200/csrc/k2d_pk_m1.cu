// k2d_pk_m1.cu -- instantiations of recon2d_pk_kernel<NPT, 1, REUSE, LOCKSTEP> (one translation unit per method: parallel build)
#include "recon2d_pk.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_2d_pk_m1(int npt, int reuse) {
    // (the least-squares kernels run node reuse only with the CTA-wide event rounds: it loses without them)
#define ANTS_K2(NP)                                                                    \
    if (npt == NP)                                                                     \
        return reuse ? (const void *)recon2d_pk_kernel<NP, 1, true, true>                \
                     : (const void *)recon2d_pk_kernel<NP, 1, false, false>
    ANTS_K2(1); ANTS_K2(2); ANTS_K2(3); ANTS_K2(4); ANTS_K2(8);
#undef ANTS_K2
    return nullptr;
}
}  // namespace ants
