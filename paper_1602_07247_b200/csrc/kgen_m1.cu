// kgen_m1.cu -- instantiations of recon_gen_kernel<1, LRFK> (the general kernel: any LRF parameterisation)
#include "recon_gen.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_gen_m1(int lrf_kind) {
    switch (lrf_kind) {
        case kAxial: return (const void *)recon_gen_kernel<1, kAxial>;
        case kXY: return (const void *)recon_gen_kernel<1, kXY>;
        case kComposite: return (const void *)recon_gen_kernel<1, kComposite>;
        case kSliced: return (const void *)recon_gen_kernel<1, kSliced>;
    }
    return nullptr;
}
}  // namespace ants
