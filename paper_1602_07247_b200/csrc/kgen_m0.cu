// kgen_m0.cu -- instantiations of recon_gen_kernel<0, LRFK> (the general kernel: any LRF parameterisation)
#include "recon_gen.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_gen_m0(int lrf_kind) {
    switch (lrf_kind) {
        case kAxial: return (const void *)recon_gen_kernel<0, kAxial>;
        case kXY: return (const void *)recon_gen_kernel<0, kXY>;
        case kComposite: return (const void *)recon_gen_kernel<0, kComposite>;
        case kSliced: return (const void *)recon_gen_kernel<0, kSliced>;
    }
    return nullptr;
}
}  // namespace ants
