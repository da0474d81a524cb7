// krefine.cu -- instantiations of refine_kernel<METHOD> (continuous refinement, refine.cuh)
#include "refine.cuh"
#include "kernels.h"

namespace ants {
const void *kernel_refine(int method) {
    switch (method) {
        case 0: return (const void *)refine_kernel<0>;
        case 1: return (const void *)refine_kernel<1>;
        case 2: return (const void *)refine_kernel<2>;
    }
    return nullptr;
}
}  // namespace ants
