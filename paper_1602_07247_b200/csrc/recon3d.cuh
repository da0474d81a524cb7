// recon3d.cuh -- contracting grids over (x, y, z) with axial+z LRFs
// (section 6.1.2).  Placeholder until the 3-D kernel lands.
#pragma once
#include "../../include/ants_recon.h"
#include "recon_common.cuh"

namespace ants {
inline int make_plan3d(bool, double, double, double, const ModelDev &, const ants_grid_params_t *, int32_t,
                       int &, int &, int &, size_t &, int &, const void *&) {
    return ANTS_ERR_UNSUPPORTED;
}
}  // namespace ants
