// kernels.h -- the reconstruction kernels are instantiated in their own translation units (k_*.cu, compiled in
// parallel by build.py); the host logic in ants_recon.cu picks one through these look-ups.  Each returns
// nullptr for a combination that is not compiled.
#pragma once

namespace ants {

// axial LRFs, strictly positive: sensor-pair-packed kernel (recon2d_pk.cuh).  method 0/1/2, npt in {1,2,3,4,8}
const void *kernel_2d_pk(int method, int npt);
// axial LRFs that are not positive everywhere: scalar kernel with per-pair validity tests (recon2d.cuh)
const void *kernel_2d_gen(int method, int npt);
// axial+z LRFs (recon3d.cuh).  method 0/1, (cpl, gzm) in {(1,1),(2,1),(3,1),(4,1),(8,1),(1,4),(2,4),(1,8),(2,8)}
const void *kernel_3d(int method, int cpl, int gzm);

}  // namespace ants
