// kernels.h -- the reconstruction kernels are instantiated in their own translation units (k2d_pk_m*.cu, k3d_m*.cu, kgen_m*.cu, compiled in
// parallel by build.py); the host logic in ants_recon.cu picks one through these look-ups.  Each returns
// nullptr for a combination that is not compiled.
#pragma once

namespace ants {

// axial LRFs, strictly positive: sensor-pair-packed kernel (recon2d_pk.cuh).  method 0/1/2, npt in {1,2,3,4,8}
// reuse: 0 none, 1 node reuse, 2 node reuse with the CTA's warps taking their events in rounds behind a barrier
const void *kernel_2d_pk(int method, int npt, int reuse);
// axial+z LRFs searched in 3-D, packed over pairs of z-levels (recon3d_pk.cuh).  method 0/1,
// (cpl, gzp) in {(1,1),(1,2),(1,3),(2,3),(2,4)}; cross = 1: (2,4) with the top level of an odd grid packed across the
// lane's two columns
const void *kernel_3d_pk(int method, int cpl, int gzp, int cross);
// the general kernel (recon_gen.cuh): XY, Composite and Sliced LRFs, and axial LRFs that are not positive
// everywhere.  method 0/1/2, lrf_kind 1/3/4/5
const void *kernel_gen(int method, int lrf_kind);
// axial+z LRFs (recon3d.cuh).  method 0/1, (cpl, gzm) in {(1,1),(2,1),(3,1),(4,1),(8,1),(1,4),(2,4),(1,8),(2,8)}
const void *kernel_3d(int method, int cpl, int gzm);

// continuous refinement (refine.cuh), method 0/1/2
const void *kernel_refine(int method);

}  // namespace ants
