// recon2d_pk.cuh -- the axial (x, y) contracting-grid kernel for strictly positive LRFs, with the
// per-(node, sensor) arithmetic PACKED over sensor pairs (section 5.1.2.2).
//
// Same mapping and the same two score formulations as recon2d.cuh (one warp per event, lanes over
// grid nodes, NPT nodes per lane; plain score on coarse grids, differential score on fine grids), but
// every FP32 add/mul/fma of the inner loops works on TWO sensors at once in a 64-bit register pair
// (fma.rn.f32x2 -> FFMA2: one issue slot, two lanes of FMA work).  The first kernel was issue-bound
// (profiles/r01_ncu_first.md: 80 % issue-slot use at 46 % FMA-pipe use); packing halves the issue
// slots of the FMA-pipe work, which leaves the two MUFU ops per pair (16 lanes/clk/SM) and the FMA
// pipe itself (~15 FMA-pipe lane-ops per pair) as the bound.
//
// Per-iteration sensor records are stored pair-interleaved, float4 {even, odd, even, odd}, so that an
// LDS.128 lands two packed operands in aligned register pairs.  A pad sensor (S = 0, L0 = 0, g = 0)
// completes an odd count; it contributes exactly 0 to every sum.
#pragma once
#include "recon2d.cuh"

namespace ants {

constexpr int kPkArrays = 9;    // D0..D7 and, for the least-squares methods, E0 (float4 [Np + 1] each)

struct WarpSmemPk {
    float4 *D[kPkArrays];   // per-pair records of the current iteration (plain mode uses D[0] only)
    float2 *SC;             // [N] {S_i (prepared), log2(S_i / g_i) or 0}
    float *S0, *S1;         // [nodes] node scores of the previous and of the current iteration (node reuse)
    unsigned char *L;       // [nodes] the nodes that have to be evaluated in this iteration, compacted
};

__host__ __device__ inline int pk_pairs(int N) { return (N + 1) / 2 + 1; }   // +1: a pad on each list
__host__ __device__ inline size_t warp_smem_bytes_pk(int N, int method, int nodes) {
    const int narr = method == 0 ? 8 : kPkArrays;
    const size_t np4 = ((size_t)nodes + 3) / 4 * 4;
    return ((size_t)pk_pairs(N) * 16 * narr + ((size_t)N * 8 + 15) / 16 * 16 + np4 * 9 + 15) / 16 * 16;
}
// CTA-shared: sens_s [N] float4, poly_s [rows] float4, grp_s [N] int, node_s [P] float2 (grid offsets of the nodes in
// units of the step: a table look-up instead of an integer division wherever a lane needs its nodes; P = 32 x the
// nodes per lane, the excess zero), and the static node lists of the node-reuse kernel
// (recon2d_pk_kernel.cuh): ident_s, todo_s, even_s [P] u8, evoff_s [P] s16, three counters
__host__ __device__ inline size_t cta_smem_bytes_pk(int N, int rows, int npt) {
    return cta_table_bytes(N, rows) + (size_t)(32 * npt) * (8 + 3 + 2) + 16;
}

__device__ __forceinline__ WarpSmemPk carve_pk(unsigned char *base, int N, int method, int nodes) {
    WarpSmemPk w;
    const int np1 = pk_pairs(N), narr = method == 0 ? 8 : kPkArrays;
    float4 *f = reinterpret_cast<float4 *>(base);
    for (int a = 0; a < kPkArrays; ++a) w.D[a] = f + (size_t)(a < narr ? a : 0) * np1;
    w.SC = reinterpret_cast<float2 *>(f + (size_t)narr * np1);
    const size_t np4 = ((size_t)nodes + 3) / 4 * 4;
    w.S0 = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(w.SC) + ((size_t)N * 8 + 15) / 16 * 16);
    w.S1 = w.S0 + np4;
    w.L = reinterpret_cast<unsigned char *>(w.S1 + np4);
    return w;
}

// degree-6 series of log1p(q)/q (|q| <= 0.1: truncation q^7/7 <= 1.5e-8), packed
__device__ __forceinline__ f32x2 log1p_over_q2(f32x2 q) {
    return fma2(q, fma2(q, fma2(q, fma2(q, fma2(q, pk1(-1.f / 6.f), pk1(0.2f)), pk1(-0.25f)), pk1(1.f / 3.f)),
                        pk1(-0.5f)), pk1(1.f));
}
__device__ __forceinline__ float log1p_series(float q) {
    return q * fmaf(q, fmaf(q, fmaf(q, fmaf(q, fmaf(q, -1.f / 6.f, 0.2f), -0.25f), 1.f / 3.f), -0.5f), 1.f);
}

}  // namespace ants

#include "recon2d_pk_kernel.cuh"
