// recon3d_pk.cuh -- the (x, y, z) contracting-grid kernel for axial+z LRFs s(r, z) (section 6.1.2;
// PAPER.md:328 section 5.1.2.2) with the per-node arithmetic PACKED over PAIRS OF Z-LEVELS.
//
// Same mapping and the same two score formulations as recon3d.cuh (one warp per event, lanes over the G x G
// (ix, iy) columns, the z-levels of a column inside the lane so that the distance work is shared by the levels;
// plain score on coarse grids, differential score on fine ones), but two adjacent z-levels share one 64-bit
// register pair: every add/mul/fma of the level loops is one FFMA2/FADD2/FMUL2 for two nodes, with the
// column's scalars (local coordinate, du, cubic jumps) as broadcast operands.  The round-1 kernel was bound by
// issue slots (profiles/r02_kernel_mix.md: 29.6 thread-instructions per pair, FMA pipe 38 % busy); packing halves
// the issue slots of the level loops, which makes the FMA pipe the bound of the differential iterations.
//
// Per-iteration tables are stored level-pair-interleaved so that one LDS.128 lands two packed operands in
// aligned register pairs: T2[lp][k] = {x_l, x_l+1, y_l, y_l+1}, {z_l, z_l+1, w_l, w_l+1} (the per-level axial
// cubics of recon3d.cuh), D2[lp][i] = {d1, d1', d2, d2'}, {d3, d3', e, e'}, J2[lp][i] = {j_up, j_up', j_dn, j_dn'}.
// An odd number of levels is completed by a pad level whose tables are zero and whose nodes are invalid.
#pragma once
#include "recon3d.cuh"

namespace ants {

struct WarpSmem3Dpk {
    float4 *A, *B, *C, *E;   // [N] per-sensor records of the current iteration
    float4 *D2;              // [LP][N][2]
    float4 *J2;              // [LP][N]
    float4 *T2;              // [LP][n_r + 1][2] level-pair tables
    float4 *dT;              // [2 LP][n_r + 1] T_l - T_c (scalar layout: read by the record build only)
    float4 *Tc;              // [n_r + 1] centre-z table
    float *W;                // [2 LP + 1][16] z-basis weights of the levels (build_level_tables_pk)
    float2 *SC;              // [N]
};

// (the E records serve the chi-square differential score only)
__host__ __device__ inline size_t warp_smem_bytes_3dpk(int N, int LP, int nr1, int method) {
    // (the z-basis weights W are dead before the D2 records are written: they share that region)
    size_t d2 = (size_t)LP * N * 32, wz = (size_t)(2 * LP + 1) * 64;
    size_t b = (size_t)N * ((method == 0 ? 3 : 4) * 16 + 8) + (d2 > wz ? d2 : wz) + (size_t)LP * N * 16 +
               (size_t)LP * nr1 * 32 + (size_t)(2 * LP + 1) * nr1 * 16;
    return (b + 15) / 16 * 16;
}

__device__ __forceinline__ WarpSmem3Dpk carve_3dpk(unsigned char *base, int N, int LP, int nr1, int method) {
    WarpSmem3Dpk w;
    w.A = reinterpret_cast<float4 *>(base);
    w.B = w.A + N;
    w.C = w.B + N;
    w.E = w.C + (method == 0 ? 0 : N);
    w.D2 = w.E + N;
    const size_t d2 = (size_t)2 * LP * N, wz = (size_t)(2 * LP + 1) * 4;     // in float4 units
    w.J2 = w.D2 + (d2 > wz ? d2 : wz);
    w.T2 = w.J2 + (size_t)LP * N;
    w.dT = w.T2 + (size_t)2 * LP * nr1;
    w.Tc = w.dT + (size_t)2 * LP * nr1;
    w.W = reinterpret_cast<float *>(w.D2);
    w.SC = reinterpret_cast<float2 *>(w.Tc + nr1);
    return w;
}

// Level tables of one iteration.  T_l[k] = sum_b bz_b(z_l) rows[kz_l + b][k] (the r-cubics of the z-coefficient
// rows contracted with the cubic z-basis at the level), Tc the same at the grid centre, dT_l = T_l - Tc.  The basis
// weights are formed in FP64 -- for dT as the DIFFERENCE of the level's and the centre's weights on a common window
// of six rows, which is what keeps dT accurate relative to itself -- by one lane per level, rounded to float, and
// the contraction itself runs in FP32 over all lanes (no conversions in the loop).  On differential grids a level
// lies within one z-knot of the centre (host-checked), so the window rows kz_c - 1 .. kz_c + 4 cover both.
__device__ __forceinline__ void build_level_tables_pk(const ModelDev &m, const float4 *poly_s, const WarpSmem3Dpk &w,
                                                      int lane, double sczd, int Gz, int LP, float cz, float hz, float halfz,
                                                      bool need_dT) {
    const int nr1 = m.n_r + 1, n_rows = m.n_z + 3;
    float *W = w.W;                         // [2 LP + 1][16]: {kz0 (as int bits), -, wT[6], wD[6], -, -}
    if (lane <= 2 * LP) {
        int kzc;
        double bc[4];
        zbasis(m, sczd, cz, kzc, bc);
        float *dst = W + lane * 16;
        double wt[6] = {0, 0, 0, 0, 0, 0}, wd[6] = {0, 0, 0, 0, 0, 0};
        int kz0 = kzc;
        if (lane == 2 * LP) {               // the centre's own table
#pragma unroll
            for (int b = 0; b < 4; ++b) wt[b] = bc[b];
        } else if (lane < Gz) {
            const float zl = fmaf((float)lane - halfz, hz, cz);
            int kzl;
            double bl[4];
            zbasis(m, sczd, zl, kzl, bl);
            if (need_dT) {
                kz0 = kzc - 1;
                const int s = kzl - kz0;    // 0, 1 or 2
#pragma unroll
                for (int j = 0; j < 6; ++j) {
#pragma unroll
                    for (int b = 0; b < 4; ++b)
                        if (s + b == j) { wt[j] += bl[b]; wd[j] += bl[b]; }
                    if (j >= 1 && j <= 4) wd[j] -= bc[j - 1];
                }
            } else {
                kz0 = kzl;
#pragma unroll
                for (int b = 0; b < 4; ++b) wt[b] = bl[b];
            }
        }
        dst[0] = __int_as_float(kz0);
#pragma unroll
        for (int j = 0; j < 6; ++j) { dst[2 + j] = (float)wt[j]; dst[8 + j] = (float)wd[j]; }
    }
    __syncwarp();
    float *T2f = reinterpret_cast<float *>(w.T2);
    for (int it = lane; it < (2 * LP + 1) * nr1; it += 32) {
        const int l = it / nr1, k = it - l * nr1;
        const float *wl = W + l * 16;
        const int kz0 = __float_as_int(wl[0]);
        float4 t = make_float4(0.f, 0.f, 0.f, 0.f), d = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const float4 r = poly_s[min(max(kz0 + j, 0), n_rows - 1) * nr1 + k];     // weight 0 outside the table
            const float a = wl[2 + j], b = wl[8 + j];
            t.x = fmaf(a, r.x, t.x); t.y = fmaf(a, r.y, t.y); t.z = fmaf(a, r.z, t.z); t.w = fmaf(a, r.w, t.w);
            d.x = fmaf(b, r.x, d.x); d.y = fmaf(b, r.y, d.y); d.z = fmaf(b, r.z, d.z); d.w = fmaf(b, r.w, d.w);
        }
        if (l == 2 * LP) {
            w.Tc[k] = t;
        } else {
            // T2[lp][k]: floats {x_l, x_l', y_l, y_l', z_l, z_l', w_l, w_l'}
            float *dst = T2f + ((size_t)(l >> 1) * nr1 + k) * 8 + (l & 1);
            dst[0] = t.x;
            dst[2] = t.y;
            dst[4] = t.z;
            dst[6] = t.w;
            w.dT[it] = d;
        }
    }
    __syncwarp();
}

// one level's cubic row out of the pair layout
__device__ __forceinline__ float4 level_row(const WarpSmem3Dpk &w, int nr1, int l, int k) {
    const float *src = reinterpret_cast<const float *>(w.T2) + ((size_t)(l >> 1) * nr1 + k) * 8 + (l & 1);
    return make_float4(src[0], src[2], src[4], src[6]);
}

// CPL columns per lane, GZP level PAIRS of the grid ((Gz + 1) / 2), METHOD 0 Poisson ML / 1 weighted chi-square.
// CROSS (odd Gz, two columns per lane): the top level, which has no partner within its column, is packed ACROSS the
// lane's two columns -- one packed unit {column 0, column 1} at level Gz - 1 with the level's table entries as
// broadcast operands and the columns' scalars packed -- instead of one half-idle pair per column: 2 (Gz - 1) / 2 + 1
// packed units per sensor instead of Gz + 1 (7 x 7 x 7: seven instead of eight).  Its accumulators, scores and
// auxiliaries live in the [0][GZP - 1] entries of the per-(column, pair) arrays ([1][GZP - 1] is unused), half hl =
// column hl.  Without CROSS an odd Gz leaves the last half pair of every column idle.
template <int CPL, int GZP, int METHOD, bool CROSS = false>
__global__ void __launch_bounds__(256, 2) recon3d_pk_kernel(const Params p) {
    static_assert(!CROSS || CPL == 2, "the cross-column unit pairs the two columns of a lane");
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = p.m;
    const int N = m.N, nr1 = m.n_r + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Gz = p.G;
    constexpr int LP = GZP;                 // level pairs: the host picks the instantiation with GZP = (Gz + 1) / 2
    const int ncol = p.G * p.G;
    const int rows = (m.n_z + 3) * nr1;
    const double sczd = (double)m.n_z / ((double)m.z_hi - (double)m.z_lo);

    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *poly_s = sens_s + N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) sens_s[i] = m.sens[i];
    for (int i = threadIdx.x; i < rows; i += blockDim.x) poly_s[i] = m.poly[i];
    __syncthreads();
    WarpSmem3Dpk w = carve_3dpk(smem + (size_t)(N + rows) * 16 + (size_t)warp * warp_smem_bytes_3dpk(N, LP, nr1, METHOD),
                                N, LP, nr1, METHOD);
    const unsigned t2_base = (unsigned)__cvta_generic_to_shared(w.T2);

    const float half = 0.5f * (float)(p.G - 1);
    float fx[CPL], fy[CPL];
    bool cv[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) {
        const int c = lane + 32 * j;
        cv[j] = c < ncol;
        const int iy = c / p.G, ix = c - iy * p.G;
        fx[j] = cv[j] ? (float)ix - half : 0.f;
        fy[j] = cv[j] ? (float)iy - half : 0.f;
    }
    const float half_diag_units = 1.41421356f * half;
    const float z_start = (p.z_seed == p.z_seed) ? p.z_seed : 0.5f * (m.z_lo + m.z_hi);   // R10

    long long e_next = grab_event(p.ctr, lane);
    for (long long e = e_next; e < p.n_events; e = e_next) {
        e_next = grab_event(p.ctr, lane);
        // ---- a1: signals, centroid / strongest-sensor start, selection (recon_common.cuh) ----
        float sumS, cx, cy;
        if (!prepare_event<METHOD>(p, sens_s, w.SC, e, lane, sumS, cx, cy)) continue;
        float cz = z_start, A_ref = 1.f;

        float h = p.h0_xy, hz = p.h0_z;
        for (int k = 0; k < p.K; ++k) {
            const bool centre_ok = cz >= m.z_lo && cz <= m.z_hi;
            const bool plain = k < p.k_diff || !centre_ok;
            build_level_tables_pk(m, poly_s, w, lane, sczd, Gz, LP, cz, hz, half, !plain);
            if (k == 0) {
                // reference energy for the plain score: A at the seed
                float sl = 0.f;
                for (int i = lane; i < N; i += 32) {
                    const float4 sn = sens_s[i];
                    const float dx = cx - sn.x, dy = cy - sn.y;
                    const float t = fminf(fmaxf(fmaf(sqrtf(fmaf(dx, dx, dy * dy)), m.sc, m.of), -0.5f), m.tmax);
                    int kk;
                    float v;
                    split_t(t, kk, v);
                    if (w.SC[i].y == w.SC[i].y) sl = fmaf(sn.z, horner(w.Tc[kk], v), sl);
                }
                sl = warp_sum(sl);
                A_ref = sl > 0.f ? sumS / sl : 1.f;
            }
            f32x2 sc_node[CPL][GZP];       // node scores of a level pair (lower is better), +inf = invalid
            f32x2 aux_node[CPL][GZP];      // plain mode: sum L (Poisson) / A (chi2) at the nodes
            if (plain) {
#include "recon3d_pk_plain.inc"
            } else {
#include "recon3d_pk_diff.inc"
            }

            // ---- a5: argmin over the G^2 * Gz nodes, recentre, contract ----
            // node code (l << 10) | column keeps the order of the linear index l * G^2 + column (R9)
            float bs = kInf;
            int bi = 0x7fffffff;
#pragma unroll
            for (int lp = 0; lp < GZP; ++lp) {
                const bool cross = CROSS && lp == GZP - 1;       // (level Gz - 1: half hl is column hl)
#pragma unroll
                for (int hl = 0; hl < 2; ++hl)
#pragma unroll
                    for (int j = 0; j < (cross ? 1 : CPL); ++j) {
                        float s_lo, s_hi;
                        upk(sc_node[j][lp], s_lo, s_hi);
                        const float s = hl ? s_hi : s_lo;
                        const int code = cross ? ((2 * lp) << 10) | (lane + 32 * hl) : ((2 * lp + hl) << 10) | (lane + 32 * j);
                        if (s < bs) { bs = s; bi = code; }
                    }
            }
            warp_argmin_redux(bs, bi);
            const bool found = bs < kInf;
            const int wl = bi >> 10, wc = bi & 1023;
            if (found) {
                float wx = 0.f, wy = 0.f, mine = 0.f;
#pragma unroll
                for (int j = 0; j < CPL; ++j)
                    if ((wc >> 5) == j) {
                        wx = fx[j];
                        wy = fy[j];
#pragma unroll
                        for (int lp = 0; lp < (CROSS ? GZP - 1 : GZP); ++lp) {
                            float a_lo, a_hi;
                            upk(aux_node[j][lp], a_lo, a_hi);
                            if (2 * lp == wl) mine = a_lo;
                            if (2 * lp + 1 == wl) mine = a_hi;
                        }
                        if (CROSS) {
                            float a_c0, a_c1;
                            upk(aux_node[0][GZP - 1], a_c0, a_c1);
                            if (wl == 2 * (GZP - 1)) mine = j ? a_c1 : a_c0;
                        }
                    }
                if (plain) {
                    const float v = __shfl_sync(kFull, mine, wc & 31);
                    A_ref = METHOD == 0 ? sumS / v : v;
                }
                cx = fmaf(__shfl_sync(kFull, wx, wc & 31), h, cx);
                cy = fmaf(__shfl_sync(kFull, wy, wc & 31), h, cy);
                cz = fmaf((float)wl - half, hz, cz);
            }
            if (p.out_path && lane == 0)
                p.out_path[e * p.K + k] = found ? (uint16_t)(wl * ncol + wc) : (uint16_t)0xFFFF;
            h *= p.factor;
            hz *= p.factor;
            __syncwarp();
        }

        // ---- a6: FP64 energy and score at the final node, store ----
        float A_fin, score_fin;
        WarpSmem3D w3;                 // final_score_3d needs N doubles of scratch (A, B) and SC
        w3.A = w.A;
        w3.SC = w.SC;
        final_score_3d<METHOD>(m, sens_s, w3, lane, sczd, cx, cy, cz, A_fin, score_fin);
        if (lane == 0) {
            reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(cx, cy, cz, A_fin);
            p.out_score[e] = score_fin;
        }
    }
    retire_warp(p.ctr, p.total_warps, lane);
}

}  // namespace ants
