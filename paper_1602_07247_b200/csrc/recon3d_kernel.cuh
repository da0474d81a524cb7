// recon3d_kernel.cuh -- the axial+z kernel (included by recon3d.cuh, which documents the mapping).
#pragma once

namespace ants {

// CPL columns per lane, GZM compiled maximum of z-levels, METHOD 0 Poisson ML / 1 weighted chi-square.
template <int CPL, int GZM, int METHOD>
__global__ void __launch_bounds__(256) recon3d_kernel(const Params p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = p.m;
    const int N = m.N, nr1 = m.n_r + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Gz = p.dim == 3 ? p.G : 1;
    const int ncol = p.G * p.G;
    const int rows = (m.n_z + 3) * nr1;
    const double sczd = (double)m.n_z / ((double)m.z_hi - (double)m.z_lo);

    // CTA-shared tables: sensor records and the per-z-coefficient spline rows
    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *poly_s = sens_s + N;
    for (int i = threadIdx.x; i < N; i += blockDim.x) sens_s[i] = m.sens[i];
    for (int i = threadIdx.x; i < rows; i += blockDim.x) poly_s[i] = m.poly[i];
    __syncthreads();
    WarpSmem3D w = carve_3d(smem + (size_t)(N + rows) * 16 + (size_t)warp * warp_smem_bytes_3d(N, Gz, nr1), N, Gz, nr1);

    // this lane's columns: offsets from the grid centre in units of the step
    const float half = 0.5f * (float)(p.G - 1);
    const float halfz = p.dim == 3 ? half : 0.f;
    float fx[CPL], fy[CPL];
    bool cv[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) {
        int c = lane + 32 * j;
        cv[j] = c < ncol;
        int iy = c / p.G, ix = c - iy * p.G;
        fx[j] = cv[j] ? (float)ix - half : 0.f;
        fy[j] = cv[j] ? (float)iy - half : 0.f;
    }
    const float half_diag_units = 1.41421356f * half;
    const float z_start = (p.z_seed == p.z_seed) ? p.z_seed : 0.5f * (m.z_lo + m.z_hi);   // R10

    long long e_next = grab_event(p.ctr, lane);
    for (long long e = e_next; e < p.n_events; e = e_next) {
        e_next = grab_event(p.ctr, lane);
        // ---- a1: signals, centroid / strongest-sensor start, selection (prepare_event, recon_common.cuh) ----
        float sumS, cx, cy;
        if (!prepare_event<METHOD>(p, sens_s, w.SC, e, lane, sumS, cx, cy)) continue;
        float cz = z_start, A_ref = 1.f;

        float h = p.h0_xy, hz = p.h0_z;
        for (int k = 0; k < p.K; ++k) {
            build_level_tables(m, poly_s, w, lane, sczd, Gz, cz, hz, halfz);
            if (k == 0) {
                // reference energy for the plain score: A at the seed
                float sl = 0.f;
                for (int i = lane; i < N; i += 32) {
                    float4 sn = sens_s[i];
                    float dx = cx - sn.x, dy = cy - sn.y;
                    float t = fminf(fmaxf(fmaf(sqrtf(fmaf(dx, dx, dy * dy)), m.sc, m.of), -0.5f), m.tmax);
                    int kk;
                    float v;
                    split_t(t, kk, v);
                    if (w.SC[i].y == w.SC[i].y) sl = fmaf(sn.z, horner(w.Tc[kk], v), sl);
                }
                sl = warp_sum(sl);
                A_ref = sl > 0.f ? sumS / sl : 1.f;
            }
            const bool centre_ok = cz >= m.z_lo && cz <= m.z_hi;
            float sc_node[CPL][GZM];       // node scores (lower is better), +inf = invalid
            float aux_node[CPL][GZM];      // plain mode: sum L (Poisson) / A (chi2) at the node
            const bool plain = k < p.k_diff || !centre_ok;
            if (plain) {
#include "recon3d_plain.inc"
            } else {
#include "recon3d_diff.inc"
            }

            // ---- a5: argmin over the G^2 * Gz nodes, recentre, contract ----
            // node code (l << 10) | column keeps the order of the linear index l * G^2 + column (R9)
            float bs = kInf;
            int bi = 0x7fffffff;
#pragma unroll
            for (int l = 0; l < GZM; ++l)
#pragma unroll
                for (int j = 0; j < CPL; ++j)
                    if (sc_node[j][l] < bs) { bs = sc_node[j][l]; bi = (l << 10) | (lane + 32 * j); }
            warp_argmin_redux(bs, bi);
            const bool found = bs < kInf;
            const int wl = bi >> 10, wc = bi & 1023;
            if (found) {
                // the winner's column offsets (and, in plain mode, its energy) live in the owner lane
                float wx = 0.f, wy = 0.f, mine = 0.f;
#pragma unroll
                for (int j = 0; j < CPL; ++j)
                    if ((wc >> 5) == j) {
                        wx = fx[j];
                        wy = fy[j];
#pragma unroll
                        for (int ll = 0; ll < GZM; ++ll)
                            if (ll == wl) mine = aux_node[j][ll];
                    }
                if (plain) {
                    float v = __shfl_sync(kFull, mine, wc & 31);
                    A_ref = METHOD == 0 ? sumS / v : v;
                }
                cx = fmaf(__shfl_sync(kFull, wx, wc & 31), h, cx);
                cy = fmaf(__shfl_sync(kFull, wy, wc & 31), h, cy);
                cz = fmaf((float)wl - halfz, hz, cz);
            }
            if (p.out_path && lane == 0)
                p.out_path[e * p.K + k] = found ? (uint16_t)(wl * ncol + wc) : (uint16_t)0xFFFF;
            h *= p.factor;
            hz *= p.factor;
            __syncwarp();
        }

        // ---- a6: FP64 energy and score at the final node, store ----
        float A_fin, score_fin;
        final_score_3d<METHOD>(m, sens_s, w, lane, sczd, cx, cy, cz, A_fin, score_fin);
        if (lane == 0) {
            reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(cx, cy, cz, A_fin);
            p.out_score[e] = score_fin;
        }
    }
    retire_warp(p.ctr, p.total_warps, lane);
}

}  // namespace ants
