// recon3d.cuh -- contracting grids with axial+z LRFs s(r, z) (PAPER.md:394 section
// 6.1.2 "Axial+Z"; section 5.1.2.2): search over (x, y, z), or over
// (x, y) at a fixed z.
//
// Mapping: one warp per event; lanes over the G*G (ix, iy) COLUMNS of the grid
// (CPL columns per lane, column = lane + 32 j), the Gz z-levels of a column looped
// inside the lane (GZM = compiled maximum), sensors looped outermost with
// warp-broadcast shared-memory records.  The distance work (sqrt, knot interval,
// local coordinate) is done once per (column, sensor) and shared by the z-levels.
//
// Per iteration the warp contracts the tensor-product table with the cubic z-basis
// of every level (FP64, a few hundred FMAs) into per-level axial tables T_l[k]
// (per-interval cubics in r) and the differences dT_l = T_l - T_centre.  After that
// a node is an axial spline lookup, exactly as in recon2d.cuh:
//   plain        (coarse grids)  s = T_l[k](v); same log2-domain Poisson sum /
//                residual-form chi-square as the 2-D kernel.
//   differential (fine grids)    dL = [T_l(r) - T_l(r0)] + dT_l(r0): Taylor form of
//                T_l about the centre radius plus the cubic jump at an adjacent r-knot,
//                plus the exactly contracted z-difference at the centre radius.
//                Poisson uses S log1p(dL/L0): degree-6 series when |dL/L0| <= 0.1 on all of a sensor's
//                nodes, lg2(1 + dL/L0) for that sensor otherwise (one warp vote per sensor).
// The reported score and energy are one FP64 evaluation at the final node.
#pragma once
#include "../../include/ants_recon.h"
#include "recon2d.cuh"
#include "recon2d_pk.cuh"

namespace ants {

struct WarpSmem3D {
    float4 *A, *B, *C, *E;   // [N] per-sensor records of the current iteration
    float4 *D;               // [Gz][N] per (level, sensor): {d1, d2, d3, e} (scaled)
    float2 *J;               // [Gz][N] per (level, sensor): cubic jumps {up, down} (scaled)
    float4 *T;               // [Gz][n_r + 1] level tables
    float4 *dT;              // [Gz][n_r + 1] T_l - T_c
    float4 *Tc;              // [n_r + 1] centre-z table
    float2 *SC;              // [N] {S_i (prepared), log2(S_i / g_i) or 0}
};

__host__ __device__ inline size_t warp_smem_bytes_3d(int N, int Gz, int nr1) {
    size_t b = (size_t)N * (4 * 16 + 8) + (size_t)Gz * N * (16 + 8) + (size_t)(2 * Gz + 1) * nr1 * 16;
    return (b + 15) / 16 * 16;
}

__device__ __forceinline__ WarpSmem3D carve_3d(unsigned char *base, int N, int Gz, int nr1) {
    WarpSmem3D w;
    w.A = reinterpret_cast<float4 *>(base);
    w.B = w.A + N;
    w.C = w.B + N;
    w.E = w.C + N;
    w.D = w.E + N;
    w.T = w.D + (size_t)Gz * N;
    w.dT = w.T + (size_t)Gz * nr1;
    w.Tc = w.dT + (size_t)Gz * nr1;
    w.J = reinterpret_cast<float2 *>(w.Tc + nr1);
    w.SC = w.J + (size_t)Gz * N;
    return w;
}

// cubic B-spline z-basis in FP64: interval kz and the four weights of coefficients kz..kz+3
__device__ __forceinline__ void zbasis(const ModelDev &m, double sczd, float z, int &kz, double b[4]) {
    double t = ((double)z - (double)m.z_lo) * sczd;
    t = fmin(fmax(t, 0.0), (double)m.n_z);
    kz = min((int)t, m.n_z - 1);
    const double u = t - (double)kz, u2 = u * u, u3 = u2 * u, o = 1.0 - u;
    b[0] = o * o * o * (1.0 / 6.0);
    b[1] = (3.0 * u3 - 6.0 * u2 + 4.0) * (1.0 / 6.0);
    b[2] = (-3.0 * u3 + 3.0 * u2 + 3.0 * u + 1.0) * (1.0 / 6.0);
    b[3] = u3 * (1.0 / 6.0);
}

// ---- FP64 evaluation of (A, score) at the final node (step a6) ----------------
template <int METHOD>
__device__ void final_score_3d(const ModelDev &m, const float4 *sens_s, const WarpSmem3D &w, int lane,
                               double sczd, float cx, float cy, float cz, float &A_out, float &score_out) {
    double *Ld = reinterpret_cast<double *>(w.A);
    const double r_lo = (double)m.r_lo, r_hi = (double)m.r_hi;
    const double hstep = (r_hi - r_lo) / (double)m.n_r;
    int kz;
    double bz[4];
    zbasis(m, sczd, cz, kz, bz);
    double sumL = 0.0, sumS = 0.0, swsl = 0.0, swll = 0.0;
    __syncwarp();
    for (int i = lane; i < m.N; i += 32) {
        Ld[i] = 0.0;
        if (!(w.SC[i].y == w.SC[i].y)) continue;            // R19: inactive sensor
        float4 sn = sens_s[i];
        double dx = (double)cx - (double)sn.x, dy = (double)cy - (double)sn.y;
        double r = sqrt(dx * dx + dy * dy);
        double rc = fmin(fmax(r, r_lo), r_hi);
        double t = (rc - r_lo) / hstep;
        int k = min(max((int)floor(t), 0), m.n_r - 1);
        double u = t - (double)k, s = 0.0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double *p = m.polyd + ((size_t)(kz + b) * m.n_r + k) * 4;
            s += bz[b] * (p[0] + u * (p[1] + u * (p[2] + u * p[3])));
        }
        double L = (double)sn.z * s;
        double S = (double)w.SC[i].x;
        Ld[i] = L;
        sumL += L;
        sumS += S;
        if (METHOD == 1) {
            double wi = 1.0 / fmax(S, 1.0);
            swsl += wi * S * L;
            swll += wi * L * L;
        }
    }
    sumL = warp_sum(sumL);
    sumS = warp_sum(sumS);
    __syncwarp();
    double A, sc = 0.0;
    bool bad = !(sumL > 0.0) || !(cz >= m.z_lo && cz <= m.z_hi);
    if (METHOD == 0) {
        A = sumS / sumL;
        for (int i = lane; i < m.N; i += 32) {
            if (!(w.SC[i].y == w.SC[i].y)) continue;
            double L = Ld[i], S = (double)w.SC[i].x, mu = A * L;
            if (S > 0.0) {
                if (!(L > 0.0)) bad = true;
                else sc += mu - S - S * log(mu / S);
            } else {
                sc += mu;
            }
        }
        sc = 2.0 * warp_sum(sc);
    } else {
        swsl = warp_sum(swsl);
        swll = warp_sum(swll);
        if (!(swll > 0.0)) bad = true;
        A = swsl / swll;
        for (int i = lane; i < m.N; i += 32) {
            if (!(w.SC[i].y == w.SC[i].y)) continue;
            double L = Ld[i], S = (double)w.SC[i].x;
            double d = S - A * L;
            sc += d * d / fmax(S, 1.0);
        }
        sc = warp_sum(sc);
    }
    bad = __any_sync(kFull, bad);
    A_out = bad ? __int_as_float(0x7fc00000) : (float)A;
    score_out = bad ? kInf : (float)sc;
    __syncwarp();
}

// ---- per-iteration level tables (FP64 z-contraction of the coefficient rows) ----
// T_l[k] = sum_b bz_b(z_l) rows[kz_l + b][k];  dT_l = T_l - T_c (exact to FP64 rounding);  Tc[k].
__device__ __forceinline__ void build_level_tables(const ModelDev &m, const float4 *poly_s, const WarpSmem3D &w,
                                                   int lane, double sczd, int Gz, float cz, float hz, float halfz) {
    const int nr1 = m.n_r + 1;
    int kzc;
    double bc[4];
    zbasis(m, sczd, cz, kzc, bc);
    for (int it = lane; it < Gz * nr1; it += 32) {
        const int l = it / nr1, k = it - l * nr1;
        const float zl = fmaf((float)l - halfz, hz, cz);
        int kzl;
        double bl[4];
        zbasis(m, sczd, zl, kzl, bl);
        double tl[4] = {0, 0, 0, 0}, tc[4] = {0, 0, 0, 0};
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const float4 r1 = poly_s[(kzl + b) * nr1 + k], r2 = poly_s[(kzc + b) * nr1 + k];
            tl[0] += bl[b] * (double)r1.x; tl[1] += bl[b] * (double)r1.y;
            tl[2] += bl[b] * (double)r1.z; tl[3] += bl[b] * (double)r1.w;
            tc[0] += bc[b] * (double)r2.x; tc[1] += bc[b] * (double)r2.y;
            tc[2] += bc[b] * (double)r2.z; tc[3] += bc[b] * (double)r2.w;
        }
        w.T[it] = make_float4((float)tl[0], (float)tl[1], (float)tl[2], (float)tl[3]);
        w.dT[it] = make_float4((float)(tl[0] - tc[0]), (float)(tl[1] - tc[1]), (float)(tl[2] - tc[2]),
                               (float)(tl[3] - tc[3]));
        if (l == 0) w.Tc[k] = make_float4((float)tc[0], (float)tc[1], (float)tc[2], (float)tc[3]);
    }
    __syncwarp();
}

}  // namespace ants

#include "recon3d_kernel.cuh"
