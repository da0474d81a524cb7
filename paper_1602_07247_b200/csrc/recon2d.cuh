// recon2d.cuh -- pieces shared by the axial (x, y) kernels (section 5.1.2.2; PAPER.md:388
// "Axial"): spline look-ups from the per-interval tables and the FP64 final score.  The kernels are
// recon2d_pk.cuh (strictly positive LRFs, packed) and recon_gen.cuh (everything else).
//
// Mapping of the kernels: one warp per event, lanes over grid nodes (node = lane + 32 j, linear index
// iy*G + ix), sensors looped inside with warp-broadcast shared-memory records; persistent CTAs.
//
// Two score formulations, both FP32 and exact rewrites of the same node score
// (DESIGN.md "Kernels"):
//   plain        (coarse grids)  spline looked up per (node, sensor);
//                Poisson: sum_i S_i (c_i - log2 s_i) + sumS log2(A_ref sumL / sumS),
//                         c_i = log2(S_i / (A_ref g_i));
//                chi2:    sum w d^2 - (sum w d L)^2 / sum w L^2, d = S - A_ref L.
//   differential (fine grids, k >= k_diff)  score minus the score at the grid
//                centre from dL_i = L_i(node) - L_i(centre), computed from
//                dr = (2 d0.delta + |delta|^2)/(r + r0) and the Taylor form of the
//                cubic at the centre plus the cubic jump at an adjacent knot.
// The reported score and energy are one FP64 evaluation at the final node.
#pragma once
#include <type_traits>

#include "recon_common.cuh"

namespace ants {

// ---- per-warp shared-memory view -------------------------------------------
struct WarpSmem2D {
    float4 *A, *B, *C, *D, *E;   // [N] each: per-sensor records of the current iteration
    float2 *SC;                  // [N] {S_i (prepared), log2(S_i / g_i) or 0}
};

__host__ __device__ inline size_t warp_smem_bytes_2d(int N) { return ((size_t)N * (5 * 16 + 8) + 15) / 16 * 16; }

__device__ __forceinline__ WarpSmem2D carve_2d(unsigned char *base, int N) {
    WarpSmem2D w;
    w.A = reinterpret_cast<float4 *>(base);
    w.B = w.A + N;
    w.C = w.B + N;
    w.D = w.C + N;
    w.E = w.D + N;
    w.SC = reinterpret_cast<float2 *>(w.E + N);
    return w;
}

// one plain spline evaluation s_m(i)(r) (no gain) from the shared-memory table
__device__ __forceinline__ float eval_axial(const ModelDev &m, const float4 *row, float r) {
    float t = fminf(fmaxf(fmaf(r, m.sc, m.of), -0.5f), m.tmax);
    int k;
    float v;
    split_t(t, k, v);
    return horner(row[k], v);
}

// spline s_m(i) at the grid centre, split so that the Taylor coefficients can follow:
// returns s0 and the interval row q, local coordinate v0 (in [-0.5, 0.5], the last
// interval takes r = r_hi as v0 = +0.5) and clamped radius r0c
__device__ __forceinline__ float centre_eval(const ModelDev &m, const float4 *row, float r0,
                                             int &k0, float &v0, float &r0c, float4 &q) {
    r0c = fminf(fmaxf(r0, m.r_lo), m.r_hi);
    float t0 = fminf(fmaxf(fmaf(r0c, m.sc, m.of), -0.5f), m.tmax);
    split_t(t0, k0, v0);
    if (k0 >= m.n_r) { k0 = m.n_r - 1; v0 += 1.0f; }
    q = row[k0];
    return horner(q, v0);
}

// ---- FP64 evaluation of (A, score) at the final node (step a6) --------------
// Follows the definitions directly: Poisson A = sumS/sumL, D = 2 sum[mu - S - S ln(mu/S)];
// chi2 w = 1/max(S,1), A = sum wSL / sum wLL, chi2 = sum w (S - A L)^2.
template <int METHOD>
__device__ void final_score_2d(const ModelDev &m, const float4 *sens_s, const int *grp_s, const WarpSmem2D &w, int lane,
                               float cx, float cy, float &A_out, float &score_out) {
    double *Ld = reinterpret_cast<double *>(w.A);
    const double r_lo = (double)m.r_lo, r_hi = (double)m.r_hi;
    const double hstep = (r_hi - r_lo) / (double)m.n_r;
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
        double u = t - (double)k;
        const double *p = m.polyd + ((size_t)grp_s[i] * m.n_r + k) * 4;
        double s = p[0] + u * (p[1] + u * (p[2] + u * p[3]));
        double L = (double)sn.z * s;
        double S = (double)w.SC[i].x;
        Ld[i] = L;
        sumL += L;
        sumS += S;
        if (METHOD >= 1) {
            double wi = 1.0 / fmax(S, 1.0);
            swsl += wi * S * L;
            swll += wi * L * L;
        }
    }
    sumL = warp_sum(sumL);
    sumS = warp_sum(sumS);
    __syncwarp();
    double A, sc = 0.0;
    bool bad = !(sumL > 0.0);
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
        A = METHOD == 2 ? sumS / sumL : swsl / swll;          // R27 / R3
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

}  // namespace ants
