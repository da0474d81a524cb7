// recon2d.cuh -- contracting-grid reconstruction over (x, y) with axial LRFs
// (section 5.1.2.2; "Axial"; PAPER.md:306 centroid).
//
// Mapping: one warp per event, lanes over grid nodes (NPT nodes per lane,
// node = lane + 32 j, linear index iy*G + ix), sensors looped inside with
// warp-broadcast shared-memory records; persistent CTAs stride over events.
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

// ---- the kernel --------------------------------------------------------------
// METHOD 0 Poisson ML, 1 weighted chi-square.  POS: every LRF is strictly
// positive (checked on the host at create), so no (node, sensor) pair can be
// invalid and the per-pair sign test is compiled out.
template <int NPT, int METHOD, bool POS>
__global__ void __launch_bounds__(256) recon2d_kernel(const Params p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = p.m;
    const int N = m.N, nr1 = m.n_r + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows = m.n_lrf * nr1;

    // CTA-shared tables: sensor records, the spline rows, the sensors' table indices
    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *poly_s = sens_s + N;
    int *grp_s = reinterpret_cast<int *>(poly_s + rows);
    for (int i = threadIdx.x; i < N; i += blockDim.x) { sens_s[i] = m.sens[i]; grp_s[i] = m.grp[i]; }
    for (int i = threadIdx.x; i < rows; i += blockDim.x) poly_s[i] = m.poly[i];
    __syncthreads();
    WarpSmem2D w = carve_2d(smem + cta_table_bytes(N, rows) + (size_t)warp * warp_smem_bytes_2d(N), N);

    // this lane's nodes: offsets from the grid centre in units of the step (exact small numbers)
    const float half = 0.5f * (float)(p.G - 1);
    float fx[NPT], fy[NPT];
    bool nv[NPT];
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        int n = lane + 32 * j;
        nv[j] = n < p.nodes;
        int iy = n / p.G, ix = n - iy * p.G;
        fx[j] = nv[j] ? (float)ix - half : 0.f;
        fy[j] = nv[j] ? (float)iy - half : 0.f;
    }
    const float half_diag_units = 1.41421356f * half;   // farthest node from the centre, in steps

    long long e_next = grab_event(p.ctr, lane);
    for (long long e = e_next; e < p.n_events; e = e_next) {
        e_next = grab_event(p.ctr, lane);
        // ---- a1: load signals (coalesced), prepare, centroid ----
        const float *sig = p.signals + e * N;
        float sumS = 0.f, sw = 0.f, sxw = 0.f, syw = 0.f;
        bool finite = true;
        for (int i = lane; i < N; i += 32) {
            float S = __ldg(sig + i);
            finite = finite && (fabsf(S) <= 3.402823466e38f);
            if (METHOD == 0) S = fmaxf(S, 0.f);          // R18
            float4 sn = sens_s[i];
            float wgt = S * sn.w;
            sumS += S;
            sw += wgt;
            sxw = fmaf(sn.x, wgt, sxw);
            syw = fmaf(sn.y, wgt, syw);
            float cs = 0.f;
            if (METHOD == 0 && S > 0.f) cs = log2f(S * sn.w);
            w.SC[i] = make_float2(S, cs);
        }
        finite = __all_sync(kFull, finite);
        sumS = warp_sum(sumS);
        sw = warp_sum(sw);
        sxw = warp_sum(sxw);
        syw = warp_sum(syw);
        __syncwarp();
        if (!finite || !(sumS > 0.f) || (p.seed_mode == 0 && !(sw > 0.f))) {
            if (lane == 0) {
                const float qnan = __int_as_float(0x7fc00000);
                reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(qnan, qnan, qnan, qnan);
                p.out_score[e] = kInf;
            }
            if (p.out_path)
                for (int k = lane; k < p.K; k += 32) p.out_path[e * p.K + k] = 0xFFFF;
            continue;
        }
        float cx = sxw / sw, cy = syw / sw;
        if (p.seed_mode == 1) strongest_sensor(w.SC, sens_s, N, lane, cx, cy);    // R20

        // reference energy for the plain score: A at the seed
        float A_ref;
        {
            float sl = 0.f;
            for (int i = lane; i < N; i += 32) {
                float4 sn = sens_s[i];
                float dx = cx - sn.x, dy = cy - sn.y;
                float s = eval_axial(m, poly_s + grp_s[i] * nr1, sqrtf(fmaf(dx, dx, dy * dy)));
                sl += sn.z * s;
            }
            sl = warp_sum(sl);
            A_ref = sl > 0.f ? sumS / sl : 1.f;
        }

        float h = p.h0_xy;
        for (int k = 0; k < p.K; ++k) {
            float sc_node[NPT];          // node scores (lower is better), +inf = invalid
            float sumL_node[NPT];        // plain mode: sum L (Poisson) / A (chi2) at the node
            if (METHOD == 2 || k < p.k_diff) {
                // =================== plain iteration =========================
                const float lA = log2f(A_ref);
                for (int i = lane; i < N; i += 32) {
                    float4 sn = sens_s[i];
                    float2 sc2 = w.SC[i];
                    float fourth;
                    if (METHOD == 0) fourth = sc2.x > 0.f ? sc2.y - lA : 0.f;      // c_i
                    else fourth = 1.f / fmaxf(sc2.x, 1.f);                          // w_i
                    w.A[i] = make_float4(sn.x, sn.y, sc2.x, fourth);
                }
                __syncwarp();
                float x[NPT], y[NPT], a1[NPT], a2[NPT], a3[NPT], a4[NPT];
                bool bad[NPT];
#pragma unroll
                for (int j = 0; j < NPT; ++j) {
                    x[j] = fmaf(fx[j], h, cx);
                    y[j] = fmaf(fy[j], h, cy);
                    a1[j] = a2[j] = a3[j] = a4[j] = 0.f;
                    bad[j] = false;
                }
#pragma unroll 2
                for (int i = 0; i < N; ++i) {
                    const float4 a = w.A[i];
                    const float4 *row = poly_s + grp_s[i] * nr1;
                    const float g = sens_s[i].z;
#pragma unroll
                    for (int j = 0; j < NPT; ++j) {
                        float dx = x[j] - a.x, dy = y[j] - a.y;
                        float r = sqrt_approx(fmaf(dx, dx, dy * dy));
                        float t = fminf(fmaxf(fmaf(r, m.sc, m.of), -0.5f), m.tmax);
                        int kk;
                        float v;
                        split_t(t, kk, v);
                        float s = horner(row[kk], v);
                        if (METHOD == 0) {
                            if (!POS) {
                                bad[j] = bad[j] || (s <= 0.f && a.z > 0.f);
                                a2[j] = fmaf(g, s, a2[j]);
                                s = fmaxf(s, 1e-37f);
                            } else {
                                a2[j] = fmaf(g, s, a2[j]);
                            }
                            a1[j] = fmaf(a.z, a.w - lg2_approx(s), a1[j]);
                        } else {
                            float L = g * s;
                            float d = fmaf(-A_ref, L, a.z);
                            float wd = a.w * d;
                            a1[j] = fmaf(wd, d, a1[j]);
                            a2[j] = fmaf(wd, L, a2[j]);
                            a3[j] = fmaf(a.w * L, L, a3[j]);
                            if (!POS || METHOD == 2) a4[j] += L;
                        }
                    }
                }
#pragma unroll
                for (int j = 0; j < NPT; ++j) {
                    float sc;
                    if (METHOD == 0) {
                        // D/(2 ln 2) = sum S_i (c_i - log2 s_i) + sumS log2(A_ref sumL / sumS)
                        sc = fmaf(sumS, log2f(a2[j] * (A_ref / sumS)), a1[j]);
                        sumL_node[j] = a2[j];
                        if (!(a2[j] > 0.f) || bad[j]) sc = kInf;
                    } else if (METHOD == 1) {
                        // chi2 = sum w d^2 - (sum w d L)^2 / sum w L^2; A = A_ref + sum w d L / sum w L^2
                        sc = a1[j] - a2[j] * a2[j] / a3[j];
                        sumL_node[j] = A_ref + a2[j] / a3[j];
                        if (!(a3[j] > 0.f) || (!POS && !(a4[j] > 0.f))) sc = kInf;
                    } else {
                        // R27: A = sumS / sumL; chi2 = sum w (d - delta L)^2, delta = A - A_ref
                        const float An = sumS / a4[j], dl = An - A_ref;
                        sc = fmaf(dl, fmaf(dl, a3[j], -2.f * a2[j]), a1[j]);
                        sumL_node[j] = An;
                        if (!(a4[j] > 0.f)) sc = kInf;
                    }
                    if (!nv[j] || !(sc == sc)) sc = kInf;
                    sc_node[j] = sc;
                }
            } else {
                // =================== differential iteration ==================
                const float reach = half_diag_units * h * 1.001f;      // mm
                const float reach_u = reach * m.sc;
                float L0sum = 0.f, P0 = 0.f, Q0 = 0.f;
                int n_simple = 0, n_knot = 0;
                // pass 1 (chi2 only): A0 = P0/Q0 at the centre needs all sensors first
                float A0 = 0.f;
                if (METHOD >= 1) {
                    for (int i = lane; i < N; i += 32) {
                        float4 sn = sens_s[i];
                        float dx0 = cx - sn.x, dy0 = cy - sn.y;
                        int k0;
                        float v0, r0c;
                        float4 q;
                        float s0 = centre_eval(m, poly_s + grp_s[i] * nr1,
                                               sqrtf(fmaf(dx0, dx0, dy0 * dy0)), k0, v0, r0c, q);
                        float L0 = sn.z * s0;
                        float S = w.SC[i].x, wi = 1.f / fmaxf(S, 1.f);
                        P0 = fmaf(wi * S, L0, P0);
                        Q0 = fmaf(wi * L0, L0, Q0);
                    }
                    P0 = warp_sum(P0);
                    Q0 = warp_sum(Q0);
                    A0 = P0 / Q0;
                }
                for (int i0 = 0; i0 < N; i0 += 32) {
                    const int i = i0 + lane;
                    const bool act = i < N;
                    float4 rA = make_float4(0, 0, 0, 1e-30f), rB = make_float4(0, 0, 0, 0);
                    float4 rC = make_float4(0, 0, 0, 0), rD = make_float4(0, 0, 0, 0), rE = make_float4(0, 0, 0, 0);
                    bool knot = false;
                    if (act) {
                        float4 sn = sens_s[i];
                        float S = w.SC[i].x;
                        float g = sn.z;
                        float dx0 = cx - sn.x, dy0 = cy - sn.y;
                        float r0sq = fmaf(dx0, dx0, dy0 * dy0);
                        float r0 = sqrtf(r0sq);
                        const float4 *row = poly_s + grp_s[i] * nr1;
                        int k0;
                        float v0, r0c;
                        float4 q;
                        float s0 = centre_eval(m, row, r0, k0, v0, r0c, q);
                        float d1 = fmaf(v0, fmaf(3.f * q.w, v0, 2.f * q.z), q.y);
                        float d2 = fmaf(3.f * q.w, v0, q.z);
                        float d3 = q.w;
                        float j_up = (k0 + 1 <= m.n_r - 1) ? row[k0 + 1].w - q.w : 0.f;
                        float j_dn = (k0 >= 1) ? row[k0 - 1].w - q.w : 0.f;
                        float a_up = 0.5f - v0, a_dn = 0.5f + v0;
                        float lo_i = m.r_lo - r0, hi_i = m.r_hi - r0;
                        float off_i = (r0 - r0c) * m.sc;
                        if (hi_i < -reach || lo_i > reach) { d1 = d2 = d3 = j_up = j_dn = 0.f; }
                        knot = (a_up < reach_u && j_up != 0.f) || (a_dn < reach_u && j_dn != 0.f);
                        rA = make_float4(2.f * dx0, 2.f * dy0, r0sq, fmaxf(r0, 1e-30f));
                        if (METHOD == 0) {
                            float inv = 1.f / s0;
                            rB = make_float4(lo_i, hi_i, off_i, S);
                            rC = make_float4(d1 * inv, d2 * inv, d3 * inv, g * s0);
                            rD = make_float4(a_up, j_up * inv, a_dn, j_dn * inv);
                            L0sum += g * s0;
                        } else {
                            float wi = 1.f / fmaxf(S, 1.f);
                            float L0 = g * s0;
                            float res = fmaf(-A0, L0, S);
                            rB = make_float4(lo_i, hi_i, off_i, wi);
                            rC = make_float4(g * d1, g * d2, g * d3, 2.f * L0);
                            rD = make_float4(a_up, g * j_up, a_dn, g * j_dn);
                            rE = make_float4(wi * A0 * A0, -2.f * wi * A0 * res, wi * S, 0.f);
                        }
                    }
                    // compaction: sensors with no knot in reach fill from the front, the others from the back
                    unsigned mk = __ballot_sync(kFull, act && knot), ms = __ballot_sync(kFull, act && !knot);
                    unsigned lt = (1u << lane) - 1u;
                    if (act) {
                        int pos = knot ? (N - 1 - n_knot - __popc(mk & lt)) : (n_simple + __popc(ms & lt));
                        w.A[pos] = rA;
                        w.B[pos] = rB;
                        w.C[pos] = rC;
                        w.D[pos] = rD;
                        if (METHOD >= 1) w.E[pos] = rE;
                    }
                    n_knot += __popc(mk);
                    n_simple += __popc(ms);
                }
                if (METHOD == 0) L0sum = warp_sum(L0sum);
                __syncwarp();

                float ddx[NPT], ddy[NPT], dd2[NPT], a1[NPT], a2[NPT], a3[NPT];
#pragma unroll
                for (int j = 0; j < NPT; ++j) {
                    ddx[j] = fx[j] * h;
                    ddy[j] = fy[j] * h;
                    dd2[j] = fmaf(ddx[j], ddx[j], ddy[j] * ddy[j]);
                    a1[j] = a2[j] = a3[j] = 0.f;
                }
                // KNOT = false: simple list [0, n_simple); KNOT = true: knot list [N - n_knot, N)
                auto body = [&](int i, auto knot_tag) {
                    constexpr bool KNOT = decltype(knot_tag)::value;
                    const float4 a = w.A[i], b = w.B[i], c = w.C[i];
                    float4 d, ee;
                    if (KNOT) d = w.D[i];
                    if (METHOD >= 1) ee = w.E[i];
#pragma unroll
                    for (int j = 0; j < NPT; ++j) {
                        float num = fmaf(ddx[j], a.x, fmaf(ddy[j], a.y, dd2[j]));   // r^2 - r0^2, accurate
                        float r = sqrt_approx(fabsf(a.z + num));
                        float dr = num * rcp_approx(r + a.w);                       // r - r0
                        dr = fminf(fmaxf(dr, b.x), b.y);                            // clamp r to [r_lo, r_hi]
                        float du = fmaf(dr, m.sc, b.z);
                        float q = du * fmaf(du, fmaf(du, c.z, c.y), c.x);           // Taylor form about the centre
                        if (KNOT) {
                            float ou = fmaxf(du - d.x, 0.f), od = fminf(du + d.z, 0.f);
                            q = fmaf(d.y * ou, ou * ou, q);                          // cubic jump above
                            q = fmaf(d.w * od, od * od, q);                          // cubic jump below
                        }
                        if (METHOD == 0) {
                            // q = dL_i/L0_i; accumulate L0_i q and S_i log1p(q) (degree-6 series)
                            a2[j] = fmaf(c.w, q, a2[j]);
                            float hq = fmaf(q, fmaf(q, fmaf(q, fmaf(q, fmaf(q, -1.f / 6.f, 0.2f), -0.25f),
                                                            1.f / 3.f), -0.5f), 1.f);
                            a1[j] = fmaf(b.w * q, hq, a1[j]);
                        } else {
                            // q = dL_i
                            a1[j] = fmaf(q, fmaf(ee.x, q, ee.y), a1[j]);             // sum w dmu (dmu - 2 res)
                            a2[j] = fmaf(ee.z, q, a2[j]);                            // dP = sum w S dL
                            a3[j] = fmaf(b.w * q, c.w + q, a3[j]);                   // dQ = sum w dL (2 L0 + dL)
                        }
                    }
                };
                for (int i = 0; i < n_simple; ++i) body(i, std::false_type{});
                for (int i = N - n_knot; i < N; ++i) body(i, std::true_type{});
#pragma unroll
                for (int j = 0; j < NPT; ++j) {
                    float sc;
                    if (METHOD == 0) {
                        // (D - D_centre)/2 = sumS log1p(sum dL / sum L0) - sum S_i log1p(q_i)
                        float ratio = a2[j] / L0sum;
                        sc = fmaf(sumS, log1pf(ratio), -a1[j]);
                        if (!(ratio > -1.f)) sc = kInf;
                    } else {
                        // chi2 - chi2_centre = Q0 (T - dP^2/Q0) / (Q0 + dQ)
                        float den = Q0 + a3[j];
                        sc = (a1[j] - a2[j] * a2[j] / Q0) * (Q0 / den);
                        if (!(den > 0.f)) sc = kInf;
                    }
                    if (!nv[j] || !(sc == sc)) sc = kInf;
                    sc_node[j] = sc;
                    sumL_node[j] = 0.f;
                }
            }

            // ---- a5: argmin over the G^2 nodes, recentre, contract ------------
            float bs = kInf;
            int bi = 0x7fffffff;
#pragma unroll
            for (int j = 0; j < NPT; ++j)
                if (sc_node[j] < bs) { bs = sc_node[j]; bi = lane + 32 * j; }
            warp_argmin(bs, bi);
            const bool found = bs < kInf;
            if (found) {
                if (METHOD == 2 || k < p.k_diff) {
                    float mine = 0.f;
#pragma unroll
                    for (int j = 0; j < NPT; ++j)
                        if ((bi >> 5) == j) mine = sumL_node[j];
                    float v = __shfl_sync(kFull, mine, bi & 31);
                    A_ref = METHOD == 0 ? sumS / v : v;
                }
                int iy = bi / p.G, ix = bi - iy * p.G;
                cx = fmaf((float)ix - half, h, cx);
                cy = fmaf((float)iy - half, h, cy);
            }
            if (p.out_path && lane == 0) p.out_path[e * p.K + k] = found ? (uint16_t)bi : (uint16_t)0xFFFF;
            h *= p.factor;
            __syncwarp();
        }

        // ---- a6: FP64 energy and score at the final node, store --------------
        float A_fin, score_fin;
        final_score_2d<METHOD>(m, sens_s, grp_s, w, lane, cx, cy, A_fin, score_fin);
        if (lane == 0) {
            reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(cx, cy, 0.f, A_fin);
            p.out_score[e] = score_fin;
        }
    }
    retire_warp(p.ctr, p.total_warps, lane);
}

}  // namespace ants
