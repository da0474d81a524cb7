// refine.cuh -- continuous refinement of reconstructed positions (include/ants_recon.h, ants_refine; DESIGN.md
// R34): the gradient-based minimisation "versus two (XY) or three (XYZ) spatial coordinates" that Minuit2
// performs in ANTS2, started from a contracting-grid result.  Levenberg-Marquardt with
// Nielsen's damping update on the node score with the energy eliminated by its closed form; analytic spline
// derivatives; every LRF parameterisation.
//
// Mapping: one warp per event, LANES OVER SENSORS (one evaluation of F, g, H costs N LRF evaluations with
// derivatives -- 1/G^d of a grid iteration), everything in FP64: B200 runs DFMA at half the FP32 rate
// (profiles/r02_fp32_peak.md) and a step is a few hundred DFMA per lane, so the whole refinement costs about as
// much as one FP32 grid iteration and needs none of the centre-relative algebra the FP32 grid scores need.  The LM
// bookkeeping is computed redundantly by all lanes from warp-reduced sums, so no lane diverges.
#pragma once
#include "recon_gen.cuh"

namespace ants {

struct RefineParams {
    ModelDev m;
    const float *signals;   // [E][N]
    long long n_events;
    float *xyzA;            // [E][4] in: start position; out: refined position and its energy
    float *score;           // [E] out
    int dim;                // 2: (x, y); 3: (x, y, z)
    int seed_mode, n_steps;
    int dtab;               // a double copy of the XY coefficients sits in shared memory
    // fields prepare_event reads through a Params view
    unsigned long long *ctr;
    int total_warps;
};

template <typename T>
__device__ __forceinline__ void dbasis4(T f, T d[4]) {
    const T o = T(1) - f;
    d[0] = -o * o * T(0.5);
    d[1] = (T(9) * f * f - T(12) * f) * T(1.0 / 6.0);
    d[2] = (T(-9) * f * f + T(6) * f + T(3)) * T(1.0 / 6.0);
    d[3] = f * f * T(0.5);
}

// tensor-product spline value and partial derivatives (per unit of the local coordinates) from c [.][nu3]
template <typename TC>
__device__ __forceinline__ double xy_value_grad(const TC *c, int nu3, int ku, int kv, const double bu[4],
                                                const double bv[4], const double du[4], const double dv[4],
                                                double &s_u, double &s_v) {
    const TC *q = c + kv * nu3 + ku;
    double s = 0.0;
    s_u = s_v = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const double c0 = (double)q[0], c1 = (double)q[1], c2 = (double)q[2], c3 = (double)q[3];
        const double row = c0 * bu[0] + c1 * bu[1] + c2 * bu[2] + c3 * bu[3];
        const double drow = c0 * du[0] + c1 * du[1] + c2 * du[2] + c3 * du[3];
        s += row * bv[b];
        s_u += drow * bv[b];
        s_v += row * dv[b];
        q += nu3;
    }
    return s;
}

// L_i / gL_i and its gradient with respect to (x, y, z), FP64, any parameterisation
static __device__ double lrf_value_grad(const ModelDev &m, const float *cxy_s, const double *cxyd_s, const float4 sn, const float4 xf, int tab,
                                 double x, double y, double z, double grad[3]) {
    const double dx = x - (double)sn.x, dy = y - (double)sn.y;
    double s = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    const int kind = m.lrf_kind;
    if (kind == kAxial || kind == kComposite || kind == kAxialZ) {
        const double r = sqrt(dx * dx + dy * dy);
        const double ex = r > 0.0 ? dx / r : 0.0, ey = r > 0.0 ? dy / r : 0.0;
        const double r_lo = (double)m.r_lo, r_hi = (double)m.r_hi;
        const double sc = (double)m.n_r / (r_hi - r_lo);
        const double rc = fmin(fmax(r, r_lo), r_hi);
        const double t = (rc - r_lo) * sc;
        const int k = min(max((int)t, 0), m.n_r - 1);
        const double u = t - (double)k;
        const bool inside = r >= r_lo && r <= r_hi;
        if (kind == kAxialZ) {
            const double z_lo = (double)m.z_lo, z_hi = (double)m.z_hi;
            const double scz = (double)m.n_z / (z_hi - z_lo);
            const double zc = fmin(fmax(z, z_lo), z_hi);
            const double tz = (zc - z_lo) * scz;
            const int kz = min(max((int)tz, 0), m.n_z - 1);
            const double fz = tz - (double)kz;
            double bz[4], dz[4];
            basis4<double>(fz, bz);
            dbasis4<double>(fz, dz);
            double sr = 0.0, sz = 0.0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const double *p = m.polyd + ((size_t)(kz + b) * m.n_r + k) * 4;
                const double f = p[0] + u * (p[1] + u * (p[2] + u * p[3]));
                const double d = p[1] + u * (2.0 * p[2] + 3.0 * u * p[3]);
                s += bz[b] * f;
                sr += bz[b] * d;
                sz += dz[b] * f;
            }
            sr = inside ? sr * sc : 0.0;
            gx += sr * ex;
            gy += sr * ey;
            gz += (z >= z_lo && z <= z_hi) ? sz * scz : 0.0;
        } else {
            const double *p = m.polyd + ((size_t)tab * m.n_r + k) * 4;
            s += p[0] + u * (p[1] + u * (p[2] + u * p[3]));
            const double ds = inside ? (p[1] + u * (2.0 * p[2] + 3.0 * u * p[3])) * sc : 0.0;
            gx += ds * ex;
            gy += ds * ey;
        }
    }
    if (kind >= kXY) {
        const double T0 = (double)xf.x, T1 = (double)xf.y, T2 = (double)xf.z, T3 = (double)xf.w;
        const double u = T0 * dx + T1 * dy, v = T2 * dx + T3 * dy;
        int ku, kv;
        double fu, fv, bu[4], bv[4], du[4], dv[4];
        locate(u, (double)m.u_lo, (double)m.su, m.nx, ku, fu);
        locate(v, (double)m.v_lo, (double)m.sv, m.ny, kv, fv);
        basis4<double>(fu, bu);
        basis4<double>(fv, bv);
        dbasis4<double>(fu, du);
        dbasis4<double>(fv, dv);
        const double u_hi = (double)m.u_lo + (double)m.nx / (double)m.su, v_hi = (double)m.v_lo + (double)m.ny / (double)m.sv;
        const double ku_in = (u >= (double)m.u_lo && u <= u_hi) ? (double)m.su : 0.0;     // a clamped coordinate: zero slope
        const double kv_in = (v >= (double)m.v_lo && v <= v_hi) ? (double)m.sv : 0.0;
        const int nu3 = m.nx + 3, per_plane = nu3 * (m.ny + 3);
        double val, su, sv;
        if (kind == kSliced) {
            const double z_lo = (double)m.z_lo, z_hi = (double)m.z_hi;
            const double dzp = (z_hi - z_lo) / (double)(m.n_planes - 1);
            const double zc = fmin(fmax(z, z_lo), z_hi);
            const int pz = min(max((int)floor((zc - z_lo) / dzp), 0), m.n_planes - 2);
            const double w = (zc - (z_lo + (double)pz * dzp)) / dzp;
            const size_t off = ((size_t)tab * m.n_planes + pz) * per_plane;
            double su0, sv0, su1, sv1, s0, s1;
            if (cxyd_s) {
                s0 = xy_value_grad(cxyd_s + off, nu3, ku, kv, bu, bv, du, dv, su0, sv0);
                s1 = xy_value_grad(cxyd_s + off + per_plane, nu3, ku, kv, bu, bv, du, dv, su1, sv1);
            } else {
                s0 = xy_value_grad(cxy_s + off, nu3, ku, kv, bu, bv, du, dv, su0, sv0);
                s1 = xy_value_grad(cxy_s + off + per_plane, nu3, ku, kv, bu, bv, du, dv, su1, sv1);
            }
            val = (1.0 - w) * s0 + w * s1;
            su = (1.0 - w) * su0 + w * su1;
            sv = (1.0 - w) * sv0 + w * sv1;
            gz += (z >= z_lo && z <= z_hi) ? (s1 - s0) / dzp : 0.0;
        } else {
            val = cxyd_s ? xy_value_grad(cxyd_s + (size_t)tab * per_plane, nu3, ku, kv, bu, bv, du, dv, su, sv)
                         : xy_value_grad(cxy_s + (size_t)tab * per_plane, nu3, ku, kv, bu, bv, du, dv, su, sv);
        }
        su *= ku_in;
        sv *= kv_in;
        s += val;
        gx += su * T0 + sv * T2;
        gy += su * T1 + sv * T3;
    }
    grad[0] = gx;
    grad[1] = gy;
    grad[2] = gz;
    return s;
}

// solve (H + lambda I) delta = -g for the leading dim x dim block (H symmetric: {xx, xy, xz, yy, yz, zz});
// false when a pivot is not positive
__device__ __forceinline__ bool lm_step(const double Hs[6], const double g[3], double lambda, int dim, double delta[3]) {
    double M[3][4] = {{Hs[0] + lambda, Hs[1], Hs[2], -g[0]}, {Hs[1], Hs[3] + lambda, Hs[4], -g[1]},
                      {Hs[2], Hs[4], Hs[5] + lambda, -g[2]}};
    if (dim == 2) { M[0][2] = M[0][3]; M[1][2] = M[1][3]; }      // the right-hand side moves into column dim
    for (int a = 0; a < dim; ++a) {
        if (!(M[a][a] > 0.0) || !(fabs(M[a][a]) <= 1.7e308)) return false;
        for (int r = a + 1; r < dim; ++r) {
            const double f = M[r][a] / M[a][a];
            for (int c = a; c <= dim; ++c) M[r][c] -= f * M[a][c];
        }
    }
    delta[0] = delta[1] = delta[2] = 0.0;
    for (int a = dim - 1; a >= 0; --a) {
        double s = M[a][dim];
        for (int c = a + 1; c < dim; ++c) s -= M[a][c] * delta[c];
        delta[a] = s / M[a][a];
    }
    for (int a = 0; a < dim; ++a)
        if (!(fabs(delta[a]) <= 1.7e308)) return false;
    return true;
}

template <int METHOD>
__global__ void __launch_bounds__(256, 2) refine_kernel(const RefineParams rp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = rp.m;
    const int N = m.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int ncxy = m.lrf_kind >= kXY ? m.n_lrf * max(m.n_planes, 1) * (m.nx + 3) * (m.ny + 3) : 0;

    // ---- CTA-shared tables (layout of recon_gen.cuh without the FP32 axial rows: FP64 reads m.polyd) ----
    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *xf_s = sens_s + N;
    int *grp_s = reinterpret_cast<int *>(xf_s + N);
    float *cxy_s = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(grp_s) + ((size_t)N * 4 + 15) / 16 * 16);
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        sens_s[i] = m.sens[i];
        grp_s[i] = m.grp[i];
        xf_s[i] = m.xf ? m.xf[i] : make_float4(1.f, 0.f, 0.f, 1.f);
    }
    double *cxyd_s = rp.dtab ? reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(cxy_s) + ((size_t)ncxy * 4 + 15) / 16 * 16)
                             : nullptr;
    for (int i = threadIdx.x; i < ncxy; i += blockDim.x) {
        cxy_s[i] = m.cxy[i];
        if (cxyd_s) cxyd_s[i] = (double)m.cxy[i];
    }
    __syncthreads();
    unsigned char *wbase = smem + cta_smem_bytes_gen(N, 0, ncxy, rp.dtab) + (size_t)warp * ((size_t)N * 40 + 8);
    double *LG = reinterpret_cast<double *>(wbase);                       // [N][4] {L, dL/dx, dL/dy, dL/dz}
    float2 *SC = reinterpret_cast<float2 *>(LG + (size_t)4 * N);          // [N] prepared signals

    // prepare_event reads its inputs through a Params view of this launch
    Params pv{};
    pv.m = m;
    pv.signals = rp.signals;
    pv.n_events = rp.n_events;
    pv.out_xyzA = rp.xyzA;
    pv.out_score = rp.score;
    pv.out_path = nullptr;
    pv.seed_mode = rp.seed_mode;
    pv.K = 0;

    const bool zdep = m.lrf_kind == kAxialZ || m.lrf_kind == kSliced;
    const double z_lo = (double)m.z_lo, z_hi = (double)m.z_hi;
    const int dim = rp.dim;

    for (long long eb = (long long)blockIdx.x * warps; eb < rp.n_events; eb += (long long)gridDim.x * warps) {
        // the CTA's warps start their events together (rounds of one event per warp): they run the same parts of this
        // large kernel at the same time and share the instruction caches (+2 ... 7 % on the refine workloads)
        __syncthreads();
        const long long e = eb + warp;
        if (e >= rp.n_events) continue;
        const float4 start = reinterpret_cast<const float4 *>(rp.xyzA)[e];
        // a failed event (NaN row) is left as it is
        if (!(fabsf(start.x) <= 3.402823466e38f && fabsf(start.y) <= 3.402823466e38f && fabsf(start.z) <= 3.402823466e38f)) {
            continue;
        }
        float sumS32, sx0, sy0;
        if (!prepare_event<METHOD>(pv, sens_s, SC, e, lane, sumS32, sx0, sy0)) continue;

        // F, A, g, H at p (false: invalid point)
        auto evaluate = [&](const double p[3], double &A, double &F, double g[3], double Hs[6]) -> bool {
            A = 0.0;
            F = 0.0;
            g[0] = g[1] = g[2] = 0.0;
#pragma unroll
            for (int a = 0; a < 6; ++a) Hs[a] = 0.0;
            if (zdep && !(p[2] >= z_lo && p[2] <= z_hi)) return false;                  // R6
            double sumL = 0.0, sumS = 0.0, P = 0.0, Q = 0.0, sd[3] = {0, 0, 0}, dP[3] = {0, 0, 0}, dQ[3] = {0, 0, 0};
            __syncwarp();
            for (int i = lane; i < N; i += 32) {
                if (!(SC[i].y == SC[i].y)) continue;                                     // R19
                const float4 sn = sens_s[i];
                double gr[3];
                const double gL = (double)sn.z;
                const double L = gL * lrf_value_grad(m, cxy_s, cxyd_s, sn, xf_s[i], grp_s[i], p[0], p[1], p[2], gr);
                gr[0] *= gL;
                gr[1] *= gL;
                gr[2] = dim == 3 ? gr[2] * gL : 0.0;
                LG[4 * i] = L;
                LG[4 * i + 1] = gr[0];
                LG[4 * i + 2] = gr[1];
                LG[4 * i + 3] = gr[2];
                const double S = (double)SC[i].x, w = 1.0 / fmax(S, 1.0);
                sumL += L;
                sumS += S;
                P += w * S * L;
                Q += w * L * L;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    sd[a] += gr[a];
                    dP[a] += w * S * gr[a];
                    dQ[a] += 2.0 * w * L * gr[a];
                }
            }
            sumL = warp_sum(sumL);
            sumS = warp_sum(sumS);
            P = warp_sum(P);
            Q = warp_sum(Q);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                sd[a] = warp_sum(sd[a]);
                dP[a] = warp_sum(dP[a]);
                dQ[a] = warp_sum(dQ[a]);
            }
            if (!(sumL > 0.0) || (METHOD == 1 && !(Q > 0.0))) return false;
            double dA[3];
            if (METHOD == 1) {
                A = P / Q;
#pragma unroll
                for (int a = 0; a < 3; ++a) dA[a] = (dP[a] * Q - P * dQ[a]) / (Q * Q);
            } else {
                A = sumS / sumL;
#pragma unroll
                for (int a = 0; a < 3; ++a) dA[a] = -A * sd[a] / sumL;
            }
            bool bad = false;
            double f = 0.0, gl[3] = {0, 0, 0}, hl[6] = {0, 0, 0, 0, 0, 0};
            for (int i = lane; i < N; i += 32) {
                if (!(SC[i].y == SC[i].y)) continue;
                const double L = LG[4 * i], S = (double)SC[i].x, mu = A * L;
                double mi[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) mi[a] = A * LG[4 * i + 1 + a] + L * dA[a];
                double cg, ch;
                if (METHOD == 0) {
                    if (S > 0.0) {
                        if (!(L > 0.0)) { bad = true; continue; }
                        f += mu - S - S * log(mu / S);
                    } else {
                        f += mu;
                    }
                    if (!(mu > 0.0)) continue;
                    cg = 2.0 * (1.0 - S / mu);
                    ch = 2.0 / mu;
                } else {
                    const double w = 1.0 / fmax(S, 1.0), d = S - mu;
                    f += w * d * d;
                    cg = -2.0 * w * d;
                    ch = 2.0 * w;
                }
                gl[0] += cg * mi[0];
                gl[1] += cg * mi[1];
                gl[2] += cg * mi[2];
                hl[0] += ch * mi[0] * mi[0];
                hl[1] += ch * mi[0] * mi[1];
                hl[2] += ch * mi[0] * mi[2];
                hl[3] += ch * mi[1] * mi[1];
                hl[4] += ch * mi[1] * mi[2];
                hl[5] += ch * mi[2] * mi[2];
            }
            bad = __any_sync(kFull, bad);
            F = warp_sum(f);
            if (METHOD == 0) F *= 2.0;
#pragma unroll
            for (int a = 0; a < 3; ++a) g[a] = warp_sum(gl[a]);
#pragma unroll
            for (int a = 0; a < 6; ++a) Hs[a] = warp_sum(hl[a]);
            return !bad;
        };

        double p[3] = {(double)start.x, (double)start.y, (double)start.z}, A, F, g[3], Hs[6];
        if (!evaluate(p, A, F, g, Hs)) {
            // the start point itself is invalid: position kept, no energy, no score
            if (lane == 0) {
                reinterpret_cast<float4 *>(rp.xyzA)[e] = make_float4(start.x, start.y, start.z, ANTS_QNAN);
                rp.score[e] = kInf;
            }
            continue;
        }
        double hmax = fmax(Hs[0], Hs[3]);
        if (dim == 3) hmax = fmax(hmax, Hs[5]);
        double lambda = 1e-3 * hmax, nu = 2.0;
        for (int it = 0; it < rp.n_steps; ++it) {
            double delta[3], q[3], A2 = 0.0, F2 = 0.0, g2[3], H2[6], rho = -1.0;
            bool ok = lm_step(Hs, g, lambda, dim, delta);
            if (ok) {
                q[0] = p[0] + delta[0];
                q[1] = p[1] + delta[1];
                q[2] = p[2] + delta[2];
                if (dim == 3 && zdep) {                      // projected step: z stays in its range
                    q[2] = fmin(fmax(q[2], z_lo), z_hi);
                    delta[2] = q[2] - p[2];
                }
                ok = evaluate(q, A2, F2, g2, H2);
            }
            if (ok) {
                double pred = 0.0;
                for (int a = 0; a < dim; ++a) pred += 0.5 * delta[a] * (lambda * delta[a] - g[a]);
                rho = pred > 0.0 ? (F - F2) / pred : -1.0;
            }
            if (ok && rho > 0.0) {
#pragma unroll
                for (int a = 0; a < 3; ++a) { p[a] = q[a]; g[a] = g2[a]; }
#pragma unroll
                for (int a = 0; a < 6; ++a) Hs[a] = H2[a];
                A = A2;
                F = F2;
                const double t = 2.0 * rho - 1.0, f = 1.0 - t * t * t;
                lambda *= fmax(f, 1.0 / 3.0);
                nu = 2.0;
            } else {
                lambda *= nu;
                nu *= 2.0;
            }
        }
        if (lane == 0) {
            reinterpret_cast<float4 *>(rp.xyzA)[e] = make_float4((float)p[0], (float)p[1], (float)p[2], (float)A);
            rp.score[e] = (float)F;
        }
        __syncwarp();
    }
}

}  // namespace ants
