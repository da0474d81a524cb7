// recon_gen.cuh -- the GENERAL contracting-grid kernel (section 5.1.2.2): any LRF parameterisation
// of PAPER.md:386-396 (Axial, XY, Composite = Axial + XY, Sliced = XY LRFs on z planes with linear interpolation),
// any sign of the LRF (per-pair validity rules), sensor groups with per-sensor frames, sensor
// selection and both start options.  The packed kernels (recon2d_pk.cuh, recon3d.cuh) are the fast paths for
// strictly positive Axial and Axial+Z LRFs; everything else runs here.
//
// Mapping: one warp per event, lanes over grid nodes (node = lane + 32 j, linear index (iz G + iy) G + ix), nodes
// taken in chunks of kNB per lane so that any grid size runs without a compiled limit; the event's active sensors
// are looped inside with warp-broadcast shared-memory records.
//
// Precision: coarse grids (k < k_fine) are scored in FP32 -- the same well-conditioned forms as the packed kernels
// (Poisson in the log2 domain about a reference energy, chi-square in residual form).  Fine grids, whose
// neighbouring nodes differ by ~1e-6 of the score, are scored in FP64: B200 runs DFMA at half the FP32 rate
// (profiles/r02_fp32_peak.md), so the generic path simply evaluates the definition in double -- spline basis,
// energy, deviance -- with the grid centre kept in double, instead of the centre-relative FP32 algebra that the
// packed kernels need an LRF-specific Taylor form for.  The reported energy and score are the FP64 evaluation at
// the final node.
#pragma once
#include "recon2d.cuh"

namespace ants {

constexpr int kNB = 3;   // nodes per lane per chunk

enum LrfKind { kAxial = 1, kAxialZ = 2, kXY = 3, kComposite = 4, kSliced = 5 };

// per-warp shared memory of the general kernel: the least-squares weights in double, prepared signals and the list of
// active sensors
__host__ __device__ inline size_t warp_smem_bytes_gen(int N) {
    return ((size_t)N * 8 + (size_t)N * 8 + (size_t)N * 2 + 15) / 16 * 16;
}
// CTA-shared tables: sens_s [N] float4, xf_s [N] float4, poly_s [rows] float4, grp_s [N] int, cxy_s [ncxy] float
// and, when it fits (dtab), cxyd_s [ncxy] double: the FP64 evaluations then read their coefficients without a
// conversion (F2F runs on the XU pipe at 16 lanes/clk/SM: 16 conversions per pair made the FP64 grids XU-bound,
// 71 % XU-pipe busy in the first round-2 capture)
__host__ __device__ inline size_t cta_smem_bytes_gen(int N, int rows, int ncxy, int dtab) {
    return (size_t)(2 * N + rows) * 16 + ((size_t)N * 4 + 15) / 16 * 16 + ((size_t)ncxy * 4 + 15) / 16 * 16 +
           (dtab ? (size_t)ncxy * 8 : 0);
}

// uniform cubic B-spline basis weights of the local coordinate f in [0, 1] (R7)
template <typename T>
__device__ __forceinline__ void basis4(T f, T b[4]) {
    // the two middle weights mirror each other: b1(f) = 2/3 - f^2 + f^3/2, b2(f) = b1(1 - f)
    const T o = T(1) - f, f2 = f * f, o2 = o * o;
    b[0] = o2 * o * T(1.0 / 6.0);
    b[1] = f2 * (T(0.5) * f - T(1)) + T(2.0 / 3.0);
    b[2] = o2 * (T(0.5) * o - T(1)) + T(2.0 / 3.0);
    b[3] = f2 * f * T(1.0 / 6.0);
}

// interval and local coordinate of x on [lo, lo + n / sc], clamped into the range (R5).  (A magic-number rounding
// in place of the two conversions was measured slower in round 2: it trades two XU-pipe conversions for five more
// FP32 / FP64 adds, and once the coefficients need no conversion the XU pipe is no longer the bound.)
template <typename T>
__device__ __forceinline__ void locate(T x, T lo, T sc, int n, int &k, T &f) {
    T t = (x - lo) * sc;
    t = t < T(0) ? T(0) : (t > T(n) ? T(n) : t);
    k = min((int)t, n - 1);
    f = t - T(k);
}

// tensor-product spline value from the coefficient table c [ny + 3][nx + 3] (u fastest), R30
template <typename T, typename TC>
__device__ __forceinline__ T xy_value(const TC *c, int nu3, int ku, int kv, const T bu[4], const T bv[4]) {
    const TC *q = c + kv * nu3 + ku;
    T s = T(0);
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const T row = T(q[0]) * bu[0] + T(q[1]) * bu[1] + T(q[2]) * bu[2] + T(q[3]) * bu[3];
        s += row * bv[b];
        q += nu3;
    }
    return s;
}

// axial spline in double from the power-basis rows (m.polyd), r clamped (R5)
__device__ __forceinline__ double axial_value64(const ModelDev &m, int tab, double r) {
    const double r_lo = (double)m.r_lo, r_hi = (double)m.r_hi;
    const double rc = fmin(fmax(r, r_lo), r_hi);
    const double t = (rc - r_lo) * ((double)m.n_r / (r_hi - r_lo));
    const int k = min(max((int)t, 0), m.n_r - 1);
    const double u = t - (double)k;
    const double *p = m.polyd + ((size_t)tab * m.n_r + k) * 4;
    return p[0] + u * (p[1] + u * (p[2] + u * p[3]));
}

// L_i / g_i at a node, in T = float (coarse grids) or double (fine grids)
template <int LRFK, typename T>
struct NodeLrf {
    // z-plane interpolation of the node (Sliced): plane index and weight, set once per node
    int pz;
    T wz;
};

template <int LRFK, typename T>
__device__ __forceinline__ T lrf_value(const ModelDev &m, const float4 *poly_s, const float *cxy_s, const double *cxyd_s,
                                       const float4 sn, const float4 xf, int tab, T x, T y, int pz, T wz) {
    const T dx = x - T(sn.x), dy = y - T(sn.y);
    T s = T(0);
    if (LRFK == kAxial || LRFK == kComposite) {
        if (sizeof(T) == 4) {
            s += T(eval_axial(m, poly_s + tab * (m.n_r + 1), sqrt_approx(fmaf((float)dx, (float)dx, (float)dy * (float)dy))));
        } else {
            s += T(axial_value64(m, tab, sqrt((double)dx * (double)dx + (double)dy * (double)dy)));
        }
    }
    if (LRFK >= kXY) {
        const T u = T(xf.x) * dx + T(xf.y) * dy, v = T(xf.z) * dx + T(xf.w) * dy;
        int ku, kv;
        T fu, fv, bu[4], bv[4];
        locate(u, T(m.u_lo), T(m.su), m.nx, ku, fu);
        locate(v, T(m.v_lo), T(m.sv), m.ny, kv, fv);
        basis4<T>(fu, bu);
        basis4<T>(fv, bv);
        const int nu3 = m.nx + 3, per_plane = nu3 * (m.ny + 3);
        const size_t off = LRFK == kSliced ? ((size_t)tab * m.n_planes + pz) * per_plane : (size_t)tab * per_plane;
        if (sizeof(T) == 8 && cxyd_s) {
            const double *c0 = cxyd_s + off;
            if (LRFK == kSliced) {
                const T s0 = xy_value<T, double>(c0, nu3, ku, kv, bu, bv), s1 = xy_value<T, double>(c0 + per_plane, nu3, ku, kv, bu, bv);
                s += (T(1) - wz) * s0 + wz * s1;
            } else {
                s += xy_value<T, double>(c0, nu3, ku, kv, bu, bv);
            }
        } else {
            const float *c0 = cxy_s + off;
            if (LRFK == kSliced) {
                const T s0 = xy_value<T, float>(c0, nu3, ku, kv, bu, bv), s1 = xy_value<T, float>(c0 + per_plane, nu3, ku, kv, bu, bv);
                s += (T(1) - wz) * s0 + wz * s1;               // R32: linear interpolation between the two planes
            } else {
                s += xy_value<T, float>(c0, nu3, ku, kv, bu, bv);
            }
        }
    }
    return s;
}

__device__ __forceinline__ void warp_argmin_d(double &s, int &idx) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double os = __shfl_xor_sync(kFull, s, o);
        const int oi = __shfl_xor_sync(kFull, idx, o);
        const bool take = (os < s) || (os == s && oi < idx);
        s = take ? os : s;
        idx = take ? oi : idx;
    }
}

template <int METHOD, int LRFK>
__global__ void __launch_bounds__(256, 2) recon_gen_kernel(const Params p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = p.m;
    const int N = m.N, nr1 = m.n_r + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows = (LRFK == kAxial || LRFK == kComposite) ? m.n_lrf * nr1 : 0;
    const int ncxy = LRFK >= kXY ? m.n_lrf * max(m.n_planes, 1) * (m.nx + 3) * (m.ny + 3) : 0;

    // ---- CTA-shared tables ----
    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *xf_s = sens_s + N;
    float4 *poly_s = xf_s + N;
    int *grp_s = reinterpret_cast<int *>(poly_s + rows);
    float *cxy_s = reinterpret_cast<float *>(reinterpret_cast<unsigned char *>(grp_s) + ((size_t)N * 4 + 15) / 16 * 16);
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        sens_s[i] = m.sens[i];
        grp_s[i] = m.grp[i];
        xf_s[i] = m.xf ? m.xf[i] : make_float4(1.f, 0.f, 0.f, 1.f);
    }
    for (int i = threadIdx.x; i < rows; i += blockDim.x) poly_s[i] = m.poly[i];
    double *cxyd_s = p.gen_dtab ? reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(cxy_s) + ((size_t)ncxy * 4 + 15) / 16 * 16)
                                : nullptr;
    for (int i = threadIdx.x; i < ncxy; i += blockDim.x) {
        cxy_s[i] = m.cxy[i];
        if (cxyd_s) cxyd_s[i] = (double)m.cxy[i];
    }
    __syncthreads();
    unsigned char *wbase = smem + cta_smem_bytes_gen(N, rows, ncxy, p.gen_dtab) + (size_t)warp * warp_smem_bytes_gen(N);
    double *Wd = reinterpret_cast<double *>(wbase);                       // least squares: w_i = 1 / max(S_i, 1)
    float2 *SC = reinterpret_cast<float2 *>(Wd + N);                      // {S_i prepared, log2(S_i / gL_i) or 0}
    unsigned short *act = reinterpret_cast<unsigned short *>(SC + N);     // indices of the event's active sensors

    const int G = p.G, GG = G * G;
    const bool zsearch = p.dim == 3;
    const bool zdep = LRFK == kSliced;
    const double half = 0.5 * (double)(G - 1);
    const double z_lo = (double)m.z_lo, z_hi = (double)m.z_hi;
    const double dzp = zdep ? (z_hi - z_lo) / (double)(m.n_planes - 1) : 1.0;
    const int chunks = (p.nodes + 32 * kNB - 1) / (32 * kNB);

    // Event distribution: every warp on its own, or (p.lockstep, a run-time flag here) the CTA in rounds of one event per
    // warp behind a barrier, which keeps its warps in the same phase of the search -- the FP32 and FP64 node loops of the
    // Composite LRF are two large bodies of code (recon2d_pk_kernel.cuh explains the mechanism; config 8 +15 %, no
    // change on the 37- and 64-sensor configs 7 and 6: the plan sets it for arrays of up to 32 sensors)
    __shared__ long long round_s;
    const int warps_cta = blockDim.x >> 5, warp_id = threadIdx.x >> 5;
    const bool LOCKSTEP = p.lockstep != 0;
    long long b_next = LOCKSTEP ? grab_round(p.ctr, warps_cta, &round_s) : 0;
    long long e_next = LOCKSTEP ? b_next + warp_id : grab_event(p.ctr, lane);
    for (long long e = e_next; LOCKSTEP ? b_next < p.n_events : e < p.n_events; e = e_next) {
        if (LOCKSTEP) {
            b_next = grab_round(p.ctr, warps_cta, &round_s);
            e_next = b_next + warp_id;
            if (e >= p.n_events) continue;
        } else {
            e_next = grab_event(p.ctr, lane);
        }
        // ---- a1: load signals (coalesced), prepare, centroid, start position, selection ----
        float sumS, sx0, sy0;
        if (!prepare_event<METHOD>(p, sens_s, SC, e, lane, sumS, sx0, sy0)) continue;
        // active list (R19) and the event constants of the FP64 scores
        int n_act = 0;
        double sumSd = 0.0, SlnS = 0.0, wSS = 0.0;
        for (int i0 = 0; i0 < N; i0 += 32) {
            const int i = i0 + lane;
            const bool on = i < N && (SC[i < N ? i : 0].y == SC[i < N ? i : 0].y);
            const unsigned mk = __ballot_sync(kFull, on);
            if (on) {
                act[n_act + __popc(mk & ((1u << lane) - 1u))] = (unsigned short)i;
                const double S = (double)SC[i].x;
                sumSd += S;
                if (METHOD == 0) {
                    if (S > 0.0) SlnS += S * log(S);
                } else {
                    const double w = 1.0 / fmax(S, 1.0);
                    Wd[i] = w;
                    wSS += S * S * w;
                }
            }
            n_act += __popc(mk);
        }
        sumSd = warp_sum(sumSd);
        SlnS = warp_sum(SlnS);
        wSS = warp_sum(wSS);
        __syncwarp();

        double cx = (double)sx0, cy = (double)sy0;
        double cz = zdep ? ((p.z_seed == p.z_seed) ? (double)p.z_seed : 0.5 * (z_lo + z_hi)) : 0.0;   // R10
        double h = (double)p.h0_xy, hz = (double)p.h0_z;

        // FP64 score of one node from single-pass sums (exact rewrites of the definitions, R2-R4, R27):
        //   Poisson  D = 2 [sum S ln S - sum S_i ln L_i - sumS ln(sumS / sumL)]      (mu = A L, A sumL = sumS)
        //   chi2     sum w S^2 - (sum w S L)^2 / sum w L^2;   sum-ratio: sum w S^2 - 2 A sum w S L + A^2 sum w L^2
        auto score64 = [&](double x, double y, double z, double &A_out) -> double {
            A_out = 0.0;
            if (zdep && !(z >= z_lo && z <= z_hi)) return (double)kInf;                               // R6
            int pz = 0;
            double wz = 0.0;
            if (zdep) {
                pz = min(max((int)floor((z - z_lo) / dzp), 0), m.n_planes - 2);
                wz = (z - (z_lo + (double)pz * dzp)) / dzp;
            }
            double sumL = 0.0, a1 = 0.0, a2 = 0.0;
            bool bad = false;
            for (int q = 0; q < n_act; ++q) {
                const int i = act[q];
                const float4 sn = sens_s[i];
                const double L = (double)sn.z * lrf_value<LRFK, double>(m, poly_s, cxy_s, cxyd_s, sn, xf_s[i], grp_s[i], x, y, pz, wz);
                const double S = (double)SC[i].x;
                sumL += L;
                if (METHOD == 0) {
                    if (S > 0.0) {
                        if (!(L > 0.0)) bad = true;
                        else a1 += S * log(L);
                    }
                } else {
                    const double w = Wd[i];
                    a1 += w * S * L;
                    a2 += w * L * L;
                }
            }
            if (bad || !(sumL > 0.0)) return (double)kInf;
            if (METHOD == 0) {
                A_out = sumSd / sumL;
                return 2.0 * (SlnS - a1 - sumSd * log(A_out));
            }
            if (METHOD == 1) {
                if (!(a2 > 0.0)) return (double)kInf;
                A_out = a1 / a2;
                return wSS - a1 * a1 / a2;
            }
            A_out = sumSd / sumL;
            return wSS - 2.0 * A_out * a1 + A_out * A_out * a2;
        };

        // reference energy of the FP32 score: A at the start position
        float A_ref = 1.f;
        if (p.k_diff > 0) {
            float sl = 0.f;
            const float czf = (float)cz;
            int pz = 0;
            float wz = 0.f;
            if (zdep) {
                pz = min(max((int)floorf((czf - m.z_lo) / (float)dzp), 0), m.n_planes - 2);
                wz = (czf - (m.z_lo + (float)pz * (float)dzp)) / (float)dzp;
            }
            for (int q = lane; q < n_act; q += 32) {
                const int i = act[q];
                const float4 sn = sens_s[i];
                sl += sn.z * lrf_value<LRFK, float>(m, poly_s, cxy_s, cxyd_s, sn, xf_s[i], grp_s[i], (float)cx, (float)cy, pz, wz);
            }
            sl = warp_sum(sl);
            A_ref = sl > 0.f ? sumS / sl : 1.f;
        }

        for (int k = 0; k < p.K; ++k) {
            double bs = (double)kInf;        // this lane's best score, its node and (FP32 mode) the energy there
            int bi = 0x7fffffff;
            float baux = 0.f;
            const bool fine = k >= p.k_diff;
            const float lA = log2f(A_ref);
            for (int c = 0; c < chunks; ++c) {
                int nn[kNB];
                bool nv[kNB];
                double x[kNB], y[kNB], z[kNB];
#pragma unroll
                for (int j = 0; j < kNB; ++j) {
                    const int n = lane + 32 * (c * kNB + j);
                    nn[j] = n;
                    nv[j] = n < p.nodes;
                    const int iz = n / GG, rem = n - iz * GG, iy = rem / G, ix = rem - iy * G;
                    x[j] = cx + ((double)ix - half) * h;
                    y[j] = cy + ((double)iy - half) * h;
                    z[j] = zsearch ? cz + ((double)iz - half) * hz : cz;
                }
                if (fine) {
#pragma unroll
                    for (int j = 0; j < kNB; ++j) {
                        if (!nv[j]) continue;
                        double A;
                        const double sc = score64(x[j], y[j], z[j], A);
                        if (sc < bs) { bs = sc; bi = nn[j]; }
                    }
                } else {
                    // FP32: Poisson sum_i S_i (c_i - log2 s_i) + sumS log2(A_ref sumL / sumS), c_i = log2(S_i/(A_ref gL_i));
                    //       chi2 sum w d^2 - (sum w d L)^2 / sum w L^2, d = S - A_ref L  (recon2d.cuh)
                    float xf32[kNB], yf32[kNB], wzf[kNB], a1[kNB], a2[kNB], a3[kNB], a4[kNB];
                    int pzf[kNB];
                    bool bad[kNB];
#pragma unroll
                    for (int j = 0; j < kNB; ++j) {
                        xf32[j] = (float)x[j];
                        yf32[j] = (float)y[j];
                        a1[j] = a2[j] = a3[j] = a4[j] = 0.f;
                        bad[j] = zdep && !(z[j] >= z_lo && z[j] <= z_hi);                          // R6
                        pzf[j] = 0;
                        wzf[j] = 0.f;
                        if (zdep) {
                            const float zz = (float)z[j];
                            pzf[j] = min(max((int)floorf((zz - m.z_lo) / (float)dzp), 0), m.n_planes - 2);
                            wzf[j] = (zz - (m.z_lo + (float)pzf[j] * (float)dzp)) / (float)dzp;
                        }
                    }
                    for (int q = 0; q < n_act; ++q) {
                        const int i = act[q];
                        const float4 sn = sens_s[i], xf = xf_s[i];
                        const float2 sc2 = SC[i];
                        const int tab = grp_s[i];
                        const float fourth = METHOD == 0 ? (sc2.x > 0.f ? sc2.y - lA : 0.f) : 1.f / fmaxf(sc2.x, 1.f);
#pragma unroll
                        for (int j = 0; j < kNB; ++j) {
                            float s = lrf_value<LRFK, float>(m, poly_s, cxy_s, cxyd_s, sn, xf, tab, xf32[j], yf32[j], pzf[j], wzf[j]);
                            if (METHOD == 0) {
                                bad[j] = bad[j] || (s <= 0.f && sc2.x > 0.f);
                                a2[j] = fmaf(sn.z, s, a2[j]);
                                s = fmaxf(s, 1e-37f);
                                a1[j] = fmaf(sc2.x, fourth - lg2_approx(s), a1[j]);
                            } else {
                                const float L = sn.z * s, d = fmaf(-A_ref, L, sc2.x), wd = fourth * d;
                                a1[j] = fmaf(wd, d, a1[j]);
                                a2[j] = fmaf(wd, L, a2[j]);
                                a3[j] = fmaf(fourth * L, L, a3[j]);
                                a4[j] += L;
                            }
                        }
                    }
#pragma unroll
                    for (int j = 0; j < kNB; ++j) {
                        float sc, aux;
                        if (METHOD == 0) {
                            sc = fmaf(sumS, log2f(a2[j] * (A_ref / sumS)), a1[j]);
                            aux = sumS / a2[j];
                            if (!(a2[j] > 0.f)) sc = kInf;
                        } else if (METHOD == 1) {
                            sc = a1[j] - a2[j] * a2[j] / a3[j];
                            aux = A_ref + a2[j] / a3[j];
                            if (!(a3[j] > 0.f) || !(a4[j] > 0.f)) sc = kInf;
                        } else {
                            const float An = sumS / a4[j], dl = An - A_ref;
                            sc = fmaf(dl, fmaf(dl, a3[j], -2.f * a2[j]), a1[j]);
                            aux = An;
                            if (!(a4[j] > 0.f)) sc = kInf;
                        }
                        if (!nv[j] || bad[j] || !(sc == sc)) sc = kInf;
                        if ((double)sc < bs) { bs = (double)sc; bi = nn[j]; baux = aux; }
                    }
                }
            }
            // ---- a5: argmin over all nodes (ties -> lowest linear index, R9), recentre, contract ----
            const int mine = bi;
            warp_argmin_d(bs, bi);
            const bool found = bs < (double)kInf;
            if (found) {
                if (!fine) {
                    // the winner's energy lives in the lane that scored it (nodes n = lane + 32 j)
                    const float v = __shfl_sync(kFull, mine == bi ? baux : 0.f, bi & 31);
                    if (v > 0.f && v == v) A_ref = v;
                }
                const int iz = bi / GG, rem = bi - iz * GG, iy = rem / G, ix = rem - iy * G;
                cx += ((double)ix - half) * h;
                cy += ((double)iy - half) * h;
                if (zsearch) cz += ((double)iz - half) * hz;
            }
            if (p.out_path && lane == 0) p.out_path[e * p.K + k] = found ? (uint16_t)bi : (uint16_t)0xFFFF;
            h *= (double)p.factor;
            hz *= (double)p.factor;
            __syncwarp();
        }

        // ---- a6: FP64 energy and score at the final node (sensors split over the lanes), store ----
        {
            const bool z_ok = !zdep || (cz >= z_lo && cz <= z_hi);
            int pz = 0;
            double wz = 0.0;
            if (zdep && z_ok) {
                pz = min(max((int)floor((cz - z_lo) / dzp), 0), m.n_planes - 2);
                wz = (cz - (z_lo + (double)pz * dzp)) / dzp;
            }
            double sumL = 0.0, swsl = 0.0, swll = 0.0;
            bool bad = !z_ok;
            double Lq[8];                                    // this lane's L values (N <= 256 per pass)
            for (int q0 = 0; q0 < n_act; q0 += 256) {
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const int q = q0 + lane + 32 * t;
                    Lq[t] = 0.0;
                    if (q < n_act) {
                        const int i = act[q];
                        const float4 sn = sens_s[i];
                        const double L = (double)sn.z * lrf_value<LRFK, double>(m, poly_s, cxy_s, cxyd_s, sn, xf_s[i], grp_s[i], cx, cy, pz, wz);
                        const double S = (double)SC[i].x, wi = 1.0 / fmax(S, 1.0);
                        Lq[t] = L;
                        sumL += L;
                        swsl += wi * S * L;
                        swll += wi * L * L;
                    }
                }
            }
            sumL = warp_sum(sumL);
            swsl = warp_sum(swsl);
            swll = warp_sum(swll);
            if (!(sumL > 0.0)) bad = true;
            if (METHOD >= 1 && !(swll > 0.0)) bad = true;
            const double A = METHOD == 1 ? swsl / swll : sumSd / sumL;
            double sc = 0.0;
            // second pass with the energy known (N <= 256: from the kept values; else recomputed)
            for (int q0 = 0; q0 < n_act; q0 += 256) {
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const int q = q0 + lane + 32 * t;
                    if (q < n_act) {
                        const int i = act[q];
                        double L = Lq[t];
                        if (n_act > 256) {
                            const float4 sn = sens_s[i];
                            L = (double)sn.z * lrf_value<LRFK, double>(m, poly_s, cxy_s, cxyd_s, sn, xf_s[i], grp_s[i], cx, cy, pz, wz);
                        }
                        const double S = (double)SC[i].x;
                        if (METHOD == 0) {
                            const double mu = A * L;
                            if (S > 0.0) {
                                if (!(L > 0.0)) bad = true;
                                else sc += mu - S - S * log(mu / S);
                            } else {
                                sc += mu;
                            }
                        } else {
                            const double d = S - A * L;
                            sc += d * d / fmax(S, 1.0);
                        }
                    }
                }
            }
            sc = warp_sum(sc);
            if (METHOD == 0) sc *= 2.0;
            bad = __any_sync(kFull, bad);
            if (lane == 0) {
                reinterpret_cast<float4 *>(p.out_xyzA)[e] =
                    make_float4((float)cx, (float)cy, (float)cz, bad ? ANTS_QNAN : (float)A);
                p.out_score[e] = bad ? kInf : (float)sc;
            }
        }
        __syncwarp();
    }
    retire_warp(p.ctr, p.total_warps, lane);
}

}  // namespace ants
